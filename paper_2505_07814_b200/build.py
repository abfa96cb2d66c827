"""Build libpty.so (the product) and libpty_benchutil.so (bench.py's FP32 microbenchmark) in-tree with nvcc
for sm_100a (cross-compiles without a GPU)."""
from __future__ import annotations

import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(HERE, "libpty.so")
BENCH_LIB = os.path.join(HERE, "libpty_benchutil.so")
HEADERS = ["pty_port.cuh", "pty_pointwise.cuh", "pty_fft.cuh", "pty_kernels.cuh", "pty_fft128.cuh", "pty_kernels128.cuh",
           "pty_kernels128g2.cuh", os.path.join("..", "..", "include", "pty.h")]
TARGETS = {LIB: (["pty_lib.cu"], HEADERS), BENCH_LIB: (["pty_bench_util.cu"], [])}
NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-O3", "-std=c++17",
              "--shared", "-Xcompiler", "-fPIC", "-Xptxas", "-v"]


def _stale(lib, sources, headers):
    if not os.path.exists(lib):
        return True
    t = os.path.getmtime(lib)
    deps = [os.path.join(CSRC, f) for f in sources + headers] + [os.path.abspath(__file__)]
    return any(os.path.getmtime(d) > t for d in deps)


def build(force=False, verbose=False):
    """Compile every CUDA source; returns the path of libpty.so."""
    nvcc = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
    for lib, (sources, headers) in TARGETS.items():
        if not force and not _stale(lib, sources, headers):
            continue
        cmd = [nvcc] + NVCC_FLAGS + ["-o", lib] + [os.path.join(CSRC, s) for s in sources]
        res = subprocess.run(cmd, capture_output=True, text=True)
        log = res.stdout + res.stderr
        with open(os.path.join(HERE, "build.log" if lib == LIB else "build_benchutil.log"), "w") as f:
            f.write(" ".join(cmd) + "\n" + log)
        if res.returncode != 0:
            raise RuntimeError("nvcc failed:\n" + log[-4000:])
        if verbose:
            print(log)
    return LIB


def build_variant(name, defines, force=False):
    """Compile pty_lib.cu once more with extra -D switches into paper_2505_07814_b200/<name> (not part of build()):
    used by tests that compare a compile-time switch of the kernels against the product build, e.g.
    build_variant("libpty_strict.so", ["-DPTY_CLUSTER_RELAXED=0"]).  Load it with PTY_LIB=<path> (binding.py)."""
    lib = os.path.join(HERE, name)
    sources, headers = TARGETS[LIB]
    if force or _stale(lib, sources, headers):
        nvcc = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
        cmd = [nvcc] + NVCC_FLAGS + list(defines) + ["-o", lib] + [os.path.join(CSRC, s) for s in sources]
        res = subprocess.run(cmd, capture_output=True, text=True)
        if res.returncode != 0:
            raise RuntimeError("nvcc failed:\n" + (res.stdout + res.stderr)[-4000:])
    return lib


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose=True))
