"""CPU check of the butterfly algebra of the N = 128 FFT core: csrc/pty_fft128.cuh compiles for the host (g++, the
packed FP32x2 intrinsics replaced by their definitions) and fft32 / the FMA-form radix-4 stage are compared with a
float64 DFT.  This pins the twiddle constants, signs and index maps of the device code without a GPU; the kernels
that use them are compared with the oracle in the -m gpu tests."""
import os
import re
import shutil
import subprocess

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
CUDA_INC = os.path.join(os.environ.get("CUDA_HOME", "/usr/local/cuda"), "include")


@pytest.mark.skipif(shutil.which("g++") is None or not os.path.exists(os.path.join(CUDA_INC, "vector_types.h")),
                    reason="needs g++ and the CUDA headers (float2)")
def test_register_fft_blocks_match_a_float64_dft(tmp_path):
    exe = str(tmp_path / "fft_check")
    cmd = ["g++", "-O1", "-std=c++17", "-I", CUDA_INC,
           "-I", os.path.join(ROOT, "paper_2505_07814_b200", "csrc"), os.path.join(ROOT, "tests", "host", "fft_check.cpp"),
           "-o", exe]
    res = subprocess.run(cmd, capture_output=True, text=True)
    assert res.returncode == 0, res.stderr[-2000:]
    out = subprocess.run([exe], capture_output=True, text=True, check=True).stdout
    errs = [float(x) for x in re.findall(r"[0-9]\.[0-9]+e[+-][0-9]+", out)]
    assert len(errs) == 3, out
    assert all(e < 5e-7 for e in errs), out       # float32 butterflies, 5 (fft32) / 2 (radix-4) stages deep
