"""The N = 256 kernels exchange wave tiles between the four CTAs of a cluster (pty_fft.cuh).  Before a CTA's tile is
overwritten by its peers' st.async, every thread of the cluster must have finished READING the old contents; the
product build orders that with `barrier.cluster.arrive.relaxed` + `wait` (no release fence, PTY_CLUSTER_RELAXED = 1).
That is an argument from how the hardware executes the barrier, not from the PTX memory model, which gives a relaxed
arrive no happens-before edge (round-2 advisor finding), and compute-sanitizer's racecheck does
not model DSMEM.  So the switch stays a compile-time one and this test is the evidence kept in the suite: the same
case, whose outputs receive one contribution each and are therefore bit-reproducible, is run 40 times under the product
build and under a build with the fenced barrier (-DPTY_CLUSTER_RELAXED=0); every run of both must give the same bits."""
import json
import os
import subprocess
import sys

import pytest

torch = pytest.importorskip("torch")
pytestmark = pytest.mark.gpu

HERE = os.path.dirname(os.path.abspath(__file__))


@pytest.mark.timeout(900)
def test_relaxed_and_fenced_cluster_barrier_give_the_same_bits():
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    from paper_2505_07814_b200 import build
    product = build.build()
    fenced = build.build_variant("libpty_strict.so", ["-DPTY_CLUSTER_RELAXED=0"])
    results = []
    for lib in (product, fenced):
        env = dict(os.environ, PTY_LIB=lib)
        out = subprocess.run([sys.executable, os.path.join(HERE, "cluster_order_worker.py"), "40"], env=env,
                             capture_output=True, text=True, timeout=600)
        assert out.returncode == 0, out.stderr[-2000:]
        results.append(json.loads(out.stdout.strip().splitlines()[-1]))
    assert results[0]["lib"] == "libpty.so" and results[1]["lib"] == "libpty_strict.so"
    for name in ("intensity", "loss_per_pos", "g_object"):
        a, b = results[0]["digests"][name], results[1]["digests"][name]
        assert len(a) == 1, (name, "product build not bit-reproducible", a)
        assert len(b) == 1, (name, "fenced build not bit-reproducible", b)
        assert a == b, (name, "the two barriers give different bits")
