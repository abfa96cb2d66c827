"""Seeded random shapes through the C ABI against the oracle: every window size (64 / 128 / 256), odd and even item
counts, one to four slices and modes, the three tilt modes with the dz gradient, and the opt-in plan flags of the
N = 128 kernels.  Each case is a few positions of a cut-down config 1 / 3 / 5, so the oracle needs a second or two."""
import os
import sys

import numpy as np
import pytest

torch = pytest.importorskip("torch")
sys.path.insert(0, os.path.dirname(os.path.abspath(__file__)))

import oracle  # noqa: E402
from cases import geom_of, make_case  # noqa: E402
from paper_2505_07814_b200 import synth  # noqa: E402

pytestmark = pytest.mark.gpu


def _cases():
    rng = np.random.default_rng(20260505)
    out = []
    for k in range(18):
        c = int(rng.choice([1, 3, 3, 3, 5, 5]))
        base = synth.get_config(c)
        Nz = 1 if c == 1 else int(rng.integers(1, 5))
        M = 1 if c == 1 else int(rng.integers(1, min(base.M, 4) + 1))
        B = int(rng.integers(1, 7 if c == 5 else 10))
        tm = 0 if c == 1 else int(rng.integers(0, 3))
        flag = int(rng.choice([0, 16, 32, 48])) if c == 3 else 0
        batch = int(rng.integers(0, 4))
        out.append((k, c, Nz, M, B, tm, flag, batch))
    return out


@pytest.fixture(scope="module")
def pty():
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    from paper_2505_07814_b200 import build
    build.build()
    from paper_2505_07814_b200 import binding
    return binding


@pytest.mark.timeout(600)
@pytest.mark.parametrize("k,c,Nz,M,B,tm,flag,batch", _cases())
def test_random_shape_matches_the_oracle(pty, k, c, Nz, M, B, tm, flag, batch):
    from test_gpu_parity import check_against_oracle, run_gpu
    base = synth.get_config(c)
    cfg = synth.get_config(c, Nz=Nz, M=M, tilt_mode=tm)
    idx = synth.minibatch(base, batch, base.B)[:B]
    case = make_case(c, "A", idx, tilt_mode=tm)
    case = dict(case, cfg=cfg, object=np.ascontiguousarray(case["object"][:Nz]),
                probe=np.ascontiguousarray(case["probe"][:M]))
    tr = synth.truth(base)
    I_true = oracle.intensity_batch(tr["object"][:Nz], tr["probe"][:M], tr["positions"][idx],
                                    tr["tilt"] if base.tilt_mode else None, geom_of(cfg))
    case["meas"] = synth.poisson_amplitudes(cfg, I_true, idx)
    want_dz = bool(tm == 0 and Nz > 1 and k % 2 == 0)
    ref = oracle.grad_batch(case["object"], case["probe"], case["positions"], case["tilt"], case["meas"], geom_of(cfg))
    res = run_gpu(pty, case, want_dz=want_dz, flags=flag)
    _, _, I_ref = oracle.forward_loss_batch(case["object"], case["probe"], case["positions"], case["tilt"], case["meas"],
                                            geom_of(cfg))
    assert np.max(np.abs(res["intensity"] - I_ref)) <= 1e-4 * I_ref.max()
    check_against_oracle(res, ref, case)
