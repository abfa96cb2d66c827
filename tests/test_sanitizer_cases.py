"""Tiny GPU cases, one per kernel family, sized to run under compute-sanitizer (racecheck / synccheck / memcheck
slow a kernel down 10-100x):  N = 64 shared-memory passes;  N = 128 two-items-per-CTA kernels with an odd item
count (the padding item, named-barrier hand-over of the transpose buffer, TMEM slots);  N = 256 on the 4-CTA
cluster (DSMEM transposes between cluster barriers), with tilt so that the kept spectra and D-sums run.
Each case is still compared with the oracle.  profiles/r02_sanitizer.md holds the commands and summaries."""
import numpy as np
import pytest

torch = pytest.importorskip("torch")
pytestmark = pytest.mark.gpu

import oracle  # noqa: E402
from cases import geom_of, rel_l2  # noqa: E402
from paper_2505_07814_b200 import synth  # noqa: E402

CASES = {
    "n64": (synth.get_config(1), 4),
    "n128_odd_items": (synth.get_config(3, Nz=2, M=3, tilt_mode=1, true_tilt=(3e-4, -2e-4), eval_tilt=(1e-4, 2e-4)), 3),
    "n256_cluster": (synth.get_config(5, Nz=2, M=2), 2),
}


@pytest.mark.parametrize("name", list(CASES))
def test_small_case(name):
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    from paper_2505_07814_b200 import build
    build.build()
    from paper_2505_07814_b200 import binding
    cfg, B = CASES[name]
    geom = geom_of(cfg)
    tr, ev = synth.truth(cfg), synth.eval_point(cfg, "A")
    if cfg.M != tr["probe"].shape[0]:
        raise AssertionError("probe modes")
    idx = synth.minibatch(cfg, 0, cfg.B)[:B]
    tilt_t = tr["tilt"] if cfg.tilt_mode else None
    tilt_e = ev["tilt"] if cfg.tilt_mode else None
    meas = synth.poisson_amplitudes(cfg, oracle.intensity_batch(tr["object"], tr["probe"], tr["positions"][idx],
                                                                tilt_t, geom), idx)
    pos = np.ascontiguousarray(ev["positions"][idx])
    ref = oracle.grad_batch(ev["object"], ev["probe"], pos, tilt_e, meas, geom)
    plan = binding.plan_for(cfg, Bmax=B)
    d = lambda x: None if x is None else torch.from_numpy(np.ascontiguousarray(x)).cuda()
    obj, probe, dpos, dtilt, dmeas = d(ev["object"]), d(ev["probe"]), d(pos), d(tilt_e), d(meas)
    g_obj, g_probe = torch.zeros_like(obj), torch.zeros_like(probe)
    g_pos = torch.zeros(B, 2, device="cuda")
    g_tilt = torch.zeros(2, device="cuda") if cfg.tilt_mode else None
    loss = plan.forward_loss(obj, probe, dpos, dtilt, dmeas)
    plan.backward(obj, probe, dpos, dtilt, dmeas, g_obj, g_probe, g_pos, g_tilt, flags=binding.PTY_BWD_REUSE_FORWARD)
    rc, _ = plan.status()
    assert rc == 0, plan.last_error()
    assert abs(loss.item() - ref["loss"]) <= 1e-4 * ref["loss"]
    assert rel_l2(g_obj.cpu().numpy(), ref["g_object"]) <= 1e-3
    assert rel_l2(g_probe.cpu().numpy(), ref["g_probe"]) <= 1e-3
    assert rel_l2(g_pos.cpu().numpy(), ref["g_positions"]) <= 1e-3
    if cfg.tilt_mode:
        assert rel_l2(g_tilt.cpu().numpy(), ref["g_tilt"].sum(0)) <= 1e-3
    plan.close()
