"""GPU parity: the CUDA path (through the C ABI) against the float64 oracle, element by element,
on the same seeded inputs.  Bar (BASELINE.json north_star): loss within 1e-4 relative, every
gradient within 1e-3 relative L2.  Integer work (crop origin) is checked through the results."""
import numpy as np
import pytest

torch = pytest.importorskip("torch")
pytestmark = pytest.mark.gpu

import oracle  # noqa: E402
from cases import WORKERS, geom_of, make_case, oracle_grad, rel_l2  # noqa: E402
from paper_2505_07814_b200 import synth  # noqa: E402

LOSS_RTOL = 1e-4
GRAD_RTOL = 1e-3


@pytest.fixture(scope="module")
def pty():
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    from paper_2505_07814_b200 import build
    build.build()
    from paper_2505_07814_b200 import binding
    return binding


def dev(x, dtype=None):
    if x is None:
        return None
    t = torch.from_numpy(np.ascontiguousarray(x)).cuda()
    return t.to(dtype) if dtype is not None else t


def run_gpu(pty, case, want_dz=False, flags=0, plan=None, bwd_flags=0, outputs=None):
    cfg = case["cfg"]
    B = len(case["positions"])
    tm = case["tilt_mode"]
    if plan is None:
        plan = pty.Plan(cfg.Nz, cfg.H, cfg.W, cfg.M, cfg.N, max(B, 1), cfg.dz, cfg.lam, cfg.dx, tilt_mode=tm,
                        flags=flags | (pty.PTY_FLAG_SPECTRA if want_dz else 0))
    obj, probe = dev(case["object"]), dev(case["probe"])
    pos, tilt, meas = dev(case["positions"]), dev(case["tilt"]), dev(case["meas"])
    out = outputs or {
        "loss": torch.zeros(1, dtype=torch.float64, device="cuda"),
        "loss_per_pos": torch.zeros(B, dtype=torch.float32, device="cuda"),
        "intensity": torch.zeros(B, cfg.N, cfg.N, dtype=torch.float32, device="cuda"),
        "g_object": torch.full(obj.shape, 7.0, dtype=torch.complex64, device="cuda"),   # must be overwritten
        "g_probe": torch.full(probe.shape, 7.0, dtype=torch.complex64, device="cuda"),
        "g_positions": torch.full((B, 2), 7.0, dtype=torch.float32, device="cuda"),
        "g_tilt": (torch.full((B, 2) if tm == 2 else (2,), 7.0, dtype=torch.float32, device="cuda") if tm else None),
        "g_dz": torch.full((1,), 7.0, dtype=torch.float32, device="cuda") if (want_dz or tm) else None,
    }
    plan.forward_loss(obj, probe, pos, tilt, meas, out["loss"], out["loss_per_pos"], out["intensity"])
    plan.backward(obj, probe, pos, tilt, meas, out["g_object"], out["g_probe"], out["g_positions"], out["g_tilt"],
                  out["g_dz"], flags=bwd_flags)
    rc, fl = plan.status()
    res = {k: (v.cpu().numpy() if v is not None else None) for k, v in out.items()}
    res["status"] = rc
    res["plan"] = plan
    return res


def check_against_oracle(res, ref, case, scale_ref=None):
    """Loss within 1e-4, every gradient within 1e-3 relative L2.  `scale_ref` (evaluation point B
    only, R26): position / tilt / dz gradients vanish analytically for a vacuum object, so their
    error is measured against the same gradient's norm at evaluation point A when that is larger."""
    cfg = case["cfg"]
    assert res["status"] == 0
    assert abs(res["loss"][0] - ref["loss"]) <= LOSS_RTOL * abs(ref["loss"]), (res["loss"][0], ref["loss"])
    np.testing.assert_allclose(res["loss_per_pos"], ref["loss_per_pos"], rtol=LOSS_RTOL)

    def err(x, r, key=None, reduce=lambda a: a):
        den = np.linalg.norm(np.ravel(reduce(r)))
        if scale_ref is not None and key is not None:
            den = max(den, np.linalg.norm(np.ravel(reduce(scale_ref[key]))))
        return float(np.linalg.norm(np.ravel(x - reduce(r))) / max(den, 1e-300))

    errs = {"g_object": err(res["g_object"], ref["g_object"]),
            "g_probe": err(res["g_probe"], ref["g_probe"]),
            "g_positions": err(res["g_positions"], ref["g_positions"], "g_positions")}
    if case["tilt_mode"] == 2:
        errs["g_tilt"] = err(res["g_tilt"], ref["g_tilt"], "g_tilt")
    elif case["tilt_mode"] == 1:
        errs["g_tilt"] = err(res["g_tilt"], ref["g_tilt"], "g_tilt", reduce=lambda a: a.sum(0))
    if res["g_dz"] is not None and cfg.Nz > 1:
        errs["g_dz"] = err(res["g_dz"][0], np.float64(ref["g_dz"]), "g_dz")
    bad = {k: v for k, v in errs.items() if not v <= GRAD_RTOL}
    assert not bad, f"gradients outside {GRAD_RTOL}: {bad} (all: {errs})"
    return errs


# (config, evaluation point, number of positions): sizes the oracle finishes in seconds that still
# span several CTAs / clusters and leave a ragged last wave of CTAs.
SMALL = [(1, "A", 32), (1, "B", 32), (2, "A", 40), (2, "B", 12), (3, "A", 20), (3, "B", 6),
         (4, "A", 14), (4, "B", 5), (5, "A", 5), (5, "B", 3)]


@pytest.mark.parametrize("c,which,B", SMALL)
def test_parity_all_configs(pty, c, which, B):
    cfg = synth.get_config(c)
    idx = synth.minibatch(cfg, 0, cfg.B)[:B]
    case = make_case(c, which, idx)
    if which == "B":      # ill-conditioned dark-field pixels: loss on the full data, gradients masked (R26)
        full = run_gpu(pty, case)
        L, lb, _ = oracle.forward_loss_batch(case["object"], case["probe"], case["positions"], case["tilt"],
                                             case["meas"], geom_of(cfg))
        assert abs(full["loss"][0] - L) <= LOSS_RTOL * L
        np.testing.assert_allclose(full["loss_per_pos"], lb, rtol=LOSS_RTOL)
        case = dict(case, meas=case["meas_masked"])
        scale_ref = oracle_grad(make_case(c, "A", idx))
    else:
        scale_ref = None
    ref = oracle_grad(case)
    res = run_gpu(pty, case, want_dz=cfg.Nz > 1)
    # intensities element by element (forward output), relative to the pattern's peak
    _, _, I_ref = oracle.forward_loss_batch(case["object"], case["probe"], case["positions"], case["tilt"],
                                            case["meas"], geom_of(cfg)) if B <= 8 else (None, None, None)
    if I_ref is not None:
        assert np.max(np.abs(res["intensity"] - I_ref)) <= 1e-4 * I_ref.max()
    errs = check_against_oracle(res, ref, case, scale_ref)
    print(f"c{c}{which} B={B}: loss rel {abs(res['loss'][0]-ref['loss'])/ref['loss']:.2e} " +
          " ".join(f"{k} {v:.2e}" for k, v in errs.items()))


@pytest.mark.parametrize("family", ["g2", "reg", "smem"])
def test_n128_kernel_families(pty, family, monkeypatch):
    """The three N = 128 kernel families (PTY_FFT128, read by pty_create): two items per CTA (default), one item
    per CTA on the register FFT, shared-memory passes.  B x M is odd here (7 x 3 after trimming the probe), so
    the two-item kernels run their padding item; with the dz gradient so that the kept spectra are covered."""
    monkeypatch.setenv("PTY_FFT128", family)
    cfg = synth.get_config(3, M=3)
    case = make_case(3, "A", synth.minibatch(cfg, 2, cfg.B)[:7])
    case = dict(case, cfg=cfg, probe=np.ascontiguousarray(case["probe"][:3]))
    ref = oracle_grad(case)
    res = run_gpu(pty, case, want_dz=True)
    check_against_oracle(res, ref, case)


def test_per_position_tilt_and_dz(pty):
    """tilt_mode 2 (one tilt per position) on the multislice config, with the dz gradient."""
    cfg = synth.get_config(3)
    case = make_case(3, "A", synth.minibatch(cfg, 1, cfg.B)[:7], tilt_mode=2)
    ref = oracle_grad(case)
    res = run_gpu(pty, case, want_dz=True)
    check_against_oracle(res, ref, case)


def test_full_minibatch_config1_and_2(pty):
    """Whole default minibatches (c1: 32, c2: 256) against the oracle."""
    for c in (1, 2):
        cfg = synth.get_config(c)
        case = make_case(c, "A", synth.minibatch(cfg, 2, cfg.B))
        check_against_oracle(run_gpu(pty, case), oracle_grad(case), case)


def test_headline_config4_batch64_compact(pty):
    """c4 with B = 64 consecutive raster positions (maximal patch overlap: the atomics' worst case)."""
    cfg = synth.get_config(4)
    case = make_case(4, "A", synth.compact_minibatch(cfg, 3, 64))
    check_against_oracle(run_gpu(pty, case), oracle_grad(case), case)


def test_headline_config4_full_batch_sampled(pty):
    """c4 at B = 1024 (the launch configuration bench.py times): per-position outputs on a sample of
    positions against the oracle; the summed gradients against the sum of sub-batch gradients."""
    cfg = synth.get_config(4)
    idx = synth.minibatch(cfg, 0, 1024)
    sample = np.arange(0, 1024, 64)
    case = make_case(4, "A", idx[sample])                 # oracle measurements for the sample only
    ev = synth.eval_point(cfg, "A")
    meas = np.zeros((1024, cfg.N, cfg.N), np.float32)
    rng = np.random.default_rng(5)
    meas[:] = np.sqrt(rng.poisson(2.0, size=(1, cfg.N, cfg.N))).astype(np.float32)   # filler for the rest
    meas[sample] = case["meas"]
    full = dict(case, positions=np.ascontiguousarray(ev["positions"][idx]), meas=meas, indices=idx)
    res = run_gpu(pty, full)
    ref = oracle_grad(case)
    np.testing.assert_allclose(res["loss_per_pos"][sample], ref["loss_per_pos"], rtol=LOSS_RTOL)
    assert rel_l2(res["g_positions"][sample], ref["g_positions"]) <= GRAD_RTOL
    assert abs(res["loss"][0] - res["loss_per_pos"].astype(np.float64).sum()) <= 1e-6 * res["loss"][0]
    # linearity over positions: gradient of the batch = sum over four disjoint quarters
    acc_obj = np.zeros_like(res["g_object"], dtype=np.complex128)
    acc_probe = np.zeros_like(res["g_probe"], dtype=np.complex128)
    for q in range(4):
        sl = slice(256 * q, 256 * (q + 1))
        part = dict(full, positions=full["positions"][sl], meas=meas[sl])
        r = run_gpu(pty, part)
        acc_obj += r["g_object"]
        acc_probe += r["g_probe"]
    assert rel_l2(res["g_object"], acc_obj) <= 1e-5
    assert rel_l2(res["g_probe"], acc_probe) <= 1e-5


def test_config3_and_5_default_batches_sampled(pty):
    """c3 (B = 512) and c5 (B = 128, 256^2 cluster path) at full minibatch size, sampled per-position outputs."""
    for c, nsample in ((3, 12), (5, 4)):
        cfg = synth.get_config(c)
        idx = synth.minibatch(cfg, 0, cfg.B)
        sample = np.linspace(0, cfg.B - 1, nsample).astype(int)
        case = make_case(c, "A", idx[sample])
        ev = synth.eval_point(cfg, "A")
        meas = np.ones((cfg.B, cfg.N, cfg.N), np.float32)
        meas[sample] = case["meas"]
        full = dict(case, positions=np.ascontiguousarray(ev["positions"][idx]), meas=meas, indices=idx)
        res = run_gpu(pty, full)
        ref = oracle_grad(case)
        np.testing.assert_allclose(res["loss_per_pos"][sample], ref["loss_per_pos"], rtol=LOSS_RTOL)
        assert rel_l2(res["g_positions"][sample], ref["g_positions"]) <= GRAD_RTOL
        assert np.all(np.isfinite(res["g_object"])) and np.all(np.isfinite(res["g_probe"]))


# ----------------------------------------------------------------------------- edge cases
def test_empty_batch_and_single_position(pty):
    cfg = synth.get_config(1)
    case = make_case(1, "A", np.array([5]))
    res = run_gpu(pty, case)
    check_against_oracle(res, oracle_grad(case), case)
    empty = dict(case, positions=np.zeros((0, 2), np.float32), meas=np.zeros((0, cfg.N, cfg.N), np.float32))
    r0 = run_gpu(pty, empty, plan=res["plan"])
    assert r0["status"] == 0 and r0["loss"][0] == 0.0
    assert np.all(r0["g_object"] == 0) and np.all(r0["g_probe"] == 0)


def test_patches_at_the_object_border_and_out_of_bounds_flag(pty):
    cfg = synth.get_config(1)
    case = make_case(1, "A", np.arange(4))
    edge = np.array([[0.0, 0.0], [cfg.H - cfg.N, cfg.W - cfg.N], [0.3, cfg.W - cfg.N - 0.4], [cfg.H - cfg.N + 0.2, 0.49]],
                    np.float32)
    case["positions"] = edge
    res = run_gpu(pty, case)
    check_against_oracle(res, oracle_grad(case), case)
    bad = dict(case, positions=np.array([[-3.0, 5.0], [10.0, cfg.W - cfg.N + 2.0], [5, 5], [6, 6]], np.float32))
    r = run_gpu(pty, bad)
    assert r["status"] == pty.PTY_ERR_BOUNDS and np.all(np.isfinite(r["g_object"]))
    assert r["plan"].status()[0] == 0            # the flag is cleared once reported


def test_argument_errors(pty):
    cfg = synth.get_config(1)
    case = make_case(1, "A", np.arange(4))
    plan = pty.Plan(cfg.Nz, cfg.H, cfg.W, cfg.M, cfg.N, 2, cfg.dz, cfg.lam, cfg.dx)
    with pytest.raises(pty.PtyError) as e:
        run_gpu(pty, case, plan=plan)            # B = 4 > Bmax = 2
    assert e.value.code == pty.PTY_ERR_INVALID_ARG
    with pytest.raises(pty.PtyError):
        pty.Plan(1, 160, 160, 1, 96, 4, 1.0, 0.02, 0.1)      # unsupported N


def test_accumulate_recompute_and_backward_without_forward(pty):
    cfg = synth.get_config(3)
    idx = synth.minibatch(cfg, 4, cfg.B)[:6]
    case = make_case(3, "A", idx)
    ref = oracle_grad(case)
    res = run_gpu(pty, case)
    plan = res["plan"]
    obj, probe = dev(case["object"]), dev(case["probe"])
    pos, meas = dev(case["positions"]), dev(case["meas"])
    # backward alone (no forward before it on these pointers) must run the forward itself
    g1 = torch.zeros_like(obj); p1 = torch.zeros_like(probe); q1 = torch.zeros(6, 2, device="cuda")
    plan.backward(obj, probe, pos, None, meas, g1, p1, q1)
    assert rel_l2(g1.cpu().numpy(), ref["g_object"]) <= GRAD_RTOL
    # accumulate: a second call adds
    plan.backward(obj, probe, pos, None, meas, g1, p1, q1, flags=pty.PTY_BWD_ACCUMULATE | pty.PTY_BWD_RECOMPUTE)
    assert rel_l2(g1.cpu().numpy(), 2 * ref["g_object"]) <= GRAD_RTOL
    assert rel_l2(p1.cpu().numpy(), 2 * ref["g_probe"]) <= GRAD_RTOL
    assert rel_l2(q1.cpu().numpy(), 2 * ref["g_positions"]) <= GRAD_RTOL


def test_run_to_run_repeatability_bound(pty):
    """Atomic accumulation order is not fixed: two runs agree to float32 rounding (reading R25)."""
    cfg = synth.get_config(2)
    case = make_case(2, "A", synth.compact_minibatch(cfg, 0, 48))
    a = run_gpu(pty, case)
    b = run_gpu(pty, case, plan=a["plan"])
    assert rel_l2(a["g_object"], b["g_object"]) <= 1e-5
    assert rel_l2(a["g_probe"], b["g_probe"]) <= 1e-5
    assert a["loss"][0] == pytest.approx(b["loss"][0], rel=1e-6)


def test_grad_host_end_to_end(pty):
    cfg = synth.get_config(1)
    case = make_case(1, "A", synth.minibatch(cfg, 1, cfg.B))
    ref = oracle_grad(case)
    plan = pty.Plan(cfg.Nz, cfg.H, cfg.W, cfg.M, cfg.N, cfg.B, cfg.dz, cfg.lam, cfg.dx, flags=pty.PTY_FLAG_HOST)
    pin = lambda x: torch.from_numpy(np.ascontiguousarray(x)).pin_memory()
    h_loss = torch.zeros(1, dtype=torch.float64).pin_memory()
    h_go = torch.zeros(case["object"].shape, dtype=torch.complex64).pin_memory()
    h_gp = torch.zeros(case["probe"].shape, dtype=torch.complex64).pin_memory()
    h_gq = torch.zeros(cfg.B, 2).pin_memory()
    plan.grad_host(pin(case["object"]), pin(case["probe"]), pin(case["positions"]), None, pin(case["meas"]),
                   h_loss, h_go, h_gp, h_gq)
    assert abs(h_loss[0].item() - ref["loss"]) <= LOSS_RTOL * ref["loss"]
    assert rel_l2(h_go.numpy(), ref["g_object"]) <= GRAD_RTOL
    assert rel_l2(h_gp.numpy(), ref["g_probe"]) <= GRAD_RTOL
    assert rel_l2(h_gq.numpy(), ref["g_positions"]) <= GRAD_RTOL


# ----------------------------------------------------------------------------- Adam / pty_step
def test_adam_update_kernel_single_step(pty):
    plan = pty.Plan(1, 160, 160, 1, 64, 4, 1.0, 0.02, 0.1)
    rng = np.random.default_rng(3)
    for n in (1, 7, 4096 + 3):
        th = rng.standard_normal(n).astype(np.float32)
        g = (rng.standard_normal(n) * 10.0 ** rng.integers(-4, 3, n)).astype(np.float32)
        m = (0.1 * rng.standard_normal(n)).astype(np.float32)
        v = (0.01 * rng.random(n)).astype(np.float32)
        tth, tg, tm, tv = dev(th), dev(g), dev(m), dev(v)
        b1, b2, lr = float(np.float32(0.9)), float(np.float32(0.999)), float(np.float32(5e-4))
        plan.adam_update(tth, tg, tm, tv, lr=lr, beta1=b1, beta2=b2, t=3)
        rth, rm, rv = oracle.adam_step(th, g, m, v, 3, lr=lr, beta1=b1, beta2=b2)
        np.testing.assert_allclose(tth.cpu().numpy(), rth, rtol=2e-6, atol=2e-8)
        np.testing.assert_allclose(tm.cpu().numpy(), rm, rtol=2e-6, atol=2e-7 * np.abs(rm).max())
        np.testing.assert_allclose(tv.cpu().numpy(), rv, rtol=2e-6, atol=2e-7 * np.abs(rv).max())


def test_pty_step_matches_oracle_adam_over_steps(pty):
    """pty_step on c1: after 1 step the update is pinned tightly; after 10 steps loosely (B9)."""
    cfg = synth.get_config(1)
    idx = synth.minibatch(cfg, 0, cfg.B)
    case = make_case(1, "A", idx)
    plan = pty.Plan(cfg.Nz, cfg.H, cfg.W, cfg.M, cfg.N, cfg.B, cfg.dz, cfg.lam, cfg.dx, flags=pty.PTY_FLAG_STEP)
    obj, probe, pos, meas = dev(case["object"]), dev(case["probe"]), dev(case["positions"]), dev(case["meas"])
    state = {}
    for name, t in (("object", obj), ("probe", probe), ("positions", pos)):
        n = t.numel() * (2 if t.is_complex() else 1)
        state["m_" + name] = torch.zeros(n, device="cuda")
        state["v_" + name] = torch.zeros(n, device="cuda")
    lr = {"object": 5e-4, "probe": 1e-4, "positions": 1e-3}
    o_obj, o_probe, o_pos = (case["object"].astype(np.complex128), case["probe"].astype(np.complex128),
                             case["positions"].astype(np.float64))
    om = {"object": np.zeros(o_obj.size * 2), "probe": np.zeros(o_probe.size * 2), "positions": np.zeros(o_pos.shape)}
    ov = {k: np.zeros_like(v) for k, v in om.items()}
    geom = geom_of(cfg)
    losses = []
    for t in range(1, 11):
        hp = pty.pty_adam(lr["object"], lr["probe"], lr["positions"], 0.0, 0.9, 0.999, 1e-8, t)
        loss = plan.step(obj, probe, pos, None, meas, hp, state)
        losses.append(loss.item())
        g = oracle.grad_batch(o_obj, o_probe, o_pos, None, case["meas"], geom, workers=WORKERS)
        assert abs(losses[-1] - g["loss"]) <= (1e-4 if t == 1 else 2e-3) * g["loss"]
        o_obj, om["object"], ov["object"] = oracle.adam_step(o_obj, g["g_object"], om["object"], ov["object"], t, lr["object"])
        o_obj = o_obj.reshape(case["object"].shape)
        o_probe, om["probe"], ov["probe"] = oracle.adam_step(o_probe, g["g_probe"], om["probe"], ov["probe"], t, lr["probe"])
        o_probe = o_probe.reshape(case["probe"].shape)
        o_pos, om["positions"], ov["positions"] = oracle.adam_step(o_pos, g["g_positions"], om["positions"], ov["positions"], t, lr["positions"])
        if t == 1:
            # first step: every touched coordinate moves by ~lr*sign(g); compare where |g| is not tiny
            gobj = g["g_object"].view(np.float64)
            big = np.abs(gobj) > 1e-3 * np.abs(gobj).max()
            d_gpu = obj.cpu().numpy().astype(np.complex128).view(np.float64) - case["object"].astype(np.complex128).view(np.float64)
            np.testing.assert_allclose(d_gpu[big], -lr["object"] * np.sign(gobj[big]), rtol=1e-3, atol=1e-7)
            assert rel_l2(pos.cpu().numpy() - case["positions"], o_pos - case["positions"]) <= 1e-3
    assert rel_l2(obj.cpu().numpy(), o_obj) <= 1e-5
    assert rel_l2(probe.cpu().numpy(), o_probe) <= 1e-5
    assert rel_l2(obj.cpu().numpy() - case["object"], o_obj - case["object"]) <= 0.05
    assert rel_l2(probe.cpu().numpy() - case["probe"], o_probe - case["probe"]) <= 0.05
    assert losses[-1] < losses[0]
