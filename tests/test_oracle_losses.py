"""Pins for oracle/losses.py (Eq. 5-9; mixed object states Eq. 2) and
oracle/constraints.py (PAPER.md:147, :289, :301-312 Eq. 13, :539): literal values written out from the printed
formulas, closed forms, invariants, central finite differences on tiny inputs and torch.autograd (float64) as an
independent third opinion."""
import math

import numpy as np
import pytest

import oracle
from oracle import Geometry
from oracle import constraints as oc
from oracle import losses as ol

GEOM = Geometry(dz=2.0, lam=0.0197, dx=0.1)


def crandn(rng, *shape):
    return rng.standard_normal(shape) + 1j * rng.standard_normal(shape)


def tiny(seed=5, N=8, H=14, Nz=2, M=2, B=3, states=None):
    rng = np.random.default_rng(seed)
    shp = (Nz, H, H) if states is None else (states, Nz, H, H)
    amp = 1 - 0.1 * rng.random(shp)
    phase = 0.4 * rng.standard_normal(shp)
    probe = crandn(rng, M, N, N)
    pos = np.floor(rng.uniform(0.6, H - N - 0.6, (B, 2))) + rng.uniform(-0.4, 0.4, (B, 2))
    tilt = rng.normal(0, 2e-3, (B, 2))
    a = np.sqrt(rng.poisson(3.0 * np.ones((B, N, N)))).astype(np.float64) + 0.1
    return amp, phase, probe, pos, tilt, a


# ------------------------------------------------------------------ Eq. 5-7 values, written out by hand
def test_data_terms_literal_values():
    """Two patterns of two pixels: every average of Eq. 5-7 typed out."""
    I = np.array([[[4.0, 9.0]], [[1.0, 16.0]]])
    a = np.array([[[1.0, 2.0]], [[2.0, 3.0]]])                  # I_meas = 1, 4, 4, 9
    t, _ = ol.data_terms(I, a, ol.LossWeights())
    # Eq. 5: sqrt(mean((2-1)^2, (3-2)^2, (1-2)^2, (4-3)^2)) / mean(1, 2, 2, 3) = 1 / 2
    assert t["gaussian"] == pytest.approx(0.5)
    # Eq. 6: -mean(I_m log(I + eps) - I) / mean(I_m)
    eps = 1e-6
    num = np.mean([1 * math.log(4 + eps) - 4, 4 * math.log(9 + eps) - 9, 4 * math.log(1 + eps) - 1, 9 * math.log(16 + eps) - 16])
    assert t["poisson"] == pytest.approx(-num / np.mean([1, 4, 4, 9]))
    # Eq. 7: <I>_B = (2.5, 12.5), <I_meas>_B = (2.5, 6.5); sqrt(mean((sqrt(2.5)-sqrt(2.5))^2, (sqrt(12.5)-sqrt(6.5))^2)) / 2
    assert t["pacbed"] == pytest.approx(math.sqrt(0.5 * (math.sqrt(12.5) - math.sqrt(6.5)) ** 2) / 2.0)


def test_gaussian_term_equals_eq5_of_the_plain_sum_and_scales():
    rng = np.random.default_rng(0)
    I, a = rng.random((3, 4, 4)) * 5 + 0.1, rng.random((3, 4, 4)) * 2
    t, _ = ol.data_terms(I, a, ol.LossWeights())
    S = sum(oracle.loss_from_intensity(I[b], a[b]) for b in range(3))
    assert t["gaussian"] == pytest.approx(oracle.loss_gaussian_eq5(S, I.size, a.mean()))
    # NRMSE: scaling model and data intensities by c^2 leaves Eq. 5 and Eq. 7 unchanged
    t2, _ = ol.data_terms(9.0 * I, 3.0 * a, ol.LossWeights())
    assert t2["gaussian"] == pytest.approx(t["gaussian"]) and t2["pacbed"] == pytest.approx(t["pacbed"])
    # exact model: Gaussian and PACBED vanish, and the Poisson term is stationary (dL_P/dI = 0 up to eps)
    a1 = a + 1.0                                                         # I >= 1 so that eps / (I + eps) <= 1e-6
    t3, g3 = ol.data_terms(a1 * a1, a1, ol.LossWeights(gaussian=0, poisson=1))
    assert t3["gaussian"] == pytest.approx(0, abs=1e-12) and t3["pacbed"] == pytest.approx(0, abs=1e-12)
    assert np.max(np.abs(g3)) < 1e-6 / a1.size


@pytest.mark.parametrize("w", [ol.LossWeights(1, 0, 0, 0), ol.LossWeights(0, 1, 0, 0), ol.LossWeights(0, 0, 1, 0),
                               ol.LossWeights(0.7, 0.3, 0.5, 0)])
def test_data_terms_gradient_by_finite_differences(w):
    rng = np.random.default_rng(2)
    I, a = rng.random((3, 3, 4)) * 5 + 0.5, rng.random((3, 3, 4)) * 2 + 0.1
    val = lambda I_: sum(wt * v for wt, v in zip((w.gaussian, w.poisson, w.pacbed), ol.data_terms(I_, a, w)[0].values()))
    _, g = ol.data_terms(I, a, w)
    h = 1e-6
    for idx in np.ndindex(I.shape):
        Ip, Im = I.copy(), I.copy()
        Ip[idx] += h; Im[idx] -= h
        assert g[idx] == pytest.approx((val(Ip) - val(Im)) / (2 * h), rel=1e-6, abs=1e-10)


# ------------------------------------------------------------------ Eq. 8 and the amplitude / phase chain rule
def test_sparse_term_counts_overlaps_and_matches_brute_force():
    rng = np.random.default_rng(3)
    phase = rng.standard_normal((2, 10, 10))
    pos = np.array([[1.0, 2.0], [1.0, 2.0], [2.3, 0.2]])       # first two patches coincide: counted twice
    L, g = ol.sparse_term(phase, pos, 4)
    brute = np.mean([np.abs(phase[:, 1:5, 2:6]), np.abs(phase[:, 1:5, 2:6]), np.abs(phase[:, 2:6, 0:4])])
    assert L == pytest.approx(brute)
    n = 3 * 2 * 16
    assert g[0, 1, 2] == pytest.approx(2 * np.sign(phase[0, 1, 2]) / n)       # covered twice
    assert g[0, 5, 0] == pytest.approx(np.sign(phase[0, 5, 0]) / n)           # covered once
    assert g[0, 9, 9] == 0.0
    assert ol.sparse_term(np.full((1, 6, 6), -0.25), np.array([[0.0, 0.0]]), 4)[0] == pytest.approx(0.25)


def test_amp_phase_chain_rule_matches_directional_derivative():
    rng = np.random.default_rng(4)
    amp, phase = 1 + 0.1 * rng.standard_normal((2, 5, 5)), rng.standard_normal((2, 5, 5))
    c = crandn(rng, 2, 5, 5)
    f = lambda A, p: float(np.sum(np.abs(ol.object_from_amp_phase(A, p) - c) ** 2))     # any real function of O
    g_O = 2 * (ol.object_from_amp_phase(amp, phase) - c)                               # dL/dRe + i dL/dIm
    gA, gp = ol.amp_phase_gradients(g_O, amp, phase)
    h = 1e-6
    for idx in [(0, 1, 2), (1, 4, 0)]:
        d = np.zeros_like(amp); d[idx] = h
        assert gA[idx] == pytest.approx((f(amp + d, phase) - f(amp - d, phase)) / (2 * h), rel=1e-6)
        assert gp[idx] == pytest.approx((f(amp, phase + d) - f(amp, phase - d)) / (2 * h), rel=1e-6)
    # unit amplitude, zero phase: O = 1, g_A = Re g_O, g_phi = Im g_O
    one, zero = np.ones((1, 2, 2)), np.zeros((1, 2, 2))
    gA, gp = ol.amp_phase_gradients(np.full((1, 2, 2), 3 - 2j), one, zero)
    assert np.allclose(gA, 3) and np.allclose(gp, -2)


# ------------------------------------------------------------------ Eq. 9 end to end
W_ALL = ol.LossWeights(gaussian=1.0, poisson=0.4, pacbed=0.6, sparse=0.1)


def _total(amp, phase, probe, pos, tilt, a, w=W_ALL, geom=GEOM):
    return ol.total_loss_and_gradients(None, probe, pos, tilt, a, geom, w, amp=amp, phase=phase)


def test_total_loss_gradients_by_finite_differences():
    amp, phase, probe, pos, tilt, a = tiny()
    ref = _total(amp, phase, probe, pos, tilt, a)
    L = lambda **kw: _total(**{**dict(amp=amp, phase=phase, probe=probe, pos=pos, tilt=tilt, a=a), **kw})["loss"]
    h = 1e-6
    rng = np.random.default_rng(9)
    for name, arr, g in (("amp", amp, ref["g_amp"]), ("phase", phase, ref["g_phase"])):
        for _ in range(12):
            idx = tuple(rng.integers(0, s) for s in arr.shape)
            d = np.zeros_like(arr); d[idx] = h
            fd = (L(**{name: arr + d}) - L(**{name: arr - d})) / (2 * h)
            assert g[idx] == pytest.approx(fd, rel=2e-5, abs=1e-9), (name, idx)
    for _ in range(8):
        idx = tuple(rng.integers(0, s) for s in probe.shape)
        for unit, part in ((1.0, np.real), (1j, np.imag)):
            d = np.zeros_like(probe); d[idx] = h * unit
            fd = (L(probe=probe + d) - L(probe=probe - d)) / (2 * h)
            assert part(ref["g_probe"][idx]) == pytest.approx(fd, rel=2e-5, abs=1e-9)
    for b in range(len(pos)):
        for ax in range(2):
            d = np.zeros_like(pos); d[b, ax] = h
            assert ref["g_positions"][b, ax] == pytest.approx((L(pos=pos + d) - L(pos=pos - d)) / (2 * h), rel=2e-5, abs=1e-9)
            d = np.zeros_like(tilt); d[b, ax] = 1e-7
            assert ref["g_tilt"][b, ax] == pytest.approx((L(tilt=tilt + d) - L(tilt=tilt - d)) / 2e-7, rel=1e-4, abs=1e-7)
    fd = (_total(amp, phase, probe, pos, tilt, a, geom=Geometry(GEOM.dz + 1e-5, GEOM.lam, GEOM.dx))["loss"]
          - _total(amp, phase, probe, pos, tilt, a, geom=Geometry(GEOM.dz - 1e-5, GEOM.lam, GEOM.dx))["loss"]) / 2e-5
    assert ref["g_dz"] == pytest.approx(fd, rel=1e-5)


def test_gaussian_only_total_is_a_positive_multiple_of_the_plain_sum_gradient():
    """Reading R13: Eq. 5's gradient = plain-sum gradient / (2 B N^2 <a>^2 L_G)."""
    amp, phase, probe, pos, tilt, a = tiny(seed=8)
    obj = ol.object_from_amp_phase(amp, phase)
    ref = oracle.grad_batch(obj, probe, pos, tilt, a, GEOM)
    tot = ol.total_loss_and_gradients(obj, probe, pos, tilt, a, GEOM, ol.LossWeights(1, 0, 0, 0))
    c = 1.0 / (2.0 * a.size * a.mean() ** 2 * tot["terms"]["gaussian"])
    assert tot["terms"]["gaussian"] == pytest.approx(oracle.loss_gaussian_eq5(ref["loss"], a.size, a.mean()))
    for k in ("g_object", "g_probe", "g_positions", "g_tilt"):
        assert np.allclose(tot[k], c * ref[k], rtol=1e-10, atol=1e-14)


def test_mixed_object_states_sum_incoherently_and_split_the_gradient():
    """Eq. 2: I = sum_n sum_m |.|^2.  Two identical states double I; the gradient of state n comes from its own waves."""
    amp, phase, probe, pos, tilt, a = tiny(seed=6, states=2)
    obj = ol.object_from_amp_phase(amp, phase)
    I2 = ol.intensity_batch_states(obj, probe, pos, tilt, GEOM)
    assert np.allclose(I2, oracle.intensity_batch(obj[0], probe, pos, tilt, GEOM)
                       + oracle.intensity_batch(obj[1], probe, pos, tilt, GEOM))
    same = np.stack([obj[0], obj[0]])
    assert np.allclose(ol.intensity_batch_states(same, probe, pos, tilt, GEOM),
                       2 * oracle.intensity_batch(obj[0], probe, pos, tilt, GEOM))
    ref = ol.total_loss_and_gradients(obj, probe, pos, tilt, a, GEOM, W_ALL)
    assert ref["g_object"].shape == obj.shape
    h = 1e-6
    for idx in [(0, 1, 5, 6), (1, 0, 7, 4)]:
        d = np.zeros_like(obj); d[idx] = h
        fd = (ol.total_loss_and_gradients(obj + d, probe, pos, tilt, a, GEOM, ol.LossWeights(1, 0.4, 0.6, 0))["loss"]
              - ol.total_loss_and_gradients(obj - d, probe, pos, tilt, a, GEOM, ol.LossWeights(1, 0.4, 0.6, 0))["loss"]) / (2 * h)
        assert ref["g_object"][idx].real == pytest.approx(fd, rel=2e-5, abs=1e-9)


def test_total_loss_against_torch_autograd():
    """Third opinion: Eq. 1-9 retyped in torch float64 with autograd (the paper's mechanism)."""
    torch = pytest.importorskip("torch")
    amp, phase, probe, pos, tilt, a = tiny(seed=12, B=2)
    w = W_ALL
    ref = _total(amp, phase, probe, pos, tilt, a, w)
    N = probe.shape[-1]
    tA = torch.tensor(amp, requires_grad=True)
    tp = torch.tensor(phase, requires_grad=True)
    tP = torch.tensor(probe, requires_grad=True)
    O = tA * torch.exp(1j * tp)
    kp = torch.fft.fftfreq(N, dtype=torch.float64)
    k = torch.fft.fftfreq(N, d=GEOM.dx, dtype=torch.float64)
    Is, sp = [], []
    for b in range(len(pos)):
        r = np.floor(pos[b] + 0.5).astype(int)
        d = pos[b] - r
        E = torch.exp(-2j * math.pi * (kp[:, None] * d[0] + kp[None, :] * d[1]))
        psi = torch.fft.ifft2(E * torch.fft.fft2(tP, norm="ortho"), norm="ortho")
        chi = (-math.pi * GEOM.lam * (k[None, :] ** 2 + k[:, None] ** 2) * GEOM.dz
               + 2 * math.pi * GEOM.dz * (k[None, :] * math.tan(tilt[b, 1]) + k[:, None] * math.tan(tilt[b, 0])))
        Mk = torch.exp(1j * chi)
        patch = O[:, r[0]:r[0] + N, r[1]:r[1] + N]
        sp.append(tp[:, r[0]:r[0] + N, r[1]:r[1] + N].abs())
        for s in range(O.shape[0]):
            phi = patch[s] * psi
            if s < O.shape[0] - 1:
                psi = torch.fft.ifft2(Mk * torch.fft.fft2(phi, norm="ortho"), norm="ortho")
        Is.append((torch.fft.fft2(phi, norm="ortho").abs() ** 2).sum(0))
    I = torch.stack(Is)
    ta = torch.tensor(a)
    LG = torch.sqrt(((I.sqrt() - ta) ** 2).mean()) / ta.mean()
    LP = -((ta ** 2) * torch.log(I + w.eps) - I).mean() / (ta ** 2).mean()
    LPB = torch.sqrt(((I.mean(0).sqrt() - (ta ** 2).mean(0).sqrt()) ** 2).mean()) / ta.mean()
    LS = torch.stack(sp).mean()
    L = w.gaussian * LG + w.poisson * LP + w.pacbed * LPB + w.sparse * LS
    L.backward()
    assert ref["loss"] == pytest.approx(L.item(), rel=1e-12)
    assert np.allclose(ref["g_amp"], tA.grad.numpy(), rtol=1e-9, atol=1e-13)
    assert np.allclose(ref["g_phase"], tp.grad.numpy(), rtol=1e-9, atol=1e-13)
    assert np.allclose(ref["g_probe"], tP.grad.numpy(), rtol=1e-9, atol=1e-13)


# ------------------------------------------------------------------ constraints
def test_orthogonalisation_invariants_and_known_case():
    rng = np.random.default_rng(1)
    P = crandn(rng, 4, 6, 6)
    Q, lam = oc.orthogonalize_modes(P)
    flat, qf = P.reshape(4, -1), Q.reshape(4, -1)
    G = np.conj(qf) @ qf.T
    assert np.allclose(G, np.diag(lam), atol=1e-10)                       # orthogonal, powers on the diagonal
    assert np.all(np.diff(lam) <= 1e-12)                                  # decreasing power
    assert np.allclose(qf.T @ np.conj(qf), flat.T @ np.conj(flat))        # same density operator sum_k |P_k><P_k|
    assert lam.sum() == pytest.approx(np.sum(np.abs(P) ** 2))             # total power
    # known case: two modes a, b with <a|b> = 0 already, |b| > |a|: the result is (b, a) up to phase
    a = np.zeros((3, 3), complex); a[0, 0] = 1.0
    b = np.zeros((3, 3), complex); b[1, 1] = 2.0j
    Q, lam = oc.orthogonalize_modes(np.stack([a, b]))
    assert np.allclose(lam, [4.0, 1.0])
    assert abs(np.vdot(Q[0], b)) == pytest.approx(4.0) and abs(np.vdot(Q[1], a)) == pytest.approx(1.0)
    # known case: P2 = P1 (fully coherent): one mode of power 2 |P1|^2 and an empty one
    Q, lam = oc.orthogonalize_modes(np.stack([P[0], P[0]]))
    assert lam[0] == pytest.approx(2 * np.sum(np.abs(P[0]) ** 2)) and lam[1] == pytest.approx(0, abs=1e-9)
    assert np.allclose(np.abs(Q[0]), math.sqrt(2) * np.abs(P[0]))


def test_rz_filter_taps_and_edges():
    g = oc.rz_taps(1.0)
    assert len(g) == 5 and g.sum() == pytest.approx(1.0)
    e = np.exp(-np.array([4, 1, 0, 1, 4]) / 2.0)
    assert np.allclose(g, e / e.sum())                                    # exp(-j^2 / 2 sigma^2), normalised
    x = np.zeros((7, 2, 2)); x[3] = 1.0
    y = oc.rz_filter(x, 1.0)
    assert np.allclose(y[1:6, 0, 0], g) and y[0, 0, 0] == 0 and y[6, 0, 0] == 0
    assert np.allclose(oc.rz_filter(np.full((4, 3, 3), 2.5), 1.0), 2.5)   # depth-constant object unchanged
    top = np.zeros((6, 1, 1)); top[0] = 1.0                               # replicate, never wrap
    yt = oc.rz_filter(top, 1.0)
    assert yt[0, 0, 0] == pytest.approx(g[2] + g[1] + g[0]) and yt[5, 0, 0] == 0.0
    z = crandn(np.random.default_rng(0), 2, 5, 3, 3)
    assert np.allclose(oc.rz_filter(z, 0.7), oc.rz_filter(z.real, 0.7) + 1j * oc.rz_filter(z.imag, 0.7))


def test_clip_and_clamp():
    assert np.array_equal(oc.clip_phase_positive(np.array([-0.2, 0.0, 0.3])), [0.0, 0.0, 0.3])
    assert np.array_equal(oc.clamp_amplitude(np.array([0.9, 0.98, 1.0, 1.5])), [0.98, 0.98, 1.0, 1.02])
