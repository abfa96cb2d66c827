"""Pins for the float64 oracle's forward model: brute force, closed forms, invariants.

Each test fixes one thing the paper / the mathematics determines, chosen so that a plausible
mistake in ``oracle/multislice.py`` (a sign, an index, a transposed axis, a dropped term)
fails at least one of them (SURVEY.md §8(c) "What pins each part").
"""
import math

import numpy as np
import pytest

import oracle
from oracle import Geometry

RNG = np.random.default_rng(7)
GEOM = Geometry(dz=2.0, lam=0.0197, dx=0.1)


def crandn(*shape):
    return RNG.standard_normal(shape) + 1j * RNG.standard_normal(shape)


# ------------------------------------------------------------------ DFT (R1)
def brute_dft2(x, sign):
    """O(N^4) definition: X[ky,kx] = (1/N) sum_{y,x} x[y,x] exp(sign 2 pi i (ky y + kx x)/N)."""
    n0, n1 = x.shape
    out = np.zeros((n0, n1), dtype=np.complex128)
    for ky in range(n0):
        for kx in range(n1):
            acc = 0j
            for y in range(n0):
                for xx in range(n1):
                    acc += x[y, xx] * np.exp(sign * 2j * math.pi * (ky * y / n0 + kx * xx / n1))
            out[ky, kx] = acc / math.sqrt(n0 * n1)
    return out


def test_dft2_matches_brute_force_8x8():
    x = crandn(8, 8)
    np.testing.assert_allclose(oracle.dft2(x), brute_dft2(x, -1), atol=1e-13)
    np.testing.assert_allclose(oracle.idft2(x), brute_dft2(x, +1), atol=1e-13)


def test_dft2_unitary_parseval_linear_batched():
    x, y = crandn(3, 16, 16), crandn(3, 16, 16)
    X = oracle.dft2(x)
    assert np.allclose(np.sum(abs(X) ** 2, axis=(1, 2)), np.sum(abs(x) ** 2, axis=(1, 2)), rtol=1e-13)
    np.testing.assert_allclose(oracle.idft2(X), x, atol=1e-13)
    np.testing.assert_allclose(oracle.dft2(2 * x - 3j * y), 2 * X - 3j * oracle.dft2(y), atol=1e-12)
    # batched transform acts on the last two axes only
    np.testing.assert_allclose(X[1], oracle.dft2(x[1]), atol=1e-13)


# ------------------------------------------------------------------ F1 split (R6)
def test_split_position():
    r, d = oracle.split_position(np.array([3.49, -0.2]))
    assert r.tolist() == [3, 0] and np.allclose(d, [0.49, -0.2])
    r, d = oracle.split_position(np.array([3.5, 7.75]))
    assert r.tolist() == [4, 8] and np.allclose(d, [-0.5, -0.25])
    assert r.dtype.kind == "i"


# ------------------------------------------------------------------ F2 shift (R2)
def test_shift_integer_is_roll_and_pins_sign_and_axis():
    P = crandn(2, 16, 16)
    np.testing.assert_allclose(oracle.shift_probe(P, np.array([3.0, 0.0])), np.roll(P, 3, axis=-2), atol=1e-12)
    np.testing.assert_allclose(oracle.shift_probe(P, np.array([0.0, -5.0])), np.roll(P, -5, axis=-1), atol=1e-12)


def test_shift_norm_composition_identity():
    P = crandn(1, 16, 16)
    a, b = np.array([0.3, -0.45]), np.array([-0.2, 0.1])
    Sa = oracle.shift_probe(P, a)
    assert np.isclose(np.linalg.norm(Sa), np.linalg.norm(P), rtol=1e-13)
    np.testing.assert_allclose(oracle.shift_probe(Sa, b), oracle.shift_probe(P, a + b), atol=1e-12)
    np.testing.assert_allclose(oracle.shift_probe(P, np.zeros(2)), P, atol=1e-13)


def test_shift_subpixel_moves_centroid():
    """A smooth blob shifted by +0.4 px along x has its centroid moved by +0.4 px."""
    y, x = np.mgrid[0:32, 0:32]
    blob = np.exp(-((y - 16) ** 2 + (x - 16) ** 2) / 18.0).astype(complex)[None]
    s = oracle.shift_probe(blob, np.array([0.0, 0.4]))
    w = abs(s[0]) ** 2
    assert abs((w * x).sum() / w.sum() - 16.4) < 1e-6
    assert abs((w * y).sum() / w.sum() - 16.0) < 1e-6


# ------------------------------------------------------------------ F3 crop
def test_crop_window_and_bounds():
    obj = np.arange(2 * 9 * 10).reshape(2, 9, 10).astype(complex)
    c = oracle.crop(obj, (2, 3), 4)
    assert c.shape == (2, 4, 4) and c[1, 0, 0] == obj[1, 2, 3] and c[0, 3, 1] == obj[0, 5, 4]
    with pytest.raises(ValueError):
        oracle.crop(obj, (6, 0), 4)
    with pytest.raises(ValueError):
        oracle.crop(obj, (0, -1), 4)


def test_translation_equivariance():
    """Shifting the object and all positions by the same integers leaves every I_b unchanged."""
    obj = np.exp(1j * RNG.standard_normal((2, 20, 22)))
    probe = crandn(2, 8, 8)
    pos = np.array([[3.2, 4.7], [6.6, 9.1]])
    I0 = oracle.intensity_batch(obj, probe, pos, None, GEOM)
    obj2 = np.roll(obj, (2, -3), axis=(1, 2))
    I1 = oracle.intensity_batch(obj2, probe, pos + np.array([2.0, -3.0]), None, GEOM)
    np.testing.assert_allclose(I1, I0, rtol=1e-12)


# ------------------------------------------------------------------ F4/F5 propagator
def test_propagator_identity_unit_modulus_composition():
    phi = crandn(2, 16, 16)
    M0 = oracle.propagator(16, Geometry(0.0, 0.0197, 0.1), (1e-3, -2e-3))
    np.testing.assert_allclose(oracle.propagate(phi, M0), phi, atol=1e-13)
    tilt = (0.7e-3, -0.4e-3)
    M1 = oracle.propagator(16, Geometry(3.0, 0.0197, 0.1), tilt)
    M2 = oracle.propagator(16, Geometry(4.5, 0.0197, 0.1), tilt)
    M3 = oracle.propagator(16, Geometry(7.5, 0.0197, 0.1), tilt)
    np.testing.assert_allclose(abs(M1), 1.0, atol=1e-14)
    np.testing.assert_allclose(M1 * M2, M3, atol=1e-12)
    out = oracle.propagate(phi, M1)
    assert np.isclose(np.linalg.norm(out), np.linalg.norm(phi), rtol=1e-13)


def test_propagator_gaussian_beam_closed_form():
    """exp(-r^2/w0^2) after z equals (1+iz/zR)^-1 exp(-r^2/(w0^2 (1+iz/zR))), zR = pi w0^2/lam.

    Pins the sign and the scale of the -i pi lam |k|^2 dz term (Eq. 4) and the unit of k (R8).
    """
    N, dx, lam, w0, z = 256, 0.1, 0.0197, 0.8, 50.0
    c = (np.arange(N) - N // 2) * dx
    r2 = c[:, None] ** 2 + c[None, :] ** 2
    beam = np.exp(-r2 / w0 ** 2).astype(complex)
    out = oracle.propagate(beam, oracle.propagator(N, Geometry(z, lam, dx), (0.0, 0.0)))
    q = 1.0 + 1j * z / (math.pi * w0 ** 2 / lam)
    np.testing.assert_allclose(out, np.exp(-r2 / (w0 ** 2 * q)) / q, atol=1e-12)


def test_propagator_tilt_is_lateral_roll():
    """lam -> 0 and dz tan(theta)/dx = n integer: propagation == roll(psi, -n) along that axis.

    Pins the sign of the tilt term and the (theta_y, theta_x) axis order.
    """
    N, dx, dz = 16, 0.1, 2.0
    psi = crandn(N, N)
    ty = math.atan(3 * dx / dz)
    tx = math.atan(-2 * dx / dz)
    My = oracle.propagator(N, Geometry(dz, 0.0, dx), (ty, 0.0))
    Mx = oracle.propagator(N, Geometry(dz, 0.0, dx), (0.0, tx))
    np.testing.assert_allclose(oracle.propagate(psi, My), np.roll(psi, -3, axis=0), atol=1e-12)
    np.testing.assert_allclose(oracle.propagate(psi, Mx), np.roll(psi, 2, axis=1), atol=1e-12)


def test_two_vacuum_slices_equal_one_thick_slice():
    """Nz slices of vacuum = one propagation over (Nz-1) dz (Eq. 3 has Nz-1 propagations, R7)."""
    probe = crandn(1, 16, 16)
    vac = np.ones((3, 24, 24), dtype=complex)
    f = oracle.forward_position(vac, probe, np.array([2.0, 3.0]), (0.0, 0.0), GEOM)
    ref = oracle.propagate(probe, oracle.propagator(16, Geometry(2 * GEOM.dz, GEOM.lam, GEOM.dx), (0, 0)))
    np.testing.assert_allclose(f["psi"][2], ref, atol=1e-12)
    assert len(f["psi"]) == 3
    # a single slice has no propagation at all: exit wave = O * shifted probe
    obj1 = np.exp(1j * RNG.standard_normal((1, 24, 24)))
    f1 = oracle.forward_position(obj1, probe, np.array([2.0, 3.0]), (0.0, 0.0), Geometry(123.0, 0.0197, 0.1))
    np.testing.assert_allclose(f1["Psi"], oracle.dft2(obj1[:, 2:18, 3:19] * probe), atol=1e-12)


def test_slice_order_first_slice_first():
    """Eq. 3: O_1 acts first.  A slice that blocks everything, placed first vs last, differs."""
    probe = crandn(1, 8, 8)
    obj = np.exp(1j * RNG.standard_normal((2, 12, 12)))
    f = oracle.forward_position(obj, probe, np.array([1.0, 2.0]), (0.0, 0.0), GEOM)
    M = oracle.propagator(8, GEOM, (0, 0))
    expect = obj[1, 1:9, 2:10] * oracle.idft2(M * oracle.dft2(obj[0, 1:9, 2:10] * probe[0]))
    np.testing.assert_allclose(f["Psi"][0], oracle.dft2(expect), atol=1e-12)


# ------------------------------------------------------------------ F6/F7 mode sum, far field
def test_mode_sum_additivity_and_intensity_conservation():
    obj = (1 - 0.1 * RNG.random((3, 20, 20))) * np.exp(1j * RNG.standard_normal((3, 20, 20)))
    probe = crandn(3, 8, 8)
    p = np.array([5.3, 6.8])
    f = oracle.forward_position(obj, probe, p, (1e-3, 2e-3), GEOM)
    singles = sum(oracle.forward_position(obj, probe[m:m + 1], p, (1e-3, 2e-3), GEOM)["I"] for m in range(3))
    np.testing.assert_allclose(f["I"], singles, rtol=1e-12)
    phi_last = f["O"][-1][None] * f["psi"][-1]
    assert np.isclose(f["I"].sum(), np.sum(abs(phi_last) ** 2), rtol=1e-12)


def test_vacuum_pattern_is_probe_spectrum():
    """O = 1, zero tilt, any Nz: I_b = sum_m |P^(m)(k)|^2 for every position (|M| = |E| = 1)."""
    probe = crandn(2, 16, 16)
    vac = np.ones((4, 30, 30), dtype=complex)
    I = oracle.intensity_batch(vac, probe, np.array([[3.3, 4.4], [10.0, 2.5]]), None, GEOM)
    expect = np.sum(abs(oracle.dft2(probe)) ** 2, axis=0)
    np.testing.assert_allclose(I[0], expect, rtol=1e-11)
    np.testing.assert_allclose(I[1], expect, rtol=1e-11)


def test_vacuum_pattern_of_generated_probe_is_flat_disc():
    from paper_2505_07814_b200 import synth
    cfg = synth.get_config(1)
    probe = synth.make_probe(cfg)
    vac = np.ones((1, cfg.H, cfg.W), dtype=complex)
    I = oracle.intensity_batch(vac, probe, np.array([[10.2, 20.7]]), None, GEOM)[0]
    kp = np.fft.fftfreq(cfg.N)
    disc = (kp[:, None] ** 2 + kp[None, :] ** 2) <= 0.125 ** 2
    assert np.isclose(I.sum(), cfg.dose, rtol=1e-5)
    np.testing.assert_allclose(I[disc], cfg.dose / disc.sum(), rtol=1e-4)
    assert I[~disc].max() < 1e-6 * I[disc].mean()


# ------------------------------------------------------------------ F8 loss
def test_loss_zero_at_truth_and_limits():
    obj = np.exp(1j * RNG.standard_normal((2, 20, 20)))
    probe = crandn(2, 8, 8)
    pos = np.array([[3.2, 4.7], [6.6, 9.1], [1.0, 2.0]])
    _, _, I = oracle.forward_loss_batch(obj, probe, pos, None, np.zeros((3, 8, 8)), GEOM)
    L0, lb0, _ = oracle.forward_loss_batch(obj, probe, pos, None, np.zeros((3, 8, 8)), GEOM)
    assert np.isclose(L0, I.sum(), rtol=1e-13)                 # a -> 0 => L = sum I
    Lt, lbt, _ = oracle.forward_loss_batch(obj, probe, pos, None, np.sqrt(I), GEOM)
    assert Lt < 1e-20 and lbt.shape == (3,)
    g = oracle.grad_batch(obj, probe, pos, None, np.sqrt(I), GEOM)
    assert g["loss"] < 1e-20
    for k in ("g_object", "g_probe", "g_positions", "g_tilt"):
        assert np.max(abs(g[k])) < 1e-8
    assert np.isclose(oracle.loss_from_intensity(np.array([4.0, 9.0]), np.array([1.0, 5.0])), 1.0 + 4.0)


def test_loss_gaussian_eq5_from_plain_sum():
    """Eq. 5 (p = 0.5): sqrt(<(sqrt(I)-a)^2>) / <a> rebuilt from S (R13)."""
    I = RNG.random((3, 8, 8)) * 5
    a = RNG.random((3, 8, 8)) * 2
    S = sum(oracle.loss_from_intensity(I[b], a[b]) for b in range(3))
    direct = math.sqrt(np.mean((np.sqrt(I) - a) ** 2)) / np.mean(a)
    assert np.isclose(oracle.loss_gaussian_eq5(S, I.size, a.mean()), direct, rtol=1e-13)


# ------------------------------------------------------------------ Adam (B9, R20)
def test_adam_first_step_is_lr_sign_g():
    theta = crandn(4, 5)
    g = crandn(4, 5)
    th1, m1, v1 = oracle.adam_step(theta, g, np.zeros((4, 10)), np.zeros((4, 10)), 1, lr=1e-3)
    gr = g.view(np.float64)
    np.testing.assert_allclose(th1.view(np.float64), theta.view(np.float64) - 1e-3 * np.sign(gr), atol=1e-9)
    np.testing.assert_allclose(m1, 0.1 * gr, rtol=1e-13)
    np.testing.assert_allclose(v1, 0.001 * gr * gr, rtol=1e-13)


def test_adam_matches_torch_optim_over_several_steps():
    torch = pytest.importorskip("torch")
    x0 = RNG.standard_normal(7)
    p = torch.tensor(x0.copy(), dtype=torch.float64, requires_grad=True)
    opt = torch.optim.Adam([p], lr=5e-4, betas=(0.9, 0.999), eps=1e-8)
    th, m, v = x0.copy(), np.zeros(7), np.zeros(7)
    for t in range(1, 6):
        g = RNG.standard_normal(7) * 10.0 ** RNG.integers(-3, 3)
        p.grad = torch.tensor(g.copy())
        opt.step()
        th, m, v = oracle.adam_step(th, g, m, v, t, lr=5e-4)
        np.testing.assert_allclose(th, p.detach().numpy(), rtol=1e-12, atol=1e-14)
