"""Pins for the oracle's hand-derived adjoint: operator-wise
dot-product tests, central finite differences of the loss on tiny inputs (every component
of every gradient), and torch.autograd in float64 as an independent third opinion
(the paper's own mechanism; test-only)."""
import math

import numpy as np
import pytest

import oracle
from oracle import Geometry

GEOM = Geometry(dz=2.0, lam=0.0197, dx=0.1)


def crandn(rng, *shape):
    return rng.standard_normal(shape) + 1j * rng.standard_normal(shape)


def rdot(a, b):
    """Real inner product <a, b> = Re sum conj(a) b (the pairing behind g = dL/dRe + i dL/dIm)."""
    return float(np.real(np.vdot(a, b)))


def tiny_problem(seed=3, N=8, H=14, Nz=3, M=2, B=3):
    rng = np.random.default_rng(seed)
    obj = (1 - 0.1 * rng.random((Nz, H, H))) * np.exp(1j * 0.5 * rng.standard_normal((Nz, H, H)))
    probe = crandn(rng, M, N, N)
    pos = rng.uniform(0.6, H - N - 0.6, (B, 2))
    pos = np.floor(pos) + rng.uniform(-0.4, 0.4, (B, 2))           # away from rounding ties
    tilt = rng.normal(0, 2e-3, (B, 2))
    a = np.sqrt(rng.poisson(3.0 * np.ones((B, N, N)))).astype(np.float64) + 0.1
    return obj, probe, pos, tilt, a


# ------------------------------------------------------------------ operator adjoints (B2-B6)
def test_adjoint_dot_products():
    rng = np.random.default_rng(11)
    N = 8
    x, y = crandn(rng, 2, N, N), crandn(rng, 2, N, N)
    delta = np.array([0.31, -0.27])
    assert np.isclose(rdot(oracle.shift_probe(x, delta), y), rdot(x, oracle.shift_probe_adjoint(y, delta)))
    Mk = oracle.propagator(N, GEOM, (1e-3, -2e-3))
    assert np.isclose(rdot(oracle.propagate(x, Mk), y), rdot(x, oracle.propagate_adjoint(y, Mk)))
    assert np.isclose(rdot(oracle.dft2(x), y), rdot(x, oracle.idft2(y)))
    obj = crandn(rng, 3, 12, 13)
    patch = crandn(rng, 3, N, N)
    back = np.zeros_like(obj)
    oracle.crop_adjoint_add(back, (2, 4), patch)
    assert np.isclose(rdot(oracle.crop(obj, (2, 4), N), patch), rdot(obj, back))
    # scatter ADDS (overlapping patches accumulate)
    oracle.crop_adjoint_add(back, (3, 4), patch)
    assert np.isclose(back[0, 3, 4], patch[0, 1, 0] + patch[0, 0, 0])


# ------------------------------------------------------------------ central finite differences
def _loss(obj, probe, pos, tilt, a, geom=GEOM):
    return oracle.forward_loss_batch(obj, probe, pos, tilt, a, geom)[0]


def test_finite_differences_every_component():
    obj, probe, pos, tilt, a = tiny_problem()
    g = oracle.grad_batch(obj, probe, pos, tilt, a, GEOM)
    h = 1e-6
    assert np.isclose(g["loss"], _loss(obj, probe, pos, tilt, a), rtol=1e-13)

    def fd_complex(arr, setter):
        out = np.zeros(arr.shape, dtype=np.complex128)
        it = np.nditer(arr, flags=["multi_index"])
        for _ in it:
            i = it.multi_index
            for unit, part in ((1.0, "re"), (1j, "im")):
                ap, am = arr.copy(), arr.copy()
                ap[i] += h * unit
                am[i] -= h * unit
                d = (setter(ap) - setter(am)) / (2 * h)
                out[i] += d if part == "re" else 1j * d
        return out

    fd_probe = fd_complex(probe, lambda p: _loss(obj, p, pos, tilt, a))
    np.testing.assert_allclose(g["g_probe"], fd_probe, rtol=2e-6, atol=2e-6 * abs(fd_probe).max())
    fd_obj = fd_complex(obj, lambda o: _loss(o, probe, pos, tilt, a))
    np.testing.assert_allclose(g["g_object"], fd_obj, rtol=2e-6, atol=2e-6 * abs(fd_obj).max())
    assert abs(fd_obj).max() > 1e-2           # the test is not vacuous

    for b in range(len(pos)):
        for ax in range(2):
            pp, pm = pos.copy(), pos.copy()
            pp[b, ax] += h
            pm[b, ax] -= h
            fd = (_loss(obj, probe, pp, tilt, a) - _loss(obj, probe, pm, tilt, a)) / (2 * h)
            assert np.isclose(g["g_positions"][b, ax], fd, rtol=1e-6, atol=1e-6)
            ht = 1e-7
            tp, tm = tilt.copy(), tilt.copy()
            tp[b, ax] += ht
            tm[b, ax] -= ht
            fd = (_loss(obj, probe, pos, tp, a) - _loss(obj, probe, pos, tm, a)) / (2 * ht)
            assert np.isclose(g["g_tilt"][b, ax], fd, rtol=1e-5, atol=1e-4)
    hz = 1e-6
    fd = (_loss(obj, probe, pos, tilt, a, Geometry(GEOM.dz + hz, GEOM.lam, GEOM.dx))
          - _loss(obj, probe, pos, tilt, a, Geometry(GEOM.dz - hz, GEOM.lam, GEOM.dx))) / (2 * hz)
    assert np.isclose(g["g_dz"], fd, rtol=1e-6, atol=1e-6)


def test_global_tilt_gradient_is_sum_over_positions():
    obj, probe, pos, _, a = tiny_problem(seed=5)
    t = np.array([1.5e-3, -0.7e-3])
    g = oracle.grad_batch(obj, probe, pos, t, a, GEOM)
    ht = 1e-7
    for ax in range(2):
        tp, tm = t.copy(), t.copy()
        tp[ax] += ht
        tm[ax] -= ht
        fd = (_loss(obj, probe, pos, tp, a) - _loss(obj, probe, pos, tm, a)) / (2 * ht)
        assert np.isclose(g["g_tilt"][:, ax].sum(), fd, rtol=1e-5, atol=1e-4)


def test_directional_derivative_larger_problem():
    """<g, delta> vs central difference for random directions, N = 32, Nz = 4, M = 3."""
    rng = np.random.default_rng(21)
    obj, probe, pos, tilt, a = tiny_problem(seed=9, N=32, H=48, Nz=4, M=3, B=4)
    g = oracle.grad_batch(obj, probe, pos, tilt, a, GEOM)
    h = 1e-6
    for _ in range(2):
        do, dp = crandn(rng, *obj.shape), crandn(rng, *probe.shape)
        fd = (_loss(obj + h * do, probe, pos, tilt, a) - _loss(obj - h * do, probe, pos, tilt, a)) / (2 * h)
        assert np.isclose(rdot(g["g_object"], do), fd, rtol=1e-6)
        fd = (_loss(obj, probe + h * dp, pos, tilt, a) - _loss(obj, probe - h * dp, pos, tilt, a)) / (2 * h)
        assert np.isclose(rdot(g["g_probe"], dp), fd, rtol=1e-6)


# ------------------------------------------------------------------ torch.autograd third opinion
def test_against_torch_autograd_float64():
    torch = pytest.importorskip("torch")
    obj, probe, pos, tilt, a = tiny_problem(seed=13, N=16, H=26, Nz=3, M=2, B=3)
    N = probe.shape[-1]
    Nz = obj.shape[0]
    to = torch.tensor(obj, dtype=torch.complex128, requires_grad=True)
    tp = torch.tensor(probe, dtype=torch.complex128, requires_grad=True)
    r = np.floor(pos + 0.5).astype(int)
    td = torch.tensor(pos - r, dtype=torch.float64, requires_grad=True)
    tt = torch.tensor(tilt, dtype=torch.float64, requires_grad=True)
    tdz = torch.tensor(GEOM.dz, dtype=torch.float64, requires_grad=True)
    kp = torch.fft.fftfreq(N, dtype=torch.float64)
    k = kp / GEOM.dx
    loss = 0.0
    for b in range(len(pos)):
        E = torch.exp(-2j * math.pi * (kp[:, None] * td[b, 0] + kp[None, :] * td[b, 1]))
        psi = torch.fft.ifft2(E * torch.fft.fft2(tp, norm="ortho"), norm="ortho")
        chi = (-math.pi * GEOM.lam * (k[None, :] ** 2 + k[:, None] ** 2) * tdz
               + 2 * math.pi * tdz * (k[None, :] * torch.tan(tt[b, 1]) + k[:, None] * torch.tan(tt[b, 0])))
        Mk = torch.exp(1j * chi)
        for s in range(Nz):
            phi = to[s, r[b, 0]:r[b, 0] + N, r[b, 1]:r[b, 1] + N] * psi
            if s < Nz - 1:
                psi = torch.fft.ifft2(Mk * torch.fft.fft2(phi, norm="ortho"), norm="ortho")
        I = (torch.fft.fft2(phi, norm="ortho").abs() ** 2).sum(0)
        loss = loss + ((torch.sqrt(I) - torch.tensor(a[b])) ** 2).sum()
    loss.backward()
    g = oracle.grad_batch(obj, probe, pos, tilt, a, GEOM)
    assert np.isclose(g["loss"], loss.item(), rtol=1e-13)
    np.testing.assert_allclose(g["g_object"], to.grad.numpy(), rtol=1e-9, atol=1e-9)
    np.testing.assert_allclose(g["g_probe"], tp.grad.numpy(), rtol=1e-9, atol=1e-9)
    np.testing.assert_allclose(g["g_positions"], td.grad.numpy(), rtol=1e-9, atol=1e-9)
    np.testing.assert_allclose(g["g_tilt"], tt.grad.numpy(), rtol=1e-9, atol=1e-7)
    assert np.isclose(g["g_dz"], tdz.grad.item(), rtol=1e-9)


# ------------------------------------------------------------------ batch plumbing
def test_grad_batch_workers_and_float32_inputs():
    obj, probe, pos, tilt, a = tiny_problem(seed=17, N=16, H=40, Nz=2, M=2, B=7)
    obj32, probe32 = obj.astype(np.complex64), probe.astype(np.complex64)
    pos32, a32 = pos.astype(np.float32), a.astype(np.float32)
    g1 = oracle.grad_batch(obj32, probe32, pos32, tilt[0], a32, GEOM, workers=1)
    g3 = oracle.grad_batch(obj32, probe32, pos32, tilt[0], a32, GEOM, workers=3)
    for k in ("g_object", "g_probe", "g_positions", "g_tilt", "loss_per_pos"):
        np.testing.assert_allclose(g3[k], g1[k], rtol=1e-11, atol=1e-11)
    assert np.isclose(g3["g_dz"], g1["g_dz"], rtol=1e-11)
    L, lb, I = oracle.forward_loss_batch(obj32, probe32, pos32, tilt[0], a32, GEOM)
    assert np.isclose(L, g1["loss"], rtol=1e-13)
    np.testing.assert_allclose(lb, g1["loss_per_pos"], rtol=1e-13)
    # positions outside any patch get exactly zero object gradient
    cover = np.zeros(obj.shape[1:], bool)
    for p in np.floor(pos32 + 0.5).astype(int):
        cover[p[0]:p[0] + 16, p[1]:p[1] + 16] = True
    assert np.all(g1["g_object"][:, ~cover] == 0)


def test_zero_intensity_pixels_have_zero_weight():
    """R14: w = 0 where I = 0 (no epsilon); a dark probe gives zero gradient, loss = sum a^2."""
    obj, probe, pos, tilt, a = tiny_problem(seed=19)
    g = oracle.grad_batch(obj, 0 * probe, pos, tilt, a, GEOM)
    assert np.isclose(g["loss"], np.sum(a ** 2))
    assert np.all(g["g_object"] == 0) and np.all(np.isfinite(g["g_probe"]))
