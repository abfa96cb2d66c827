"""Seeded synthetic 4D-STEM-shaped inputs (stand-ins for the paper's datasets).

This module holds NONE of the method's arithmetic (no forward model, loss, adjoint or
optimiser): it only draws objects, probes, scan positions and Poisson counts.  It is the
one module both the CUDA path's callers and the oracle's callers import, so that both
sides see bit-identical float32/complex64 inputs.  Whoever needs measurements supplies
the noise-free intensity (the tests take it from ``oracle/``; ``bench.py`` takes it from
the library's own forward call) and gets ``sqrt(Poisson(I))`` back.

Recipe: SURVEY.md §8(d) / DESIGN.md "Input recipe"; shapes follow BASELINE.json
``configs`` which follow the paper's Tables S3/S4: 128^2 detector,
64^2-128^2 scans, 1-21 slices, 1-12 probe modes, 1e4-1e6 e-/pattern.
Random streams: ``seed = 1000*c + k`` with k = 0 truth object, 1 evaluation object,
2 scan jitter, 3 Poisson, 4 evaluation-position perturbation, 5 minibatch permutation.
"""
from __future__ import annotations

from dataclasses import dataclass, replace

import numpy as np

__all__ = ["Config", "CONFIGS", "get_config", "make_object", "make_probe", "raster",
           "true_positions", "eval_point", "truth", "minibatch", "compact_minibatch",
           "poisson_amplitudes"]


@dataclass(frozen=True)
class Config:
    c: int            # config number 1..5 (BASELINE.json configs[c-1])
    N: int            # probe / detector window
    H: int            # object height = width
    Nz: int
    M: int
    B: int            # default minibatch
    ns: int           # scan is ns x ns
    step: int         # raster step, px
    jitter: float     # uniform +-J px true-position jitter
    dose: float       # electrons per pattern = sum |P|^2
    dz: float         # Angstrom
    lam: float = 0.0197   # Angstrom (300 kV), inherited from config 3 (R23)
    dx: float = 0.1       # Angstrom / px
    atoms: bool = False
    tilt_mode: int = 0    # 0 none, 1 global
    true_tilt: tuple = (0.0, 0.0)   # (theta_y, theta_x) rad
    eval_tilt: tuple = (0.0, 0.0)
    powers: tuple = ()

    @property
    def W(self):
        return self.H

    @property
    def n_positions(self):
        return self.ns * self.ns

    @property
    def origin(self):
        return (self.H - ((self.ns - 1) * self.step + self.N)) // 2


CONFIGS = {
    1: Config(c=1, N=64, H=160, Nz=1, M=1, B=32, ns=16, step=6, jitter=0.3, dose=1e4, dz=2.0),
    2: Config(c=2, N=128, H=576, Nz=1, M=6, B=256, ns=64, step=7, jitter=0.5, dose=1e5, dz=2.0,
              powers=(0.5, 0.2, 0.1, 0.1, 0.05, 0.05)),
    3: Config(c=3, N=128, H=576, Nz=8, M=4, B=512, ns=64, step=7, jitter=0.5, dose=1e5, dz=2.0,
              atoms=True),
    4: Config(c=4, N=128, H=1088, Nz=6, M=12, B=1024, ns=128, step=7, jitter=0.5, dose=1e5,
              dz=5.0, atoms=True),
    # (theta_x, theta_y) = (0.5, -0.3) mrad true, (0.3, -0.1) mrad at evaluation point A (R11)
    5: Config(c=5, N=256, H=1280, Nz=20, M=8, B=128, ns=96, step=10, jitter=1.0, dose=1e6,
              dz=1.0, atoms=True, tilt_mode=1, true_tilt=(-0.3e-3, 0.5e-3),
              eval_tilt=(-0.1e-3, 0.3e-3)),
}


def get_config(c, **overrides):
    return replace(CONFIGS[int(c)], **overrides)


def _blur_periodic(img, sigma):
    """Periodic Gaussian blur (unit DC gain) of the last two axes, via the convolution theorem."""
    h, w = img.shape[-2:]
    fy = np.fft.fftfreq(h)[:, None]
    fx = np.fft.fftfreq(w)[None, :]
    g = np.exp(-2.0 * np.pi ** 2 * sigma ** 2 * (fx * fx + fy * fy))
    return np.real(np.fft.ifft2(np.fft.fft2(img) * g))


def make_object(cfg, stream, phase_scale=1.0):
    """[Nz,H,W] complex64 transmission t = A exp(i phi) (BASELINE.json configs)."""
    rng = np.random.default_rng(1000 * cfg.c + stream)
    out = np.empty((cfg.Nz, cfg.H, cfg.W), dtype=np.complex64)
    for s in range(cfg.Nz):
        phi = _blur_periodic(rng.standard_normal((cfg.H, cfg.W)), 2.0)
        phi *= 0.5 / np.max(np.abs(phi))
        if cfg.atoms:
            n_atoms = int(round(0.02 * cfg.H * cfg.W))
            pts = np.zeros((cfg.H, cfg.W))
            iy = rng.integers(0, cfg.H, n_atoms)
            ix = rng.integers(0, cfg.W, n_atoms)
            np.add.at(pts, (iy, ix), 1.0)
            # a unit impulse blurred with sigma has peak 1/(2 pi sigma^2): rescale to 0.3 rad
            phi += 0.3 * (2.0 * np.pi * 1.5 ** 2) * _blur_periodic(pts, 1.5)
        phi *= phase_scale
        amp = 1.0 - 0.05 * np.abs(phi)
        out[s] = (amp * np.exp(1j * phi)).astype(np.complex64)
    return out


_HG_ORDERS = [(1, 0), (0, 1), (1, 1), (2, 0), (0, 2), (2, 1), (1, 2), (2, 2), (3, 0), (0, 3), (3, 1)]


def _hermite(n, x):
    return [np.ones_like(x), 2 * x, 4 * x * x - 2, 8 * x ** 3 - 12 * x][n]


def make_probe(cfg, defocus_coeff=0.3):
    """[M,N,N] complex64 orthogonal probe modes, sum |P|^2 = dose, centred at (N/2, N/2)."""
    N, M = cfg.N, cfg.M
    kp = np.fft.fftfreq(N)
    k2 = kp[:, None] ** 2 + kp[None, :] ** 2
    aperture = (k2 <= 0.125 ** 2).astype(np.float64)
    p0 = np.fft.fftshift(np.fft.ifft2(aperture * np.exp(1j * np.pi * defocus_coeff * k2 / 0.25)))
    yy = (np.arange(N) - N // 2)[:, None] / 6.0
    xx = (np.arange(N) - N // 2)[None, :] / 6.0
    env = np.exp(-0.5 * (xx * xx + yy * yy))
    modes = [p0]
    for a, b in _HG_ORDERS[:M - 1]:
        modes.append(p0 * _hermite(a, yy) * _hermite(b, xx) * env)
    ortho = []
    for v in modes:                                   # Gram-Schmidt, in order
        for u in ortho:
            v = v - u * np.vdot(u, v)
        ortho.append(v / np.sqrt(np.vdot(v, v).real))
    if cfg.powers:
        pw = np.array(cfg.powers[:M], dtype=np.float64)
    else:
        pw = 0.6 ** np.arange(M)
    pw = pw / pw.sum() * cfg.dose
    return np.stack([u * np.sqrt(q) for u, q in zip(ortho, pw)]).astype(np.complex64)


def raster(cfg):
    """[ns*ns, 2] float64 integer raster corners (p_y, p_x), row-major scan order."""
    g = cfg.origin + cfg.step * np.arange(cfg.ns, dtype=np.float64)
    yy, xx = np.meshgrid(g, g, indexing="ij")
    return np.stack([yy.ravel(), xx.ravel()], axis=1)


def true_positions(cfg):
    rng = np.random.default_rng(1000 * cfg.c + 2)
    return (raster(cfg) + rng.uniform(-cfg.jitter, cfg.jitter, (cfg.n_positions, 2))).astype(np.float32)


def truth(cfg):
    """Ground truth: dict(object, probe, positions, tilt) as float32/complex64."""
    return {"object": make_object(cfg, 0), "probe": make_probe(cfg, 0.3),
            "positions": true_positions(cfg), "tilt": np.array(cfg.true_tilt, dtype=np.float32)}


def eval_point(cfg, which="A"):
    """Evaluation point A (perturbed: parity + timing), B (the paper's default start,
    PAPER.md:102-104: unit amplitude, phase U[0,1e-8], un-jittered raster; parity only) or
    Bp (B with phase U[0,1e-2]: a near-vacuum start whose dark field is above float32 noise)."""
    if which == "A":
        rng = np.random.default_rng(1000 * cfg.c + 4)
        pert = np.clip(rng.normal(0.0, 0.2, (cfg.n_positions, 2)), -0.6, 0.6)
        return {"object": make_object(cfg, 1, phase_scale=0.5), "probe": make_probe(cfg, 0.35),
                "positions": (true_positions(cfg).astype(np.float64) + pert).astype(np.float32),
                "tilt": np.array(cfg.eval_tilt, dtype=np.float32)}
    if which == "B":
        rng = np.random.default_rng(1000 * cfg.c + 1)
        phase = rng.uniform(0.0, 1e-8, (cfg.Nz, cfg.H, cfg.W))
        return {"object": np.exp(1j * phase).astype(np.complex64), "probe": make_probe(cfg, 0.3),
                "positions": raster(cfg).astype(np.float32),
                "tilt": np.zeros(2, dtype=np.float32)}
    if which == "Bp":
        # B': the same start with the phase range raised to U[0, 1e-2] -- still "unit amplitude, small random
        # phase", but the dark field it scatters sits well above float32 rounding noise (R26)
        rng = np.random.default_rng(1000 * cfg.c + 1)
        phase = rng.uniform(0.0, 1e-2, (cfg.Nz, cfg.H, cfg.W))
        return {"object": np.exp(1j * phase).astype(np.complex64), "probe": make_probe(cfg, 0.3),
                "positions": raster(cfg).astype(np.float32),
                "tilt": np.zeros(2, dtype=np.float32)}
    raise ValueError(which)


def minibatch(cfg, j=0, B=None):
    """Indices of minibatch j of the seeded random permutation (reading R18)."""
    B = cfg.B if B is None else B
    perm = np.random.default_rng(1000 * cfg.c + 5).permutation(cfg.n_positions)
    nb = max(1, cfg.n_positions // B)
    j = j % nb
    return perm[j * B:(j + 1) * B]


def compact_minibatch(cfg, j=0, B=None):
    """B consecutive raster positions: the atomic-contention worst case (R18)."""
    B = cfg.B if B is None else B
    nb = max(1, cfg.n_positions // B)
    j = j % nb
    return np.arange(j * B, (j + 1) * B)


def poisson_amplitudes(cfg, intensity, indices):
    """sqrt(Poisson(I)) as float32, DC at [0,0].  One independent stream per position
    (seeded by the position's index in the scan), so any subset reproduces the same counts."""
    intensity = np.asarray(intensity, dtype=np.float64)
    out = np.empty(intensity.shape, dtype=np.float32)
    for i, idx in enumerate(np.asarray(indices).ravel()):
        rng = np.random.default_rng([1000 * cfg.c + 3, int(idx)])
        out[i] = np.sqrt(rng.poisson(np.maximum(intensity[i], 0.0)))
    return out
