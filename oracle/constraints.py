"""Plain float64 CPU oracle for the per-iteration physical constraints of the paper's timed runs
(PAPER.md:145-147, :289, :301-312 Eq. 13, :539) -- SURVEY.md §8(f) NEXT-3.

TEST INFRASTRUCTURE ONLY (see ``oracle/__init__.py``): the product never imports this.

  * probe-mode orthogonalisation (Thibault & Menzel 2013): the modes are replaced by the
    eigen-decomposition of the mixed state they span.  With the Gram matrix G_ij = <P_i|P_j> = sum_r conj(P_i) P_j
    (Hermitian, positive semi-definite) and its unit eigenvectors G v_k = lambda_k v_k, the new modes are
    P'_k = sum_j (v_k)_j P_j: mutually orthogonal, <P'_k|P'_k> = lambda_k, same density operator
    sum_k |P'_k><P'_k|, ordered by decreasing power lambda_k.  A mode is defined up to a unit phase factor
    (and up to a rotation inside a degenerate eigenspace); lambda_k and the density operator are unique.
  * r_z filter, Eq. 13: O'(r) = O(r) * G_sigma_z(r_z), a 1-D Gaussian blur along depth.
    Reading R31 (the paper gives neither the truncation nor the edge rule; "without intermixing the top and
    bottom slices" rules out a periodic one): taps g_j = exp(-j^2 / (2 sigma_z^2)) for |j| <= R = max(1,
    ceil(2 sigma_z)), normalised to sum 1, slices beyond the ends replaced by the end slice ("replicate"), so a
    depth-constant object is unchanged.  The kernel is real: applied to a complex array it blurs real and
    imaginary parts (Eq. 13 as printed); PtyRAD stores amplitude and phase and blurs each array.
  * positivity: negative object-phase values are clipped to 0 after the iteration.
  * amplitude threshold: the object amplitude is clamped to [0.98, 1.02].
"""
from __future__ import annotations

import math

import numpy as np

__all__ = ["orthogonalize_modes", "rz_taps", "rz_filter", "clip_phase_positive", "clamp_amplitude"]


def orthogonalize_modes(probe):
    """probe [M,N,N] complex -> (orthogonal modes [M,N,N] sorted by decreasing power, powers lambda [M])."""
    P = np.asarray(probe, dtype=np.complex128)
    M = P.shape[0]
    flat = P.reshape(M, -1)
    G = np.conj(flat) @ flat.T                      # G_ij = sum_r conj(P_i) P_j
    lam, V = np.linalg.eigh(G)                      # ascending; columns are the eigenvectors v_k
    order = np.argsort(lam)[::-1]
    lam, V = lam[order], V[:, order]
    new = (V.T @ flat).reshape(P.shape)             # P'_k = sum_j (v_k)_j P_j
    return new, np.maximum(lam, 0.0)


def rz_taps(sigma_z):
    """Normalised Gaussian taps g_j, j = -R..R, R = max(1, ceil(2 sigma_z)) (reading R31)."""
    R = max(1, int(math.ceil(2.0 * sigma_z)))
    j = np.arange(-R, R + 1, dtype=np.float64)
    g = np.exp(-j * j / (2.0 * sigma_z * sigma_z))
    return g / g.sum()


def rz_filter(x, sigma_z):
    """Eq. 13: blur along the depth axis (axis -3 of [..., Nz, H, W]) with replicated end slices."""
    x = np.asarray(x)
    x = x.astype(np.complex128 if np.iscomplexobj(x) else np.float64)
    g = rz_taps(sigma_z)
    R = (len(g) - 1) // 2
    Nz = x.shape[-3]
    out = np.zeros_like(x)
    for z in range(Nz):
        for j in range(-R, R + 1):
            zz = min(max(z + j, 0), Nz - 1)
            out[..., z, :, :] += g[j + R] * x[..., zz, :, :]
    return out


def clip_phase_positive(phase):
    """Positivity constraint on the object phase: max(phase, 0)."""
    return np.maximum(np.asarray(phase, dtype=np.float64), 0.0)


def clamp_amplitude(amp, lo=0.98, hi=1.02):
    """Amplitude threshold: clamp to [lo, hi]."""
    return np.clip(np.asarray(amp, dtype=np.float64), lo, hi)
