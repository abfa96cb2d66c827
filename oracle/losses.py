"""Plain float64 CPU oracle for the paper's loss family (Eq. 5-9), the amplitude / phase object
parameterisation and mixed object states -- SURVEY.md §8(f) NEXT-2 / NEXT-4.

TEST INFRASTRUCTURE ONLY (see ``oracle/__init__.py``): the product never imports this.

Notation: ``I`` = I_model [B,N,N], ``a`` = sqrt(I_meas) [B,N,N] (the ABI's ``meas_amp``),
``<.>_{D,B}`` = mean over the detector pixels and the minibatch, ``<.>_B`` = mean over the minibatch.

  Eq. 5  L_Gaussian = sqrt(<(I^p - I_meas^p)^2>_{D,B}) / <I_meas^p>_{D,B},         p = 1/2
  Eq. 6  L_Poisson  = -<I_meas^p log(I^p + eps) - I^p>_{D,B} / <I_meas^p>_{D,B},   p = 1, eps = 1e-6
  Eq. 7  L_PACBED   = sqrt(<(<I>_B^p - <I_meas>_B^p)^2>_D) / <I_meas^p>_{D,B},     p = 1/2
  Eq. 8  L_sparse   = <|O_p|^p>_{R,B}^{1/p}, O_p = phase of the object patches,     p = 1
  Eq. 9  L_total    = w1 L_Gaussian + w2 L_Poisson + w3 L_PACBED + w4 L_sparse

Readings (R27-R31): the powers are the paper's defaults (Gaussian 1/2, Poisson 1, sparse 1) and the
PACBED term uses the Gaussian's p = 1/2 (the paper gives it no default of its own); Eq. 8 averages |phase| over
the cropped object patches O_b[s] of the minibatch (spatial dimension R = the N x N window and the Nz slices,
B = the batch), so a pixel under c patches counts c times; where I = 0 the derivative of I^(1/2) is taken as 0
(R14) -- the Poisson term needs no such rule thanks to eps.

The object is stored as two real arrays, amplitude A and phase phi, O = A exp(i phi); with
g_O = dL/dRe O + i dL/dIm O:  g_A = Re(conj(g_O) exp(i phi)),  g_phi = Im(g_O conj(O)).

Mixed object states (Eq. 2): object [N_o, Nz, H, W]; I_b = sum_m sum_n |F[psi^(m)(n)]|^2.
"""
from __future__ import annotations

from dataclasses import dataclass

import numpy as np

from . import multislice as ms

__all__ = ["LossWeights", "data_terms", "sparse_term", "object_from_amp_phase", "amp_phase_gradients",
           "intensity_batch_states", "total_loss_and_gradients"]


@dataclass(frozen=True)
class LossWeights:
    """Eq. 9 weights w1..w4 and the Poisson epsilon."""
    gaussian: float = 1.0
    poisson: float = 0.0
    pacbed: float = 0.0
    sparse: float = 0.0
    eps: float = 1e-6


def data_terms(I, a, w: LossWeights):
    """Eq. 5-7 on one minibatch.  Returns (dict of the three term values, dL_data/dI [B,N,N]) where
    L_data = w1 L_Gaussian + w2 L_Poisson + w3 L_PACBED."""
    I = np.asarray(I, dtype=np.float64)
    a = np.asarray(a, dtype=np.float64)
    B = I.shape[0]
    n = I.size                                     # |D| |B|
    nD = I[0].size
    I_meas = a * a
    dLdI = np.zeros_like(I)
    # Eq. 5, p = 1/2:  I^p = sqrt(I), I_meas^p = a
    sqrtI = np.sqrt(I)
    mean_a = a.mean()
    mse = np.mean((sqrtI - a) ** 2)
    L_G = np.sqrt(mse) / mean_a
    if w.gaussian != 0.0 and mse > 0.0:
        d_sqrt = np.zeros_like(I)                  # d sqrt(I) / dI = 1 / (2 sqrt(I)), 0 where I = 0 (R14)
        nz = I > 0
        d_sqrt[nz] = 0.5 / sqrtI[nz]
        dLdI += w.gaussian * (1.0 / (2.0 * np.sqrt(mse) * mean_a)) * (2.0 * (sqrtI - a) / n) * d_sqrt
    # Eq. 6, p = 1
    mean_Im = I_meas.mean()
    L_P = -np.mean(I_meas * np.log(I + w.eps) - I) / mean_Im
    if w.poisson != 0.0:
        dLdI += w.poisson * (-(I_meas / (I + w.eps) - 1.0) / n) / mean_Im
    # Eq. 7, p = 1/2 (reading R28): position-averaged patterns
    Ibar, Imbar = I.mean(axis=0), I_meas.mean(axis=0)
    diff = np.sqrt(Ibar) - np.sqrt(Imbar)
    mse_pb = np.mean(diff ** 2)
    L_PB = np.sqrt(mse_pb) / mean_a
    if w.pacbed != 0.0 and mse_pb > 0.0:
        d_sqrt = np.zeros_like(Ibar)
        nz = Ibar > 0
        d_sqrt[nz] = 0.5 / np.sqrt(Ibar[nz])
        dL_dIbar = (1.0 / (2.0 * np.sqrt(mse_pb) * mean_a)) * (2.0 * diff / nD) * d_sqrt
        dLdI += w.pacbed * dL_dIbar[None] / B      # d<I>_B / dI_b = 1 / B
    return {"gaussian": float(L_G), "poisson": float(L_P), "pacbed": float(L_PB)}, dLdI


def sparse_term(phase, positions, N):
    """Eq. 8 with p = 1 (reading R27): mean |phase| over the cropped patches of the minibatch.
    ``phase`` [..., Nz, H, W] (any leading object-state axis).  Returns (L_sparse, dL_sparse/dphase)."""
    phase = np.asarray(phase, dtype=np.float64)
    positions = np.asarray(positions, dtype=np.float64)
    B = len(positions)
    total = 0.0
    g = np.zeros_like(phase)
    n_patch = B * int(np.prod(phase.shape[:-2])) * N * N
    for b in range(B):
        r, _ = ms.split_position(positions[b])
        patch = ms.crop(phase, r, N)
        total += np.sum(np.abs(patch))
        ms.crop_adjoint_add(g, r, np.sign(patch) / n_patch)
    return float(total / n_patch), g


def object_from_amp_phase(amp, phase):
    """O = A exp(i phi)."""
    return np.asarray(amp, dtype=np.float64) * np.exp(1j * np.asarray(phase, dtype=np.float64))


def amp_phase_gradients(g_obj, amp, phase):
    """Chain rule of O = A exp(i phi): g_A = Re(conj(g_O) e^{i phi}), g_phi = Im(g_O conj(O))."""
    e = np.exp(1j * np.asarray(phase, dtype=np.float64))
    O = np.asarray(amp, dtype=np.float64) * e
    return np.real(np.conj(g_obj) * e), np.imag(g_obj * np.conj(O))


def _states(obj):
    obj = np.asarray(obj, dtype=np.complex128)
    return obj if obj.ndim == 4 else obj[None]


def intensity_batch_states(obj, probe, positions, tilt, geom):
    """Eq. 2 with object states: I_b = sum_n sum_m |F[psi^(m)(n)]|^2; obj [N_o,Nz,H,W] or [Nz,H,W]."""
    return sum(ms.intensity_batch(o, probe, positions, tilt, geom) for o in _states(obj))


def total_loss_and_gradients(obj, probe, positions, tilt, meas_amp, geom, w: LossWeights, amp=None, phase=None):
    """Eq. 9 and all its gradients for one minibatch.

    Either ``obj`` (complex [Nz,H,W] or [N_o,Nz,H,W]) or the pair ``amp``, ``phase`` (same shapes, real) gives
    the object; the sparsity term needs the phase array (with a complex object it uses ``angle(obj)`` for the
    VALUE only and contributes no gradient).  Returns dict(loss, terms, g_object, g_probe, g_positions [B,2],
    g_tilt [B,2], g_dz, and g_amp, g_phase when amp / phase were given).
    """
    if amp is not None:
        obj = object_from_amp_phase(amp, phase)
    objs = _states(obj)
    probe = np.asarray(probe, dtype=np.complex128)
    positions = np.asarray(positions, dtype=np.float64)
    B = len(positions)
    tilts = ms._tilt_per_position(tilt, B)
    N = probe.shape[-1]
    # pass 1: model intensities (the normalisations of Eq. 5-7 couple the whole minibatch)
    fwd = [[ms.forward_position(o, probe, positions[b], tilts[b], geom) for o in objs] for b in range(B)]
    I = np.stack([sum(f["I"] for f in fb) for fb in fwd])
    terms, dLdI = data_terms(I, meas_amp, w)
    # pass 2: the adjoint B2-B8 seeded with dL/dI, per position and object state
    g_obj = np.zeros(objs.shape, dtype=np.complex128)
    g_probe = np.zeros(probe.shape, dtype=np.complex128)
    g_pos, g_tilt, g_dz = np.zeros((B, 2)), np.zeros((B, 2)), 0.0
    for b in range(B):
        for n, f in enumerate(fwd[b]):
            gp, gt, gz = ms.backprop_position(f, probe, dLdI[b], tilts[b], geom, g_obj[n], g_probe)
            g_pos[b] += gp
            g_tilt[b] += gt
            g_dz += gz
    ph = np.asarray(phase, dtype=np.float64) if phase is not None else np.angle(np.asarray(obj))
    L_s, g_s = sparse_term(ph, positions, N)
    terms["sparse"] = L_s
    loss = (w.gaussian * terms["gaussian"] + w.poisson * terms["poisson"] + w.pacbed * terms["pacbed"]
            + w.sparse * L_s)
    out = {"loss": float(loss), "terms": terms, "intensity": I,
           "g_object": g_obj if np.asarray(obj).ndim == 4 else g_obj[0],
           "g_probe": g_probe, "g_positions": g_pos, "g_tilt": g_tilt, "g_dz": g_dz}
    if amp is not None:
        g_a, g_p = amp_phase_gradients(out["g_object"], amp, phase)
        out["g_amp"], out["g_phase"] = g_a, g_p + w.sparse * g_s
    return out
