"""Plain float64 CPU oracle: mixed-state multislice forward model, amplitude loss,
hand-derived adjoint and Adam, step by step in the paper's order and notation.

TEST INFRASTRUCTURE ONLY (see ``oracle/__init__.py``): the product never imports this.

Citations are ``PAPER.md:<line>`` (= /root/reference/PAPER.md) and the SURVEY.md §8(c)
step names (F1..F8 forward, B1..B9 adjoint, R1..R25 readings of silent points; the
readings are listed again in DESIGN.md).

Conventions (readings R1, R2, R4, R5, R8, R15):
  * arrays are row-major ``(y, x)``; DC of every spectrum sits at index ``[0, 0]``;
  * ``F`` is the unitary 2-D DFT with kernel ``exp(-2 pi i k.r)`` (numpy ``norm="ortho"``);
  * ``positions[b] = (p_y, p_x)`` in pixels, top-left corner of the N x N crop;
  * ``tilt = (theta_y, theta_x)`` in radians, global ``[2]`` or per position ``[B, 2]``;
  * complex gradients are ``g = dL/dRe + i dL/dIm`` (what torch.autograd returns).

All inputs are upcast to float64/complex128 on entry, so the float32 arrays the GPU
receives are seen bit-identically here.  ``numpy.fft`` is the one library primitive used
as a step; it is pinned against a brute-force O(N^4) DFT in tests/test_oracle_pins.py.
"""
from __future__ import annotations

import math
from dataclasses import dataclass

import numpy as np

__all__ = [
    "Geometry", "dft2", "idft2", "split_position", "shift_kernel", "shift_probe",
    "shift_probe_adjoint", "crop", "crop_adjoint_add", "propagator_phase", "propagator",
    "propagate", "propagate_adjoint", "forward_position", "intensity_batch",
    "loss_from_intensity", "forward_loss_batch", "backprop_position", "grad_position", "grad_batch",
    "loss_gaussian_eq5", "adam_step",
]


@dataclass(frozen=True)
class Geometry:
    """Physical constants of the propagator, Angstrom (Eq. 4)."""
    dz: float
    lam: float
    dx: float


# --------------------------------------------------------------------------- DFT
def dft2(x):
    """Unitary 2-D DFT over the last two axes, kernel exp(-2 pi i k.r) (R1)."""
    return np.fft.fft2(x, norm="ortho")


def idft2(x):
    """Inverse of :func:`dft2` (kernel exp(+2 pi i k.r), unitary)."""
    return np.fft.ifft2(x, norm="ortho")


# --------------------------------------------------------------------------- F1
def split_position(p):
    """F1: r = floor(p + 0.5) (integer crop origin), Delta = p - r in [-0.5, 0.5).

    PAPER.md:81 ("rho_j - round(rho_j) = Delta r_j"); tie-break R6.
    """
    p = np.asarray(p, dtype=np.float64)
    r = np.floor(p + 0.5)
    return r.astype(np.int64), p - r


# --------------------------------------------------------------------------- F2
def shift_kernel(N, delta):
    """F2: E(k) = exp(-2 pi i (k_py Delta_y + k_px Delta_x)), k_p = fftfreq(N) (R2)."""
    kp = np.fft.fftfreq(N)
    return np.exp(-2j * np.pi * (kp[:, None] * delta[0] + kp[None, :] * delta[1]))


def shift_probe(probe, delta):
    """F2: S_Delta P = F^-1[E . F[P]], i.e. (S_Delta P)(r) = P(r - Delta) (R2)."""
    N = probe.shape[-1]
    return idft2(shift_kernel(N, delta) * dft2(probe))


def shift_probe_adjoint(g, delta):
    """Adjoint of :func:`shift_probe` (B6): F^-1[conj(E) . F[g]]."""
    N = g.shape[-1]
    return idft2(np.conj(shift_kernel(N, delta)) * dft2(g))


# --------------------------------------------------------------------------- F3
def crop(obj, r, N):
    """F3: O_b[s] = object[s, r_y:r_y+N, r_x:r_x+N].  Never wraps (R22)."""
    ry, rx = int(r[0]), int(r[1])
    H, W = obj.shape[-2:]
    if ry < 0 or rx < 0 or ry + N > H or rx + N > W:
        raise ValueError(f"patch at ({ry},{rx}) size {N} leaves the {H}x{W} object (R22)")
    return obj[..., ry:ry + N, rx:rx + N]


def crop_adjoint_add(g_obj, r, patch):
    """Adjoint of :func:`crop` (B3): scatter-add a patch gradient into the full object."""
    ry, rx = int(r[0]), int(r[1])
    N = patch.shape[-1]
    g_obj[..., ry:ry + N, rx:rx + N] += patch


# --------------------------------------------------------------------------- F4
def propagator_phase(N, geom, tilt):
    """F4: chi(k) = -pi lam |k|^2 dz + 2 pi dz (k_x tan th_x + k_y tan th_y), k = fftfreq(N, dx).

    PAPER.md:89, Eq. 4; k in cycles/Angstrom (R8); no band limit (R9).  tilt = (th_y, th_x).
    """
    k = np.fft.fftfreq(N, d=geom.dx)
    ky, kx = k[:, None], k[None, :]
    ty, tx = float(tilt[0]), float(tilt[1])
    return (-np.pi * geom.lam * (kx * kx + ky * ky) * geom.dz
            + 2.0 * np.pi * geom.dz * (kx * math.tan(tx) + ky * math.tan(ty)))


def propagator(N, geom, tilt):
    """F4: M_{theta,dz}(k) = exp(i chi(k)) (Eq. 4)."""
    return np.exp(1j * propagator_phase(N, geom, tilt))


def propagate(phi, Mk):
    """F5: psi = F^-1[M . F[phi]] (Eq. 3)."""
    return idft2(Mk * dft2(phi))


def propagate_adjoint(g, Mk):
    """Adjoint of :func:`propagate` (B5): F^-1[conj(M) . F[g]]."""
    return idft2(np.conj(Mk) * dft2(g))


# --------------------------------------------------------------------------- F1-F7
def forward_position(obj, probe, p, tilt, geom):
    """F1-F7 for one scan position: all M probe modes through the Nz slices.

    obj [Nz,H,W], probe [M,N,N] complex; p = (p_y, p_x); tilt = (th_y, th_x).
    Returns a dict with the integer origin ``r``, sub-pixel ``delta``, the waves incident
    on every slice ``psi[s]`` ([Nz][M,N,N]), the far field ``Psi`` [M,N,N] and the
    mode-summed intensity ``I`` [N,N] (Eq. 1-4).
    """
    obj = np.asarray(obj, dtype=np.complex128)
    probe = np.asarray(probe, dtype=np.complex128)
    Nz = obj.shape[0]
    N = probe.shape[-1]
    r, delta = split_position(p)                       # F1
    psi = shift_probe(probe, delta)                    # F2  psi_0^(m)
    O = crop(obj, r, N)                                # F3
    Mk = propagator(N, geom, tilt)                     # F4
    incident = []
    phi = None
    for s in range(Nz):                                # F5 (Eq. 3: Nz transmissions,
        incident.append(psi)                           #     Nz-1 propagations, R7)
        phi = O[s][None, :, :] * psi
        if s < Nz - 1:
            psi = propagate(phi, Mk)
    Psi = dft2(phi)                                    # F6
    I = np.sum(Psi.real ** 2 + Psi.imag ** 2, axis=0)  # F7 (Eq. 2)
    return {"r": r, "delta": delta, "O": O, "M": Mk, "psi": incident, "Psi": Psi, "I": I}


def intensity_batch(obj, probe, positions, tilt, geom):
    """I_b(k) for every position of a batch -> [B,N,N] float64 (Eq. 1-2)."""
    positions = np.asarray(positions, dtype=np.float64)
    tilt = _tilt_per_position(tilt, len(positions))
    return np.stack([forward_position(obj, probe, positions[b], tilt[b], geom)["I"]
                     for b in range(len(positions))])


# --------------------------------------------------------------------------- F8
def loss_from_intensity(I, a):
    """F8: L = sum_k (sqrt(I(k)) - a(k))^2 (amplitude loss; Eq. 5 with p = 0.5, reading R13)."""
    d = np.sqrt(I) - np.asarray(a, dtype=np.float64)
    return float(np.sum(d * d))


def loss_gaussian_eq5(S, n_pixels_total, mean_a):
    """Eq. 5 from the plain sum S: sqrt(S / (B N^2)) / <a> (R13)."""
    return math.sqrt(S / n_pixels_total) / mean_a


def _tilt_per_position(tilt, B):
    tilt = np.asarray(tilt if tilt is not None else (0.0, 0.0), dtype=np.float64)
    if tilt.ndim == 1:
        tilt = np.broadcast_to(tilt, (B, 2))
    return tilt


def forward_loss_batch(obj, probe, positions, tilt, meas_amp, geom):
    """F1-F8 over a minibatch.  Returns (L, loss_per_position [B], I [B,N,N])."""
    positions = np.asarray(positions, dtype=np.float64)
    B = len(positions)
    tilt = _tilt_per_position(tilt, B)
    I = np.empty((B,) + tuple(np.shape(meas_amp)[1:]), dtype=np.float64)
    lb = np.empty(B, dtype=np.float64)
    for b in range(B):
        I[b] = forward_position(obj, probe, positions[b], tilt[b], geom)["I"]
        lb[b] = loss_from_intensity(I[b], meas_amp[b])
    return float(lb.sum()), lb, I


# --------------------------------------------------------------------------- B1-B8
def backprop_position(f, probe, dLdI, tilt, geom, g_obj, g_probe):
    """B2-B8 for one position, for ANY loss that depends on the model through I_b(k) only:
    ``dLdI`` [N,N] = dL/dI_b(k), so that g_Psi^(m) = 2 dLdI Psi^(m) (I = sum_m |Psi|^2, convention R15).

    ``f`` is the dict of :func:`forward_position`.  Adds into ``g_obj`` [Nz,H,W] and ``g_probe`` [M,N,N]
    (complex128) and returns (g_pos [2], g_tilt [2], g_dz).  Used with dLdI = 1 - a/sqrt(I) for the amplitude
    loss (B1) and with the weighted total of Eq. 5-9 (oracle/losses.py).
    """
    probe = np.asarray(probe, dtype=np.complex128)
    Nz = len(f["psi"])
    N = probe.shape[-1]
    Psi, O, Mk = f["Psi"], f["O"], f["M"]
    g = idft2(2.0 * np.asarray(dLdI, dtype=np.float64)[None] * Psi)    # B2: g wrt phi_Nz
    D = np.zeros((N, N))
    for s in range(Nz - 1, -1, -1):
        crop_adjoint_add(g_obj[s], f["r"],                             # B3
                         np.sum(np.conj(f["psi"][s]) * g, axis=0))
        g = np.conj(O[s])[None] * g                                    # B4: g wrt psi_{s-1}
        if s > 0:                                                      # B5
            ghat = dft2(g)
            D += np.sum(np.imag(np.conj(dft2(f["psi"][s])) * ghat), axis=0)
            g = idft2(np.conj(Mk) * ghat)
    ghat0 = dft2(g)                                                    # B6
    E = shift_kernel(N, f["delta"])
    g_probe += idft2(np.conj(E)[None] * ghat0)
    kp = np.fft.fftfreq(N)                                             # B7
    T = np.sum(np.imag(np.conj(ghat0) * E[None] * dft2(probe)), axis=0)
    g_pos = 2.0 * np.pi * np.array([np.sum(kp[:, None] * T), np.sum(kp[None, :] * T)])
    k = np.fft.fftfreq(N, d=geom.dx)                                   # B8
    ky, kx = k[:, None], k[None, :]
    ty, tx = float(tilt[0]), float(tilt[1])
    g_tilt = 2.0 * np.pi * geom.dz * np.array([np.sum(D * ky) / math.cos(ty) ** 2,
                                               np.sum(D * kx) / math.cos(tx) ** 2])
    g_dz = float(np.sum(D * (-np.pi * geom.lam * (kx * kx + ky * ky)
                             + 2.0 * np.pi * (kx * math.tan(tx) + ky * math.tan(ty)))))
    return g_pos, g_tilt, g_dz


def grad_position(obj, probe, p, tilt, a, geom, g_obj, g_probe):
    """B1-B8 for one position.  Adds into ``g_obj`` [Nz,H,W] and ``g_probe`` [M,N,N]
    (complex128) and returns (loss_b, g_pos [2], g_tilt [2], g_dz).

    Hand-derived adjoint of F1-F8 (the paper uses reverse-mode AD; the
    formulas are SURVEY.md §8(c) B1-B8, convention R15, position gradient R3).
    """
    f = forward_position(obj, probe, p, tilt, geom)
    a = np.asarray(a, dtype=np.float64)
    I = f["I"]
    sqrtI = np.sqrt(I)
    loss_b = float(np.sum((sqrtI - a) ** 2))                           # F8
    w = np.zeros_like(I)                                               # B1 (R14): dL/dI = 1 - a/sqrt(I)
    nz = I > 0
    w[nz] = 1.0 - a[nz] / sqrtI[nz]
    g_pos, g_tilt, g_dz = backprop_position(f, probe, w, tilt, geom, g_obj, g_probe)
    return loss_b, g_pos, g_tilt, g_dz


# Inputs of the grad_batch call in flight.  Worker processes are forked AFTER this is set and read it from their copy
# of the parent's memory, so the arrays (114 MB of complex128 object on config 4) are not pickled to every worker;
# only the chunk's index list travels.  A parallelisation aid: no arithmetic of the method lives here.
_SHARED = None


def _grad_chunk(idx):
    obj, probe, positions, tilt, meas_amp, geom = _SHARED
    Nz, H, W = obj.shape
    N = probe.shape[-1]
    r = np.floor(positions[idx] + 0.5).astype(np.int64)
    y0, y1 = int(r[:, 0].min()), int(r[:, 0].max()) + N     # row band touched by this chunk
    g_band = np.zeros((Nz, y1 - y0, W), dtype=np.complex128)
    g_probe = np.zeros(probe.shape, dtype=np.complex128)
    out = []
    for b in idx:
        p = positions[b] - np.array([y0, 0.0])
        out.append(grad_position(obj[:, y0:y1], probe, p, tilt[b], meas_amp[b], geom,
                                 g_band, g_probe))
    return idx, y0, y1, g_band, g_probe, out


def grad_batch(obj, probe, positions, tilt, meas_amp, geom, workers=1):
    """B1-B8 summed over a minibatch (positions are independent).

    Returns dict(loss, loss_per_pos [B], g_object [Nz,H,W], g_probe [M,N,N],
    g_positions [B,2], g_tilt [B,2] (per position; a global tilt's gradient is the sum
    over b, R10), g_dz).  ``workers`` > 1 splits the positions over forked processes and
    sums the partial gradients (used for timing and for the larger parity cases).
    """
    obj = np.asarray(obj, dtype=np.complex128)
    probe = np.asarray(probe, dtype=np.complex128)
    positions = np.asarray(positions, dtype=np.float64)
    meas_amp = np.asarray(meas_amp, dtype=np.float64)
    B = len(positions)
    tilt = np.array(_tilt_per_position(tilt, B))
    order = np.argsort(np.floor(positions[:, 0] + 0.5), kind="stable")
    workers = max(1, min(int(workers), B)) if B else 1
    global _SHARED
    jobs = [c for c in np.array_split(order, workers) if len(c)]
    _SHARED = (obj, probe, positions, tilt, meas_amp, geom)
    try:
        if len(jobs) > 1:
            import multiprocessing as mp
            with mp.get_context("fork").Pool(len(jobs)) as pool:      # forked here: the children see _SHARED
                results = pool.map(_grad_chunk, jobs)
        else:
            results = [_grad_chunk(j) for j in jobs]
    finally:
        _SHARED = None
    g_object = np.zeros(obj.shape, dtype=np.complex128)
    g_probe = np.zeros(probe.shape, dtype=np.complex128)
    lb = np.zeros(B)
    g_pos = np.zeros((B, 2))
    g_tilt = np.zeros((B, 2))
    g_dz = 0.0
    for idx, y0, y1, g_band, gp, out in results:
        g_object[:, y0:y1] += g_band
        g_probe += gp
        for b, (l, gpos, gt, gz) in zip(idx, out):
            lb[b], g_pos[b], g_tilt[b] = l, gpos, gt
            g_dz += gz
    return {"loss": float(lb.sum()), "loss_per_pos": lb, "g_object": g_object,
            "g_probe": g_probe, "g_positions": g_pos, "g_tilt": g_tilt, "g_dz": g_dz}


# --------------------------------------------------------------------------- B9
def adam_step(theta, g, m, v, t, lr, beta1=0.9, beta2=0.999, eps=1e-8):
    """B9: one bias-corrected Adam step (Kingma & Ba; reading R20).

    Complex parameters are treated as two reals (views).  ``t`` is the 1-based step
    count.  Returns the new (theta, m, v) as float64/complex128 arrays.
    """
    theta = np.array(theta, dtype=np.complex128 if np.iscomplexobj(theta) else np.float64)
    cplx = np.iscomplexobj(theta)
    th = theta.view(np.float64) if cplx else theta
    gg = np.ascontiguousarray(g, dtype=theta.dtype)
    gg = gg.view(np.float64) if cplx else gg
    m = np.array(m, dtype=np.float64).reshape(th.shape)
    v = np.array(v, dtype=np.float64).reshape(th.shape)
    m = beta1 * m + (1.0 - beta1) * gg
    v = beta2 * v + (1.0 - beta2) * gg * gg
    mhat = m / (1.0 - beta1 ** t)
    vhat = v / (1.0 - beta2 ** t)
    th = th - lr * mhat / (np.sqrt(vhat) + eps)
    theta = th.view(np.complex128) if cplx else th
    return theta, m, v
