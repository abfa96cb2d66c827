"""Shared helpers for the GPU parity tests: build a seeded case (inputs for both sides) and the
oracle's answer.  Measurements come from the ORACLE forward at the ground truth plus Poisson noise
(SURVEY.md §8(d)); no input or expected value ever comes from the CUDA path."""
from __future__ import annotations

import functools
import os

import numpy as np

import oracle
from paper_2505_07814_b200 import synth

WORKERS = max(1, min(16, len(os.sched_getaffinity(0))))


def rel_l2(x, ref):
    x = np.asarray(x)
    ref = np.asarray(ref)
    return float(np.linalg.norm((x - ref).ravel()) / max(np.linalg.norm(ref.ravel()), 1e-300))


def geom_of(cfg):
    return oracle.Geometry(cfg.dz, cfg.lam, cfg.dx)


@functools.lru_cache(maxsize=8)
def _truth(c):
    return synth.truth(synth.get_config(c))


@functools.lru_cache(maxsize=8)
def _eval(c, which):
    return synth.eval_point(synth.get_config(c), which)


def make_case(c, which, indices, tilt_mode=None):
    """Inputs for config c at evaluation point `which` on scan positions `indices`."""
    cfg = synth.get_config(c)
    indices = np.asarray(indices)
    tr, ev = _truth(c), _eval(c, which)
    tm = cfg.tilt_mode if tilt_mode is None else tilt_mode
    I_true = oracle.intensity_batch(tr["object"], tr["probe"], tr["positions"][indices],
                                    tr["tilt"] if cfg.tilt_mode else None, geom_of(cfg))
    meas = synth.poisson_amplitudes(cfg, I_true, indices)
    tilt = ev["tilt"] if tm else None
    if tm == 2:
        rng = np.random.default_rng(1000 * c + 77)
        tilt = (ev["tilt"][None, :] + rng.normal(0, 2e-4, (len(indices), 2))).astype(np.float32)
    case = {"cfg": cfg, "object": ev["object"], "probe": ev["probe"],
            "positions": np.ascontiguousarray(ev["positions"][indices]), "tilt": tilt, "tilt_mode": tm,
            "meas": meas, "indices": indices}
    if which == "B":
        # DESIGN.md reading R26: at the exact-vacuum start the model's dark field is float32 rounding
        # noise (I ~ 1e-14 of the peak), and d/dPsi (|Psi| - a)^2 = 2 (1 - a/|Psi|) Psi has a phase set
        # by that noise wherever counts a > 0 were measured: the gradient is ill-conditioned there in
        # any float32 arithmetic.  Gradients at point B are therefore compared with the counts of those
        # pixels (model intensity below 1e-9 of the pattern's peak, per the ORACLE) set to zero; the
        # loss and the intensities are compared on the full measurements.
        I_B = oracle.intensity_batch(case["object"], case["probe"], case["positions"], tilt, geom_of(cfg))
        dark = I_B < 1e-9 * I_B.max(axis=(1, 2), keepdims=True)
        case["meas_masked"] = np.where(dark, 0.0, meas).astype(np.float32)
    return case


def oracle_grad(case, workers=None):
    cfg = case["cfg"]
    return oracle.grad_batch(case["object"], case["probe"], case["positions"], case["tilt"], case["meas"],
                             geom_of(cfg), workers=WORKERS if workers is None else workers)
