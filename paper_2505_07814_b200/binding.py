"""Thin ctypes binding of ``include/pty.h``: argument marshalling only.

Every step of the hot path runs in the CUDA kernels of ``libpty.so``; PyTorch is used here for
device memory and streams (``tensor.data_ptr()``, ``torch.cuda.current_stream()``).  Importing
this module fails loudly if the library has not been built (``python -m
paper_2505_07814_b200.build``): there is no CPU or PyTorch fallback.
"""
from __future__ import annotations

import ctypes as C
import os

import torch

_HERE = os.path.dirname(os.path.abspath(__file__))
# PTY_LIB names another build of the same library (build.build_variant: a compile-time switch under test); the default
# is the in-tree product build.  Either way a missing file is an error: there is no fallback path.
LIB_PATH = os.environ.get("PTY_LIB") or os.path.join(_HERE, "libpty.so")

if not os.path.exists(LIB_PATH):
    raise ImportError(f"{LIB_PATH} is missing: build it with `python -m paper_2505_07814_b200.build` "
                      "(nvcc, sm_100a).  There is no fallback path.")

lib = C.CDLL(LIB_PATH)

PTY_OK, PTY_ERR_INVALID_ARG, PTY_ERR_UNSUPPORTED = 0, -1, -2
PTY_ERR_WORKSPACE, PTY_ERR_CUDA, PTY_ERR_BOUNDS, PTY_ERR_ZERO_DATA = -3, -4, -5, -6
PTY_FLAG_SPECTRA, PTY_FLAG_STEP, PTY_FLAG_HOST, PTY_FLAG_AMP_PHASE, PTY_FLAG_TMA_OBJECT, PTY_FLAG_PAIR_SUM = 1, 2, 4, 8, 16, 32
PTY_BWD_ACCUMULATE, PTY_BWD_REUSE_FORWARD = 1, 4

EXPORTS = ["pty_workspace_bytes", "pty_create", "pty_destroy", "pty_forward_loss", "pty_backward",
           "pty_step", "pty_adam_update", "pty_grad_host", "pty_status", "pty_profile",
           "pty_profile_read", "pty_set_loss", "pty_loss_terms", "pty_forward_loss_ap", "pty_backward_ap",
           "pty_step_ap", "pty_constrain", "pty_rz_filter_object", "pty_grad_host_async", "pty_grad_host_wait",
           "pty_ortho_probe_noalloc", "pty_launch_count", "pty_last_error", "pty_version"]
_INT_RETURNS = EXPORTS[:21]


class pty_dims(C.Structure):
    _fields_ = [("Nz", C.c_int32), ("H", C.c_int32), ("W", C.c_int32), ("M", C.c_int32), ("N", C.c_int32),
                ("Bmax", C.c_int32), ("dz", C.c_float), ("lam", C.c_float), ("dx", C.c_float),
                ("tilt_mode", C.c_int32), ("flags", C.c_int32), ("n_obj", C.c_int32)]


class pty_loss(C.Structure):
    _fields_ = [("mode", C.c_int32), ("w_gaussian", C.c_float), ("w_poisson", C.c_float), ("w_pacbed", C.c_float),
                ("w_sparse", C.c_float), ("eps", C.c_float)]


class pty_adam_ap(C.Structure):
    _fields_ = [("lr_amp", C.c_float), ("lr_phase", C.c_float), ("lr_probe", C.c_float), ("lr_positions", C.c_float),
                ("lr_tilt", C.c_float), ("beta1", C.c_float), ("beta2", C.c_float), ("eps", C.c_float), ("t", C.c_int32)]


class pty_adam_state_ap(C.Structure):
    _fields_ = [(n, C.c_void_p) for n in ("m_amp", "v_amp", "m_phase", "v_phase", "m_probe", "v_probe", "m_positions",
                                          "v_positions", "m_tilt", "v_tilt")]


class pty_constraints(C.Structure):
    _fields_ = [("ortho_probe", C.c_int32), ("sigma_z", C.c_float), ("phase_positive", C.c_int32),
                ("clamp_amp", C.c_int32), ("amp_min", C.c_float), ("amp_max", C.c_float)]


class pty_adam(C.Structure):
    _fields_ = [("lr_object", C.c_float), ("lr_probe", C.c_float), ("lr_positions", C.c_float),
                ("lr_tilt", C.c_float), ("beta1", C.c_float), ("beta2", C.c_float), ("eps", C.c_float),
                ("t", C.c_int32)]


class pty_adam_state(C.Structure):
    _fields_ = [(n, C.c_void_p) for n in ("m_object", "v_object", "m_probe", "v_probe", "m_positions",
                                          "v_positions", "m_tilt", "v_tilt")]


_vp = C.c_void_p
lib.pty_workspace_bytes.argtypes = [C.POINTER(pty_dims), C.POINTER(C.c_size_t)]
lib.pty_create.argtypes = [C.POINTER(_vp), C.POINTER(pty_dims), _vp, C.c_size_t, C.c_int]
lib.pty_destroy.argtypes = [_vp]
lib.pty_forward_loss.argtypes = [_vp, _vp, _vp, _vp, _vp, _vp, C.c_int32, _vp, _vp, _vp, _vp]
lib.pty_backward.argtypes = [_vp, _vp, _vp, _vp, _vp, _vp, C.c_int32, _vp, _vp, _vp, _vp, _vp, C.c_int32, _vp]
lib.pty_step.argtypes = [_vp, _vp, _vp, _vp, _vp, _vp, C.c_int32, C.POINTER(pty_adam),
                         C.POINTER(pty_adam_state), _vp, _vp]
lib.pty_adam_update.argtypes = [_vp, _vp, _vp, _vp, _vp, C.c_size_t, C.c_float, C.c_float, C.c_float,
                                C.c_float, C.c_int32, _vp]
lib.pty_grad_host.argtypes = [_vp, _vp, _vp, _vp, _vp, _vp, C.c_int32, _vp, _vp, _vp, _vp, _vp, _vp]
lib.pty_grad_host_async.argtypes = lib.pty_grad_host.argtypes
lib.pty_grad_host_wait.argtypes = [_vp]
lib.pty_status.argtypes = [_vp, C.POINTER(C.c_int32)]
lib.pty_profile.argtypes = [_vp, C.c_int32]
lib.pty_profile_read.argtypes = [_vp, C.POINTER(C.c_float), C.POINTER(C.c_int32), C.POINTER(C.c_float),
                                 C.POINTER(C.c_int32)]
lib.pty_launch_count.argtypes = [_vp]
lib.pty_launch_count.restype = C.c_int64
lib.pty_last_error.argtypes = [_vp]
lib.pty_last_error.restype = C.c_char_p
lib.pty_version.restype = C.c_char_p
lib.pty_set_loss.argtypes = [_vp, C.POINTER(pty_loss)]
lib.pty_loss_terms.argtypes = [_vp, C.POINTER(C.c_double)]
lib.pty_forward_loss_ap.argtypes = [_vp, _vp, _vp, _vp, _vp, _vp, _vp, C.c_int32, _vp, _vp, _vp, _vp]
lib.pty_backward_ap.argtypes = [_vp, _vp, _vp, _vp, _vp, _vp, _vp, C.c_int32, _vp, _vp, _vp, _vp, _vp, _vp, C.c_int32, _vp]
lib.pty_step_ap.argtypes = [_vp, _vp, _vp, _vp, _vp, _vp, _vp, C.c_int32, C.POINTER(pty_adam_ap),
                            C.POINTER(pty_adam_state_ap), _vp, _vp]
lib.pty_constrain.argtypes = [_vp, _vp, _vp, _vp, C.POINTER(pty_constraints), _vp]
lib.pty_rz_filter_object.argtypes = [_vp, _vp, C.c_float, _vp]
lib.pty_ortho_probe_noalloc.argtypes = [_vp, C.c_int32, C.c_int32, C.c_int, _vp]
for _n in _INT_RETURNS:
    getattr(lib, _n).restype = C.c_int


class PtyError(RuntimeError):
    def __init__(self, code, msg):
        super().__init__(f"pty error {code}: {msg}")
        self.code = code


def _ptr(t, dtype=None, device=None):
    """Device (or host) address of a contiguous tensor; None -> NULL."""
    if t is None:
        return None
    if not t.is_contiguous():
        raise ValueError("tensors passed to the pty C ABI must be contiguous")
    if dtype is not None and t.dtype != dtype:
        raise TypeError(f"expected {dtype}, got {t.dtype}")
    if device is not None and t.device.type != device:
        raise ValueError(f"expected a {device} tensor, got {t.device}")
    return t.data_ptr()


def _stream():
    return torch.cuda.current_stream().cuda_stream


class Plan:
    """Owns a pty_plan and its workspace (a torch uint8 CUDA tensor)."""

    def __init__(self, Nz, H, W, M, N, Bmax, dz, lam, dx, tilt_mode=0, flags=0, device=0, n_obj=1):
        if not torch.cuda.is_available():
            raise RuntimeError("pty needs a CUDA device (sm_100a); there is no CPU fallback")
        self.dims = pty_dims(Nz, H, W, M, N, Bmax, dz, lam, dx, tilt_mode, flags, n_obj)
        nbytes = C.c_size_t(0)
        rc = lib.pty_workspace_bytes(C.byref(self.dims), C.byref(nbytes))
        if rc != PTY_OK:
            raise PtyError(rc, lib.pty_last_error(None).decode())
        self.workspace_bytes = nbytes.value
        self.device = torch.device("cuda", device)
        self.workspace = torch.empty(nbytes.value + 256, dtype=torch.uint8, device=self.device)
        base = (self.workspace.data_ptr() + 255) & ~255
        self._h = _vp(None)
        rc = lib.pty_create(C.byref(self._h), C.byref(self.dims), base, nbytes.value, device)
        if rc != PTY_OK:
            raise PtyError(rc, lib.pty_last_error(None).decode())
        self._loss = torch.zeros(1, dtype=torch.float64, device=self.device)

    def _check(self, rc):
        if rc != PTY_OK:
            raise PtyError(rc, lib.pty_last_error(self._h).decode())

    def close(self):
        if getattr(self, "_h", None) is not None and self._h.value:
            lib.pty_destroy(self._h)
            self._h = _vp(None)

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    # ---- the calls of include/pty.h -------------------------------------------------------
    def forward_loss(self, obj, probe, positions, tilt, meas_amp, loss=None, loss_per_pos=None, intensity=None):
        loss = self._loss if loss is None else loss
        self._check(lib.pty_forward_loss(
            self._h, _ptr(obj, torch.complex64, "cuda"), _ptr(probe, torch.complex64, "cuda"),
            _ptr(positions, torch.float32, "cuda"), _ptr(tilt, torch.float32, "cuda"),
            _ptr(meas_amp, torch.float32, "cuda"), positions.shape[0], _ptr(loss, torch.float64, "cuda"),
            _ptr(loss_per_pos, torch.float32, "cuda"), _ptr(intensity, torch.float32, "cuda"), _stream()))
        return loss

    def backward(self, obj, probe, positions, tilt, meas_amp, g_object, g_probe=None, g_positions=None,
                 g_tilt=None, g_dz=None, flags=0):
        self._check(lib.pty_backward(
            self._h, _ptr(obj, torch.complex64, "cuda"), _ptr(probe, torch.complex64, "cuda"),
            _ptr(positions, torch.float32, "cuda"), _ptr(tilt, torch.float32, "cuda"),
            _ptr(meas_amp, torch.float32, "cuda"), positions.shape[0], _ptr(g_object, torch.complex64, "cuda"),
            _ptr(g_probe, torch.complex64, "cuda"), _ptr(g_positions, torch.float32, "cuda"),
            _ptr(g_tilt, torch.float32, "cuda"), _ptr(g_dz, torch.float32, "cuda"), flags, _stream()))

    def step(self, obj, probe, positions, tilt, meas_amp, hp: pty_adam, state: dict, loss=None):
        loss = self._loss if loss is None else loss
        st = pty_adam_state(*[_ptr(state.get(n), torch.float32, "cuda") for n, _ in pty_adam_state._fields_])
        self._check(lib.pty_step(
            self._h, _ptr(obj, torch.complex64, "cuda"), _ptr(probe, torch.complex64, "cuda"),
            _ptr(positions, torch.float32, "cuda"), _ptr(tilt, torch.float32, "cuda"),
            _ptr(meas_amp, torch.float32, "cuda"), positions.shape[0], C.byref(hp), C.byref(st),
            _ptr(loss, torch.float64, "cuda"), _stream()))
        return loss

    def set_loss(self, mode=0, w_gaussian=1.0, w_poisson=0.0, w_pacbed=0.0, w_sparse=0.0, eps=1e-6):
        cfg = pty_loss(mode, w_gaussian, w_poisson, w_pacbed, w_sparse, eps)
        self._check(lib.pty_set_loss(self._h, C.byref(cfg)))

    def loss_terms(self):
        """{'gaussian', 'poisson', 'pacbed', 'sparse'} of the last loss-mode-1 forward (synchronises)."""
        out = (C.c_double * 4)()
        self._check(lib.pty_loss_terms(self._h, out))
        return dict(zip(("gaussian", "poisson", "pacbed", "sparse"), list(out)))

    def forward_loss_ap(self, amp, phase, probe, positions, tilt, meas_amp, loss=None, loss_per_pos=None, intensity=None):
        loss = self._loss if loss is None else loss
        self._check(lib.pty_forward_loss_ap(
            self._h, _ptr(amp, torch.float32, "cuda"), _ptr(phase, torch.float32, "cuda"),
            _ptr(probe, torch.complex64, "cuda"), _ptr(positions, torch.float32, "cuda"),
            _ptr(tilt, torch.float32, "cuda"), _ptr(meas_amp, torch.float32, "cuda"), positions.shape[0],
            _ptr(loss, torch.float64, "cuda"), _ptr(loss_per_pos, torch.float32, "cuda"),
            _ptr(intensity, torch.float32, "cuda"), _stream()))
        return loss

    def backward_ap(self, amp, phase, probe, positions, tilt, meas_amp, g_amp, g_phase, g_probe=None, g_positions=None,
                    g_tilt=None, g_dz=None, flags=0):
        self._check(lib.pty_backward_ap(
            self._h, _ptr(amp, torch.float32, "cuda"), _ptr(phase, torch.float32, "cuda"),
            _ptr(probe, torch.complex64, "cuda"), _ptr(positions, torch.float32, "cuda"),
            _ptr(tilt, torch.float32, "cuda"), _ptr(meas_amp, torch.float32, "cuda"), positions.shape[0],
            _ptr(g_amp, torch.float32, "cuda"), _ptr(g_phase, torch.float32, "cuda"),
            _ptr(g_probe, torch.complex64, "cuda"), _ptr(g_positions, torch.float32, "cuda"),
            _ptr(g_tilt, torch.float32, "cuda"), _ptr(g_dz, torch.float32, "cuda"), flags, _stream()))

    def step_ap(self, amp, phase, probe, positions, tilt, meas_amp, hp: pty_adam_ap, state: dict, loss=None):
        loss = self._loss if loss is None else loss
        st = pty_adam_state_ap(*[_ptr(state.get(n), torch.float32, "cuda") for n, _ in pty_adam_state_ap._fields_])
        self._check(lib.pty_step_ap(
            self._h, _ptr(amp, torch.float32, "cuda"), _ptr(phase, torch.float32, "cuda"),
            _ptr(probe, torch.complex64, "cuda"), _ptr(positions, torch.float32, "cuda"),
            _ptr(tilt, torch.float32, "cuda"), _ptr(meas_amp, torch.float32, "cuda"), positions.shape[0],
            C.byref(hp), C.byref(st), _ptr(loss, torch.float64, "cuda"), _stream()))
        return loss

    def constrain(self, amp=None, phase=None, probe=None, ortho_probe=False, sigma_z=0.0, phase_positive=False,
                  clamp_amp=None):
        lo, hi = clamp_amp if clamp_amp is not None else (0.0, 0.0)
        c = pty_constraints(1 if ortho_probe else 0, sigma_z, 1 if phase_positive else 0,
                            1 if clamp_amp is not None else 0, lo, hi)
        self._check(lib.pty_constrain(self._h, _ptr(amp, torch.float32, "cuda"), _ptr(phase, torch.float32, "cuda"),
                                      _ptr(probe, torch.complex64, "cuda"), C.byref(c), _stream()))

    def rz_filter_object(self, obj, sigma_z):
        self._check(lib.pty_rz_filter_object(self._h, _ptr(obj, torch.complex64, "cuda"), sigma_z, _stream()))

    def adam_update(self, theta, grad, m, v, lr, beta1=0.9, beta2=0.999, eps=1e-8, t=1):
        n = theta.numel() * (2 if theta.is_complex() else 1)
        self._check(lib.pty_adam_update(self._h, theta.data_ptr(), grad.data_ptr(), _ptr(m, torch.float32, "cuda"),
                                        _ptr(v, torch.float32, "cuda"), n, lr, beta1, beta2, eps, t, _stream()))

    def grad_host(self, h_obj, h_probe, h_positions, h_tilt, h_meas_amp, h_loss, h_g_object, h_g_probe=None,
                  h_g_positions=None, h_g_tilt=None, wait=True):
        """wait=False: pty_grad_host_async (enqueue only); call grad_host_wait() before reading the outputs."""
        self._check((lib.pty_grad_host if wait else lib.pty_grad_host_async)(
            self._h, _ptr(h_obj, torch.complex64, "cpu"), _ptr(h_probe, torch.complex64, "cpu"),
            _ptr(h_positions, torch.float32, "cpu"), _ptr(h_tilt, torch.float32, "cpu"),
            _ptr(h_meas_amp, torch.float32, "cpu"), h_positions.shape[0], _ptr(h_loss, torch.float64, "cpu"),
            _ptr(h_g_object, torch.complex64, "cpu"), _ptr(h_g_probe, torch.complex64, "cpu"),
            _ptr(h_g_positions, torch.float32, "cpu"), _ptr(h_g_tilt, torch.float32, "cpu"), _stream()))

    def grad_host_wait(self):
        self._check(lib.pty_grad_host_wait(self._h))

    def status(self):
        flags = C.c_int32(0)
        rc = lib.pty_status(self._h, C.byref(flags))
        return rc, flags.value

    def profile(self, enable=True):
        self._check(lib.pty_profile(self._h, 1 if enable else 0))

    def profile_read(self):
        """{'fwd': (ms_total, launches), 'bwd': (ms_total, launches)} since the last read."""
        f, b = C.c_float(0), C.c_float(0)
        nf, nb = C.c_int32(0), C.c_int32(0)
        self._check(lib.pty_profile_read(self._h, C.byref(f), C.byref(nf), C.byref(b), C.byref(nb)))
        return {"fwd": (f.value, nf.value), "bwd": (b.value, nb.value)}

    def launch_count(self):
        return int(lib.pty_launch_count(self._h))

    def last_error(self):
        return lib.pty_last_error(self._h).decode()


def plan_for(cfg, Bmax=None, flags=0, device=0, n_obj=1):
    """Plan for a ``synth.Config``."""
    return Plan(cfg.Nz, cfg.H, cfg.W, cfg.M, cfg.N, cfg.B if Bmax is None else Bmax, cfg.dz, cfg.lam, cfg.dx,
                tilt_mode=cfg.tilt_mode, flags=flags, device=device, n_obj=n_obj)


ORTHO_NOALLOC_MAX_MODES = 32


def ortho_probe_noalloc(probe):
    """pty_ortho_probe_noalloc: orthogonalise the modes of ``probe`` [M, N, N] (complex64, CUDA) in place without a
    plan or a workspace -- for callers that have no device memory to give the library (a host application whose pool
    already owns the whole GPU, a hook that only receives the probe).  The scratch is a fixed 33 KB array inside
    libpty.so, one per GPU and shared by every call: M <= 32, and calls that can overlap on one GPU race, so keep them
    on one stream.  Make the first call on each device at start-up, outside stream capture (it looks the array up).
    Enqueued on torch's current stream of the probe's device; does not synchronise."""
    if probe.dim() != 3 or probe.shape[1] != probe.shape[2]:
        raise ValueError("probe must be [M, N, N]")
    with torch.cuda.device(probe.device):
        rc = lib.pty_ortho_probe_noalloc(_ptr(probe, torch.complex64, "cuda"), probe.shape[0], probe.shape[1],
                                         probe.device.index, _stream())
    if rc != PTY_OK:
        raise PtyError(rc, lib.pty_last_error(None).decode())
