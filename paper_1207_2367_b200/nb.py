"""ctypes binding of libnb.so -- same names as include/nb.h, argument marshalling only.

Every function takes the context handle first and accepts, for [dev|host] pointers, either a
contiguous float64/int32 torch tensor (CUDA or CPU, pinned or not) or a contiguous numpy
array; the raw address goes straight to the C call.  Outputs are caller-provided buffers, or
are allocated here as torch CUDA tensors when omitted.  PyTorch is used for device memory
and the stream only.  A non-zero return code raises NBError carrying nb_last_error().
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

from . import _build

__all__ = [
    "NBError", "lib", "lib_path", "exported_symbols", "NBody",
    "nb_init", "nb_free", "nb_set_limits", "nb_startup", "nb_startup_commit", "nb_next_block", "nb_get_active", "nb_predict",
    "nb_force", "nb_correct_and_step", "nb_run_until", "nb_run_steps", "nb_energy", "nb_get_state",
    "nb_get_derivs", "nb_get_pred", "nb_set_pred_acc", "nb_set_pred", "nb_get_full_state",
    "nb_set_full_state", "nb_get_stats", "nb_set_tuning", "nb_set_loop_mode", "nb_get_loop_mode", "nb_set_precision", "nb_set_j_range", "nb_get_forces", "nb_set_forces", "nb_get_launch", "nb_probe_fp64_peak",
    "nb_set_debug", "nb_version", "nb_last_error", "nb_force_static", "NB_STATIC_MAX_N",
]

NB_OK, NB_EINVAL, NB_ESTATE, NB_ECUDA, NB_ENOMEM = 0, -1, -2, -3, -4
_CODES = {NB_EINVAL: "NB_EINVAL", NB_ESTATE: "NB_ESTATE", NB_ECUDA: "NB_ECUDA", NB_ENOMEM: "NB_ENOMEM"}


class NBError(RuntimeError):
    def __init__(self, code, msg):
        super().__init__("%s (%d): %s" % (_CODES.get(code, "NB_E?"), code, msg))
        self.code = code


_vp = C.c_void_p
_i64 = C.c_int64
_dbl = C.c_double
_SIGS = {
    "nb_init": (C.c_int, [C.POINTER(_vp), _i64, _vp, _vp, _vp, _dbl, _dbl, _vp]),
    "nb_set_limits": (C.c_int, [_vp, _dbl, _dbl, _dbl]),
    "nb_startup": (C.c_int, [_vp]),
    "nb_startup_commit": (C.c_int, [_vp, C.c_int]),
    "nb_next_block": (C.c_int, [_vp, C.POINTER(_dbl), C.POINTER(_i64)]),
    "nb_get_active": (C.c_int, [_vp, _vp]),
    "nb_predict": (C.c_int, [_vp, _dbl]),
    "nb_force": (C.c_int, [_vp, _vp, _i64, _vp, _vp, _vp]),
    "nb_correct_and_step": (C.c_int, [_vp]),
    "nb_run_until": (C.c_int, [_vp, _dbl, C.POINTER(_i64)]),
    "nb_run_steps": (C.c_int, [_vp, _i64, _vp, _vp, _vp]),
    "nb_energy": (C.c_int, [_vp, C.POINTER(_dbl)]),
    "nb_get_state": (C.c_int, [_vp, _vp, _vp, _vp, _vp]),
    "nb_get_derivs": (C.c_int, [_vp, _vp, _vp, _vp, _vp]),
    "nb_get_pred": (C.c_int, [_vp, _vp, _vp, _vp]),
    "nb_set_pred_acc": (C.c_int, [_vp, _vp]),
    "nb_set_pred": (C.c_int, [_vp, _vp, _vp, _vp]),
    "nb_get_full_state": (C.c_int, [_vp, _vp]),
    "nb_set_full_state": (C.c_int, [_vp, _vp]),
    "nb_get_stats": (C.c_int, [_vp, C.POINTER(_dbl), C.POINTER(_i64)]),
    "nb_set_tuning": (C.c_int, [_vp, C.c_int, C.c_int]),
    "nb_set_loop_mode": (C.c_int, [_vp, C.c_int]),
    "nb_get_loop_mode": (C.c_int, [_vp, C.POINTER(C.c_int)]),
    "nb_set_precision": (C.c_int, [_vp, C.c_int]),
    "nb_set_j_range": (C.c_int, [_vp, _i64, _i64]),
    "nb_get_forces": (C.c_int, [_vp, _vp]),
    "nb_set_forces": (C.c_int, [_vp, _vp]),
    "nb_get_launch": (C.c_int, [_vp, C.POINTER(_i64)]),
    "nb_probe_fp64_peak": (C.c_int, [_vp, _i64, C.POINTER(_dbl), C.POINTER(C.c_float)]),
    "nb_set_debug": (C.c_int, [_vp, C.c_int]),
    "nb_force_static": (C.c_int, [_i64, _vp, _vp, _vp, _vp, _dbl, _vp, _i64, _vp, _vp, _vp, _vp, C.c_char_p, _i64]),
    "nb_last_error": (C.c_char_p, [_vp]),
    "nb_free": (None, [_vp]),
    "nb_version": (C.c_char_p, []),
}
_lib = None


def exported_symbols():
    """Names include/nb.h declares (the binding's signature table mirrors the header)."""
    return sorted(_SIGS)


def lib_path() -> str:
    return _build.LIB


def lib():
    """Load libnb.so (building it in-tree with nvcc if it is missing or stale).  Fails loudly."""
    global _lib
    if _lib is None:
        path = _build.build()
        if not os.path.exists(path):
            raise ImportError("libnb.so is missing and could not be built: %s" % path)
        L = C.CDLL(path)
        for name, (res, args) in _SIGS.items():
            fn = getattr(L, name)  # AttributeError if the library does not export it
            fn.restype = res
            fn.argtypes = args
        _lib = L
    return _lib


# ---------------------------------------------------------------------------- marshalling
def _torch():
    import torch
    return torch


def _ptr(x, dtype=np.float64, n=None):
    """Raw address of a contiguous tensor/array (None -> NULL); checks dtype and size."""
    if x is None:
        return None
    if isinstance(x, np.ndarray):
        if x.dtype != dtype or not x.flags["C_CONTIGUOUS"]:
            raise TypeError("numpy argument must be C-contiguous %s" % np.dtype(dtype).name)
        if n is not None and x.size != n:
            raise ValueError("argument has %d elements, expected %d" % (x.size, n))
        return x.ctypes.data
    torch = _torch()
    if isinstance(x, torch.Tensor):
        want = {np.float64: torch.float64, np.int32: torch.int32, np.int64: torch.int64,
                np.float32: torch.float32}[dtype]
        if x.dtype != want or not x.is_contiguous():
            raise TypeError("tensor argument must be contiguous %s" % want)
        if n is not None and x.numel() != n:
            raise ValueError("argument has %d elements, expected %d" % (x.numel(), n))
        return x.data_ptr()
    raise TypeError("expected a torch tensor or numpy array, got %r" % type(x))


def _check(ctx, rc):
    if rc != NB_OK:
        msg = lib().nb_last_error(ctx).decode() if ctx else "no context"
        raise NBError(rc, msg)


def _dev_empty(shape, dtype=None):
    torch = _torch()
    return torch.empty(shape, dtype=dtype or torch.float64, device="cuda")


# ---------------------------------------------------------------------------- the C-ABI, by name
def nb_version() -> str:
    return lib().nb_version().decode()


def nb_last_error(ctx) -> str:
    return lib().nb_last_error(ctx).decode()


def nb_init(pos, vel, mass, eps, eta, stream=None):
    """nb_init -> opaque context handle.  stream: a torch.cuda.Stream, a raw cudaStream_t or None."""
    N = int(mass.shape[0])
    if stream is not None and hasattr(stream, "cuda_stream"):
        stream = stream.cuda_stream
    h = _vp()
    rc = lib().nb_init(C.byref(h), N, _ptr(pos, n=3 * N), _ptr(vel, n=3 * N), _ptr(mass, n=N), float(eps),
                       float(eta), _vp(stream or 0))
    if rc != NB_OK:
        raise NBError(rc, "nb_init failed (N=%d, eps=%g, eta=%g)" % (N, eps, eta))
    return h


def nb_free(ctx):
    lib().nb_free(ctx)


def nb_set_limits(ctx, dt_min, dt_max, eta_init=0.01):
    _check(ctx, lib().nb_set_limits(ctx, float(dt_min), float(dt_max), float(eta_init)))


def nb_startup(ctx):
    _check(ctx, lib().nb_startup(ctx))


def nb_startup_commit(ctx, npass):
    _check(ctx, lib().nb_startup_commit(ctx, int(npass)))


def nb_next_block(ctx):
    t, m = _dbl(), _i64()
    _check(ctx, lib().nb_next_block(ctx, C.byref(t), C.byref(m)))
    return t.value, m.value


def nb_get_active(ctx, idx):
    _check(ctx, lib().nb_get_active(ctx, _ptr(idx, np.int32)))
    return idx


def nb_predict(ctx, t):
    _check(ctx, lib().nb_predict(ctx, float(t)))


def nb_force(ctx, active_idx, n_active, acc=None, jerk=None, snap=None):
    n = int(n_active)
    _check(ctx, lib().nb_force(ctx, _ptr(active_idx, np.int32, n if active_idx is not None else None), n,
                               _ptr(acc, n=3 * n), _ptr(jerk, n=3 * n), _ptr(snap, n=3 * n)))
    return acc, jerk, snap


def nb_correct_and_step(ctx):
    _check(ctx, lib().nb_correct_and_step(ctx))


def nb_run_until(ctx, t_end) -> int:
    n = _i64()
    _check(ctx, lib().nb_run_until(ctx, float(t_end), C.byref(n)))
    return n.value


def nb_run_steps(ctx, n, log=True):
    n = int(n)
    lt = np.zeros(max(n, 1)); lm = np.zeros(max(n, 1), dtype=np.int64); ms = np.zeros(max(n, 1), dtype=np.float32)
    if log:
        _check(ctx, lib().nb_run_steps(ctx, n, lt.ctypes.data, lm.ctypes.data, ms.ctypes.data))
    else:
        _check(ctx, lib().nb_run_steps(ctx, n, None, None, None))
    return lt[:n], lm[:n], ms[:n]


def nb_energy(ctx):
    out = (_dbl * 9)()
    _check(ctx, lib().nb_energy(ctx, out))
    return np.array(out[:], dtype=np.float64)


def nb_get_state(ctx, pos=None, vel=None, t=None, dt=None):
    _check(ctx, lib().nb_get_state(ctx, _ptr(pos), _ptr(vel), _ptr(t), _ptr(dt)))


def nb_get_derivs(ctx, acc=None, jerk=None, snap=None, crackle=None):
    _check(ctx, lib().nb_get_derivs(ctx, _ptr(acc), _ptr(jerk), _ptr(snap), _ptr(crackle)))


def nb_get_pred(ctx, pos=None, vel=None, acc=None):
    _check(ctx, lib().nb_get_pred(ctx, _ptr(pos), _ptr(vel), _ptr(acc)))


def nb_set_pred_acc(ctx, acc_pred):
    _check(ctx, lib().nb_set_pred_acc(ctx, _ptr(acc_pred)))


def nb_set_pred(ctx, pos, vel, acc=None):
    _check(ctx, lib().nb_set_pred(ctx, _ptr(pos), _ptr(vel), _ptr(acc)))


def nb_get_full_state(ctx, state):
    _check(ctx, lib().nb_get_full_state(ctx, _ptr(state)))
    return state


def nb_set_full_state(ctx, state):
    _check(ctx, lib().nb_set_full_state(ctx, _ptr(state)))


def nb_get_stats(ctx):
    out = (_dbl * 4)()
    hist = (_i64 * 64)()
    _check(ctx, lib().nb_get_stats(ctx, out, hist))
    return dict(n_steps=int(out[0]), n_pairs=float(out[1]), n_launch=int(out[2]), t_now=float(out[3]),
                hist=np.array(hist[:], dtype=np.int64))


def nb_set_tuning(ctx, split=0, jlanes=0):
    _check(ctx, lib().nb_set_tuning(ctx, int(split), int(jlanes)))


def nb_set_loop_mode(ctx, device_driven=1):
    _check(ctx, lib().nb_set_loop_mode(ctx, int(device_driven)))


def nb_get_loop_mode(ctx) -> int:
    mode = C.c_int()
    _check(ctx, lib().nb_get_loop_mode(ctx, C.byref(mode)))
    return mode.value


def nb_set_precision(ctx, mode=0):
    _check(ctx, lib().nb_set_precision(ctx, int(mode)))


def nb_set_j_range(ctx, j_begin, j_end):
    _check(ctx, lib().nb_set_j_range(ctx, int(j_begin), int(j_end)))


def nb_get_forces(ctx, buf):
    _check(ctx, lib().nb_get_forces(ctx, _ptr(buf)))
    return buf


def nb_set_forces(ctx, buf):
    _check(ctx, lib().nb_set_forces(ctx, _ptr(buf)))


def nb_get_launch(ctx):
    out = (_i64 * 5)()
    _check(ctx, lib().nb_get_launch(ctx, out))
    return dict(threads=out[0], jlanes=out[1], splits=out[2], ctas=out[3], tile=out[4])


def nb_probe_fp64_peak(ctx, iters=1 << 16):
    f, ms = _dbl(), C.c_float()
    _check(ctx, lib().nb_probe_fp64_peak(ctx, int(iters), C.byref(f), C.byref(ms)))
    return f.value, ms.value


def nb_set_debug(ctx, on=1):
    _check(ctx, lib().nb_set_debug(ctx, int(on)))


NB_STATIC_MAX_N = 65536


def _dev_ptr(x, dtype=np.float64, n=None):
    """Raw address of a contiguous CUDA tensor (None -> NULL): nb_force_static takes device pointers only."""
    if x is None:
        return None
    if not hasattr(x, "is_cuda") or not x.is_cuda:
        raise TypeError("nb_force_static takes CUDA tensors only (device pointers)")
    return _ptr(x, dtype, n)


def nb_force_static(pos, vel, acc_pred, mass, eps, active_idx, n_active, acc=None, jerk=None, snap=None, stream=None):
    """nb_force_static: the evaluation without a context and without any allocation (include/nb.h).  Every
    array is a CUDA tensor the caller owns, outputs included; nothing is allocated here either."""
    N, n = int(mass.shape[0]), int(n_active)
    if stream is not None and hasattr(stream, "cuda_stream"):
        stream = stream.cuda_stream
    err = C.create_string_buffer(512)
    rc = lib().nb_force_static(N, _dev_ptr(pos, n=3 * N), _dev_ptr(vel, n=3 * N), _dev_ptr(acc_pred, n=3 * N),
                               _dev_ptr(mass, n=N), float(eps), _dev_ptr(active_idx, np.int32, n if active_idx is not None else None),
                               n, _dev_ptr(acc, n=3 * n), _dev_ptr(jerk, n=3 * n), _dev_ptr(snap, n=3 * n),
                               _vp(stream or 0), err, len(err))
    if rc != NB_OK:
        raise NBError(rc, err.value.decode())
    return acc, jerk, snap


# ---------------------------------------------------------------------------- convenience wrapper
class NBody:
    """Owns one context; methods are the C calls with device tensors allocated for outputs."""

    def __init__(self, pos, vel, mass, eps, eta, dt_min=None, dt_max=None, eta_init=0.01, stream=None):
        torch = _torch()
        if not torch.cuda.is_available():
            raise RuntimeError("paper_1207_2367_b200 needs a CUDA device (sm_100a); there is no CPU path")
        self.N = int(mass.shape[0])
        if stream is None:
            stream = torch.cuda.current_stream()
        self._stream = stream
        self.ctx = nb_init(pos, vel, mass, eps, eta, stream)
        if dt_min is not None or dt_max is not None:
            nb_set_limits(self.ctx, dt_min if dt_min is not None else 2.0 ** -25,
                          dt_max if dt_max is not None else 2.0 ** -3, eta_init)

    def close(self):
        if getattr(self, "ctx", None):
            nb_free(self.ctx)
            self.ctx = None

    __del__ = close

    def sync(self):
        self._stream.synchronize()

    def startup(self):
        nb_startup(self.ctx)

    def next_block(self):
        return nb_next_block(self.ctx)

    def active(self, n_active):
        idx = _dev_empty((int(n_active),), _torch().int32)
        nb_get_active(self.ctx, idx)
        self.sync()
        return idx

    def predict(self, t):
        nb_predict(self.ctx, t)

    def force(self, active_idx=None, n_active=None):
        n = self.N if n_active is None and active_idx is None else (
            int(n_active) if n_active is not None else int(active_idx.shape[0]))
        acc, jerk, snap = _dev_empty((n, 3)), _dev_empty((n, 3)), _dev_empty((n, 3))
        nb_force(self.ctx, active_idx, n, acc, jerk, snap)
        return acc, jerk, snap

    def correct_and_step(self):
        nb_correct_and_step(self.ctx)

    def run_until(self, t_end):
        return nb_run_until(self.ctx, t_end)

    def run_steps(self, n, log=True):
        return nb_run_steps(self.ctx, n, log)

    def energy(self):
        return nb_energy(self.ctx)

    def state(self):
        pos, vel = _dev_empty((self.N, 3)), _dev_empty((self.N, 3))
        t, dt = _dev_empty((self.N,)), _dev_empty((self.N,))
        nb_get_state(self.ctx, pos, vel, t, dt)
        self.sync()
        return pos, vel, t, dt

    def derivs(self):
        out = [_dev_empty((self.N, 3)) for _ in range(4)]
        nb_get_derivs(self.ctx, *out)
        self.sync()
        return out

    def pred(self):
        out = [_dev_empty((self.N, 3)) for _ in range(3)]
        nb_get_pred(self.ctx, *out)
        self.sync()
        return out

    def stats(self):
        return nb_get_stats(self.ctx)
