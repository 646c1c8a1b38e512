"""Thin ctypes binding of include/mas_pcg.h: same names, argument marshalling only.

Every step of the numerical path runs in the CUDA kernels of lib/libmas_pcg.so.  There is no
Python or CPU fallback: if the library is missing (and cannot be built) importing fails loudly,
and without a CUDA device `mas_pcg_create` returns MAS_ECUDA.
PyTorch is used by callers for device buffers and streams only; this module takes raw pointers.
"""
from __future__ import annotations

import ctypes
import os

import numpy as np

from . import build as _build

MAS_OK, MAS_MAXIT, MAS_EINVAL, MAS_ENOMEM, MAS_ECUDA, MAS_EBREAKDOWN = 0, 1, -1, -2, -3, -4
MAS_BC_DIRICHLET, MAS_BC_NEUMANN = 0, 1

_dp = ctypes.POINTER(ctypes.c_double)


class mas_grid_t(ctypes.Structure):
    _fields_ = [("nr", ctypes.c_int), ("nt", ctypes.c_int), ("np", ctypes.c_int)]


class mas_metric_t(ctypes.Structure):
    _fields_ = [(n, _dp) for n in ("r_c", "dr_c", "r_f", "dr_f", "sin_c", "dth_c", "sin_f", "dth_f",
                                   "dph_c", "dph_f")]


class mas_bc_t(ctypes.Structure):
    _fields_ = [("r_inner", ctypes.c_int), ("r_outer", ctypes.c_int)]


class mas_nu_t(ctypes.Structure):
    _fields_ = [("kind", ctypes.c_int), ("v", _dp)]


def _load():
    path = _build.LIB
    if not _build.up_to_date():
        try:
            path = _build.build()
        except Exception as e:  # no nvcc on this machine: use the shipped .so if there is one
            if not os.path.exists(path):
                raise ImportError(f"libmas_pcg.so is missing and could not be built: {e}") from e
    L = ctypes.CDLL(path)
    vp = ctypes.c_void_p
    L.mas_pcg_create.restype = ctypes.c_int
    L.mas_pcg_create.argtypes = [ctypes.POINTER(mas_grid_t), ctypes.POINTER(mas_metric_t), ctypes.c_double,
                                 ctypes.POINTER(mas_nu_t), ctypes.POINTER(mas_bc_t), ctypes.POINTER(vp)]
    L.mas_pcg_set_dt.restype = ctypes.c_int
    L.mas_pcg_set_dt.argtypes = [vp, ctypes.c_double, vp]
    for name in ("mas_pcg_solve", "mas_pcg_solve_host"):
        f = getattr(L, name)
        f.restype = ctypes.c_int
        f.argtypes = [vp, vp, vp, ctypes.c_double, ctypes.c_int, vp, ctypes.POINTER(ctypes.c_int), _dp]
    L.mas_pcg_apply.restype = ctypes.c_int
    L.mas_pcg_apply.argtypes = [vp, vp, vp, vp]
    L.mas_pcg_profile.restype = ctypes.c_int
    L.mas_pcg_profile.argtypes = [vp, vp, vp, ctypes.c_int, vp, _dp]
    L.mas_pcg_lop.restype = ctypes.c_int
    L.mas_pcg_lop.argtypes = [vp, vp, vp, vp]
    L.mas_pcg_lambda_max.restype = ctypes.c_int
    L.mas_pcg_lambda_max.argtypes = [vp, _dp]
    L.mas_sts_stages.restype = ctypes.c_int
    L.mas_sts_stages.argtypes = [vp, ctypes.c_double, ctypes.POINTER(ctypes.c_int)]
    L.mas_sts_advance.restype = ctypes.c_int
    L.mas_sts_advance.argtypes = [vp, vp, ctypes.c_double, ctypes.c_int, vp]
    L.mas_pcg_mix_probe.restype = ctypes.c_int
    L.mas_pcg_mix_probe.argtypes = [vp, ctypes.c_int, ctypes.c_int, vp, _dp]
    L.mas_pcg_stats.restype = ctypes.c_int
    L.mas_pcg_stats.argtypes = [vp, ctypes.POINTER(ctypes.c_longlong)]
    L.mas_pcg_set_option.restype = ctypes.c_int
    L.mas_pcg_set_option.argtypes = [vp, ctypes.c_char_p, ctypes.c_int]
    L.mas_pcg_destroy.restype = None
    L.mas_pcg_destroy.argtypes = [vp]
    L.mas_pcg_strerror.restype = ctypes.c_char_p
    L.mas_pcg_strerror.argtypes = [ctypes.c_int]
    return L


_lib = None


def lib():
    global _lib
    if _lib is None:
        _lib = _load()
    return _lib


def mas_pcg_strerror(status: int) -> str:
    return lib().mas_pcg_strerror(int(status)).decode()


class MasError(RuntimeError):
    def __init__(self, status, where):
        super().__init__(f"{where}: {mas_pcg_strerror(status)} ({status})")
        self.status = status


def _f64(a):
    return np.ascontiguousarray(a, dtype=np.float64)


def mas_pcg_create(grid, metric_arrays, dt, nu_kind, nu, bc=(0, 0)) -> int:
    """grid = (nr, nt, np); metric_arrays = the ten HOST arrays of mas_metric_t in declaration order.
    Returns the opaque handle (an int); raises MasError on a negative status."""
    arrs = [_f64(a) for a in metric_arrays]
    nu_h = _f64(nu)
    g = mas_grid_t(*[int(v) for v in grid])
    m = mas_metric_t(*[a.ctypes.data_as(_dp) for a in arrs])
    n = mas_nu_t(int(nu_kind), nu_h.ctypes.data_as(_dp))
    b = mas_bc_t(int(bc[0]), int(bc[1]))
    out = ctypes.c_void_p()
    st = lib().mas_pcg_create(ctypes.byref(g), ctypes.byref(m), float(dt), ctypes.byref(n), ctypes.byref(b),
                              ctypes.byref(out))
    if st != MAS_OK:
        raise MasError(st, "mas_pcg_create")
    return out.value


def mas_pcg_destroy(handle):
    lib().mas_pcg_destroy(handle)


def mas_pcg_set_dt(handle, dt, stream=0):
    st = lib().mas_pcg_set_dt(handle, float(dt), stream)
    if st != MAS_OK:
        raise MasError(st, "mas_pcg_set_dt")


def mas_pcg_set_option(handle, name: str, value: int):
    st = lib().mas_pcg_set_option(handle, name.encode(), int(value))
    if st != MAS_OK:
        raise MasError(st, f"mas_pcg_set_option({name}={value})")


def mas_pcg_apply(handle, x_ptr, y_ptr, stream=0):
    st = lib().mas_pcg_apply(handle, x_ptr, y_ptr, stream)
    if st != MAS_OK:
        raise MasError(st, "mas_pcg_apply")


def _solve(fn, where, handle, b_ptr, x_ptr, rtol, maxit, stream, want_hist):
    it = ctypes.c_int(0)
    hist = np.empty(maxit + 1) if want_hist else None
    st = fn(handle, b_ptr, x_ptr, float(rtol), int(maxit), stream, ctypes.byref(it),
            hist.ctypes.data_as(_dp) if want_hist else None)
    if st < 0:
        err = MasError(st, where)
        if st == MAS_EBREAKDOWN:                 # x holds the last iterate; the count and history are meaningful
            err.iters = it.value
            err.hist = hist[: it.value + 1].copy() if want_hist else None
        raise err
    return st, it.value, (hist[: it.value + 1].copy() if want_hist else None)


def mas_pcg_solve(handle, b_ptr, x_ptr, rtol, maxit, stream=0, want_hist=True):
    """DEVICE pointers (ints).  Returns (status, iters, hist[0..iters])."""
    return _solve(lib().mas_pcg_solve, "mas_pcg_solve", handle, b_ptr, x_ptr, rtol, maxit, stream, want_hist)


def mas_pcg_solve_host(handle, b_ptr, x_ptr, rtol, maxit, stream=0, want_hist=True):
    """HOST pointers (ints); copies are inside the call."""
    return _solve(lib().mas_pcg_solve_host, "mas_pcg_solve_host", handle, b_ptr, x_ptr, rtol, maxit, stream,
                  want_hist)


def mas_pcg_profile(handle, b_ptr, x_ptr, nit, stream=0):
    """Per-kernel CUDA-event timing of nit iterations: {k1_ms, k2_ms, k1_min_ms, k2_min_ms}."""
    out = np.zeros(4)
    st = lib().mas_pcg_profile(handle, b_ptr, x_ptr, int(nit), stream, out.ctypes.data_as(_dp))
    if st != MAS_OK:
        raise MasError(st, "mas_pcg_profile")
    return {"k1_ms": out[0], "k2_ms": out[1], "k1_min_ms": out[2], "k2_min_ms": out[3]}


def mas_pcg_lop(handle, u_ptr, y_ptr, stream=0):
    st = lib().mas_pcg_lop(handle, u_ptr, y_ptr, stream)
    if st != MAS_OK:
        raise MasError(st, "mas_pcg_lop")


def mas_pcg_lambda_max(handle) -> float:
    out = ctypes.c_double(0.0)
    st = lib().mas_pcg_lambda_max(handle, ctypes.byref(out))
    if st != MAS_OK:
        raise MasError(st, "mas_pcg_lambda_max")
    return out.value


def mas_sts_stages(handle, tau) -> int:
    out = ctypes.c_int(0)
    st = lib().mas_sts_stages(handle, float(tau), ctypes.byref(out))
    if st != MAS_OK:
        raise MasError(st, "mas_sts_stages")
    return out.value


def mas_sts_advance(handle, u_ptr, tau, s, stream=0):
    st = lib().mas_sts_advance(handle, u_ptr, float(tau), int(s), stream)
    if st != MAS_OK:
        raise MasError(st, "mas_sts_advance")


def mas_pcg_mix_probe(handle, which, reps, stream=0) -> float:
    """ms per launch of a trivial linear kernel with K1's (which=6) or K2's (which=3) DRAM read/write mix."""
    out = ctypes.c_double(0.0)
    st = lib().mas_pcg_mix_probe(handle, int(which), int(reps), stream, ctypes.byref(out))
    if st != MAS_OK:
        raise MasError(st, "mas_pcg_mix_probe")
    return out.value


def mas_pcg_stats(handle):
    out = (ctypes.c_longlong * 8)()
    st = lib().mas_pcg_stats(handle, out)
    if st != MAS_OK:
        raise MasError(st, "mas_pcg_stats")
    return {"loop_launches": out[0], "other_launches": out[1], "loop_mode": out[2], "bytes_per_cell_iter": out[3],
            "k1_doubles_per_cell": out[4], "k2_doubles_per_cell": out[5]}
