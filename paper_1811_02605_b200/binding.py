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
MAS_ETOOBIG = -5
MAS_PCG_STATIC_MAX_CELLS = 1 << 25   # include/mas_pcg.h: the largest mesh mas_pcg_residual_static serves
MAS_BC_DIRICHLET, MAS_BC_NEUMANN = 0, 1
MAX_RHS = 3

_dp = ctypes.POINTER(ctypes.c_double)
_ip = ctypes.POINTER(ctypes.c_int)
_vpp = ctypes.POINTER(ctypes.c_void_p)


class mas_grid_t(ctypes.Structure):
    _fields_ = [("nr", ctypes.c_int), ("nt", ctypes.c_int), ("np", ctypes.c_int)]


class mas_metric_t(ctypes.Structure):
    _fields_ = [(n, _dp) for n in ("r_c", "dr_c", "r_f", "dr_f", "sin_c", "dth_c", "sin_f", "dth_f",
                                   "dph_c", "dph_f")]


class mas_bc_t(ctypes.Structure):
    _fields_ = [("r_inner", ctypes.c_int), ("r_outer", ctypes.c_int)]


class mas_nu_t(ctypes.Structure):
    _fields_ = [("kind", ctypes.c_int), ("v", _dp)]


def _prototypes(L):
    """argtypes / restype of every include/mas_pcg.h entry point on a loaded library."""
    vp, ci, cd = ctypes.c_void_p, ctypes.c_int, ctypes.c_double
    create_args = [ctypes.POINTER(mas_grid_t), ctypes.POINTER(mas_metric_t), cd, ctypes.POINTER(mas_nu_t),
                   ctypes.POINTER(mas_bc_t)]
    sig = {
        "mas_pcg_create": (ci, create_args + [_vpp]),
        "mas_pcg_set_dt": (ci, [vp, cd, vp]),
        "mas_pcg_solve": (ci, [vp, vp, vp, cd, ci, vp, _ip, _dp]),
        "mas_pcg_solve_host": (ci, [vp, vp, vp, cd, ci, vp, _ip, _dp]),
        "mas_pcg_solve_multi": (ci, [vp, ci, _vpp, _vpp, cd, ci, vp, _ip, _ip, _dp]),
        "mas_pcg_apply": (ci, [vp, vp, vp, vp]),
        "mas_pcg_residual_static": (ci, [vp, vp, vp, vp, vp, vp]),
        "mas_pcg_lop": (ci, [vp, vp, vp, vp]),
        "mas_pcg_lambda_max": (ci, [vp, _dp]),
        "mas_sts_stages": (ci, [vp, cd, _ip]),
        "mas_sts_advance": (ci, [vp, vp, cd, ci, vp]),
        "mas_pcg_stats": (ci, [vp, ctypes.POINTER(ctypes.c_longlong)]),
        "mas_pcg_set_option": (ci, [vp, ctypes.c_char_p, ci]),
        "mas_pcg_set_preconditioner": (ci, [vp, ci, ci, ci, ci]),
        "mas_pcg_destroy": (None, [vp]),
        "mas_pcg_strerror": (ctypes.c_char_p, [ci]),
        "mas_pcg_slabs_create": (ci, create_args + [ci, _ip, _vpp]),
        "mas_pcg_slabs_set_dt": (ci, [vp, cd, vp]),
        "mas_pcg_slabs_set_option": (ci, [vp, ctypes.c_char_p, ci]),
        "mas_pcg_slabs_set_preconditioner": (ci, [vp, ci, ci, ci, ci]),
        "mas_pcg_slabs_solve": (ci, [vp, _vpp, _vpp, cd, ci, vp, _ip, _dp]),
        "mas_pcg_slabs_stats": (ci, [vp, ctypes.POINTER(ctypes.c_longlong)]),
        "mas_pcg_slabs_destroy": (None, [vp]),
    }
    for name, (res, args) in sig.items():
        f = getattr(L, name)
        f.restype = res
        f.argtypes = args
    return L


def _load():
    path = _build.LIB
    if not _build.up_to_date():
        try:
            path = _build.build()
        except Exception as e:  # no nvcc on this machine: use the shipped .so if there is one
            if not os.path.exists(path):
                raise ImportError(f"libmas_pcg.so is missing and could not be built: {e}") from e
    return _prototypes(ctypes.CDLL(path))


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


def _create_args(grid, metric_arrays, dt, nu_kind, nu, bc):
    arrs = [_f64(a) for a in metric_arrays]
    nu_h = _f64(nu)
    g = mas_grid_t(*[int(v) for v in grid])
    m = mas_metric_t(*[a.ctypes.data_as(_dp) for a in arrs])
    n = mas_nu_t(int(nu_kind), nu_h.ctypes.data_as(_dp))
    b = mas_bc_t(int(bc[0]), int(bc[1]))
    keep = (arrs, nu_h, g, m, n, b)              # alive until the call returns
    return keep, (ctypes.byref(g), ctypes.byref(m), float(dt), ctypes.byref(n), ctypes.byref(b))


def mas_pcg_create(grid, metric_arrays, dt, nu_kind, nu, bc=(0, 0), L=None) -> int:
    """grid = (nr, nt, np); metric_arrays = the ten HOST arrays of mas_metric_t in declaration order.
    Returns the opaque handle (an int); raises MasError on a negative status."""
    keep, args = _create_args(grid, metric_arrays, dt, nu_kind, nu, bc)
    out = ctypes.c_void_p()
    st = (L or lib()).mas_pcg_create(*args, ctypes.byref(out))
    if st != MAS_OK:
        raise MasError(st, "mas_pcg_create")
    return out.value


def mas_pcg_destroy(handle, L=None):
    (L or lib()).mas_pcg_destroy(handle)


def mas_pcg_set_dt(handle, dt, stream=0):
    st = lib().mas_pcg_set_dt(handle, float(dt), stream)
    if st != MAS_OK:
        raise MasError(st, "mas_pcg_set_dt")


def mas_pcg_set_option(handle, name: str, value: int, L=None):
    st = (L or lib()).mas_pcg_set_option(handle, name.encode(), int(value))
    if st != MAS_OK:
        raise MasError(st, f"mas_pcg_set_option({name}={value})")


MAS_PC1, MAS_PC2 = 1, 2


def mas_pcg_set_preconditioner(handle, kind: int, boxes=(1, 1, 0), L=None):
    st = (L or lib()).mas_pcg_set_preconditioner(handle, int(kind), int(boxes[0]), int(boxes[1]), int(boxes[2]))
    if st != MAS_OK:
        raise MasError(st, f"mas_pcg_set_preconditioner({kind}, {tuple(boxes)})")


def mas_pcg_apply(handle, x_ptr, y_ptr, stream=0):
    st = lib().mas_pcg_apply(handle, x_ptr, y_ptr, stream)
    if st != MAS_OK:
        raise MasError(st, "mas_pcg_apply")


def mas_pcg_residual_static(handle, b_ptr, ax_ptr, r_ptr, sums_ptr, stream=0):
    """r = V.b - ax and the three sums (||V.b||^2, ||r||^2, r.D^-1 r) into the DEVICE array at sums_ptr, for callers
    that must not allocate device memory (include/mas_pcg.h has the full contract: the scratch is a fixed array in
    the library, N <= MAS_PCG_STATIC_MAX_CELLS, calls that overlap on the GPU race, make the first call on a device
    before any stream capture).  Enqueues only; raises MasError on a non-zero status (MAS_ETOOBIG past the limit)."""
    st = lib().mas_pcg_residual_static(handle, b_ptr, ax_ptr, r_ptr, sums_ptr, stream)
    if st != MAS_OK:
        raise MasError(st, "mas_pcg_residual_static")


def _raise(st, where, iters=None, hist=None):
    err = MasError(st, where)
    if st == MAS_EBREAKDOWN:                     # x holds the last iterate; the count and history are meaningful
        err.iters, err.hist = iters, hist
    raise err


def _solve(fn, where, handle, b_ptr, x_ptr, rtol, maxit, stream, want_hist):
    it = ctypes.c_int(0)
    hist = np.empty(maxit + 1) if want_hist else None
    st = fn(handle, b_ptr, x_ptr, float(rtol), int(maxit), stream, ctypes.byref(it),
            hist.ctypes.data_as(_dp) if want_hist else None)
    if st < 0:
        _raise(st, where, it.value, hist[: it.value + 1].copy() if want_hist else None)
    return st, it.value, (hist[: it.value + 1].copy() if want_hist else None)


def mas_pcg_solve(handle, b_ptr, x_ptr, rtol, maxit, stream=0, want_hist=True):
    """DEVICE pointers (ints).  Returns (status, iters, hist[0..iters])."""
    return _solve(lib().mas_pcg_solve, "mas_pcg_solve", handle, b_ptr, x_ptr, rtol, maxit, stream, want_hist)


def mas_pcg_solve_host(handle, b_ptr, x_ptr, rtol, maxit, stream=0, want_hist=True):
    """HOST pointers (ints); copies are inside the call."""
    return _solve(lib().mas_pcg_solve_host, "mas_pcg_solve_host", handle, b_ptr, x_ptr, rtol, maxit, stream,
                  want_hist)


def _ptr_array(ptrs):
    return (ctypes.c_void_p * len(ptrs))(*[int(p) for p in ptrs])


def mas_pcg_solve_multi(handle, b_ptrs, x_ptrs, rtol, maxit, stream=0, want_hist=True):
    """nrhs = len(b_ptrs) <= 3 DEVICE pointers each.  Returns (worst status, [status_j], [iters_j], [hist_j]);
    raises MasError only on argument / runtime errors (a per-right-hand-side breakdown is reported in status_j)."""
    nrhs = len(b_ptrs)
    it = (ctypes.c_int * nrhs)()
    sj = (ctypes.c_int * nrhs)()
    hist = np.empty((nrhs, maxit + 1)) if want_hist else None
    st = lib().mas_pcg_solve_multi(handle, nrhs, _ptr_array(b_ptrs), _ptr_array(x_ptrs), float(rtol), int(maxit),
                                   stream, it, sj, hist.ctypes.data_as(_dp) if want_hist else None)
    if st < 0 and st != MAS_EBREAKDOWN:
        raise MasError(st, "mas_pcg_solve_multi")
    hists = [hist[j, : it[j] + 1].copy() for j in range(nrhs)] if want_hist else None
    return st, list(sj), list(it), hists


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


def _stats_dict(out):
    return {"loop_launches": out[0], "other_launches": out[1], "loop_mode": out[2], "bytes_per_cell_iter": out[3],
            "k1_doubles_per_cell": out[4], "k2_doubles_per_cell": out[5], "persistent_grid_or_slabs": out[6],
            "coop_refused": out[7]}


def mas_pcg_stats(handle, L=None):
    out = (ctypes.c_longlong * 8)()
    st = (L or lib()).mas_pcg_stats(handle, out)
    if st != MAS_OK:
        raise MasError(st, "mas_pcg_stats")
    return _stats_dict(out)


# ---- NEXT-3: r-slab groups ----
def mas_pcg_slabs_create(grid, metric_arrays, dt, nu_kind, nu, bc, i_split) -> int:
    keep, args = _create_args(grid, metric_arrays, dt, nu_kind, nu, bc)
    split = (ctypes.c_int * len(i_split))(*[int(v) for v in i_split])
    out = ctypes.c_void_p()
    st = lib().mas_pcg_slabs_create(*args, len(i_split) - 1, split, ctypes.byref(out))
    if st != MAS_OK:
        raise MasError(st, "mas_pcg_slabs_create")
    return out.value


def mas_pcg_slabs_destroy(handle):
    lib().mas_pcg_slabs_destroy(handle)


def mas_pcg_slabs_set_dt(handle, dt, stream=0):
    st = lib().mas_pcg_slabs_set_dt(handle, float(dt), stream)
    if st != MAS_OK:
        raise MasError(st, "mas_pcg_slabs_set_dt")


def mas_pcg_slabs_set_preconditioner(handle, kind: int, boxes=(1, 1, 0)):
    st = lib().mas_pcg_slabs_set_preconditioner(handle, int(kind), int(boxes[0]), int(boxes[1]), int(boxes[2]))
    if st != MAS_OK:
        raise MasError(st, f"mas_pcg_slabs_set_preconditioner({kind}, {tuple(boxes)})")


def mas_pcg_slabs_set_option(handle, name: str, value: int):
    st = lib().mas_pcg_slabs_set_option(handle, name.encode(), int(value))
    if st != MAS_OK:
        raise MasError(st, f"mas_pcg_slabs_set_option({name}={value})")


def mas_pcg_slabs_solve(handle, b_ptrs, x_ptrs, rtol, maxit, stream=0, want_hist=True):
    it = ctypes.c_int(0)
    hist = np.empty(maxit + 1) if want_hist else None
    st = lib().mas_pcg_slabs_solve(handle, _ptr_array(b_ptrs), _ptr_array(x_ptrs), float(rtol), int(maxit), stream,
                                   ctypes.byref(it), hist.ctypes.data_as(_dp) if want_hist else None)
    if st < 0:
        _raise(st, "mas_pcg_slabs_solve", it.value, hist[: it.value + 1].copy() if want_hist else None)
    return st, it.value, (hist[: it.value + 1].copy() if want_hist else None)


def mas_pcg_slabs_stats(handle):
    out = (ctypes.c_longlong * 8)()
    st = lib().mas_pcg_slabs_stats(handle, out)
    if st != MAS_OK:
        raise MasError(st, "mas_pcg_slabs_stats")
    return _stats_dict(out)
