"""ctypes loader for the ORACLE (oracle/mas_pcg_ref.c).  Test infrastructure, not product code.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may
import this module.  It imports nothing from the CUDA package.
"""
from __future__ import annotations

import ctypes
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "mas_pcg_ref.c")
_LIB = os.path.join(_HERE, "libmas_pcg_ref.so")

REF_OK, REF_MAXIT, REF_EINVAL, REF_ENOMEM, REF_EBREAKDOWN = 0, 1, -1, -2, -4

_dp = ctypes.POINTER(ctypes.c_double)


def build(force: bool = False) -> str:
    """gcc -O2, one thread, no fast-math, no FMA contraction (plain IEEE fp64 + long double sums)."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        tmp = f"{_LIB}.{os.getpid()}.tmp"
        subprocess.check_call(["gcc", "-std=c99", "-O2", "-ffp-contract=off", "-fPIC", "-shared",
                               "-o", tmp, _SRC, "-lm"])
        os.replace(tmp, _LIB)
    return _LIB


_lib = None


def lib():
    global _lib
    if _lib is None:
        L = ctypes.CDLL(build())
        L.mas_ref_create.restype = ctypes.c_void_p
        L.mas_ref_create.argtypes = [ctypes.c_int] * 3 + [_dp] * 10 + [ctypes.c_double, ctypes.c_int, _dp,
                                                                    ctypes.c_int, ctypes.c_int]
        L.mas_ref_destroy.argtypes = [ctypes.c_void_p]
        L.mas_ref_set_dt.argtypes = [ctypes.c_void_p, ctypes.c_double]
        for name in ("mas_ref_volume", "mas_ref_diag"):
            getattr(L, name).argtypes = [ctypes.c_void_p, _dp]
        L.mas_ref_apply.argtypes = [ctypes.c_void_p, _dp, _dp]
        L.mas_ref_stiffness_max.restype = ctypes.c_double
        L.mas_ref_stiffness_max.argtypes = [ctypes.c_void_p]
        L.mas_ref_pcg.restype = ctypes.c_int
        L.mas_ref_pcg.argtypes = [ctypes.c_void_p, _dp, _dp, ctypes.c_double, ctypes.c_int,
                                  ctypes.POINTER(ctypes.c_int), _dp]
        L.mas_ref_pcg_multi.restype = ctypes.c_int
        L.mas_ref_pcg_multi.argtypes = [ctypes.c_void_p, ctypes.c_int, _dp, _dp, ctypes.c_double, ctypes.c_int,
                                        ctypes.POINTER(ctypes.c_int), ctypes.POINTER(ctypes.c_int), _dp]
        L.mas_ref_lop.argtypes = [ctypes.c_void_p, _dp, _dp]
        L.mas_ref_lambda_max_bound.restype = ctypes.c_double
        L.mas_ref_lambda_max_bound.argtypes = [ctypes.c_void_p]
        L.mas_ref_sts.restype = ctypes.c_int
        L.mas_ref_sts.argtypes = [ctypes.c_void_p, _dp, ctypes.c_double, ctypes.c_int]
        L.mas_ref_pc2_create.restype = ctypes.c_void_p
        L.mas_ref_pc2_create.argtypes = [ctypes.c_void_p, ctypes.c_int, ctypes.c_int, ctypes.c_int]
        L.mas_ref_pc2_destroy.argtypes = [ctypes.c_void_p]
        L.mas_ref_pc2_apply.argtypes = [ctypes.c_void_p, _dp, _dp]
        L.mas_ref_pc2_dense_factors.argtypes = [ctypes.c_void_p, _dp, _dp]
        L.mas_ref_pcg_pc2.restype = ctypes.c_int
        L.mas_ref_pcg_pc2.argtypes = [ctypes.c_void_p, ctypes.c_void_p, _dp, _dp, ctypes.c_double, ctypes.c_int,
                                      ctypes.POINTER(ctypes.c_int), _dp]
        _lib = L
    return _lib


def _p(a: np.ndarray):
    assert a.dtype == np.float64 and a.flags.c_contiguous
    return a.ctypes.data_as(_dp)


class RefOperator:
    """The oracle's operator for one mesh / nu / boundary kinds / dt."""

    def __init__(self, mesh, dt: float, nu_kind: int, nu: np.ndarray, bc=(0, 0)):
        self.shape = (mesh.nr, mesh.nt, mesh.np_)
        arrs = [np.ascontiguousarray(a, dtype=np.float64) for a in mesh.metric_arrays()]
        nu = np.ascontiguousarray(nu, dtype=np.float64)
        self._h = lib().mas_ref_create(mesh.nr, mesh.nt, mesh.np_, *[_p(a) for a in arrs],
                                       float(dt), int(nu_kind), _p(nu), int(bc[0]), int(bc[1]))
        if not self._h:
            raise ValueError("mas_ref_create rejected its arguments")

    def close(self):
        if self._h:
            lib().mas_ref_destroy(self._h)
            self._h = None

    __del__ = close

    def set_dt(self, dt: float):
        lib().mas_ref_set_dt(self._h, float(dt))

    def volume(self) -> np.ndarray:
        v = np.empty(self.shape)
        lib().mas_ref_volume(self._h, _p(v))
        return v

    def diag(self) -> np.ndarray:
        d = np.empty(self.shape)
        lib().mas_ref_diag(self._h, _p(d))
        return d

    def apply(self, u: np.ndarray) -> np.ndarray:
        """A_sym u."""
        u = np.ascontiguousarray(u, dtype=np.float64).reshape(self.shape)
        y = np.empty(self.shape)
        lib().mas_ref_apply(self._h, _p(u), _p(y))
        return y

    def apply_phys(self, u: np.ndarray) -> np.ndarray:
        """A_phys u = (A_sym u) / V   -- the caller-facing 'A = I - dt nu lap'."""
        return self.apply(u) / self.volume()

    def stiffness_max(self) -> float:
        return float(lib().mas_ref_stiffness_max(self._h))

    def pcg(self, b_phys: np.ndarray, x0: np.ndarray | None, rtol: float, maxit: int):
        """Returns (status, iters, x, hist[0..iters])."""
        b = np.ascontiguousarray(b_phys, dtype=np.float64).reshape(self.shape)
        x = np.zeros(self.shape) if x0 is None else np.array(x0, dtype=np.float64, order="C").reshape(self.shape)
        hist = np.full(maxit + 1, np.nan)
        it = ctypes.c_int(0)
        st = lib().mas_ref_pcg(self._h, _p(b), _p(x), float(rtol), int(maxit), ctypes.byref(it), _p(hist))
        return st, it.value, x, hist[: it.value + 1].copy()

    def pcg_multi(self, b_phys: np.ndarray, x0: np.ndarray | None, rtol: float, maxit: int):
        """nrhs independent solves sharing the operator; b_phys has shape (nrhs, nr, nt, np).
        Returns (worst status, [status_j], [iters_j], x (nrhs, ...), [hist_j[0..iters_j]])."""
        b = np.ascontiguousarray(b_phys, dtype=np.float64)
        nrhs = b.shape[0]
        assert b.shape[1:] == self.shape
        x = np.zeros_like(b) if x0 is None else np.array(x0, dtype=np.float64, order="C").reshape(b.shape)
        hist = np.full((nrhs, maxit + 1), np.nan)
        it = (ctypes.c_int * nrhs)()
        st = (ctypes.c_int * nrhs)()
        worst = lib().mas_ref_pcg_multi(self._h, nrhs, _p(b), _p(x), float(rtol), int(maxit), it, st, _p(hist))
        return worst, list(st), list(it), x, [hist[j, : it[j] + 1].copy() for j in range(nrhs)]

    # ---- NEXT-1: explicit operator and RKL2 super time stepping ----
    def lop(self, u: np.ndarray) -> np.ndarray:
        """M u = -(1/V) sum_f G_f (u_c - u_nb): the FD form of div(nu grad u)."""
        u = np.ascontiguousarray(u, dtype=np.float64).reshape(self.shape)
        y = np.empty(self.shape)
        lib().mas_ref_lop(self._h, _p(u), _p(y))
        return y

    def lambda_max_bound(self) -> float:
        return float(lib().mas_ref_lambda_max_bound(self._h))

    def sts(self, u: np.ndarray, tau: float, s: int) -> np.ndarray:
        """One RKL2 super-step of size tau with s stages; returns the new field."""
        y = np.array(u, dtype=np.float64, order="C").reshape(self.shape)
        st = lib().mas_ref_sts(self._h, _p(y), float(tau), int(s))
        if st != REF_OK:
            raise ValueError(f"mas_ref_sts status {st}")
        return y

    # ---- NEXT-4: PC2, block-Jacobi ILU(0) ----
    def pc2(self, boxes=(0, 0, 0)) -> "RefPc2":
        """The block-Jacobi ILU(0) preconditioner of this operator AT ITS CURRENT dt; boxes = (bi, bj, bk) cells
        per box in r, theta, phi (0 = the whole extent)."""
        return RefPc2(self, boxes)

    def pcg_pc2(self, pc: "RefPc2", b_phys: np.ndarray, x0: np.ndarray | None, rtol: float, maxit: int):
        """PCG with z = M^-1 r, M = pc.  Returns (status, iters, x, hist[0..iters])."""
        b = np.ascontiguousarray(b_phys, dtype=np.float64).reshape(self.shape)
        x = np.zeros(self.shape) if x0 is None else np.array(x0, dtype=np.float64, order="C").reshape(self.shape)
        hist = np.full(maxit + 1, np.nan)
        it = ctypes.c_int(0)
        st = lib().mas_ref_pcg_pc2(self._h, pc._h, _p(b), _p(x), float(rtol), int(maxit), ctypes.byref(it), _p(hist))
        return st, it.value, x, hist[: it.value + 1].copy()

    def dense(self) -> np.ndarray:
        """Dense A_sym, column by column from unit vectors (tiny meshes only)."""
        n = int(np.prod(self.shape))
        assert n <= 4096
        A = np.empty((n, n))
        e = np.zeros(n)
        for c in range(n):
            e[c] = 1.0
            A[:, c] = self.apply(e.reshape(self.shape)).ravel()
            e[c] = 0.0
        return A


class RefPc2:
    """PC2: zero-fill ILU of the block-diagonal part of A_sym in a box partition."""

    def __init__(self, op: RefOperator, boxes=(0, 0, 0)):
        self.shape = op.shape
        self._h = lib().mas_ref_pc2_create(op._h, int(boxes[0]), int(boxes[1]), int(boxes[2]))
        if not self._h:
            raise MemoryError("mas_ref_pc2_create failed")

    def close(self):
        if self._h:
            lib().mas_ref_pc2_destroy(self._h)
            self._h = None

    __del__ = close

    def apply(self, r: np.ndarray) -> np.ndarray:
        """z = M^-1 r."""
        r = np.ascontiguousarray(r, dtype=np.float64).reshape(self.shape)
        z = np.empty(self.shape)
        lib().mas_ref_pc2_apply(self._h, _p(r), _p(z))
        return z

    def dense_factors(self):
        """(L, U) as dense n x n arrays (tiny meshes only)."""
        n = int(np.prod(self.shape))
        assert n <= 4096
        Ld, Ud = np.empty((n, n)), np.empty((n, n))
        lib().mas_ref_pc2_dense_factors(self._h, _p(Ld), _p(Ud))
        return Ld, Ud
