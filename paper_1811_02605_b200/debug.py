"""Binding of include/mas_pcg_debug.h: the measurement probes bench.py uses for its per-kernel CUDA-event pass.
They live in lib/libmas_pcg_dbg.so (the product source compiled with -DMAS_PCG_DEBUG_PROBES), not in the
product library, so a handle used with them is created through that library."""
from __future__ import annotations

import ctypes

import numpy as np

from . import binding as B
from . import build as _build

_dbg = None
_dp = ctypes.POINTER(ctypes.c_double)


def lib_dbg():
    global _dbg
    if _dbg is None:
        if not _build.up_to_date():
            _build.build()
        L = B._prototypes(ctypes.CDLL(_build.LIB_DBG))
        vp = ctypes.c_void_p
        L.mas_pcg_dbg_profile.restype = ctypes.c_int
        L.mas_pcg_dbg_profile.argtypes = [vp, vp, vp, ctypes.c_int, vp, _dp]
        L.mas_pcg_dbg_mix_probe.restype = ctypes.c_int
        L.mas_pcg_dbg_mix_probe.argtypes = [vp, ctypes.c_int, ctypes.c_int, vp, _dp]
        _dbg = L
    return _dbg


class MasPcgProbe:
    """One operator created through the debug library; profile() and mix_probe() only."""

    def __init__(self, mesh, dt, nu_kind, nu, bc=(0, 0), options=(), precond=1):
        self.n = mesh.nr * mesh.nt * mesh.np_
        self._h = B.mas_pcg_create((mesh.nr, mesh.nt, mesh.np_), mesh.metric_arrays(), dt, nu_kind, nu, bc, L=lib_dbg())
        if precond != 1:
            B.mas_pcg_set_preconditioner(self._h, precond, L=lib_dbg())
        for name, value in options:
            B.mas_pcg_set_option(self._h, name, value, L=lib_dbg())

    def close(self):
        if getattr(self, "_h", None):
            B.mas_pcg_destroy(self._h, L=lib_dbg())
            self._h = None

    __del__ = close

    def profile(self, b, x, nit, stream_ptr=0):
        """Per-kernel CUDA-event timing of nit iterations: {k1_ms, k2_ms, k1_min_ms, k2_min_ms}."""
        out = np.zeros(4)
        st = lib_dbg().mas_pcg_dbg_profile(self._h, b.data_ptr(), x.data_ptr(), int(nit), stream_ptr, out.ctypes.data_as(_dp))
        if st != B.MAS_OK:
            raise B.MasError(st, "mas_pcg_dbg_profile")
        return {"k1_ms": out[0], "k2_ms": out[1], "k1_min_ms": out[2], "k2_min_ms": out[3]}

    def mix_probe(self, which, reps=50, stream_ptr=0) -> float:
        """ms per launch of a trivial linear kernel with K1's (which = 6, or 5 without q) or K2's (3) DRAM mix."""
        out = ctypes.c_double(0.0)
        st = lib_dbg().mas_pcg_dbg_mix_probe(self._h, int(which), int(reps), stream_ptr, ctypes.byref(out))
        if st != B.MAS_OK:
            raise B.MasError(st, "mas_pcg_dbg_mix_probe")
        return out.value

    def stats(self):
        return B.mas_pcg_stats(self._h, L=lib_dbg())
