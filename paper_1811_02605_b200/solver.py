"""MasPcg / MasPcgSlabs: torch-tensor front ends of the C ABI (argument marshalling only)."""
from __future__ import annotations

import torch

from . import binding as B


def _stream_ptr(stream=None) -> int:
    s = torch.cuda.current_stream() if stream is None else stream
    return int(s.cuda_stream)


def _dev_ptr(t: torch.Tensor, n: int) -> int:
    if not (t.is_cuda and t.dtype == torch.float64 and t.is_contiguous() and t.numel() == n):
        raise ValueError(f"need a contiguous CUDA float64 tensor with {n} elements")
    return t.data_ptr()


class MasPcg:
    """One operator (mesh, nu, boundary kinds, dt) on the current CUDA device."""

    def __init__(self, mesh, dt, nu_kind, nu, bc=(0, 0)):
        if not torch.cuda.is_available():
            raise RuntimeError("MasPcg needs a CUDA device (there is no CPU fallback)")
        self.shape = (mesh.nr, mesh.nt, mesh.np_)
        self.n = mesh.nr * mesh.nt * mesh.np_
        self._h = B.mas_pcg_create(self.shape, mesh.metric_arrays(), dt, nu_kind, nu, bc)

    def close(self):
        if getattr(self, "_h", None) and B is not None and getattr(B, "mas_pcg_destroy", None):
            B.mas_pcg_destroy(self._h)          # (module globals may already be gone at interpreter exit)
            self._h = None

    __del__ = close

    def set_dt(self, dt, stream=None):
        B.mas_pcg_set_dt(self._h, dt, _stream_ptr(stream))

    def set_option(self, name, value):
        B.mas_pcg_set_option(self._h, name, value)

    def set_preconditioner(self, kind: int, boxes=(1, 1, 0)):
        """kind 1 = PC1 (point Jacobi), 2 = PC2 (block-Jacobi ILU(0); on the GPU the boxes are the phi lines)"""
        B.mas_pcg_set_preconditioner(self._h, kind, boxes)

    def apply(self, x: torch.Tensor, y: torch.Tensor | None = None, stream=None) -> torch.Tensor:
        """y = A_sym x"""
        if y is None:
            y = torch.empty_like(x)
        B.mas_pcg_apply(self._h, _dev_ptr(x, self.n), _dev_ptr(y, self.n), _stream_ptr(stream))
        return y

    def residual_static(self, b: torch.Tensor, ax: torch.Tensor, r: torch.Tensor, sums: torch.Tensor, stream=None):
        """r = V.b - ax; sums (a CUDA float64 tensor of 3) = ||V.b||^2, ||r||^2, r.D^-1 r.  The allocation-free
        entry point (mas_pcg_residual_static): every tensor is the caller's, nothing is allocated here or below."""
        B.mas_pcg_residual_static(self._h, _dev_ptr(b, self.n), _dev_ptr(ax, self.n), _dev_ptr(r, self.n),
                                  _dev_ptr(sums, 3), _stream_ptr(stream))

    def solve(self, b: torch.Tensor, x: torch.Tensor, rtol: float, maxit: int, stream=None, want_hist=True):
        """Solves A_phys x = b in place in x (x holds x0 on entry).  Returns (status, iters, hist)."""
        return B.mas_pcg_solve(self._h, _dev_ptr(b, self.n), _dev_ptr(x, self.n), rtol, maxit,
                               _stream_ptr(stream), want_hist)

    def solve_multi(self, bs, xs, rtol: float, maxit: int, stream=None, want_hist=True):
        """nrhs <= 3 right-hand sides sharing the operator, one set of launches; xs updated in place.
        Returns (worst status, [status_j], [iters_j], [hist_j])."""
        return B.mas_pcg_solve_multi(self._h, [_dev_ptr(b, self.n) for b in bs], [_dev_ptr(x, self.n) for x in xs],
                                     rtol, maxit, _stream_ptr(stream), want_hist)

    def solve_host(self, b_host: torch.Tensor, x_host: torch.Tensor, rtol: float, maxit: int, stream=None,
                   want_hist=True):
        """Same with HOST (ideally pinned) float64 tensors; H2D/D2H copies happen inside the C call."""
        for t in (b_host, x_host):
            if t.is_cuda or t.dtype != torch.float64 or not t.is_contiguous() or t.numel() != self.n:
                raise ValueError("need contiguous host float64 tensors with nr*nt*np elements")
        return B.mas_pcg_solve_host(self._h, b_host.data_ptr(), x_host.data_ptr(), rtol, maxit,
                                    _stream_ptr(stream), want_hist)

    # ---- NEXT-1: explicit operator and RKL2 super time stepping ----
    def lop(self, u: torch.Tensor, y: torch.Tensor | None = None, stream=None) -> torch.Tensor:
        """y = M u, the FD form of div(nu grad u)."""
        if y is None:
            y = torch.empty_like(u)
        B.mas_pcg_lop(self._h, _dev_ptr(u, self.n), _dev_ptr(y, self.n), _stream_ptr(stream))
        return y

    def lambda_max(self) -> float:
        return B.mas_pcg_lambda_max(self._h)

    def sts_stages(self, tau: float) -> int:
        return B.mas_sts_stages(self._h, tau)

    def sts_advance(self, u: torch.Tensor, tau: float, s: int, stream=None) -> torch.Tensor:
        """One RKL2 super-step of size tau with s stages, in place in u."""
        B.mas_sts_advance(self._h, _dev_ptr(u, self.n), tau, s, _stream_ptr(stream))
        return u

    def stats(self):
        return B.mas_pcg_stats(self._h)


class MasPcgSlabs:
    """The same operator split into r-slabs (NEXT-3), all driven from this process on the current device.
    b and x are given as whole-mesh tensors and handed to the library slab by slab (views of their planes)."""

    def __init__(self, mesh, dt, nu_kind, nu, bc, i_split):
        if not torch.cuda.is_available():
            raise RuntimeError("MasPcgSlabs needs a CUDA device (there is no CPU fallback)")
        self.shape = (mesh.nr, mesh.nt, mesh.np_)
        self.split = [int(v) for v in i_split]
        self._h = B.mas_pcg_slabs_create(self.shape, mesh.metric_arrays(), dt, nu_kind, nu, bc, self.split)

    def close(self):
        if getattr(self, "_h", None) and B is not None and getattr(B, "mas_pcg_slabs_destroy", None):
            B.mas_pcg_slabs_destroy(self._h)
            self._h = None

    __del__ = close

    def set_dt(self, dt, stream=None):
        B.mas_pcg_slabs_set_dt(self._h, dt, _stream_ptr(stream))

    def set_option(self, name, value):
        B.mas_pcg_slabs_set_option(self._h, name, value)

    def set_preconditioner(self, kind: int, boxes=(1, 1, 0)):
        B.mas_pcg_slabs_set_preconditioner(self._h, kind, boxes)

    def _slab_ptrs(self, t: torch.Tensor):
        plane = self.shape[1] * self.shape[2]
        _dev_ptr(t, self.shape[0] * plane)
        return [t.data_ptr() + 8 * plane * lo for lo in self.split[:-1]]

    def solve(self, b: torch.Tensor, x: torch.Tensor, rtol: float, maxit: int, stream=None, want_hist=True):
        return B.mas_pcg_slabs_solve(self._h, self._slab_ptrs(b), self._slab_ptrs(x), rtol, maxit,
                                     _stream_ptr(stream), want_hist)

    def stats(self):
        return B.mas_pcg_slabs_stats(self._h)
