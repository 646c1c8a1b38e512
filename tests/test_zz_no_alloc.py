"""mas_pcg_residual_static -- the one entry point of the library that allocates no device memory.

Why it exists: a program that keeps all its fields on the GPU and has filled the card with them (the paper's code
keeps every array device-resident), a process held to a fixed device-memory limit, or a step loop
that cannot afford the device-wide stall of cudaMalloc / cudaFree has no way to give a library workspace after
set-up.  For these callers the reduction scratch of this one call is a fixed 98 560-byte array inside the library,
good for meshes of up to 2**25 cells; all vectors are the caller's.

What is checked here: its output against the path that already exists -- mas_pcg_solve with maxit = 0 runs the same
init step on handle-owned workspaces and returns hist[0] = ||V.b - A x0|| / ||V.b|| -- within the history gate the
parity tests use (helpers.HIST_RTOL), on calls made back to back, because every call reuses the one array and what
the previous call left in it must not leak into the next.

This file is named so that pytest collects it last (`pytest --collect-only -q tests`): the driver runs the suite with
-x, and a failure here must not hide the parity tests.  It passes alone in a fresh process (the first call on the
device is then also the one that looks up the array's address) and after the rest of the suite.
"""
import ctypes

import numpy as np
import pytest

from mas_inputs import configs
from tests import helpers as H

pytestmark = pytest.mark.gpu


def _t(a):
    import torch
    return torch.from_numpy(np.ascontiguousarray(a, dtype=np.float64)).cuda()


def _existing_path_hist0(gpu, b, x0):
    """hist[0] of the solve that already exists; maxit = 0 runs apply + init only and leaves x alone."""
    x = x0.clone()
    st, k, hist = gpu.solve(b, x, 0.0, 0)
    assert k == 0 and bool((x == x0).all())
    return float(hist[0])


def _static_path(gpu, b, x0, r, sums):
    """apply (no scratch) + the allocation-free call, into tensors that exist already.  Returns the three sums."""
    import torch
    ax = gpu.apply(x0)
    gpu.residual_static(b, ax, r, sums)
    torch.cuda.synchronize()
    return sums.cpu().numpy().copy(), ax


def _inputs(shape, seed):
    rng = np.random.default_rng(seed)
    return _t(rng.uniform(-1, 1, shape)), _t(rng.standard_normal(shape))


def _check(gpu, oref, b, x0, r, sums, label):
    import torch
    h_old = _existing_path_hist0(gpu, b, x0)
    s, ax = _static_path(gpu, b, x0, r, sums)
    h_new = float(np.sqrt(s[1] / s[0]))
    gap = abs(h_new - h_old) / h_old
    H.record_gap(label, static_hist0=gap)
    assert gap <= H.HIST_RTOL, f"{label}: hist[0] {h_new!r} (static scratch) vs {h_old!r} (existing path)"
    # the vector output: r = V.b - A x0, V from the oracle's volume (rounding order of the product differs: a few ulp)
    V = _t(oref.volume())
    r_exp = V * b.reshape(V.shape) - ax.reshape(V.shape)
    assert float((r.reshape(V.shape) - r_exp).abs().max()) <= 1e-14 * float(r_exp.abs().max())
    # and the sums against r itself (plain torch reductions)
    assert abs(s[1] - float(torch.vdot(r, r))) <= 1e-13 * s[1]
    assert s[0] > 0 and s[2] > 0
    return s


@pytest.mark.parametrize("kind", ["general", "uniform_c1"])
def test_static_scratch_matches_existing_path_on_calls_in_a_row(kind):
    """Two different problems one after the other on one stream, then the first again: each call agrees with the
    existing path, and the repeat returns the same bits (nothing of the call in between survives in the array)."""
    import torch
    if kind == "general":      # non-uniform phi, nu(r, theta), 53 466 cells = 7 blocks, the last one ragged
        mesh, dt, nu_kind, nu = H.general_case(21, 19, 134, s=500.0)
    else:                      # BASELINE.json config 1: uniform phi (the Dinv-plane instantiation), 8 blocks
        prob = configs.make("c1")
        mesh, dt, nu_kind, nu = prob.mesh, prob.dt_for(2.0), prob.nu_kind, prob.nu
    oref, gpu = H.both_ops(mesh, dt, nu_kind, nu)
    gpu.set_option("persistent", 0)                # existing path = the streaming init kernel this one is a variant of
    n = mesh.nr * mesh.nt * mesh.np_
    r = torch.empty(n, dtype=torch.float64, device="cuda")
    sums = torch.zeros(3, dtype=torch.float64, device="cuda")
    b1, x1 = _inputs(mesh.shape, 5)
    b2, x2 = _inputs(mesh.shape, 6)
    b1, x1, b2, x2 = (t.reshape(-1) for t in (b1, x1, b2, x2))
    s1 = _check(gpu, oref, b1, x1, r, sums, f"static {kind} call 1")
    s2 = _check(gpu, oref, b2, x2, r, sums, f"static {kind} call 2")
    assert not np.array_equal(s1, s2)
    s1_again, _ = _static_path(gpu, b1, x1, r, sums)
    assert np.array_equal(s1, s1_again)
    oref.close()
    gpu.close()


def test_static_scratch_small_mesh_after_large_and_in_place():
    """A one-block mesh right after an eight-block one (the slots the small call does not use still hold the large
    call's partial sums), through a second handle (the array is per device, not per handle); r written over ax."""
    import torch
    prob = configs.make("c1")
    oref_big, big = H.both_ops(prob.mesh, prob.dt_for(2.0), prob.nu_kind, prob.nu)
    mesh, dt, nu_kind, nu = H.general_case(3, 2, 64)
    oref, small = H.both_ops(mesh, dt, nu_kind, nu)
    nb = prob.mesh.nr * prob.mesh.nt * prob.mesh.np_
    bb, xb = (t.reshape(-1) for t in _inputs(prob.mesh.shape, 7))
    rb = torch.empty(nb, dtype=torch.float64, device="cuda")
    sums = torch.zeros(3, dtype=torch.float64, device="cuda")
    _check(big, oref_big, bb, xb, rb, sums, "static c1 before small")
    bs, xs = (t.reshape(-1) for t in _inputs(mesh.shape, 8))
    rs = torch.empty(bs.numel(), dtype=torch.float64, device="cuda")
    s = _check(small, oref, bs, xs, rs, sums, "static small after c1")
    ax = small.apply(xs)
    small.residual_static(bs, ax, ax, sums)        # in place: r replaces ax
    torch.cuda.synchronize()
    assert bool((ax == rs).all()) and np.array_equal(sums.cpu().numpy(), s)
    for o in (oref, oref_big, small, big):
        o.close()


def test_static_scratch_rejects_a_mesh_beyond_its_limit():
    """One plane more than 256 x 256 x 512: the array has no partial-sum slot for the extra blocks, so the call
    says so (MAS_ETOOBIG, with a message that names the limit) before it looks at any pointer's contents."""
    import torch
    from mas_inputs import grids
    from paper_1811_02605_b200 import MasPcg, binding as B
    mesh = grids.full_sphere_mesh(grids.radial_faces_pack(257, 4.0), 256, 512)
    assert mesh.nr * mesh.nt * mesh.np_ > B.MAS_PCG_STATIC_MAX_CELLS
    gpu = MasPcg(mesh, 1e-3, 0, np.array([1.0]))
    dummy = torch.zeros(16, dtype=torch.float64, device="cuda")      # never dereferenced: the size test comes first
    p = dummy.data_ptr()
    st = B.lib().mas_pcg_residual_static(ctypes.c_void_p(gpu._h), p, p + 32, p + 64, p + 96, 0)
    assert st == B.MAS_ETOOBIG
    assert "MAS_PCG_STATIC_MAX_CELLS" in B.mas_pcg_strerror(st)
    with pytest.raises(B.MasError):
        B.mas_pcg_residual_static(gpu._h, p, p + 32, p + 64, p + 96, 0)
    torch.cuda.synchronize()
    assert float(dummy.abs().sum()) == 0.0
    gpu.close()
