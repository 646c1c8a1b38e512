"""GPU parity on meshes that are non-uniform in r, THETA and phi (grids.random_mesh) -- the input class of the paper's
mesh ("non-uniform logically-rectangular"; "extremely non-uniform grid").  Every other GPU
test builds theta faces as pi*j/nt, so the theta-face planes CT / AT and the sin_c*dth_c factor of V2 / CR had only
been compared with the oracle for equal theta widths ("What's missing" 3).  Here every kernel family
runs on random theta widths: stencil (apply, lop: all tiles), PCG-PC1 (all K1 tiles x {72 B, 64 B} x {graph loop,
host loop, one-kernel solve}), PC2, batched right-hand sides, r-slab groups, RKL2 -- at ragged small sizes and once
at 128 x 192 x 256.  phi is taken both non-uniform (the UNIFORM=false kernel instantiations) and uniform (the
Dinv-plane instantiations the BASELINE configs time, now with non-uniform theta).  Run on the B200 box: pytest tests -m gpu"""
import numpy as np
import pytest

from mas_inputs import grids
from oracle import ref
from tests import helpers as H

pytestmark = pytest.mark.gpu

LINES = (1, 1, 0)


def _t(a):
    import torch
    return torch.from_numpy(np.ascontiguousarray(a, dtype=np.float64)).cuda()


def _case(nr, nt, np_, uniform_phi, bc=(0, 0), seed=0, s=300.0, amp=0.3):
    mesh = grids.random_mesh(nr, nt, np_, seed=7000 + seed, amp=amp, uniform_phi=uniform_phi)
    assert nt < 3 or np.ptp(mesh.dth_c) > 0.1 * mesh.dth_c.mean()    # theta really is non-uniform
    nu = 0.5 + np.random.default_rng(seed).uniform(0.0, 1.0, (nr, nt))
    dt = s / H.oracle_s1(mesh, 1, nu, bc)
    return mesh, dt, 1, nu


FORMS = [(t, 0, 0) for t in range(7)] + [(t, 1, t % 6) for t in range(7)]


@pytest.mark.parametrize("uniform_phi", [False, True])
@pytest.mark.parametrize("shape,bc", [((5, 7, 66), (0, 0)), ((6, 9, 130), (1, 1)), ((4, 15, 258), (0, 1)),
                                      ((9, 11, 70), (1, 0)), ((3, 1, 4), (0, 0))])
def test_nonuniform_theta_stencil_all_tiles(shape, bc, uniform_phi):
    mesh, dt, nu_kind, nu = _case(*shape, uniform_phi, bc, seed=shape[2])
    oref, gpu = H.both_ops(mesh, dt, nu_kind, nu, bc)
    u = np.random.default_rng(2).standard_normal(mesh.shape)
    a_ref, l_ref = oref.apply(u), oref.lop(u)
    for tile in range(6):
        gpu.set_option("stencil_tile", tile)
        a = gpu.apply(_t(u)).cpu().numpy().reshape(mesh.shape)
        l = gpu.lop(_t(u)).cpu().numpy().reshape(mesh.shape)
        assert H.apply_gap(a, a_ref, f"nonuni apply {shape} u{uniform_phi} tile {tile}") <= H.APPLY_RTOL
        assert H.apply_gap(l, l_ref, f"nonuni lop {shape} u{uniform_phi} tile {tile}") <= H.APPLY_RTOL
    assert gpu.lambda_max() == pytest.approx(oref.lambda_max_bound(), rel=1e-12)


@pytest.mark.parametrize("uniform_phi", [False, True])
@pytest.mark.parametrize("loop_mode", [1, 0])
def test_nonuniform_theta_pcg_every_k1_tile_and_traffic_form(loop_mode, uniform_phi):
    mesh, dt, nu_kind, nu = _case(21, 19, 134, uniform_phi, seed=1, s=500.0)
    oref, gpu = H.both_ops(mesh, dt, nu_kind, nu)
    gpu.set_option("persistent", 0)
    gpu.set_option("loop_mode", loop_mode)
    rng = np.random.default_rng(3)
    b, x0 = rng.uniform(-1, 1, mesh.shape), rng.standard_normal(mesh.shape)
    for tile, qrec, k2r_tile in FORMS:
        for name, val in (("tile", tile), ("qrecompute", qrec), ("k2r_tile", k2r_tile)):
            gpu.set_option(name, val)
        H.check_parity(gpu, oref, b, x0, 1e-10, 2000, label=f"nonuni u{uniform_phi} t{tile} q{qrec} m{loop_mode}")
        st = gpu.stats()
        assert st["loop_mode"] == loop_mode and st["bytes_per_cell_iter"] == (64 if qrec else 72)


@pytest.mark.parametrize("uniform_phi", [False, True])
@pytest.mark.parametrize("shape,bc", [((9, 11, 70), (0, 0)), ((16, 16, 128), (1, 0)), ((5, 6, 258), (0, 1))])
def test_nonuniform_theta_one_kernel_solve(shape, bc, uniform_phi):
    mesh, dt, nu_kind, nu = _case(*shape, uniform_phi, bc, seed=11)
    oref, gpu = H.both_ops(mesh, dt, nu_kind, nu, bc)
    rng = np.random.default_rng(4)
    b, x0 = rng.uniform(-1, 1, mesh.shape), rng.standard_normal(mesh.shape)
    H.check_parity(gpu, oref, b, x0, 1e-10, 2000, label=f"nonuni persistent {shape} u{uniform_phi}")
    assert gpu.stats()["loop_mode"] == 2


@pytest.mark.parametrize("uniform_phi", [False, True])
@pytest.mark.parametrize("shape", [(6, 5, 134), (3, 6, 260), (2, 3, 500), (9, 11, 70)])
def test_nonuniform_theta_pc2(shape, uniform_phi):
    import torch
    mesh, dt, nu_kind, nu = _case(*shape, uniform_phi, seed=shape[2], s=400.0)
    oref, gpu = H.both_ops(mesh, dt, nu_kind, nu)
    gpu.set_preconditioner(2, LINES)
    rng = np.random.default_rng(5)
    b, x0 = rng.uniform(-1, 1, mesh.shape), rng.standard_normal(mesh.shape)
    pc = oref.pc2(LINES)
    st_r, k_r, x_r, h_r = oref.pcg_pc2(pc, b, x0, 1e-10, 2000)
    bd, xd = _t(b), _t(x0)
    st_g, k_g, h_g = gpu.solve(bd, xd, 1e-10, 2000)
    assert st_g == st_r and abs(k_g - k_r) <= 1
    m = min(H.HIST_ITERS, k_r, k_g) + 1
    gated, raw = H.hist_gaps(h_g, h_r, m)
    assert gated <= H.HIST_RTOL
    if k_g != k_r:
        xd = _t(x0)
        gpu.solve(bd, xd, 0.0, k_r)
    err = np.linalg.norm(xd.cpu().numpy() - x_r) / np.linalg.norm(x_r)
    H.record_gap(f"nonuni pc2 {shape} u{uniform_phi}", hist=gated, hist_raw=raw, x_l2=float(err))
    assert err <= H.X_RTOL
    assert gpu.stats()["bytes_per_cell_iter"] == 88


@pytest.mark.parametrize("uniform_phi", [False, True])
def test_nonuniform_theta_batched_right_hand_sides(uniform_phi):
    import torch
    mesh, dt, nu_kind, nu = _case(13, 10, 134, uniform_phi, seed=21, s=200.0)
    oref, gpu = H.both_ops(mesh, dt, nu_kind, nu)
    gpu.set_option("persistent", 0)
    rng = np.random.default_rng(6)
    bs = [rng.uniform(-1, 1, mesh.shape) for _ in range(3)]
    _, st_r, k_r, x_r, h_r = oref.pcg_multi(np.stack(bs), None, 1e-10, 2000)
    bd = [_t(b) for b in bs]
    xd = [torch.zeros_like(bd[0]) for _ in range(3)]
    _, st_g, k_g, h_g = gpu.solve_multi(bd, xd, 1e-10, 2000)
    assert st_g == st_r
    for j in range(3):
        assert abs(k_g[j] - k_r[j]) <= 1
        m = min(H.HIST_ITERS, k_r[j], k_g[j]) + 1
        assert H.hist_gaps(h_g[j], h_r[j], m)[0] <= H.HIST_RTOL
        if k_g[j] == k_r[j]:
            assert np.linalg.norm(xd[j].cpu().numpy() - x_r[j]) / np.linalg.norm(x_r[j]) <= H.X_RTOL
        x1 = torch.zeros_like(bd[0])
        st1, k1, h1 = gpu.solve(bd[j], x1, 1e-10, 2000)
        assert k1 == k_g[j] and np.array_equal(h1, h_g[j]) and torch.equal(x1, xd[j])


@pytest.mark.parametrize("precond", [1, 2])
@pytest.mark.parametrize("uniform_phi", [False, True])
def test_nonuniform_theta_slab_group(uniform_phi, precond):
    from paper_1811_02605_b200 import MasPcgSlabs
    bc = (0, 1)
    mesh, dt, nu_kind, nu = _case(21, 19, 134, uniform_phi, bc, seed=31, s=500.0)
    oref = ref.RefOperator(mesh, dt, nu_kind, nu, bc)
    g = MasPcgSlabs(mesh, dt, nu_kind, nu, bc, [0, 5, 11, 16, 21])
    rng = np.random.default_rng(7)
    b, x0 = rng.uniform(-1, 1, mesh.shape), rng.standard_normal(mesh.shape)
    if precond == 1:
        H.check_parity(g, oref, b, x0, 1e-10, 2000, label=f"nonuni slabs u{uniform_phi}")
        return
    g.set_preconditioner(2, LINES)
    pc = oref.pc2(LINES)
    st_r, k_r, x_r, h_r = oref.pcg_pc2(pc, b, x0, 0.0, 25)
    xd = _t(x0)
    st_g, k_g, h_g = g.solve(_t(b), xd, 0.0, 25)
    assert (st_g, k_g) == (st_r, k_r)
    assert H.hist_gaps(h_g, h_r, 26)[0] <= H.HIST_RTOL
    assert np.linalg.norm(xd.cpu().numpy().reshape(x_r.shape) - x_r) / np.linalg.norm(x_r) <= H.X_RTOL


@pytest.mark.parametrize("uniform_phi", [False, True])
@pytest.mark.parametrize("s", [5, 16])
def test_nonuniform_theta_rkl2(s, uniform_phi):
    bc = (1, 0)
    mesh, _, nu_kind, nu = _case(13, 10, 134, uniform_phi, bc, seed=41)
    oref, gpu = H.both_ops(mesh, 1.0, nu_kind, nu, bc)
    lam = gpu.lambda_max()
    lim = lambda n: (n * n + n - 2.0) / 4.0 * 2.0 / lam
    tau = 0.5 * (lim(s - 1) + lim(s))
    assert gpu.sts_stages(tau) == s
    u = np.random.default_rng(8).standard_normal(mesh.shape)
    y_ref = oref.sts(u, tau, s)
    for tile in range(6):
        gpu.set_option("stencil_tile", tile)
        ud = _t(u)
        gpu.sts_advance(ud, tau, s)
        assert np.abs(ud.cpu().numpy().reshape(mesh.shape) - y_ref).max() <= 1e-11 * np.abs(u).max(), tile


@pytest.mark.parametrize("uniform_phi", [False, True])
def test_nonuniform_mesh_128x192x256_every_family(uniform_phi):
    """Once at a size that spans many tiles in every direction (6.3 M cells): apply, 40 fixed PCG-PC1 iterations in
    the 72 B and the 64 B form, 15 PC2 iterations, one RKL2 super-step of 8 stages, against the oracle."""
    import torch
    shape = (128, 192, 256)
    mesh, dt, nu_kind, nu = _case(*shape, uniform_phi, seed=51, s=1e4)
    oref, gpu = H.both_ops(mesh, dt, nu_kind, nu)
    rng = np.random.default_rng(9)
    u = rng.standard_normal(shape)
    assert H.apply_gap(gpu.apply(_t(u)).cpu().numpy().reshape(shape), oref.apply(u),
                       f"nonuni apply 128x192x256 u{uniform_phi}") <= H.APPLY_RTOL
    b = rng.uniform(-1, 1, shape)
    for qrec in (0, 1):
        gpu.set_option("qrecompute", qrec)
        H.check_parity(gpu, oref, b, None, 0.0, 40, label=f"nonuni 128x192x256 u{uniform_phi} q{qrec}")
        assert gpu.stats()["loop_mode"] == 1
    gpu.set_option("qrecompute", 0)
    gpu.set_preconditioner(2, LINES)
    pc = oref.pc2(LINES)
    st_r, k_r, x_r, h_r = oref.pcg_pc2(pc, b, None, 0.0, 15)
    bd, xd = _t(b), torch.zeros(shape, dtype=torch.float64, device="cuda")
    st_g, k_g, h_g = gpu.solve(bd, xd, 0.0, 15)
    assert (st_g, k_g) == (st_r, k_r)
    gated, raw = H.hist_gaps(h_g, h_r, 16)
    err = np.linalg.norm(xd.cpu().numpy() - x_r) / np.linalg.norm(x_r)
    H.record_gap(f"nonuni pc2 128x192x256 u{uniform_phi}", hist=gated, hist_raw=raw, x_l2=float(err))
    assert gated <= H.HIST_RTOL and err <= H.X_RTOL
    gpu.set_preconditioner(1)
    tau = 0.9 * (8 * 8 + 8 - 2.0) / 4.0 * 2.0 / gpu.lambda_max()
    y_ref = oref.sts(u, tau, 8)
    ud = _t(u)
    gpu.sts_advance(ud, tau, 8)
    assert np.abs(ud.cpu().numpy() - y_ref).max() <= 1e-11 * np.abs(u).max()
