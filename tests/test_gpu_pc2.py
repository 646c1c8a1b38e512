"""GPU parity for PC2 ("the second (PC2) is a block-Jacobi using a zero-fill incomplete LU
factorization [22]"; blocks = non-overlapping boxes is the reading DESIGN.md R8): mas_pcg_set_preconditioner(MAS_PC2) + mas_pcg_solve against the oracle's mas_ref_pcg_pc2 with the
same boxes (the phi lines: 1 x 1 x np), under the north_star gates.  Run on the B200 box:  pytest tests -m gpu"""
import numpy as np
import pytest

from mas_inputs import configs, grids
from oracle import ref
from tests import helpers as H

pytestmark = pytest.mark.gpu
LINES = (1, 1, 0)


def _t(a):
    import torch
    return torch.from_numpy(np.ascontiguousarray(a, dtype=np.float64)).cuda()


def _check(gpu, oref, b, x0, rtol, maxit, label):
    """status, count within +-1, history gate over the first 50 iterations, x gate at equal counts"""
    import torch
    pc = oref.pc2(LINES)
    st_r, k_r, x_r, h_r = oref.pcg_pc2(pc, b, x0, rtol, maxit)
    bd = _t(b)
    xd = torch.zeros_like(bd) if x0 is None else _t(x0)
    st_g, k_g, h_g = gpu.solve(bd, xd, rtol, maxit)
    assert st_g == st_r, f"{label}: status gpu {st_g} vs oracle {st_r}"
    assert abs(k_g - k_r) <= 1, f"{label}: iterations gpu {k_g} vs oracle {k_r}"
    m = min(H.HIST_ITERS, k_r, k_g) + 1
    hist_gated, hist_raw = H.hist_gaps(h_g, h_r, m)
    assert hist_gated <= H.HIST_RTOL, f"{label}: history gap {hist_gated:.3e} (raw {hist_raw:.3e})"
    if k_g != k_r:
        xd = torch.zeros_like(bd) if x0 is None else _t(x0)
        _, k2, _ = gpu.solve(bd, xd, 0.0, k_r)
        assert k2 == k_r
    xg = xd.cpu().numpy()
    err = np.linalg.norm(xg - x_r) / np.linalg.norm(x_r)
    emax = float(np.abs(xg - x_r).max() / np.abs(x_r).max())
    H.record_gap(label, hist=hist_gated, hist_raw=hist_raw, x_l2=float(err), x_max=emax,
                 k_ref=k_r, k_gpu=k_g)
    assert err <= H.X_RTOL and emax <= 100 * H.X_RTOL, f"{label}: x gap {err:.3e} / {emax:.3e}"
    s = gpu.stats()
    assert s["bytes_per_cell_iter"] == 88 and s["loop_mode"] in (0, 1)
    return k_r, k_g


@pytest.mark.parametrize("loop_mode", [1, 0])
@pytest.mark.parametrize("shape", [(9, 11, 70), (6, 5, 134), (7, 9, 8), (5, 4, 4), (3, 6, 260), (2, 3, 600),
                                   (2, 3, 500), (3, 2, 802), (2, 2, 1024)])
def test_pc2_general_mesh_nonuniform_phi_warm_start(shape, loop_mode):
    """odd sizes, every chunk length M -- np = 4, 8, 70 (M = 4), 134 (8), 260 (12), 500 (16), 600 (24), 802 and
    1024 (32: ragged and full) --, ragged last chunk, non-uniform phi, nu(r, theta), x0 != 0"""
    mesh, dt, nu_kind, nu = H.general_case(*shape, s=400.0)
    oref, gpu = H.both_ops(mesh, dt, nu_kind, nu)
    gpu.set_preconditioner(2, LINES)
    gpu.set_option("loop_mode", loop_mode)
    rng = np.random.default_rng(shape[2])
    b, x0 = rng.uniform(-1, 1, mesh.shape), rng.standard_normal(mesh.shape)
    k_r, k_g = _check(gpu, oref, b, x0, 1e-10, 2000, f"pc2 general {shape} m{loop_mode}")
    st1, k1, _, _ = oref.pcg(b, x0, 1e-10, 2000)
    assert k_r < k1                                              # PC2 needs fewer iterations than PC1


@pytest.mark.parametrize("bc", [(1, 1), (1, 0)])
def test_pc2_uniform_phi_neumann(bc):
    mesh = grids.full_sphere_mesh(grids.radial_faces_pack(10, 4.0), 9, 66)
    s1 = H.oracle_s1(mesh, 0, np.array([1.0]), bc)
    oref, gpu = H.both_ops(mesh, 200.0 / s1, 0, np.array([1.0]), bc)
    gpu.set_preconditioner(2)
    b = np.random.default_rng(8).uniform(-1, 1, mesh.shape)
    _check(gpu, oref, b, None, 1e-10, 2000, f"pc2 bc{bc}")


@pytest.mark.parametrize("np_", [500, 802, 1024])
def test_pc2_uniform_phi_long_lines(np_):
    """the uniform-phi instantiations of the two longest chunk lengths (M = 16: np 385..512; M = 32: np 769..1024),
    which no BASELINE.json config except config 4 (np = 512) reaches"""
    mesh = grids.full_sphere_mesh(grids.radial_faces_pack(3, 4.0), 4, np_)
    rng = np.random.default_rng(np_)
    nu = 0.5 + rng.uniform(0.0, 1.0, (3, 4))
    s1 = H.oracle_s1(mesh, 1, nu)
    oref, gpu = H.both_ops(mesh, 300.0 / s1, 1, nu)
    gpu.set_preconditioner(2)
    b, x0 = rng.uniform(-1, 1, mesh.shape), rng.standard_normal(mesh.shape)
    _check(gpu, oref, b, x0, 1e-10, 2000, f"pc2 uniform np={np_}")


def test_pc2_config1_and_rerun_bit_identity_and_back_to_pc1():
    import torch
    prob = configs.make("c1")
    oref, gpu = H.both_ops(prob.mesh, prob.dt_for(2.0), prob.nu_kind, prob.nu)
    b = configs.rhs_uniform(prob)
    gpu.set_preconditioner(2)
    _check(gpu, oref, b, None, prob.rtol, prob.maxit, "pc2 c1")
    bd = _t(b)
    runs = []
    for _ in range(3):
        x = torch.zeros_like(bd)
        st, k, h = gpu.solve(bd, x, prob.rtol, prob.maxit)
        runs.append((st, k, h.tobytes(), x.cpu().numpy().tobytes()))
    assert runs[0] == runs[1] == runs[2]
    gpu.set_preconditioner(1)                                    # and PC1 again on the same handle
    H.check_parity(gpu, oref, b, None, prob.rtol, prob.maxit, label="c1 pc1 after pc2")


@pytest.mark.parametrize("s", [10.0, 1000.0])
def test_pc2_config2_manufactured_solution(s):
    prob = configs.make("c2")
    oref, gpu = H.both_ops(prob.mesh, prob.dt_for(s), prob.nu_kind, prob.nu)
    gpu.set_preconditioner(2)
    u = configs.field_manufactured(prob)
    b = oref.apply_phys(u)
    _check(gpu, oref, b, None, 1e-10, 5000, f"pc2 c2 s={s:g}")
    import torch
    bd, xd = _t(b), torch.zeros(prob.mesh.shape, dtype=torch.float64, device="cuda")
    st, k, _ = gpu.solve(bd, xd, 1e-14, 5000)
    assert st == 0 and np.linalg.norm(xd.cpu().numpy() - u) / np.linalg.norm(u) <= 1e-10   # P1 with PC2


def test_pc2_config3_full_size():
    prob = configs.make("c3")
    oref, gpu = H.both_ops(prob.mesh, prob.dt_for(1e4), prob.nu_kind, prob.nu)
    gpu.set_preconditioner(2)
    b = configs.rhs_blob(prob)
    k_r, k_g = _check(gpu, oref, b, None, prob.rtol, prob.maxit, "pc2 c3")
    assert k_r <= 60                                             # 437 with PC1


def test_pc2_config4_full_size_first_40_iterations():
    prob = configs.make("c4")
    oref, gpu = H.both_ops(prob.mesh, prob.dt_for(1e4), prob.nu_kind, prob.nu)
    gpu.set_preconditioner(2)
    b = configs.rhs_uniform(prob)
    _check(gpu, oref, b, None, 0.0, 40, "pc2 c4/40")


@pytest.mark.parametrize("full", [False, True])
def test_pc2_config5_chain_first_3_solves_set_dt_refactors(full):
    """config 5's chain (dt varies per step, warm start) with PC2, at a reduced size and at 192 x 256 x 384"""
    import torch
    prob = configs.make("c5") if full else configs.make("c5", shape=(48, 64, 96))
    dt0 = prob.dt_for(100.0) if full else 100.0 / H.oracle_s1(prob.mesh, prob.nu_kind, prob.nu)
    oref, gpu = H.both_ops(prob.mesh, dt0, prob.nu_kind, prob.nu)
    gpu.set_preconditioner(2)
    chain = configs.Chain(prob, 100)
    b = chain.state0 + chain.noise()
    x_r, xd = None, torch.zeros(prob.mesh.shape, dtype=torch.float64, device="cuda")
    for step in range(3):
        dt = dt0 * chain.dt_factor[step]
        oref.set_dt(dt)
        gpu.set_dt(dt)                                           # refactors the ILU(0) pivots
        pc = oref.pc2(LINES)
        st_r, k_r, x_r, h_r = oref.pcg_pc2(pc, b, x_r, prob.rtol, prob.maxit)
        st_g, k_g, h_g = gpu.solve(_t(b), xd, prob.rtol, prob.maxit)
        assert st_g == st_r == 0 and abs(k_g - k_r) <= 1
        m = min(k_r, k_g) + 1
        assert (np.abs(h_g[:m] - h_r[:m]) / h_r[:m]).max() <= H.HIST_RTOL
        if k_g == k_r:
            assert np.linalg.norm(xd.cpu().numpy() - x_r) / np.linalg.norm(x_r) <= H.X_RTOL
        else:
            xd.copy_(_t(x_r))
        b = x_r + chain.noise()


def test_pc2_multi_rhs_matches_single_solves_bitwise():
    import torch
    mesh, dt, nu_kind, nu = H.general_case(12, 10, 66, s=300.0)
    oref, gpu = H.both_ops(mesh, dt, nu_kind, nu)
    gpu.set_preconditioner(2)
    rng = np.random.default_rng(5)
    bs = [rng.uniform(-1, 1, mesh.shape) for _ in range(3)]
    bd = [_t(b) for b in bs]
    xd = [torch.zeros_like(bd[0]) for _ in range(3)]
    worst, sts, ks, hs = gpu.solve_multi(bd, xd, 1e-10, 500)
    pc = oref.pc2(LINES)
    for j in range(3):
        st_r, k_r, x_r, h_r = oref.pcg_pc2(pc, bs[j], None, 1e-10, 500)
        assert sts[j] == st_r and abs(ks[j] - k_r) <= 1
        x1 = torch.zeros_like(bd[0])
        st1, k1, h1 = gpu.solve(bd[j], x1, 1e-10, 500)
        assert (st1, k1) == (sts[j], ks[j]) and np.array_equal(h1, hs[j]) and torch.equal(x1, xd[j])
        if ks[j] == k_r:
            assert np.linalg.norm(xd[j].cpu().numpy() - x_r) / np.linalg.norm(x_r) <= H.X_RTOL


def test_pc2_breakdown_zero_rhs_and_argument_errors():
    import torch
    from paper_1811_02605_b200 import MasError
    mesh, dt, nu_kind, nu = H.general_case(6, 5, 34, s=50.0)
    oref, gpu = H.both_ops(mesh, dt, nu_kind, nu)
    for boxes in [(2, 1, 0), (1, 2, 0), (1, 1, 16), (0, 0, 0)]:   # only the line boxes exist on the GPU
        with pytest.raises(MasError) as e:
            gpu.set_preconditioner(2, boxes)
        assert e.value.status == -1
    with pytest.raises(MasError):
        gpu.set_preconditioner(3)
    gpu.set_preconditioner(2, (1, 1, 34))
    b = np.random.default_rng(2).uniform(-1, 1, mesh.shape)
    x = torch.ones(mesh.shape, dtype=torch.float64, device="cuda")
    st, k, h = gpu.solve(_t(np.zeros(mesh.shape)), x, 1e-10, 10)
    assert (st, k) == (0, 0) and h[0] == 0.0 and float(x.abs().max()) == 0.0
    st, k, h = gpu.solve(_t(b), x, 1e-10, 0)
    assert (st, k) == (1, 0)
    b[1, 2, 3] = np.nan
    with pytest.raises(MasError) as e:
        gpu.solve(_t(b), x, 1e-10, 10)
    assert e.value.status == -4 and e.value.iters == 0
    mesh2 = grids.full_sphere_mesh(grids.radial_faces_ratio(3, 1.02), 3, 2)
    _, gpu2 = H.both_ops(mesh2, 1e-3, 0, np.array([1.0]))
    with pytest.raises(MasError):
        gpu2.set_preconditioner(2)                               # np < 4


@pytest.mark.parametrize("loop_mode", [1, 0])
@pytest.mark.parametrize("split", [[0, 10, 21], [0, 1, 2, 20, 21], [0, 5, 11, 16, 21]])
def test_pc2_slab_groups_parity_and_bits(split, loop_mode):
    """PC2 on an r-slab group (NEXT-3 x NEXT-4): every slab preconditions its own phi lines, K1 reads the neighbours'
    adjacent planes of z through pointers; the oracle is the undivided PC2 solve."""
    from paper_1811_02605_b200 import MasPcgSlabs
    bc = (0, 1)
    mesh, dt, nu_kind, nu = H.general_case(21, 19, 134, s=500.0, bc=bc)
    oref = ref.RefOperator(mesh, dt, nu_kind, nu, bc)
    g = MasPcgSlabs(mesh, dt, nu_kind, nu, bc, split)
    g.set_option("loop_mode", loop_mode)
    g.set_preconditioner(2)
    rng = np.random.default_rng(3)
    b, x0 = rng.uniform(-1, 1, mesh.shape), rng.standard_normal(mesh.shape)
    pc = oref.pc2(LINES)
    st_r, k_r, x_r, h_r = oref.pcg_pc2(pc, b, x0, 1e-10, 2000)
    runs = []
    for _ in range(2):
        xd = _t(x0)
        st_g, k_g, h_g = g.solve(_t(b), xd, 1e-10, 2000)
        runs.append((k_g, h_g.tobytes(), xd.cpu().numpy().tobytes()))
    assert runs[0] == runs[1]
    assert st_g == st_r and abs(k_g - k_r) <= 1
    m = min(H.HIST_ITERS, k_r, k_g) + 1
    assert H.hist_gaps(h_g, h_r, m)[0] <= H.HIST_RTOL
    if k_g == k_r:
        assert np.linalg.norm(xd.cpu().numpy() - x_r) / np.linalg.norm(x_r) <= H.X_RTOL
    s = g.stats()
    assert s["bytes_per_cell_iter"] == 88 and s["persistent_grid_or_slabs"] == len(split) - 1
    g.set_preconditioner(1)                                      # back to PC1 on the same group
    st1, k1, _ = g.solve(_t(b), _t(x0), 1e-10, 2000)
    assert st1 == 0 and k1 > k_g
