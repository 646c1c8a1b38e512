"""GPU parity tests proper: the CUDA path (through the C ABI) against the oracle, element by
element, on the same seeded inputs.  Run on the B200 box:  pytest tests -m gpu"""
import numpy as np
import pytest

from mas_inputs import configs, grids
from oracle import ref
from tests import helpers as H

pytestmark = pytest.mark.gpu


def _t(a):
    import torch
    return torch.from_numpy(np.ascontiguousarray(a, dtype=np.float64)).cuda()


# ------------------------------------------------------------------ matvec alone (build step 4)
@pytest.mark.parametrize("bc", [(0, 0), (1, 1), (0, 1)])
@pytest.mark.parametrize("shape", [(9, 11, 70), (1, 1, 2), (3, 2, 64), (5, 17, 130)])
def test_apply_matches_oracle_general_mesh(shape, bc):
    mesh, dt, nu_kind, nu = H.general_case(*shape, bc=bc)
    oref, gpu = H.both_ops(mesh, dt, nu_kind, nu, bc)
    u = np.random.default_rng(1).standard_normal(mesh.shape)
    y_ref = oref.apply(u)
    y = gpu.apply(_t(u)).cpu().numpy().reshape(mesh.shape)
    assert H.apply_gap(y, y_ref, f"apply {shape} bc{bc}") <= H.APPLY_RTOL


def test_apply_matches_oracle_uniform_phi_config1():
    prob = configs.make("c1")
    oref, gpu = H.both_ops(prob.mesh, prob.dt_for(2.0), prob.nu_kind, prob.nu)
    u = configs.rhs_uniform(prob)
    y_ref = oref.apply(u)
    y = gpu.apply(_t(u)).cpu().numpy().reshape(prob.mesh.shape)
    assert H.apply_gap(y, y_ref, "apply c1") <= H.APPLY_RTOL


@pytest.mark.parametrize("name,s", [("c3", 1e4), ("c5", 100.0)])
def test_apply_matches_oracle_full_size_stiff(name, s):
    """The standalone matvec at a BASELINE.json size and stiffness (coefficient form on the GPU against the
    oracle's flux-difference form: the cancellation in d*u - sum(c*u_nb) grows with s)."""
    prob = configs.make(name)
    oref, gpu = H.both_ops(prob.mesh, prob.dt_for(s), prob.nu_kind, prob.nu)
    u = np.random.default_rng(11).standard_normal(prob.mesh.shape)
    y_ref = oref.apply(u)
    y = gpu.apply(_t(u)).cpu().numpy().reshape(prob.mesh.shape)
    assert H.apply_gap(y, y_ref, f"apply {name} s={s:g}") <= H.APPLY_RTOL


def test_gpu_operator_symmetric_and_constant_closed_form():
    """P3 / P5 on the GPU operator itself."""
    import torch
    mesh, dt, nu_kind, nu = H.general_case(12, 13, 96, bc=(1, 1))
    oref, gpu = H.both_ops(mesh, dt, nu_kind, nu, (1, 1))
    rng = np.random.default_rng(4)
    x, y = _t(rng.standard_normal(mesh.shape)), _t(rng.standard_normal(mesh.shape))
    Ax, Ay = gpu.apply(x), gpu.apply(y)
    assert abs(float(torch.vdot(x.ravel(), Ay.ravel()) - torch.vdot(y.ravel(), Ax.ravel()))) \
        <= 1e-13 * float(x.norm() * Ay.norm())
    assert float(torch.vdot(x.ravel(), Ax.ravel())) > 0
    one = torch.ones_like(x)
    V = oref.volume()
    assert np.allclose(gpu.apply(one).cpu().numpy().reshape(mesh.shape), V, rtol=1e-13, atol=0)


# ------------------------------------------------------------------ full solves: every K1 tile / traffic form / loop mode
# (K1 tile, qrecompute, K2R tile): qrecompute = 1 is the 64 B/cell/iteration form (q not stored, K2R recomputes it)
FORMS = [(t, 0, 0) for t in range(7)] + [(t, 1, t % 6) for t in range(7)]


@pytest.mark.parametrize("loop_mode", [1, 0])
@pytest.mark.parametrize("tile,qrec,k2r_tile", FORMS)
def test_solve_parity_general_mesh_all_forms(tile, qrec, k2r_tile, loop_mode):
    mesh, dt, nu_kind, nu = H.general_case(21, 19, 134, s=500.0)   # 2 phi tiles (ragged), ragged theta
    oref, gpu = H.both_ops(mesh, dt, nu_kind, nu)
    gpu.set_option("persistent", 0)              # this test is about the streaming kernels
    gpu.set_option("tile", tile)
    gpu.set_option("qrecompute", qrec)
    gpu.set_option("k2r_tile", k2r_tile)
    gpu.set_option("loop_mode", loop_mode)
    rng = np.random.default_rng(3)
    b = rng.uniform(-1, 1, mesh.shape)
    x0 = rng.standard_normal(mesh.shape)
    H.check_parity(gpu, oref, b, x0, 1e-10, 2000, label=f"t{tile} q{qrec} m{loop_mode}")
    st = gpu.stats()
    assert st["loop_mode"] == loop_mode and st["bytes_per_cell_iter"] == (64 if qrec else 72)


@pytest.mark.parametrize("tile,qrec,k2r_tile", FORMS)
def test_solve_parity_uniform_phi_all_forms(tile, qrec, k2r_tile):
    prob = configs.make("c3", shape=(40, 37, 192))
    s1 = H.oracle_s1(prob.mesh, prob.nu_kind, prob.nu)
    oref, gpu = H.both_ops(prob.mesh, 1e3 / s1, prob.nu_kind, prob.nu)
    gpu.set_option("persistent", 0)
    gpu.set_option("tile", tile)
    gpu.set_option("qrecompute", qrec)
    gpu.set_option("k2r_tile", k2r_tile)
    H.check_parity(gpu, oref, configs.rhs_blob(prob), None, 1e-9, 3000, label=f"uniform t{tile} q{qrec}")


@pytest.mark.parametrize("qrec", [0, 1])
def test_l2_plan_hints_do_not_change_the_bits(qrec):
    """The L2 eviction-priority hints are performance-only: the same solve with and without them is bit-identical."""
    import torch
    prob = configs.make("c3", shape=(40, 37, 192))
    s1 = H.oracle_s1(prob.mesh, prob.nu_kind, prob.nu)
    from paper_1811_02605_b200 import MasPcg
    gpu = MasPcg(prob.mesh, 1e3 / s1, prob.nu_kind, prob.nu)
    gpu.set_option("persistent", 0)
    gpu.set_option("qrecompute", qrec)
    b = _t(configs.rhs_blob(prob))
    runs = []
    for first_x in (0, 1):
        gpu.set_option("l2_first_x", first_x)
        x = torch.zeros_like(b)
        st, k, h = gpu.solve(b, x, 1e-9, 3000)
        runs.append((st, k, h.tobytes(), x.cpu().numpy().tobytes()))
    assert all(r == runs[0] for r in runs[1:])


@pytest.mark.parametrize("persistent", [0, 1])
@pytest.mark.parametrize("bc", [(1, 1), (1, 0)])
def test_solve_parity_neumann(bc, persistent):
    mesh, dt, nu_kind, nu = H.general_case(10, 9, 66, s=50.0, bc=bc)
    oref, gpu = H.both_ops(mesh, dt, nu_kind, nu, bc)
    gpu.set_option("persistent", persistent)
    b = np.random.default_rng(8).uniform(-1, 1, mesh.shape)
    H.check_parity(gpu, oref, b, None, 1e-10, 2000, label=f"bc{bc}")


# ------------------------------------------------------------------ BASELINE.json configs
@pytest.mark.parametrize("persistent", [0, 1])
def test_config1_parity_and_rerun_bit_identity(persistent):
    import torch
    prob = configs.make("c1")
    oref, gpu = H.both_ops(prob.mesh, prob.dt_for(2.0), prob.nu_kind, prob.nu)
    gpu.set_option("persistent", persistent)
    b = configs.rhs_uniform(prob)
    k_r, k_g = H.check_parity(gpu, oref, b, None, prob.rtol, prob.maxit, label="c1")
    # north_star (3): a rerun gives the same bits
    bd = _t(b)
    runs = []
    for _ in range(3):
        xd = torch.zeros_like(bd)
        st, k, h = gpu.solve(bd, xd, prob.rtol, prob.maxit)
        runs.append((k, h.tobytes(), xd.cpu().numpy().tobytes()))
    assert runs[0] == runs[1] == runs[2]


@pytest.mark.parametrize("persistent", [0, 1])
@pytest.mark.parametrize("s", configs.STIFFNESS["c2"])
def test_config2_parity_and_manufactured_solution(s, persistent):
    import torch
    prob = configs.make("c2")
    oref, gpu = H.both_ops(prob.mesh, prob.dt_for(s), prob.nu_kind, prob.nu)
    gpu.set_option("persistent", persistent)
    gpu.solve(_t(np.ones(prob.mesh.shape)), _t(np.zeros(prob.mesh.shape)), 0.0, 1)
    assert gpu.stats()["loop_mode"] == (2 if persistent else 1)        # config 2 fits the one-kernel path
    u = configs.field_manufactured(prob)
    b = oref.apply_phys(u)                       # the same b for both sides
    H.check_parity(gpu, oref, b, None, 1e-10, prob.maxit, label=f"c2 s={s}")
    # P1 on the GPU path: recover u to 1e-10 at rtol 1e-14 (Q11)
    bd, xd = _t(b), torch.zeros(prob.mesh.shape, dtype=torch.float64, device="cuda")
    st, k, h = gpu.solve(bd, xd, 1e-14, 5000)
    assert st == 0
    xg = xd.cpu().numpy()
    assert np.linalg.norm(xg - u) / np.linalg.norm(u) <= 1e-10


def test_config3_parity_full_size():
    prob = configs.make("c3")
    oref, gpu = H.both_ops(prob.mesh, prob.dt_for(1e4), prob.nu_kind, prob.nu)
    H.check_parity(gpu, oref, configs.rhs_blob(prob), None, prob.rtol, prob.maxit, label="c3")


def test_config4_full_size_first_50_iterations_and_fixed_count():
    """256x256x512 in the launch configuration bench.py times: history over the first 50 iterations
    and x after 50 against the oracle; then the 500-fixed-iteration run returns MAS_MAXIT, k = 500."""
    import torch
    prob = configs.make("c4")
    oref, gpu = H.both_ops(prob.mesh, prob.dt_for(1e4), prob.nu_kind, prob.nu)
    b = configs.rhs_uniform(prob)
    H.check_parity(gpu, oref, b, None, 0.0, 50, label="c4/50")
    bd = _t(b)
    xd = torch.zeros_like(bd)
    st, k, h = gpu.solve(bd, xd, 0.0, prob.maxit)
    assert st == 1 and k == prob.maxit and np.isfinite(h).all() and h.size == prob.maxit + 1
    assert gpu.stats()["loop_launches"] == 2 * prob.maxit
    assert gpu.stats()["bytes_per_cell_iter"] in (64, 72, 80)
    # property that holds at any size: the true residual of the returned x matches the recurrence
    V = _t(oref.volume())
    r_true = V * bd - gpu.apply(xd)
    h_true = float(r_true.norm() / (V * bd).norm())
    assert h_true == pytest.approx(h[-1], rel=1e-3)


def test_config5_chain_first_3_solves():
    """Time-step proxy: dt varies per step, warm start; both sides get the SAME right-hand sides
    (built from the oracle's x_k) so that the histories are comparable to 1e-10."""
    prob = configs.make("c5", shape=(48, 64, 128))
    s1 = H.oracle_s1(prob.mesh, prob.nu_kind, prob.nu)
    dt0 = 100.0 / s1
    oref, gpu = H.both_ops(prob.mesh, dt0, prob.nu_kind, prob.nu)
    chain = configs.Chain(prob, 3)
    rhs = chain.state0 + chain.noise()
    x_prev = None
    for step in range(3):
        dt = dt0 * chain.dt_factor[step]
        oref.set_dt(dt)
        gpu.set_dt(dt)
        H.check_parity(gpu, oref, rhs, x_prev, prob.rtol, prob.maxit, label=f"c5 step {step}")
        _, _, x_prev, _ = oref.pcg(rhs, x_prev, prob.rtol, prob.maxit)
        rhs = x_prev + chain.noise()


def test_config5_full_size_first_3_solves():
    """BASELINE.json configs[4] at its stated size, 192x256x384 (18.9 M cells), with the calibrated dt0
    (s = 100): set_dt per step, warm start, the first 3 of the 100 chained solves,
    gates unchanged.  Both sides get the SAME right-hand sides, built from the oracle's x_k."""
    prob = configs.make("c5")
    dt0 = prob.dt_for(100.0)
    oref, gpu = H.both_ops(prob.mesh, dt0, prob.nu_kind, prob.nu)
    chain = configs.Chain(prob, 100)
    rhs = chain.state0 + chain.noise()
    x_prev = None
    for step in range(3):
        dt = dt0 * chain.dt_factor[step]
        oref.set_dt(dt)
        gpu.set_dt(dt)
        k_r, k_g = H.check_parity(gpu, oref, rhs, x_prev, prob.rtol, prob.maxit, label=f"c5 full step {step}")
        assert 30 <= k_r <= 120                      # the paper's "easy" regime, ~70 iterations
        _, _, x_prev, _ = oref.pcg(rhs, x_prev, prob.rtol, prob.maxit)
        rhs = x_prev + chain.noise()


# ------------------------------------------------------------------ breakdown and argument errors
def _modes(gpu, mode):
    """mode: 'persistent' (one cooperative kernel), 'graph' (CUDA-graph WHILE loop), 'host' (host chunks)."""
    gpu.set_option("persistent", 1 if mode == "persistent" else 0)
    gpu.set_option("loop_mode", 0 if mode == "host" else 1)


@pytest.mark.parametrize("mode", ["persistent", "graph", "host"])
def test_breakdown_nonfinite_rhs_at_init(mode):
    """A NaN in b makes bb non-finite: MAS_EBREAKDOWN with k = 0 on every loop path, as in the oracle
    ("non-finite scalar"); x is left as x0."""
    import torch
    from paper_1811_02605_b200 import MasError
    mesh, dt, nu_kind, nu = H.general_case(12, 10, 66, s=50.0)
    oref, gpu = H.both_ops(mesh, dt, nu_kind, nu)
    _modes(gpu, mode)
    rng = np.random.default_rng(9)
    b, x0 = rng.uniform(-1, 1, mesh.shape), rng.standard_normal(mesh.shape)
    b[3, 4, 5] = np.nan
    st_r, k_r, x_r, _ = oref.pcg(b, x0, 1e-10, 100)
    assert (st_r, k_r) == (ref.REF_EBREAKDOWN, 0) and np.array_equal(x_r, x0)
    xd = _t(x0)
    with pytest.raises(MasError) as e:
        gpu.solve(_t(b), xd, 1e-10, 100)
    assert e.value.status == -4 and e.value.iters == 0
    assert np.array_equal(xd.cpu().numpy(), x0)
    # the handle stays usable: a clean solve afterwards
    b[3, 4, 5] = 0.25
    H.check_parity(gpu, oref, b, x0, 1e-10, 500, label=f"after breakdown {mode}")


@pytest.mark.parametrize("mode", ["persistent", "graph", "host"])
def test_breakdown_sigma_overflow_in_first_matvec(mode):
    """p.Ap overflows to +Inf in the first K1 while bb, rr and rho are still finite: MAS_EBREAKDOWN raised by the
    matvec kernel's scalar step (S3) at k = 0, and x must still be x0 (nothing pending for the deferred x-update)."""
    import torch
    from paper_1811_02605_b200 import MasError
    mesh = grids.wobbly_phi_mesh(grids.radial_faces_pack(12, 4.0, 1.0, 1.3), 10, 66, 21)   # thin shell: every d < 1,
    nu = 0.5 + np.random.default_rng(22).uniform(0.0, 1.0, (12, 10))                        # so rr stays below rho
    dt, nu_kind = 50.0 / H.oracle_s1(mesh, 1, nu), 1
    oref, gpu = H.both_ops(mesh, dt, nu_kind, nu)
    assert oref.diag().max() < 1.0
    _modes(gpu, mode)
    # a right-hand side whose Jacobi-scaled residual D^-1/2 V b is a 3-D checkerboard: every neighbour has the
    # opposite sign, so the Rayleigh quotient sigma/rho of D^-1/2 A D^-1/2 is well above 1
    i, j, k = np.ogrid[:mesh.shape[0], :mesh.shape[1], :mesh.shape[2]]
    d, V = oref.diag(), oref.volume()
    b = np.where((i + j + k) % 2 == 0, 1.0, -1.0) * np.sqrt(d) / V
    b *= 1.0 + 0.1 * np.random.default_rng(3).uniform(-1, 1, mesh.shape)
    r0 = V * b
    z0 = r0 / d
    rho0, sigma0 = float(np.sum(r0 * z0)), float(np.sum(z0 * oref.apply(z0)))
    assert sigma0 > 1.1 * rho0
    scale = np.sqrt(np.finfo(np.float64).max / np.sqrt(rho0 * sigma0))      # rho finite, sigma = Inf
    b *= scale
    st_r, k_r, x_r, h_r = oref.pcg(b, None, 1e-10, 100)
    assert (st_r, k_r) == (ref.REF_EBREAKDOWN, 0) and not x_r.any() and np.isfinite(h_r[0])   # the sigma branch
    xd = torch.zeros(mesh.shape, dtype=torch.float64, device="cuda")
    with pytest.raises(MasError) as e:
        gpu.solve(_t(b), xd, 1e-10, 100)
    assert e.value.status == -4 and e.value.iters == 0
    assert e.value.hist[0] == pytest.approx(h_r[0], rel=1e-12)
    assert not xd.any()


def test_misaligned_and_aliased_vectors_are_einval():
    import torch
    from paper_1811_02605_b200 import binding as B
    mesh, dt, nu_kind, nu = H.general_case(4, 4, 8)
    _, gpu = H.both_ops(mesh, dt, nu_kind, nu)
    n = mesh.shape[0] * mesh.shape[1] * mesh.shape[2]
    buf = torch.zeros(2 * n + 2, dtype=torch.float64, device="cuda")
    base = buf.data_ptr()
    L = B.lib()
    for b_ptr, x_ptr in [(base + 8, base + 8 * (n + 2)), (base, base + 8 * (n + 1)), (base, base)]:
        assert L.mas_pcg_solve(gpu._h, b_ptr, x_ptr, 1e-10, 10, None, None, None) == B.MAS_EINVAL
    assert L.mas_pcg_apply(gpu._h, base, base, None) == B.MAS_EINVAL
    assert L.mas_pcg_apply(gpu._h, base + 8, base + 8 * (n + 2), None) == B.MAS_EINVAL
    assert L.mas_pcg_solve(gpu._h, base, base + 8 * (n + 2), -1.0, 10, None, None, None) == B.MAS_EINVAL
    assert L.mas_pcg_solve(gpu._h, base, base + 8 * (n + 2), 1e-10, -1, None, None, None) == B.MAS_EINVAL


# ------------------------------------------------------------------ edge and degenerate cases
@pytest.mark.parametrize("persistent", [0, 1])
def test_zero_rhs_maxit_zero_dt_zero(persistent):
    import torch
    mesh, dt, nu_kind, nu = H.general_case(6, 5, 8)
    oref, gpu = H.both_ops(mesh, dt, nu_kind, nu)
    gpu.set_option("persistent", persistent)
    z = torch.zeros(mesh.shape, dtype=torch.float64, device="cuda")
    x = torch.ones_like(z)
    st, k, h = gpu.solve(z, x, 1e-10, 10)                  # zero RHS: x = 0, no iterations
    assert (st, k) == (0, 0) and h[0] == 0.0 and not x.any()
    b = _t(np.random.default_rng(0).uniform(-1, 1, mesh.shape))
    x = torch.zeros_like(b)
    st, k, h = gpu.solve(b, x, 1e-10, 0)                   # maxit = 0
    assert (st, k) == (1, 0) and h.size == 1 and h[0] == pytest.approx(1.0) and not x.any()
    gpu.set_dt(0.0)                                        # P7: A = diag(V): one iteration, x = b
    st, k, h = gpu.solve(b, x, 1e-12, 10)
    assert (st, k) == (0, 1)
    assert torch.allclose(x, b, rtol=1e-15, atol=0)


@pytest.mark.parametrize("persistent", [0, 1])
def test_smallest_mesh_and_single_row(persistent):
    for shape in [(1, 1, 2), (1, 7, 4), (7, 1, 2)]:
        mesh, dt, nu_kind, nu = H.general_case(*shape, s=20.0)
        oref, gpu = H.both_ops(mesh, dt, nu_kind, nu)
        gpu.set_option("persistent", persistent)
        b = np.random.default_rng(2).uniform(-1, 1, mesh.shape)
        H.check_parity(gpu, oref, b, None, 1e-12, 200, label=str(shape))


def test_solve_host_matches_device_solve_bitwise():
    import torch
    prob = configs.make("c1")
    from paper_1811_02605_b200 import MasPcg
    gpu = MasPcg(prob.mesh, prob.dt_for(2.0), prob.nu_kind, prob.nu)
    b = torch.from_numpy(configs.rhs_uniform(prob)).pin_memory()
    xh = torch.zeros(prob.mesh.shape, dtype=torch.float64).pin_memory()
    st, k, h = gpu.solve_host(b, xh, prob.rtol, prob.maxit)
    xd = torch.zeros(prob.mesh.shape, dtype=torch.float64, device="cuda")
    st2, k2, h2 = gpu.solve(b.cuda(), xd, prob.rtol, prob.maxit)
    assert (st, k) == (st2, k2) and np.array_equal(h, h2) and torch.equal(xh, xd.cpu())


def test_history_longer_than_initial_capacity_and_stream():
    import torch
    mesh, dt, nu_kind, nu = H.general_case(4, 4, 8, s=5.0)
    oref, gpu = H.both_ops(mesh, dt, nu_kind, nu)
    b = _t(np.random.default_rng(5).uniform(-1, 1, mesh.shape))
    s = torch.cuda.Stream()
    with torch.cuda.stream(s):
        x = torch.zeros_like(b)
        st, k, h = gpu.solve(b, x, 1e-10, 20000, stream=s)      # maxit+1 > initial history capacity
    assert st == 0 and k < 200
    _, k_r, x_r, h_r = oref.pcg(b.cpu().numpy(), None, 1e-10, 20000)
    assert abs(k - k_r) <= 1


# ------------------------------------------------------------------ determinism as a race detector
@pytest.mark.parametrize("tile,qrec,k2r_tile", [(0, 0, 0), (1, 0, 0), (3, 0, 0), (0, 1, 1), (1, 1, 0), (3, 1, 2), (5, 1, 4)])
def test_rerun_bit_identity_every_kernel_family(tile, qrec, k2r_tile):
    """north_star (3): deterministic reductions => a rerun gives the same bits.  compute-sanitizer is closed on
    this GPU pool, so this doubles as the race check of the shared-memory rings: a missing barrier shows up as
    run-to-run differences on a mesh with thousands of blocks in flight."""
    import torch
    prob = configs.make("c3", shape=(96, 100, 384))
    s1 = H.oracle_s1(prob.mesh, prob.nu_kind, prob.nu)
    from paper_1811_02605_b200 import MasPcg
    gpu = MasPcg(prob.mesh, 1e3 / s1, prob.nu_kind, prob.nu)
    gpu.set_option("persistent", 0)
    gpu.set_option("tile", tile)
    gpu.set_option("qrecompute", qrec)
    gpu.set_option("k2r_tile", k2r_tile)
    b = _t(configs.rhs_blob(prob))
    runs = []
    for _ in range(4):
        x = torch.zeros_like(b)
        st, k, h = gpu.solve(b, x, 0.0, 60)
        runs.append((k, h.tobytes(), x.cpu().numpy().tobytes()))
    assert all(r == runs[0] for r in runs[1:])


# ------------------------------------------------------------------ large meshes: byte offsets beyond 4 GiB
def test_large_mesh_64bit_offsets_closed_forms():
    """320 x 1024 x 2048 = 671 M cells, 5.4 GB per vector (N < 2^31 is the documented maximum; element offsets
    fit 32 bits, byte offsets do not).  The oracle cannot run this in seconds, so the checks are properties that
    hold at any size: with Neumann radial faces A_sym 1 = V exactly (P5) and M 1 = 0; and after a few PCG
    iterations the recurrence residual equals the true residual b_s - A x."""
    import torch
    from mas_inputs import grids
    from paper_1811_02605_b200 import MasPcg
    nr, nt, np_ = 320, 1024, 2048
    if torch.cuda.mem_get_info()[0] < 60e9:
        pytest.skip("needs ~45 GB of free device memory")
    mesh = grids.full_sphere_mesh(grids.radial_faces_pack(nr, 4.0), nt, np_)
    nu = configs.nu_profile(mesh)
    gpu = MasPcg(mesh, 1.0, 1, nu, (1, 1))
    lam = gpu.lambda_max()
    gpu.set_dt(10.0 / lam)                # stiffness <= 5: A 1 = (V + dt G) - dt G cancels to ~eps * stiffness
    V = (torch.from_numpy(mesh.r_c ** 2 * mesh.dr_c)[:, None, None]
         * torch.from_numpy(mesh.sin_c * mesh.dth_c)[None, :, None]
         * torch.from_numpy(mesh.dph_c)[None, None, :]).cuda()
    one = torch.ones(mesh.shape, dtype=torch.float64, device="cuda")
    y = gpu.apply(one)
    assert float(((y - V).abs() / V).max()) <= 1e-12
    gpu.lop(one, y)
    assert float(y.abs().max()) <= 1e-12 * lam
    del one
    # a few iterations: true residual == recurrence residual, also at the far end of the arrays
    g = torch.Generator(device="cuda").manual_seed(7)
    b = torch.rand(mesh.shape, dtype=torch.float64, device="cuda", generator=g) * 2 - 1
    gpu.set_dt(50.0 / lam)
    x = torch.zeros_like(b)
    bs_norm = float((V * b).norm())
    hs = []
    for qrec, bpc in ((0, 72), (1, 64)):  # both forms: K2 (q stored) and K2R (two sums per block) on 11 840+ K1 blocks
        gpu.set_option("qrecompute", qrec)
        x.zero_()
        st, k, h = gpu.solve(b, x, 0.0, 5)
        assert (st, k) == (1, 5) and np.isfinite(h).all() and (np.diff(h) != 0).all()
        assert gpu.stats()["bytes_per_cell_iter"] == bpc
        gpu.apply(x, y)                   # y = A x
        y.neg_().add_(V * b)              # true residual b_s - A x
        assert float(y.norm()) / bs_norm == pytest.approx(h[-1], rel=1e-9)
        # last plane was really updated (a wrapped 32-bit byte offset would leave it untouched)
        assert float(x[-1].abs().max()) > 0 and float(x[0].abs().max()) > 0
        hs.append(h)
    assert np.allclose(hs[0], hs[1], rtol=1e-11, atol=0.0)


# ------------------------------------------------------------------ the one-kernel (persistent cooperative) path
@pytest.mark.parametrize("shape,bc", [((21, 19, 134), (0, 0)), ((9, 11, 70), (1, 0)), ((40, 37, 192), (0, 1)),
                                      ((3, 2, 64), (1, 1))])
def test_persistent_kernel_parity_general_mesh_warm_start_and_bits(shape, bc):
    import torch
    mesh, dt, nu_kind, nu = H.general_case(*shape, s=500.0, bc=bc)
    oref, gpu = H.both_ops(mesh, dt, nu_kind, nu, bc)
    gpu.set_option("persistent", 1)
    rng = np.random.default_rng(3)
    b = rng.uniform(-1, 1, mesh.shape)
    x0 = rng.standard_normal(mesh.shape)
    H.check_parity(gpu, oref, b, x0, 1e-10, 2000, label=f"persistent {shape}")
    assert gpu.stats()["loop_mode"] == 2 and gpu.stats()["loop_launches"] == 1
    runs = []
    for _ in range(3):
        xd = _t(x0)
        st, k, h = gpu.solve(_t(b), xd, 1e-10, 2000)
        runs.append((k, h.tobytes(), xd.cpu().numpy().tobytes()))
    assert runs[0] == runs[1] == runs[2]


def test_persistent_default_and_too_large_falls_back():
    from paper_1811_02605_b200 import MasPcg
    small = configs.make("c1")
    gpu = MasPcg(small.mesh, small.dt_for(2.0), small.nu_kind, small.nu)
    b = _t(configs.rhs_uniform(small))
    gpu.solve(b, _t(np.zeros(small.mesh.shape)), 1e-10, 100)
    assert gpu.stats()["loop_mode"] == 2                     # default: small mesh -> one kernel
    big = configs.make("c3", shape=(64, 96, 256))            # 1.6 M cells: state does not fit on chip
    s1 = H.oracle_s1(big.mesh, big.nu_kind, big.nu)
    gpu = MasPcg(big.mesh, 100.0 / s1, big.nu_kind, big.nu)
    gpu.set_option("persistent", 1)
    bb = _t(configs.rhs_blob(big))
    st, k, h = gpu.solve(bb, _t(np.zeros(big.mesh.shape)), 1e-8, 500)
    assert st == 0 and gpu.stats()["loop_mode"] == 1         # falls back to the graph loop
