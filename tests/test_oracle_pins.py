"""Pins for the ORACLE (oracle/mas_pcg_ref.c): it is checked against what the mathematics fixes,
never against itself and never against the CUDA path.  CPU only.

Pin list = DESIGN.md "Oracle pins" / SURVEY.md 8(c) C5 P1..P10 (+ Krylov optimality, volume sum).
"""
import math

import numpy as np
import pytest

from mas_inputs import configs, grids
from oracle import ref

ONE = np.array([1.0])


def tiny_op(s=2.0, bc=(0, 0), nu_kind=0, nu=ONE, mesh=None):
    """4x4x8 mesh of BASELINE.json north_star check (b), stiffness s."""
    m = mesh or grids.full_sphere_mesh(grids.radial_faces_ratio(4, 1.02), 4, 8)
    op = ref.RefOperator(m, 1.0, nu_kind, nu, bc)
    op.set_dt(s / op.stiffness_max())
    return m, op


def varnu_wobbly(nr=6, nt=5, np_=7, seed=11):
    """Odd sizes, non-uniform phi, nu varying in r AND theta: the most general operator."""
    m = grids.wobbly_phi_mesh(grids.radial_faces_pack(nr, 4.0), nt, np_, seed)
    rng = np.random.default_rng(seed + 1)
    nu = 0.5 + rng.uniform(0.0, 1.0, (nr, nt))
    return m, nu


# ------------------------------------------------------------------ P2: dense LU (north_star b)
@pytest.mark.parametrize("bc", [(0, 0), (1, 0), (0, 1)])
def test_P2_dense_lu_direct_solve(bc):
    m, op = tiny_op(s=50.0, bc=bc)
    A = op.dense()
    rng = np.random.default_rng(5)
    b = rng.uniform(-1, 1, m.shape)
    V = op.volume()
    x_lu = np.linalg.solve(A, (V * b).ravel())
    st, k, x, hist = op.pcg(b, None, 1e-14, 1000)
    assert st == ref.REF_OK
    assert np.linalg.norm(x.ravel() - x_lu) / np.linalg.norm(x_lu) <= 1e-12
    # P4 (north_star d): finite termination, k <= N = 128
    assert k <= A.shape[0]


def test_P2_general_operator_dense_lu():
    m, nu = varnu_wobbly()
    _, op = tiny_op(s=300.0, nu_kind=1, nu=nu, mesh=m)
    A = op.dense()
    rng = np.random.default_rng(6)
    b = rng.standard_normal(m.shape)
    x_lu = np.linalg.solve(A, (op.volume() * b).ravel())
    st, k, x, _ = op.pcg(b, rng.standard_normal(m.shape), 1e-14, 2000)   # nonzero x0
    assert st == ref.REF_OK and k <= A.shape[0]
    assert np.linalg.norm(x.ravel() - x_lu) / np.linalg.norm(x_lu) <= 1e-12


# ------------------------------------------------------------------ P3: symmetry, positivity (north_star c)
def test_P3_dense_bitwise_symmetric_and_spd():
    m, nu = varnu_wobbly()
    _, op = tiny_op(s=1000.0, nu_kind=1, nu=nu, mesh=m)
    A = op.dense()
    # flux form: every face conductance is ONE expression used by both of its cells
    assert np.array_equal(A, A.T)
    w = np.linalg.eigvalsh(A)
    assert w.min() > 0.0
    # diagonal of the dense matrix is mas_ref_diag
    assert np.allclose(np.diag(A), op.diag().ravel(), rtol=1e-14, atol=0)
    # 7-point sparsity: at most 6 off-diagonal entries per row
    assert ((A != 0).sum(axis=1) <= 7).all()
    # M-matrix sign pattern: positive diagonal, non-positive off-diagonals
    off = A - np.diag(np.diag(A))
    assert (off <= 0).all() and (np.diag(A) > 0).all()


def test_P3_random_vectors_midsize():
    p = configs.make("c3", shape=(20, 24, 32))
    op = ref.RefOperator(p.mesh, 1.0, p.nu_kind, p.nu, p.bc)
    op.set_dt(1e4 / op.stiffness_max())
    rng = np.random.default_rng(7)
    for _ in range(3):
        x = rng.standard_normal(p.mesh.shape)
        y = rng.standard_normal(p.mesh.shape)
        Ax, Ay = op.apply(x), op.apply(y)
        assert abs(np.vdot(x, Ay) - np.vdot(y, Ax)) <= 1e-13 * np.linalg.norm(x) * np.linalg.norm(Ay)
        assert np.vdot(x, Ax) > 0


# ------------------------------------------------------------------ P5: constant vector, volume
def test_P5_neumann_constant_in_nullspace_of_L():
    m, nu = varnu_wobbly(8, 9, 10)
    _, op = tiny_op(s=100.0, bc=(1, 1), nu_kind=1, nu=nu, mesh=m)
    one = np.ones(m.shape)
    V = op.volume()
    assert np.allclose(op.apply(one), V, rtol=1e-13, atol=0)


def test_P5_dirichlet_constant_hits_only_boundary_rows():
    m, op = tiny_op(s=10.0)
    y = op.apply(np.ones(m.shape)) - op.volume()
    assert np.abs(y[1:-1]).max() <= 1e-13 * np.abs(y).max()
    assert (y[0] > 0).all() and (y[-1] > 0).all()
    # the boundary conductance is nu r_f^2 sin dth dph / (half cell): ratio outer/inner rows
    dt = op.stiffness_max()  # placeholder to keep op alive; ratio test below is dt-free
    ratio = y[-1] / y[0]
    expect = (m.r_f[-1] ** 2 / m.dr_f[-1]) / (m.r_f[0] ** 2 / m.dr_f[0])
    assert np.allclose(ratio, expect, rtol=1e-12)
    assert dt > 0


@pytest.mark.parametrize("n", [8, 16, 32])
def test_volume_sums_to_shell_volume_second_order(n):
    """sum V -> 4 pi/3 (R^3 - 1); midpoint-rule error falls 4x per refinement."""
    errs = []
    for k in (n, 2 * n):
        m = grids.shell_wedge_mesh(k, k, k, 1.0, 2.0)
        op = ref.RefOperator(m, 0.0, 0, ONE)
        errs.append(abs(op.volume().sum() - 4.0 * math.pi / 3.0 * 7.0))
    assert errs[0] / errs[1] == pytest.approx(4.0, rel=0.05)


# ------------------------------------------------------------------ P6: phi eigenfunction
@pytest.mark.parametrize("mode", [1, 3])
def test_P6_phi_eigenfunction_is_separable(mode):
    p = configs.make("c1", shape=(6, 7, 16))
    m = p.mesh
    op = ref.RefOperator(m, 0.37, 0, ONE)
    rng = np.random.default_rng(8)
    f = rng.uniform(0.5, 1.5, (m.nr, m.nt, 1))
    c = np.cos(mode * m.ph_c)[None, None, :]
    y = op.apply(f * c)
    y0 = op.apply(f * np.ones_like(c))           # phi-independent part
    dph = 2 * math.pi / m.np_
    lam = (4.0 / dph) * math.sin(mode * dph / 2) ** 2        # eigenvalue of the periodic 3-point stencil
    gp = (m.dr_c[:, None] * m.dth_c[None, :] / m.sin_c[None, :])[:, :, None]
    expect = (y0 + 0.37 * gp * f * lam) * c
    assert np.allclose(y, expect, rtol=0, atol=1e-13 * np.abs(y).max())


# ------------------------------------------------------------------ P7: dt = 0
def test_P7_dt_zero_one_iteration_identity():
    p = configs.make("c1", shape=(5, 6, 8))
    op = ref.RefOperator(p.mesh, 0.0, 0, ONE)
    b = configs.rhs_uniform(p)
    st, k, x, hist = op.pcg(b, None, 1e-12, 10)
    assert st == ref.REF_OK and k == 1
    assert np.allclose(x, b, rtol=1e-15, atol=0)
    assert hist[0] == pytest.approx(1.0) and hist[1] <= 1e-15


def test_zero_rhs_returns_zero_and_no_iterations():
    m, op = tiny_op()
    st, k, x, hist = op.pcg(np.zeros(m.shape), np.ones(m.shape), 1e-10, 10)
    assert st == ref.REF_OK and k == 0 and not x.any() and hist[0] == 0.0


def test_maxit_return_and_history_length():
    m, op = tiny_op(s=1e3)
    b = np.random.default_rng(2).uniform(-1, 1, m.shape)
    st, k, x, hist = op.pcg(b, None, 0.0, 7)       # rtol = 0: fixed iteration count (Q8)
    assert st == ref.REF_MAXIT and k == 7 and hist.size == 8
    st, k, x, hist = op.pcg(b, None, 1e-10, 0)
    assert st == ref.REF_MAXIT and k == 0 and hist.size == 1


# ------------------------------------------------------------------ P8: equivariances
def test_P8_phi_roll_and_theta_flip():
    p = configs.make("c1", shape=(6, 8, 16))
    op = ref.RefOperator(p.mesh, 1.0, 0, ONE)
    op.set_dt(100.0 / op.stiffness_max())
    b = configs.rhs_uniform(p)
    st, k, x, h = op.pcg(b, None, 1e-12, 500)
    st2, k2, x2, h2 = op.pcg(np.roll(b, 5, axis=2), None, 1e-12, 500)
    assert k2 == k and np.allclose(np.roll(x, 5, axis=2), x2, rtol=0, atol=1e-13 * np.abs(x).max())
    st3, k3, x3, h3 = op.pcg(b[:, ::-1, :].copy(), None, 1e-12, 500)
    assert k3 == k and np.allclose(x[:, ::-1, :], x3, rtol=0, atol=1e-13 * np.abs(x).max())


# ------------------------------------------------------------------ P9: continuum consistency
def _radial(r):
    R = np.sin(math.pi * (r - 1.0))
    R1 = math.pi * np.cos(math.pi * (r - 1.0))
    R2 = -math.pi ** 2 * R
    return R, R1, R2


def _continuum_case(n, nu_slope):
    """u = R(r) sin^2(th) cos(2 phi), R(1) = R(2) = 0 (homogeneous Dirichlet on both faces).
    lap u = (R'' + 2R'/r - 6R/r^2) sin^2 cos2phi  [angular eigenvalue -l(l+1), l = 2];
    div(nu grad u) = nu lap u + nu' R' sin^2 cos2phi  for nu = 1 + nu_slope*(r-1)."""
    m = grids.shell_wedge_mesh(n, n, 2 * n, 1.0, 2.0)
    r = m.r_c[:, None, None]
    ang = (np.sin(m.th_c) ** 2)[None, :, None] * np.cos(2 * m.ph_c)[None, None, :]
    R, R1, R2 = _radial(r)
    u = R * ang
    nu_r = 1.0 + nu_slope * (r - 1.0)
    div = (nu_r * (R2 + 2 * R1 / r - 6 * R / r ** 2) + nu_slope * R1) * ang
    nu = np.ascontiguousarray(np.broadcast_to(1.0 + nu_slope * (m.r_c - 1.0)[:, None], (m.nr, m.nt)))
    return m, nu, u, div


@pytest.mark.parametrize("nu_slope", [0.0, 0.8])
def test_P9_truncation_error_second_order_interior(nu_slope):
    errs = []
    for n in (12, 24):
        m, nu, u, div = _continuum_case(n, nu_slope)
        c = 0.05
        op = ref.RefOperator(m, c, 1, nu)
        lhs = op.apply(u) / op.volume()            # A_phys u  ~  u - c div(nu grad u)
        err = np.abs(lhs - (u - c * div))[2:-2]    # away from the one-sided Dirichlet rows
        errs.append(err.max())
    assert errs[0] / errs[1] > 3.3                 # O(h^2): ratio -> 4


@pytest.mark.parametrize("nu_slope", [0.0, 0.8])
def test_P9_solution_error_second_order(nu_slope):
    errs = []
    for n in (8, 16):
        m, nu, u, div = _continuum_case(n, nu_slope)
        c = 0.05
        op = ref.RefOperator(m, c, 1, nu)
        st, k, x, _ = op.pcg(u - c * div, None, 1e-13, 5000)
        assert st == ref.REF_OK
        errs.append(np.abs(x - u).max())
    assert errs[0] / errs[1] > 3.3


# ------------------------------------------------------------------ the iteration itself
def _krylov_iterate(A, d, bs, x0, k):
    """Brute force: x_k = x0 + argmin_{y in K_k(M^-1 A, M^-1 r0)} ||x* - x0 - y||_A (dense algebra)."""
    r0 = bs - A @ x0
    cols = [r0 / d]
    for _ in range(k - 1):
        cols.append((A @ cols[-1]) / d)
    K, _ = np.linalg.qr(np.stack(cols, axis=1))
    c = np.linalg.solve(K.T @ A @ K, K.T @ r0)
    return x0 + K @ c


def test_krylov_optimality_of_each_iterate():
    m, nu = varnu_wobbly()
    _, op = tiny_op(s=200.0, nu_kind=1, nu=nu, mesh=m)
    A, d, V = op.dense(), op.diag().ravel(), op.volume()
    rng = np.random.default_rng(9)
    b = rng.standard_normal(m.shape)
    x0 = rng.standard_normal(m.shape)
    bs = (V * b).ravel()
    for k in range(1, 7):
        st, kk, xk, hist = op.pcg(b, x0, 0.0, k)
        assert kk == k
        xe = _krylov_iterate(A, d, bs, x0.ravel(), k)
        assert np.linalg.norm(xk.ravel() - xe) <= 1e-11 * np.linalg.norm(xe)
        # history entry k is the 2-norm of the TRUE residual of iterate k over ||b_s|| (Q6, Q7)
        true = np.linalg.norm(bs - A @ xk.ravel()) / np.linalg.norm(bs)
        assert hist[k] == pytest.approx(true, rel=1e-10)
    assert hist[0] == pytest.approx(np.linalg.norm(bs - A @ x0.ravel()) / np.linalg.norm(bs), rel=1e-13)


def test_P10_energy_norm_error_decreases_and_cg_bound():
    m, op = tiny_op(s=1000.0)
    A = op.dense()
    b = np.random.default_rng(3).uniform(-1, 1, m.shape)
    xs = np.linalg.solve(A, (op.volume() * b).ravel())
    prev = math.inf
    for k in range(0, 12):
        _, _, xk, _ = op.pcg(b, None, 0.0, k)
        e = xk.ravel() - xs
        en = math.sqrt(e @ A @ e)
        assert en < prev
        prev = en
    # kappa(D^-1 A) <= 1 + 2s (Gershgorin)  =>  k <= 0.5 sqrt(kappa) ln(2/rtol) + 1
    st, k, _, _ = op.pcg(b, None, 1e-10, 1000)
    assert st == ref.REF_OK and k <= 0.5 * math.sqrt(1 + 2 * 1000.0) * math.log(2 / 1e-10) + 1


# ------------------------------------------------------------------ P1: manufactured solution (north_star a)
@pytest.mark.parametrize("s", configs.STIFFNESS["c2"])
def test_P1_manufactured_solution_config2(s):
    prob = configs.make("c2")
    op = ref.RefOperator(prob.mesh, prob.dt_for(s), prob.nu_kind, prob.nu, prob.bc)
    u = configs.field_manufactured(prob)
    b = op.apply_phys(u)
    st, k, x, hist = op.pcg(b, None, 1e-14, 5000)        # Q11: rtol 1e-14
    assert st == ref.REF_OK
    assert np.linalg.norm(x - u) / np.linalg.norm(u) <= 1e-10


def test_calibration_file_matches_oracle():
    """mas_inputs/dt_calibration.json is what oracle/calibrate_dt.py would write today."""
    for name, kind in (("c1", "config"), ("c2", "config"), ("c3", "config"), ("c3", "nonuniform"), ("c3", "clustered")):
        prob = configs.make(name, mesh_kind=kind)
        op = ref.RefOperator(prob.mesh, 1.0, prob.nu_kind, prob.nu, prob.bc)
        assert op.stiffness_max() == pytest.approx(prob.s1(), rel=1e-14)
        op.close()


@pytest.mark.parametrize("kind", ["nonuniform", "clustered"])
def test_round3_mesh_kinds_are_valid_inputs_and_give_an_spd_operator(kind):
    """grids.random_mesh / grids.clustered_mesh: widths positive and summing to the domain,
    polar faces of zero area, theta really non-uniform, and -- on a reduced shape -- the oracle's operator on them
    is the symmetric positive definite M-matrix the pins above establish for the other meshes."""
    prob = configs.make("c3", shape=(5, 7, 8), mesh_kind=kind)
    m = prob.mesh
    assert prob.name == {"nonuniform": "c3n", "clustered": "c3k"}[kind]
    for w, total in ((m.dr_c, m.r_f[-1] - m.r_f[0]), (m.dth_c, np.pi), (m.dph_c, 2 * np.pi)):
        assert np.all(w > 0) and w.sum() == pytest.approx(total, rel=1e-13)
    assert m.sin_f[0] == 0.0 and m.sin_f[-1] == 0.0 and np.all(m.sin_f[1:-1] > 0)
    assert np.ptp(m.dth_c) > 0.1 * m.dth_c.mean()
    assert (np.ptp(m.dph_c) > 0) == (kind == "nonuniform")
    op = ref.RefOperator(m, 1.0, prob.nu_kind, prob.nu, prob.bc)
    op.set_dt(100.0 / op.stiffness_max())
    A = op.dense()
    assert np.array_equal(A, A.T) and np.all(np.diag(A) > 0)
    np.linalg.cholesky(A)
    assert np.allclose(A.sum(axis=1)[m.nt * m.np_:-m.nt * m.np_], op.volume().ravel()[m.nt * m.np_:-m.nt * m.np_], rtol=1e-12)
    op.close()


def test_config1_diagonal_dominance_ratio_is_1p5():
    """BASELINE.json config 1: 'diagonal-dominance ratio ~ 1.5'  <=>  s = 2 (Q12)."""
    prob = configs.make("c1")
    op = ref.RefOperator(prob.mesh, prob.dt_for(2.0), 0, ONE)
    d, V = op.diag(), op.volume()
    offsum = d - V                      # Dirichlet rows have less off-diagonal mass, so >= holds
    assert (d / offsum).min() == pytest.approx(1.5, rel=1e-12)


# ------------------------------------------------------------------ breakdown (SURVEY 8(b) MAS_EBREAKDOWN, C3)
def test_breakdown_nonfinite_rhs_keeps_x0():
    m, op = tiny_op(s=20.0)
    rng = np.random.default_rng(9)
    b, x0 = rng.uniform(-1, 1, m.shape), rng.standard_normal(m.shape)
    for bad in (np.nan, np.inf):
        bb = b.copy()
        bb[1, 2, 3] = bad
        st, k, x, hist = op.pcg(bb, x0, 1e-10, 50)
        assert (st, k) == (ref.REF_EBREAKDOWN, 0) and np.array_equal(x, x0) and hist.size == 1
    st, k, x, hist = op.pcg(b, np.where(np.arange(8) == 2, np.nan, x0), 1e-10, 50)     # NaN in x0: rr, rho non-finite
    assert (st, k) == (ref.REF_EBREAKDOWN, 0)


def test_breakdown_sigma_overflow_stops_before_any_update():
    """p.Ap = +Inf with bb, rr, rho finite: C3's `!isfinite(sigma)` branch; no iteration is counted, x = x0.
    (A thin shell r in [1, 1.2]: every d < 1, so rr = sum r^2 stays below rho = sum r^2/d.)"""
    m, op = tiny_op(s=20.0, mesh=grids.full_sphere_mesh(grids.radial_faces_ratio(4, 1.02, 1.0, 1.2), 4, 8))
    assert op.diag().max() < 1.0
    i, j, k = np.ogrid[:4, :4, :8]
    d, V = op.diag(), op.volume()
    b = np.where((i + j + k) % 2 == 0, 1.0, -1.0) * np.sqrt(d) / V
    r0 = V * b
    z0 = r0 / d
    rho0, sigma0 = float(np.sum(r0 * z0)), float(np.sum(z0 * op.apply(z0)))
    assert sigma0 > 1.1 * rho0
    b *= np.sqrt(np.finfo(np.float64).max / np.sqrt(rho0 * sigma0))
    st, kk, x, hist = op.pcg(b, None, 1e-10, 50)
    assert (st, kk) == (ref.REF_EBREAKDOWN, 0) and not x.any() and np.isfinite(hist[0])


# ------------------------------------------------------------------ NEXT-2: several right-hand sides, one operator
def test_pcg_multi_is_three_independent_textbook_solves():
    """mas_ref_pcg_multi is DEFINED as nrhs single solves (v_r, v_theta, v_phi share one coefficient
    set, nothing else): bit-equal x, history, count and status per right-hand side, including one that converges
    at once (zero RHS) and one that hits the iteration cap."""
    m, nu = varnu_wobbly()
    _, op = tiny_op(s=300.0, nu_kind=1, nu=nu, mesh=m)
    rng = np.random.default_rng(31)
    b = rng.uniform(-1, 1, (3,) + m.shape)
    b[1] = 0.0
    x0 = rng.standard_normal((3,) + m.shape)
    for maxit in (2000, 5):
        worst, sts, its, x, hists = op.pcg_multi(b, x0, 1e-12, maxit)
        for jr in range(3):
            st1, k1, x1, h1 = op.pcg(b[jr], x0[jr], 1e-12, maxit)
            assert (sts[jr], its[jr]) == (st1, k1)
            assert np.array_equal(x[jr], x1) and np.array_equal(hists[jr], h1)
        assert worst == max(sts)
    assert op.pcg_multi(b, x0, 1e-12, 5)[1] == [ref.REF_MAXIT, ref.REF_OK, ref.REF_MAXIT]
