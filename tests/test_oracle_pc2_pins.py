"""Pins for the ORACLE's PC2 (oracle/mas_pcg_ref.c, NEXT-4: "the second (PC2) is a block-Jacobi using a zero-fill
incomplete LU factorization [22]"; blocks = non-overlapping boxes is the reading DESIGN.md R8): checked against what the mathematics fixes, never against itself and
never against the CUDA path.  CPU only.

  * the defining property of ILU(0) (Saad [22]): L unit lower, U upper, both confined to the pattern of A_blk, and
    (L U)_ij = (A_blk)_ij on that pattern -- on dense copies, with A_blk rebuilt HERE from the dense A_sym and an
    independently computed box id per cell;
  * exactness where ILU(0) has no fill to drop: tridiagonal operators (1-D meshes) => M = A, one PCG iteration;
  * dt = 0 => M = diag(V);  symmetry and positivity of M^-1 (U = diag(U) L^T for a symmetric M-matrix);
  * box locality of M^-1;  the PCG solution against dense LU;  Krylov optimality of the preconditioned iterates
    against a brute-force minimiser;  hist[k] against the true residual;
  * fewer iterations than PC1, by about the factor PAPER.md:80 reports (550 -> 100-200).
"""
import numpy as np
import pytest

from mas_inputs import configs, grids
from oracle import ref

ONE = np.array([1.0])


def _op(mesh, s, nu_kind=0, nu=ONE, bc=(0, 0)):
    op = ref.RefOperator(mesh, 1.0, nu_kind, nu, bc)
    op.set_dt(s / op.stiffness_max())
    return op


def _tiny(s=50.0):
    return grids.full_sphere_mesh(grids.radial_faces_ratio(4, 1.02), 4, 8)


def _general(nr=5, nt=3, np_=6, seed=11):
    m = grids.wobbly_phi_mesh(grids.radial_faces_pack(nr, 4.0), nt, np_, seed)
    nu = 0.5 + np.random.default_rng(seed + 1).uniform(0.0, 1.0, (nr, nt))
    return m, nu


def _box_ids(shape, boxes):
    """box id of every cell, computed here (not by the oracle): boxes of bi x bj x bk cells from the origin."""
    nr, nt, np_ = shape
    bi, bj, bk = [b if 0 < b <= n else n for b, n in zip(boxes, shape)]
    i, j, k = np.meshgrid(np.arange(nr), np.arange(nt), np.arange(np_), indexing="ij")
    nbj, nbk = -(-nt // bj), -(-np_ // bk)
    return (((i // bi) * nbj + (j // bj)) * nbk + (k // bk)).ravel()


def _a_blk(op, boxes):
    A = op.dense()
    ids = _box_ids(op.shape, boxes)
    return np.where(ids[:, None] == ids[None, :], A, 0.0)


CASES = [("tiny", (0, 0, 0)), ("tiny", (2, 2, 4)), ("tiny", (1, 1, 0)), ("tiny", (3, 2, 0)), ("tiny", (1, 4, 3)),
         ("general", (0, 0, 0)), ("general", (2, 2, 0)), ("general", (1, 1, 0)), ("general", (2, 1, 4))]


def _case(kind):
    if kind == "tiny":
        m = _tiny()
        return m, _op(m, 50.0)
    m, nu = _general()
    return m, _op(m, 300.0, 1, nu)


@pytest.mark.parametrize("kind,boxes", CASES)
def test_ilu0_defining_property(kind, boxes):
    m, op = _case(kind)
    Ab = _a_blk(op, boxes)
    L, U = op.pc2(boxes).dense_factors()
    pat = Ab != 0.0
    n = Ab.shape[0]
    assert np.array_equal(np.diag(L), np.ones(n)) and np.all(np.triu(L, 1) == 0.0) and np.all(np.tril(U, -1) == 0.0)
    assert not np.any((L != 0.0) & ~pat & ~np.eye(n, dtype=bool)) and not np.any((U != 0.0) & ~pat)   # zero fill
    LU = L @ U
    scale = np.abs(Ab).max()
    assert np.abs(LU - Ab)[pat].max() <= 1e-13 * scale            # exact on the pattern ...
    if boxes == (0, 0, 0):
        assert np.abs(LU - Ab)[~pat].max() > 1e-6 * scale         # ... and genuinely incomplete off it (3-D: fill was dropped)
    assert np.all(np.diag(U) > 0.0)                                # M-matrix: positive pivots


@pytest.mark.parametrize("kind,boxes", CASES)
def test_apply_is_the_two_triangular_solves_and_is_symmetric_positive(kind, boxes):
    m, op = _case(kind)
    pc = op.pc2(boxes)
    L, U = pc.dense_factors()
    rng = np.random.default_rng(3)
    x, y = rng.standard_normal(m.shape), rng.standard_normal(m.shape)
    zx = pc.apply(x).ravel()
    z_dense = np.linalg.solve(U, np.linalg.solve(L, x.ravel()))   # library triangular solves on the dense factors
    assert np.abs(zx - z_dense).max() <= 1e-12 * np.abs(z_dense).max()
    zy = pc.apply(y).ravel()
    assert abs(x.ravel() @ zy - y.ravel() @ zx) <= 1e-12 * np.linalg.norm(x) * np.linalg.norm(zy)
    assert x.ravel() @ zx > 0.0
    D = np.diag(np.diag(U))
    assert np.abs(U - D @ L.T).max() <= 1e-13 * np.abs(U).max()   # symmetric A => U = D L^T (incomplete Cholesky form)


def test_box_locality():
    m, op = _case("tiny")
    boxes = (2, 2, 4)
    ids = _box_ids(m.shape, boxes).reshape(m.shape)
    pc = op.pc2(boxes)
    rng = np.random.default_rng(4)
    for b in (0, 3, 7):
        r = np.where(ids == b, rng.standard_normal(m.shape), 0.0)
        z = pc.apply(r)
        assert np.all(z[ids != b] == 0.0) and np.any(z[ids == b] != 0.0)


@pytest.mark.parametrize("axis", ["r", "theta"])
def test_tridiagonal_operator_is_factored_exactly(axis):
    """A 1-D mesh gives a tridiagonal A_sym; ILU(0) of a tridiagonal matrix drops nothing => M = A, M^-1 r = A^-1 r,
    and PCG converges in one iteration."""
    if axis == "r":
        m = grids.full_sphere_mesh(grids.radial_faces_pack(40, 4.0), 1, 1)
    else:
        m = grids.full_sphere_mesh(grids.radial_faces_ratio(1, 1.02), 40, 1)
    op = _op(m, 1e3)
    A = op.dense()
    assert np.count_nonzero(np.triu(A, 2)) == 0 and np.count_nonzero(np.diag(A, 1)) == 39
    rng = np.random.default_rng(5)
    r = rng.standard_normal(m.shape)
    pc = op.pc2()
    z = pc.apply(r).ravel()
    z_ref = np.linalg.solve(A, r.ravel())
    assert np.abs(z - z_ref).max() <= 1e-12 * np.abs(z_ref).max()
    b = rng.uniform(-1, 1, m.shape)
    st, k, x, h = op.pcg_pc2(pc, b, None, 1e-12, 50)
    assert st == ref.REF_OK and k == 1 and h[1] <= 1e-13
    x_ref = np.linalg.solve(A, (op.volume() * b).ravel())
    assert np.abs(x.ravel() - x_ref).max() <= 1e-12 * np.abs(x_ref).max()
    st1, k1, _, _ = op.pcg(b, None, 1e-12, 500)
    assert k1 > 5                                                  # PC1 needs many: the pin is not vacuous


def test_periodic_line_is_not_exact_but_close():
    """1-D in phi: cyclic tridiagonal.  ILU(0) keeps the wrap entries and drops their fill, so M != A, yet one
    application already reduces the residual far more than the diagonal does."""
    m = grids.full_sphere_mesh(grids.radial_faces_ratio(1, 1.02), 1, 64)
    op = _op(m, 1e3)
    A = op.dense()
    assert A[0, 63] != 0.0 and A[63, 0] != 0.0
    L, U = op.pc2().dense_factors()
    assert L[63, 0] != 0.0 and U[0, 63] != 0.0                    # the wrap coupling is inside the (whole-phi) box
    rng = np.random.default_rng(6)
    b = rng.uniform(-1, 1, m.shape)
    _, k2, x2, _ = op.pcg_pc2(op.pc2(), b, None, 1e-12, 200)
    _, k1, x1, _ = op.pcg(b, None, 1e-12, 200)
    assert 1 < k2 < k1 / 3
    Lc, Uc = op.pc2((0, 0, 32)).dense_factors()                   # two half-circle boxes: no wrap inside a box
    assert Lc[63, 0] == 0.0 and Uc[0, 63] == 0.0 and Lc[32, 31] == 0.0


def test_dt_zero_gives_the_diagonal():
    m = _tiny()
    op = ref.RefOperator(m, 0.0, 0, ONE)
    r = np.random.default_rng(7).standard_normal(m.shape)
    assert np.array_equal(op.pc2().apply(r), r / op.volume())
    st, k, x, _ = op.pcg_pc2(op.pc2(), r, None, 1e-14, 10)
    assert st == ref.REF_OK and k == 1 and np.allclose(x, r, rtol=1e-15)


@pytest.mark.parametrize("kind,boxes", [("tiny", (0, 0, 0)), ("tiny", (1, 1, 0)), ("general", (2, 2, 0)), ("general", (1, 1, 0))])
def test_pcg_pc2_against_dense_lu_and_true_residual(kind, boxes):
    m, op = _case(kind)
    A = op.dense()
    rng = np.random.default_rng(8)
    b, x0 = rng.uniform(-1, 1, m.shape), rng.standard_normal(m.shape)
    bs = (op.volume() * b).ravel()
    x_lu = np.linalg.solve(A, bs)
    pc = op.pc2(boxes)
    st, k, x, h = op.pcg_pc2(pc, b, x0, 1e-14, 500)
    assert st == ref.REF_OK and k <= A.shape[0]
    assert np.linalg.norm(x.ravel() - x_lu) / np.linalg.norm(x_lu) <= 1e-12
    assert abs(h[0] - np.linalg.norm(bs - A @ x0.ravel()) / np.linalg.norm(bs)) <= 1e-13 * h[0]
    for kk in (1, 3, 6):                                          # hist[k] is the true residual of iterate k
        _, k_, xk, hk = op.pcg_pc2(pc, b, x0, 0.0, kk)
        assert k_ == kk and np.array_equal(hk, h[: kk + 1])
        true = np.linalg.norm(bs - A @ xk.ravel()) / np.linalg.norm(bs)
        assert abs(hk[-1] - true) <= 1e-10 * true


def test_krylov_optimality_of_the_preconditioned_iterates():
    """x_k minimises the A-norm of the error over x0 + span{M^-1 r0, (M^-1 A) M^-1 r0, ...} (the defining property of
    preconditioned CG): checked for k = 1..5 against a dense brute-force minimiser built from the dense factors."""
    m, op = _case("general")
    boxes = (2, 2, 0)
    A = op.dense()
    L, U = op.pc2(boxes).dense_factors()
    Minv = np.linalg.inv(L @ U)
    rng = np.random.default_rng(9)
    b, x0 = rng.uniform(-1, 1, m.shape), rng.standard_normal(m.shape)
    bs = (op.volume() * b).ravel()
    xs = np.linalg.solve(A, bs)
    r0 = bs - A @ x0.ravel()
    pc = op.pc2(boxes)
    basis = [Minv @ r0]
    for k in range(1, 6):
        K = np.stack(basis, axis=1)
        Q, _ = np.linalg.qr(K)
        c = np.linalg.solve(Q.T @ A @ Q, Q.T @ r0)                 # minimise ||x0 + Q c - x*||_A
        x_opt = x0.ravel() + Q @ c
        _, kk, xk, _ = op.pcg_pc2(pc, b, x0, 0.0, k)
        assert kk == k
        e_opt, e_k = x_opt - xs, xk.ravel() - xs
        na = lambda e: np.sqrt(e @ A @ e)
        assert abs(na(e_k) - na(e_opt)) <= 1e-9 * na(e_opt)
        assert np.linalg.norm(xk.ravel() - x_opt) <= 1e-8 * np.linalg.norm(x_opt)
        basis.append(Minv @ (A @ basis[-1]))


def test_fewer_iterations_than_pc1_by_the_papers_factor():
    """~550 iterations with PC1 against 100-200 with PC2 on the hard (viscosity) solve: a factor
    2.75-5.5.  On a reduced config-3 mesh at the same stiffness (1e4) ILU(0) must do at least that well; smaller boxes
    can only weaken it (more couplings dropped), boxes of whole phi lines stay well ahead of PC1."""
    prob = configs.make("c3", (24, 36, 48))
    op = _op(prob.mesh, 1e4, prob.nu_kind, prob.nu)
    b = configs.rhs_blob(prob)
    _, k1, x1, _ = op.pcg(b, None, 1e-9, 5000)
    counts = {}
    for boxes in [(0, 0, 0), (1, 1, 0), (4, 4, 0), (4, 4, 12)]:
        st, k, x, _ = op.pcg_pc2(op.pc2(boxes), b, None, 1e-9, 5000)
        assert st == ref.REF_OK
        assert np.linalg.norm(x - x1) / np.linalg.norm(x1) <= 1e-6     # same solution (both stopped at rtol 1e-9)
        counts[boxes] = k
    assert k1 / counts[(0, 0, 0)] >= 2.75, (k1, counts)
    assert counts[(0, 0, 0)] <= counts[(4, 4, 0)] <= counts[(1, 1, 0)] < k1 / 2.75, (k1, counts)
    assert counts[(4, 4, 0)] <= counts[(4, 4, 12)] < k1, counts   # cutting phi lines weakens it further, still better than PC1


def test_zero_rhs_maxit_zero_and_nonfinite():
    m, op = _case("tiny")
    pc = op.pc2((1, 1, 0))
    st, k, x, h = op.pcg_pc2(pc, np.zeros(m.shape), np.ones(m.shape), 1e-10, 10)
    assert (st, k) == (ref.REF_OK, 0) and np.all(x == 0.0) and h[0] == 0.0
    b = np.random.default_rng(1).uniform(-1, 1, m.shape)
    st, k, x, h = op.pcg_pc2(pc, b, None, 1e-10, 0)
    assert (st, k) == (ref.REF_MAXIT, 0) and h[0] == 1.0
    b[1, 2, 3] = np.nan
    st, k, x, h = op.pcg_pc2(pc, b, None, 1e-10, 10)
    assert (st, k) == (ref.REF_EBREAKDOWN, 0) and np.all(x == 0.0)
