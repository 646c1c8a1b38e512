"""Randomised pins for the ORACLE: the same mathematical facts as tests/test_oracle_pins.py and
tests/test_oracle_pc2_pins.py, on seeded RANDOM meshes -- odd sizes in every direction, non-uniform widths in r, theta
AND phi, nu varying in r and theta, every combination of radial boundary kinds -- so that an index or boundary slip
that the hand-picked cases happen to miss still fails.  CPU only; every case is a few hundred cells."""
import numpy as np
import pytest

from mas_inputs import grids
from oracle import ref


def _random_case(seed):
    rng = np.random.default_rng(1000 + seed)
    nr, nt, np_ = int(rng.integers(1, 7)), int(rng.integers(1, 7)), int(rng.integers(3, 9))
    r_f = 1.0 + np.concatenate(([0.0], np.cumsum(rng.uniform(0.05, 1.0, nr))))
    w_t = rng.uniform(0.5, 1.5, nt)
    th_f = np.concatenate(([0.0], np.cumsum(w_t))) * (np.pi / w_t.sum())
    th_f[-1] = np.pi
    w_p = rng.uniform(0.5, 1.5, np_)
    ph_f = np.concatenate(([0.0], np.cumsum(w_p))) * (2.0 * np.pi / w_p.sum())
    mesh = grids.mesh_from_faces(r_f, th_f, ph_f)
    mesh.sin_f[0] = 0.0
    mesh.sin_f[nt] = 0.0
    nu = rng.uniform(0.2, 3.0, (nr, nt))
    bc = (int(rng.integers(0, 2)), int(rng.integers(0, 2)))
    s = float(10.0 ** rng.uniform(0.0, 3.5))
    op = ref.RefOperator(mesh, 1.0, 1, nu, bc)
    op.set_dt(s / op.stiffness_max())
    return rng, mesh, nu, bc, op


@pytest.mark.parametrize("seed", range(12))
def test_random_mesh_operator_is_a_symmetric_m_matrix_with_the_closed_form_row_sums(seed):
    rng, mesh, nu, bc, op = _random_case(seed)
    A = op.dense()
    n = A.shape[0]
    assert np.array_equal(A, A.T)                                   # P3: bit-wise symmetric
    assert np.all(np.diag(A) > 0) and np.all(A[~np.eye(n, dtype=bool)] <= 0.0)
    np.linalg.cholesky(A)                                           # positive definite
    assert np.count_nonzero(A, axis=1).max() <= 7
    # P5: A 1 = V + dt * (conductance of the Dirichlet boundary faces of the cell); = V exactly with Neumann faces
    V = op.volume()
    extra = np.zeros(mesh.shape)
    geom = lambda f, i: nu[i] * mesh.r_f[f] ** 2 / mesh.dr_f[f]     # per theta row, without sin dth dph
    solid = (mesh.sin_c * mesh.dth_c)[:, None] * mesh.dph_c[None, :]
    one = (A @ np.ones(n)).reshape(mesh.shape)
    resid = one - V                                                  # = dt * boundary conductances
    if bc[0] == 0:
        extra[0] += geom(0, 0)[:, None] * solid
    if bc[1] == 0:
        extra[-1] += geom(mesh.nr, mesh.nr - 1)[:, None] * solid
    if extra.any():
        ratio = resid[extra > 0] / extra[extra > 0]                  # the same dt everywhere
        assert np.allclose(ratio, ratio.flat[0], rtol=1e-9) and ratio.flat[0] > 0
        assert np.abs(resid[extra == 0]).max() <= 1e-12 * np.abs(one).max()
    else:
        assert np.abs(resid).max() <= 1e-12 * np.abs(one).max()


@pytest.mark.parametrize("seed", range(12))
def test_random_mesh_pcg_with_both_preconditioners_against_dense_lu(seed):
    rng, mesh, nu, bc, op = _random_case(seed)
    A = op.dense()
    b, x0 = rng.uniform(-1, 1, mesh.shape), rng.standard_normal(mesh.shape)
    x_lu = np.linalg.solve(A, (op.volume() * b).ravel())
    st, k, x, h = op.pcg(b, x0, 1e-14, 5000)
    assert st == ref.REF_OK and k <= A.shape[0] + 2
    assert np.linalg.norm(x.ravel() - x_lu) <= 1e-11 * np.linalg.norm(x_lu)
    boxes = (int(rng.integers(0, 4)), int(rng.integers(0, 4)), int(rng.integers(0, 5)))
    pc = op.pc2(boxes)
    st2, k2, x2, h2 = op.pcg_pc2(pc, b, x0, 1e-14, 5000)
    assert st2 == ref.REF_OK and k2 <= k + 1                        # never worse than point Jacobi (up to one iteration)
    assert np.linalg.norm(x2.ravel() - x_lu) <= 1e-11 * np.linalg.norm(x_lu)


@pytest.mark.parametrize("seed", range(12))
def test_random_mesh_random_boxes_ilu0_property(seed):
    rng, mesh, nu, bc, op = _random_case(seed)
    boxes = (int(rng.integers(0, 4)), int(rng.integers(0, 4)), int(rng.integers(0, 5)))
    nr, nt, np_ = mesh.shape
    bi, bj, bk = [b if 0 < b <= n else n for b, n in zip(boxes, mesh.shape)]
    i, j, k = np.meshgrid(np.arange(nr), np.arange(nt), np.arange(np_), indexing="ij")
    ids = (((i // bi) * 64 + (j // bj)) * 64 + (k // bk)).ravel()
    A = op.dense()
    Ab = np.where(ids[:, None] == ids[None, :], A, 0.0)
    L, U = op.pc2(boxes).dense_factors()
    pat = Ab != 0.0
    assert not np.any((L != 0.0) & ~pat & ~np.eye(len(ids), dtype=bool)) and not np.any((U != 0.0) & ~pat)
    assert np.abs(L @ U - Ab)[pat].max() <= 1e-13 * np.abs(Ab).max()
    assert np.all(np.diag(U) > 0)
