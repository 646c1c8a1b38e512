"""Pins for the oracle's RKL2 super time stepping (NEXT-1; "Runge-Kutta Legendre super
time-stepping (STS) scheme [21]").  The paper prints no formulas, so the scheme is pinned against what
its reference [21] and the mathematics fix: the closed-form stability polynomial
R_s(z) = a_s + b_s P_s(1 + w_1 z) with the Legendre polynomial P_s, second-order consistency with the
matrix exponential, conservation, and stability up to tau_max = (s^2+s-2)/4 * 2/lambda_max.  CPU only."""
import math

import numpy as np
import pytest
from numpy.polynomial import legendre

from mas_inputs import grids
from oracle import ref


def setup(bc=(0, 0), seed=11, shape=(5, 4, 6)):
    m = grids.wobbly_phi_mesh(grids.radial_faces_pack(shape[0], 4.0), shape[1], shape[2], seed)
    nu = 0.5 + np.random.default_rng(seed + 1).uniform(0, 1, shape[:2])
    op = ref.RefOperator(m, 1.0, 1, nu, bc)
    V = op.volume().ravel()
    Lsym = op.dense() - np.diag(V)                 # A_sym(dt=1) = V + Lsym
    return m, op, V, Lsym


def eig_M(V, Lsym):
    """M = -V^-1 Lsym is self-adjoint in the V inner product: symmetrise with V^1/2."""
    sv = np.sqrt(V)
    S = -(Lsym / sv[:, None]) / sv[None, :]
    lam, Q = np.linalg.eigh(S)
    return lam, Q / sv[:, None]                    # columns: eigenvectors of M


def test_lop_is_minus_Vinv_Lsym_and_lambda_bound_holds():
    m, op, V, Lsym = setup()
    u = np.random.default_rng(0).standard_normal(m.shape)
    assert np.allclose(op.lop(u).ravel(), -(Lsym @ u.ravel()) / V, rtol=1e-12, atol=1e-12)
    lam, _ = eig_M(V, Lsym)
    assert lam.max() <= 1e-9 * abs(lam.min())      # negative semidefinite
    assert abs(lam.min()) <= op.lambda_max_bound() <= 2.0 * np.max(np.diag(Lsym) / V) * (1 + 1e-12)


@pytest.mark.parametrize("s", [2, 3, 4, 7, 12])
def test_stability_polynomial_is_the_shifted_legendre_closed_form(s):
    m, op, V, Lsym = setup()
    lam, Q = eig_M(V, Lsym)
    w1 = 4.0 / (s * s + s - 2.0)
    b = 1.0 / 3.0 if s < 3 else (s * s + s - 2.0) / (2.0 * s * (s + 1.0))
    tau = 0.9 * (2.0 / w1) / abs(lam.min())        # inside the stability interval [-2/w1... ] scaled
    Ps = legendre.Legendre.basis(s)
    for idx in (0, len(lam) // 3, len(lam) // 2, len(lam) - 2):
        v = Q[:, idx].reshape(m.shape)
        out = op.sts(v, tau, s).ravel()
        R_expected = (1.0 - b) + b * Ps(1.0 + w1 * tau * lam[idx])
        R_observed = (out @ (V * Q[:, idx])) / (Q[:, idx] @ (V * Q[:, idx]))
        assert R_observed == pytest.approx(R_expected, rel=1e-10, abs=1e-12)
        assert np.allclose(out, R_expected * Q[:, idx], rtol=0, atol=1e-10 * np.abs(Q[:, idx]).max())


@pytest.mark.parametrize("s", [3, 6])
def test_local_error_against_matrix_exponential_is_third_order(s):
    m, op, V, Lsym = setup()
    lam, Q = eig_M(V, Lsym)
    u = np.random.default_rng(2).standard_normal(m.shape)
    coef = Q.T @ (V * u.ravel())                   # V-orthonormal eigenbasis
    errs = []
    for tau in (0.2 / abs(lam.min()), 0.1 / abs(lam.min())):
        exact = Q @ (np.exp(tau * lam) * coef)
        errs.append(np.linalg.norm(op.sts(u, tau, s).ravel() - exact))
    assert errs[0] / errs[1] == pytest.approx(8.0, rel=0.25)


def test_neumann_conserves_the_volume_integral_and_constants():
    m, op, V, Lsym = setup(bc=(1, 1))
    u = np.random.default_rng(3).standard_normal(m.shape)
    tau = 20.0 / op.lambda_max_bound()
    out = op.sts(u, tau, 9)
    assert (V * out.ravel()).sum() == pytest.approx((V * u.ravel()).sum(), rel=1e-12, abs=1e-12)
    one = np.ones(m.shape)
    assert np.allclose(op.sts(one, tau, 9), one, rtol=1e-13)


@pytest.mark.parametrize("s", [4, 10])
def test_stable_up_to_tau_max_and_unstable_well_beyond(s):
    m, op, V, Lsym = setup()
    lam, _ = eig_M(V, Lsym)
    tau_max = (s * s + s - 2.0) / 4.0 * 2.0 / abs(lam.min())
    u = np.random.default_rng(4).standard_normal(m.shape)
    vnorm = lambda a: math.sqrt((V * a.ravel() ** 2).sum())
    y = u
    for _ in range(20):
        y = op.sts(y, tau_max, s)
    assert vnorm(y) <= vnorm(u) * (1 + 1e-12)       # |R_s| <= 1 on the whole spectrum
    y = u
    for _ in range(6):
        y = op.sts(y, 4.0 * tau_max, s)
    assert vnorm(y) > 1e3 * vnorm(u)                # the limit is real


def test_one_super_step_approximates_the_implicit_solve_of_the_same_dt():
    """STS and the PCG path advance the same viscosity operator: for a smooth field and a
    small step, (I - tau M)^-1 u and RKL2 agree to O(tau^2)."""
    m, op, V, Lsym = setup(shape=(6, 6, 8))
    lam, Q = eig_M(V, Lsym)
    u = (np.sin(math.pi * (m.r_c - m.r_f[0]) / (m.r_f[-1] - m.r_f[0]))[:, None, None]
         * (np.sin(m.th_c) ** 2)[None, :, None] * np.cos(m.ph_c)[None, None, :])
    errs = []
    for tau in (0.4 / abs(lam.min()), 0.2 / abs(lam.min())):
        op.set_dt(tau)
        st, k, x_imp, _ = op.pcg(u, None, 1e-14, 1000)
        errs.append(np.abs(op.sts(u, tau, 5) - x_imp).max())
    assert errs[0] / errs[1] == pytest.approx(4.0, rel=0.3)
