"""GPU parity for NEXT-1 (RKL2 super time stepping) and the marching stencil kernel behind it, against
the oracle, through the C ABI.  Run on the B200 box:  pytest tests -m gpu"""
import numpy as np
import pytest

from mas_inputs import configs
from tests import helpers as H

pytestmark = pytest.mark.gpu

LOP_RTOL = 1e-14      # one stencil application: rounding-order differences only (observed <= 4e-16 in round 2)
STS_RTOL = 1e-11      # s stages of such differences (s <= 64 here), relative to max |u|


def _t(a):
    import torch
    return torch.from_numpy(np.ascontiguousarray(a, dtype=np.float64)).cuda()


@pytest.mark.parametrize("tile", list(range(6)))
@pytest.mark.parametrize("shape,bc", [((9, 11, 70), (0, 0)), ((21, 19, 134), (1, 0)), ((1, 1, 2), (0, 0)),
                                      ((5, 17, 260), (1, 1)), ((40, 9, 128), (0, 1))])
def test_lop_and_apply_match_oracle_general_mesh(shape, bc, tile):
    mesh, dt, nu_kind, nu = H.general_case(*shape, bc=bc)
    oref, gpu = H.both_ops(mesh, dt, nu_kind, nu, bc)
    gpu.set_option("stencil_tile", tile)
    u = np.random.default_rng(1).standard_normal(mesh.shape)
    for fn_ref, fn_gpu in ((oref.lop, gpu.lop), (oref.apply, gpu.apply)):
        y_ref = fn_ref(u)
        y = fn_gpu(_t(u)).cpu().numpy().reshape(mesh.shape)
        assert H.apply_gap(y, y_ref, f"lop/apply {shape} tile {tile}") <= LOP_RTOL
    assert gpu.lambda_max() == pytest.approx(oref.lambda_max_bound(), rel=1e-12)


def test_lop_and_apply_uniform_phi():
    prob = configs.make("c3", shape=(40, 37, 192))
    oref, gpu = H.both_ops(prob.mesh, 1e-3, prob.nu_kind, prob.nu)
    u = configs.rhs_blob(prob)
    y_ref = oref.lop(u)
    y = gpu.lop(_t(u)).cpu().numpy()
    assert H.apply_gap(y, y_ref, "lop uniform") <= LOP_RTOL
    a_ref = oref.apply(u)
    assert H.apply_gap(gpu.apply(_t(u)).cpu().numpy(), a_ref, "apply uniform") <= H.APPLY_RTOL


@pytest.mark.parametrize("tile", list(range(6)))
@pytest.mark.parametrize("s", [2, 3, 5, 16, 64])
@pytest.mark.parametrize("uniform", [False, True])
def test_sts_advance_matches_oracle(s, uniform, tile):
    if uniform:
        prob = configs.make("c3", shape=(24, 21, 128))
        mesh, nu_kind, nu, bc = prob.mesh, prob.nu_kind, prob.nu, (0, 0)
        u = configs.rhs_blob(prob)
    else:
        mesh, _, nu_kind, nu = H.general_case(13, 10, 134)
        bc = (0, 1)
        u = np.random.default_rng(5).standard_normal(mesh.shape)
    oref, gpu = H.both_ops(mesh, 1.0, nu_kind, nu, bc)
    gpu.set_option("stencil_tile", tile)
    lam = gpu.lambda_max()
    lim = lambda n: (n * n + n - 2.0) / 4.0 * 2.0 / lam        # largest stable tau with n stages
    tau = 0.5 * (lim(s - 1) + lim(s)) if s > 2 else 0.9 * lim(2)  # needs exactly s stages
    assert gpu.sts_stages(tau) == s
    y_ref = oref.sts(u, tau, s)
    ud = _t(u)
    gpu.sts_advance(ud, tau, s)
    y = ud.cpu().numpy().reshape(mesh.shape)
    assert np.isfinite(y).all()
    assert np.abs(y - y_ref).max() <= STS_RTOL * np.abs(u).max()


def test_sts_conserves_volume_integral_with_neumann_and_rerun_is_bit_identical():
    mesh, _, nu_kind, nu = H.general_case(12, 13, 96, bc=(1, 1))
    oref, gpu = H.both_ops(mesh, 1.0, nu_kind, nu, (1, 1))
    V = oref.volume()
    u = np.random.default_rng(6).standard_normal(mesh.shape)
    tau = 30.0 / gpu.lambda_max()
    s = gpu.sts_stages(tau)
    outs = []
    for _ in range(2):
        ud = _t(u)
        gpu.sts_advance(ud, tau, s)
        outs.append(ud.cpu().numpy())
    assert outs[0].tobytes() == outs[1].tobytes()
    assert (V * outs[0]).sum() == pytest.approx((V * u).sum(), rel=1e-11, abs=1e-11)


def test_sts_then_pcg_solve_on_the_same_handle():
    """sts_advance borrows the PCG workspaces; a following solve must be unaffected."""
    prob = configs.make("c1")
    oref, gpu = H.both_ops(prob.mesh, prob.dt_for(2.0), prob.nu_kind, prob.nu)
    b = configs.rhs_uniform(prob)
    ud = _t(b)
    gpu.sts_advance(ud, 5.0 / gpu.lambda_max(), 4)
    H.check_parity(gpu, oref, b, None, prob.rtol, prob.maxit, label="after sts")


def test_sts_config4_full_size_eight_stages():
    """RKL2 against the oracle at the size `bench.py --workload sts` times (256 x 256 x 512, config 4's mesh and nu):
    one super-step of s = 8 stages, every cell compared ("What's missing" 5)."""
    prob = configs.make("c4")
    oref, gpu = H.both_ops(prob.mesh, 1.0, prob.nu_kind, prob.nu)
    u = configs.rhs_blob(prob)
    s = 8
    tau = 0.9 * (s * s + s - 2.0) / 4.0 * 2.0 / gpu.lambda_max()
    assert gpu.sts_stages(tau) == s
    y_ref = oref.sts(u, tau, s)
    ud = _t(u)
    gpu.sts_advance(ud, tau, s)
    gap = float(np.abs(ud.cpu().numpy().reshape(y_ref.shape) - y_ref).max() / np.abs(u).max())
    H.record_gap("sts c4 s=8", sts=gap)
    assert gap <= STS_RTOL


def test_sts_viscosity_advance_production_like_mesh():
    """The paper's regime: ~200 sub-steps per step with the large uniform viscosity."""
    prob = configs.make("c3", shape=(48, 64, 128))
    oref, gpu = H.both_ops(prob.mesh, 1.0, prob.nu_kind, prob.nu)
    u = configs.rhs_blob(prob)
    s = 200
    tau = 0.9 * (s * s + s - 2.0) / 4.0 * 2.0 / gpu.lambda_max()
    y_ref = oref.sts(u, tau, s)
    ud = _t(u)
    gpu.sts_advance(ud, tau, s)
    assert np.abs(ud.cpu().numpy() - y_ref).max() <= 1e-10 * np.abs(u).max()
