"""GPU parity for batched right-hand sides (the three components of v share one
coefficient set): mas_pcg_solve_multi against the oracle's mas_ref_pcg_multi (= three independent textbook solves),
per right-hand side, and bit-identity with three single GPU solves.  Run on the B200 box:  pytest tests -m gpu"""
import numpy as np
import pytest

from mas_inputs import configs
from oracle import ref
from tests import helpers as H

pytestmark = pytest.mark.gpu


def _t(a):
    import torch
    return torch.from_numpy(np.ascontiguousarray(a, dtype=np.float64)).cuda()


def _check_multi(gpu, oref, bs, x0s, rtol, maxit, label, bitwise_vs_single=True):
    """Per right-hand side: status, count within +-1, history gate, x gate at equal counts; and the batched GPU
    solve reproduces single GPU solves bit for bit."""
    import torch
    nrhs = len(bs)
    worst_r, st_r, k_r, x_r, h_r = oref.pcg_multi(np.stack(bs), None if x0s is None else np.stack(x0s), rtol, maxit)
    bd = [_t(b) for b in bs]
    xd = [torch.zeros_like(bd[0]) if x0s is None else _t(x0s[j]) for j in range(nrhs)]
    worst_g, st_g, k_g, h_g = gpu.solve_multi(bd, xd, rtol, maxit)
    stats = gpu.stats()
    # one K1 + one K2 per iteration for the whole batch; the host-driven loop launches whole chunks of 16 iterations
    # whose kernels return at once after the end, and counts every launch
    want = 2 * max(k_g) if stats["loop_mode"] == 1 else 2 * min(maxit, 16 * ((max(k_g) + 15) // 16))
    assert stats["loop_launches"] == want, (stats, k_g)
    assert st_g == st_r, f"{label}: statuses gpu {st_g} vs oracle {st_r}"
    assert worst_g == worst_r
    for j in range(nrhs):
        assert abs(k_g[j] - k_r[j]) <= 1, f"{label} rhs {j}: iterations gpu {k_g[j]} vs oracle {k_r[j]}"
        m = min(H.HIST_ITERS, k_r[j], k_g[j]) + 1
        hist_gated, hist_raw = H.hist_gaps(h_g[j], h_r[j], m)
        assert hist_gated <= H.HIST_RTOL, f"{label} rhs {j}: history gap {hist_gated:.3e} (raw {hist_raw:.3e})"
        if k_g[j] == k_r[j] and np.abs(x_r[j]).max() > 0:
            xg = xd[j].cpu().numpy()
            err = np.linalg.norm(xg - x_r[j]) / np.linalg.norm(x_r[j])
            H.record_gap(f"{label} rhs {j}", hist=hist_gated, hist_raw=hist_raw, x_l2=float(err),
                         x_max=float(np.abs(xg - x_r[j]).max() / np.abs(x_r[j]).max()), k_ref=k_r[j], k_gpu=k_g[j])
            assert err <= H.X_RTOL, f"{label} rhs {j}: x gap {err:.3e}"
    if bitwise_vs_single:
        for j in range(nrhs):
            x1 = torch.zeros_like(bd[0]) if x0s is None else _t(x0s[j])
            st1, k1, h1 = gpu.solve(bd[j], x1, rtol, maxit)
            assert (st1, k1) == (st_g[j], k_g[j]) and np.array_equal(h1, h_g[j]) and torch.equal(x1, xd[j]), \
                f"{label} rhs {j}: batched solve differs from the single solve"
    return k_g


@pytest.mark.parametrize("qrec", [0, 1])
@pytest.mark.parametrize("loop_mode", [1, 0])
def test_multi_general_mesh_independent_convergence(loop_mode, qrec):
    """Three right-hand sides of very different difficulty: a zero one (done at once), a smooth one, a rough one
    with a warm start; each converges at its own iteration and drops out."""
    mesh, dt, nu_kind, nu = H.general_case(21, 19, 134, s=500.0)
    oref, gpu = H.both_ops(mesh, dt, nu_kind, nu)
    gpu.set_option("persistent", 0)
    gpu.set_option("loop_mode", loop_mode)
    gpu.set_option("qrecompute", qrec)
    rng = np.random.default_rng(3)
    bs = [np.zeros(mesh.shape), np.ones(mesh.shape), rng.uniform(-1, 1, mesh.shape)]
    x0s = [rng.standard_normal(mesh.shape) for _ in range(3)]
    k = _check_multi(gpu, oref, bs, x0s, 1e-10, 2000, f"multi general m{loop_mode} q{qrec}")
    assert k[0] == 0 and len(set(k)) == 3
    # two right-hand sides, and an iteration cap that only one of them hits
    _check_multi(gpu, oref, bs[1:], None, 1e-10, k[1] + 2 if k[1] < k[2] else k[2] + 2, "multi capped")


def test_multi_config1_full():
    prob = configs.make("c1")
    oref, gpu = H.both_ops(prob.mesh, prob.dt_for(2.0), prob.nu_kind, prob.nu)
    bs = []
    for j in range(3):
        prob.seed = j
        bs.append(configs.rhs_uniform(prob))
    gpu.set_option("persistent", 0)              # single solves on the same path, for the bit-identity check
    _check_multi(gpu, oref, bs, None, prob.rtol, prob.maxit, "multi c1")


def test_multi_vs_single_small_mesh_with_persistent_left_at_its_default():
    """include/mas_pcg.h, mas_pcg_solve_multi: with "persistent" at its default (1) a single solve of a small mesh
    runs in the cooperative kernel and a batched one in the streaming kernels; the header promises agreement to
    rounding there (bit-identity only when both run the same kernels, which the tests above check with persistent = 0)."""
    import torch
    prob = configs.make("c1")
    oref, gpu = H.both_ops(prob.mesh, prob.dt_for(2.0), prob.nu_kind, prob.nu)
    bs = []
    for j in range(3):
        prob.seed = 10 + j
        bs.append(configs.rhs_uniform(prob))
    k_multi = _check_multi(gpu, oref, bs, None, prob.rtol, prob.maxit, "multi c1 default", bitwise_vs_single=False)
    bd = [_t(b) for b in bs]
    xm = [torch.zeros_like(bd[0]) for _ in range(3)]
    _, st_m, k_m, h_m = gpu.solve_multi(bd, xm, prob.rtol, prob.maxit)
    assert gpu.stats()["loop_mode"] in (0, 1)
    assert k_m == k_multi
    for j in range(3):
        x1 = torch.zeros_like(bd[0])
        st1, k1, h1 = gpu.solve(bd[j], x1, prob.rtol, prob.maxit)
        assert gpu.stats()["loop_mode"] == 2, "config 1 should take the one-kernel solve by default"
        assert st1 == st_m[j] and abs(k1 - k_m[j]) <= 1
        m = min(H.HIST_ITERS, k1, k_m[j]) + 1
        rel = np.abs(h1[:m] - h_m[j][:m]) / h_m[j][:m]
        assert rel.max() <= H.HIST_RTOL, f"rhs {j}: history gap {rel.max():.3e} between the two kernel families"
        if k1 == k_m[j]:
            gap = float((x1 - xm[j]).norm() / xm[j].norm())
            H.record_gap(f"multi-vs-persistent c1 rhs {j}", multi_x_l2=gap, multi_hist=float(rel.max()))
            assert gap <= H.X_RTOL


def test_multi_config3_full_size_first_60_iterations():
    prob = configs.make("c3")
    oref, gpu = H.both_ops(prob.mesh, prob.dt_for(1e4), prob.nu_kind, prob.nu)
    bs = []
    for j in range(3):
        prob.seed = 2 + j
        bs.append(configs.rhs_blob(prob))
    _check_multi(gpu, oref, bs, None, 0.0, 60, "multi c3/60")


def test_multi_config5_full_size_three_steps_of_the_chain_as_one_batch():
    """config 5's mesh and stiffness; the batch = the chain's first right-hand side with three noise draws."""
    prob = configs.make("c5")
    oref, gpu = H.both_ops(prob.mesh, prob.dt_for(100.0), prob.nu_kind, prob.nu)
    chain = configs.Chain(prob, 100)
    bs = [chain.state0 + chain.noise() for _ in range(3)]
    k = _check_multi(gpu, oref, bs, None, prob.rtol, prob.maxit, "multi c5", bitwise_vs_single=False)
    assert all(30 <= kj <= 120 for kj in k)


def test_multi_breakdown_in_one_rhs_leaves_the_others_alone():
    import torch
    mesh, dt, nu_kind, nu = H.general_case(12, 10, 66, s=50.0)
    oref, gpu = H.both_ops(mesh, dt, nu_kind, nu)
    rng = np.random.default_rng(5)
    bs = [rng.uniform(-1, 1, mesh.shape) for _ in range(3)]
    bs[1][2, 3, 4] = np.nan
    worst_r, st_r, k_r, x_r, h_r = oref.pcg_multi(np.stack(bs), None, 1e-10, 500)
    assert st_r == [0, ref.REF_EBREAKDOWN, 0] and worst_r == ref.REF_EBREAKDOWN
    bd = [_t(b) for b in bs]
    xd = [torch.zeros_like(bd[0]) for _ in range(3)]
    worst_g, st_g, k_g, h_g = gpu.solve_multi(bd, xd, 1e-10, 500)
    assert (worst_g, st_g) == (worst_r, st_r) and k_g[1] == 0
    for j in (0, 2):
        assert abs(k_g[j] - k_r[j]) <= 1
        if k_g[j] == k_r[j]:
            assert np.linalg.norm(xd[j].cpu().numpy() - x_r[j]) / np.linalg.norm(x_r[j]) <= H.X_RTOL


def test_multi_argument_errors():
    import torch
    from paper_1811_02605_b200 import MasError
    mesh, dt, nu_kind, nu = H.general_case(4, 4, 8)
    _, gpu = H.both_ops(mesh, dt, nu_kind, nu)
    v = [torch.zeros(mesh.shape, dtype=torch.float64, device="cuda") for _ in range(5)]
    for bs, xs in [(v[:4], v[:4]), ([v[0], v[1]], [v[2], v[2]]), ([v[0], v[1]], [v[1], v[2]]), ([], [])]:
        with pytest.raises(MasError) as e:
            gpu.solve_multi(bs, xs, 1e-10, 10)
        assert e.value.status == -1
