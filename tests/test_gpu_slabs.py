"""GPU parity for the r-slab decomposition: the mesh split into slabs with
their own vectors, neighbours' boundary planes read through pointers inside the kernels, per-slab partial sums
combined in slab order.  The oracle is unchanged -- the undivided solve is the definition.  All slabs are driven
from one process on one device (the form testable with one GPU).  Run on the B200 box:  pytest tests -m gpu"""
import numpy as np
import pytest

from mas_inputs import configs
from tests import helpers as H

pytestmark = pytest.mark.gpu


def _t(a):
    import torch
    return torch.from_numpy(np.ascontiguousarray(a, dtype=np.float64)).cuda()


def _slabs(mesh, dt, nu_kind, nu, bc, split):
    from paper_1811_02605_b200 import MasPcgSlabs
    return MasPcgSlabs(mesh, dt, nu_kind, nu, bc, split)


SPLITS = {21: [[0, 21], [0, 10, 21], [0, 1, 2, 20, 21], [0, 5, 11, 16, 21], [0, 3, 6, 9, 12, 15, 18, 21]],
          40: [[0, 20, 40], [0, 7, 19, 33, 40]]}


@pytest.mark.parametrize("qrec", [0, 1])
@pytest.mark.parametrize("loop_mode", [1, 0])
@pytest.mark.parametrize("split", SPLITS[21])
def test_slabs_general_mesh_parity_and_bits(split, loop_mode, qrec):
    import torch
    bc = (0, 1)
    mesh, dt, nu_kind, nu = H.general_case(21, 19, 134, s=500.0, bc=bc)
    from oracle import ref
    oref = ref.RefOperator(mesh, dt, nu_kind, nu, bc)
    g = _slabs(mesh, dt, nu_kind, nu, bc, split)
    g.set_option("loop_mode", loop_mode)
    g.set_option("qrecompute", qrec)
    rng = np.random.default_rng(3)
    b, x0 = rng.uniform(-1, 1, mesh.shape), rng.standard_normal(mesh.shape)
    H.check_parity(g, oref, b, x0, 1e-10, 2000, label=f"slabs {len(split) - 1} m{loop_mode} q{qrec}")
    st = g.stats()
    assert st["loop_mode"] == loop_mode and st["persistent_grid_or_slabs"] == len(split) - 1
    runs = []
    for _ in range(3):
        xd = _t(x0)
        s_, k, h = g.solve(_t(b), xd, 1e-10, 2000)
        runs.append((k, h.tobytes(), xd.cpu().numpy().tobytes()))
    assert runs[0] == runs[1] == runs[2]


@pytest.mark.parametrize("split", SPLITS[40])
def test_slabs_uniform_phi_against_oracle_and_undivided_gpu_solve(split):
    import torch
    prob = configs.make("c3", shape=(40, 37, 192))
    s1 = H.oracle_s1(prob.mesh, prob.nu_kind, prob.nu)
    oref, gpu = H.both_ops(prob.mesh, 1e3 / s1, prob.nu_kind, prob.nu)
    g = _slabs(prob.mesh, 1e3 / s1, prob.nu_kind, prob.nu, prob.bc, split)
    b = configs.rhs_blob(prob)
    k_r, k_g = H.check_parity(g, oref, b, None, 1e-9, 3000, label=f"slabs uniform {len(split) - 1}")
    gpu.set_option("persistent", 0)
    bd, x1, x2 = _t(b), torch.zeros(prob.mesh.shape, dtype=torch.float64, device="cuda"), None
    st1, k1, h1 = gpu.solve(bd, x1, 1e-9, 3000)
    x2 = torch.zeros_like(x1)
    st2, k2, h2 = g.solve(bd, x2, 1e-9, 3000)
    assert (st1, k1) == (st2, k2)
    m = min(len(h1), len(h2))
    assert np.abs(h1[:m] - h2[:m]).max() <= 1e-11 * h1[0]          # same iterates up to the order of the sums
    assert float((x1 - x2).norm() / x1.norm()) <= 1e-10


def test_slabs_separate_allocations_zero_rhs_set_dt_and_breakdown():
    """The slabs' b and x need not be views of one array; zero RHS, dt = 0, and a NaN right-hand side behave as in
    the undivided solve."""
    import torch
    from paper_1811_02605_b200 import binding as B, MasError
    mesh, dt, nu_kind, nu = H.general_case(9, 6, 70, s=80.0)
    from oracle import ref
    oref = ref.RefOperator(mesh, dt, nu_kind, nu)
    split = [0, 4, 5, 9]
    g = _slabs(mesh, dt, nu_kind, nu, (0, 0), split)
    rng = np.random.default_rng(8)
    b = rng.uniform(-1, 1, mesh.shape)
    st_r, k_r, x_r, h_r = oref.pcg(b, None, 1e-11, 500)
    bs = [_t(b[lo:hi]) for lo, hi in zip(split[:-1], split[1:])]          # three independent allocations
    xs = [torch.zeros_like(t) for t in bs]
    st, k, h = B.mas_pcg_slabs_solve(g._h, [t.data_ptr() for t in bs], [t.data_ptr() for t in xs], 1e-11, 500,
                                     int(torch.cuda.current_stream().cuda_stream))
    assert st == st_r and abs(k - k_r) <= 1
    if k == k_r:
        xg = torch.cat(xs).cpu().numpy()
        assert np.linalg.norm(xg - x_r) / np.linalg.norm(x_r) <= H.X_RTOL
    z = torch.zeros(mesh.shape, dtype=torch.float64, device="cuda")
    x = torch.ones_like(z)
    st, k, h = g.solve(z, x, 1e-10, 10)
    assert (st, k) == (0, 0) and not x.any()
    g.set_dt(0.0)                                                          # A = diag(V): one iteration, x = b
    bd = _t(b)
    st, k, h = g.solve(bd, x, 1e-12, 10)
    assert (st, k) == (0, 1) and torch.allclose(x, bd, rtol=1e-15, atol=0)
    g.set_dt(dt)
    bad = b.copy()
    bad[7, 1, 2] = np.nan
    x.zero_()
    with pytest.raises(MasError) as e:
        g.solve(_t(bad), x, 1e-10, 10)
    assert e.value.status == -4 and e.value.iters == 0 and not x.any()


def test_slabs_config3_full_size_4_slabs_first_60_iterations():
    prob = configs.make("c3")
    from oracle import ref
    dt = prob.dt_for(1e4)
    oref = ref.RefOperator(prob.mesh, dt, prob.nu_kind, prob.nu, prob.bc)
    g = _slabs(prob.mesh, dt, prob.nu_kind, prob.nu, prob.bc, [0, 32, 64, 96, 128])
    H.check_parity(g, oref, configs.rhs_blob(prob), None, 0.0, 60, label="slabs c3/60 4 slabs")


def test_slabs_create_rejects_bad_splits():
    from paper_1811_02605_b200 import MasError
    mesh, dt, nu_kind, nu = H.general_case(6, 4, 8)
    for split in ([0, 3, 3, 6], [1, 6], [0, 5], [0, 7], list(range(0, 7)) + [6] * 12):
        with pytest.raises(MasError) as e:
            _slabs(mesh, dt, nu_kind, nu, (0, 0), split)
        assert e.value.status == -1
