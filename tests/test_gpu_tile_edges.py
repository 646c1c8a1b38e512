"""Ragged-tile sweep: phi sizes that straddle the 128-cell tile rows (tile-row remainders 2, 62, 64, 66,
126, 0, 2 ...), theta sizes around the tile heights, short r extents, both radial boundary kinds -- for every kernel
family, against the oracle.  Run on the B200 box:  pytest tests -m gpu"""
import numpy as np
import pytest

from mas_inputs import grids
from tests import helpers as H

pytestmark = pytest.mark.gpu

NPS = [2, 4, 62, 64, 66, 126, 128, 130, 190, 194, 254, 256, 258, 322]
NTS = [1, 2, 5, 6, 7, 8, 9, 15]


def _t(a):
    import torch
    return torch.from_numpy(np.ascontiguousarray(a, dtype=np.float64)).cuda()


def _case(nr, nt, np_, uniform, bc, seed):
    if uniform:
        mesh = grids.full_sphere_mesh(grids.radial_faces_pack(nr, 4.0), nt, np_)
        rng = np.random.default_rng(seed)
        nu = 0.5 + rng.uniform(0.0, 1.0, (nr, nt))
        dt = 200.0 / H.oracle_s1(mesh, 1, nu, bc)
        return mesh, dt, 1, nu
    return H.general_case(nr, nt, np_, seed=seed, s=200.0, bc=bc)


@pytest.mark.parametrize("uniform", [True, False])
@pytest.mark.parametrize("np_", NPS)
def test_stencil_kernels_all_tiles_ragged_phi(np_, uniform):
    """apply (A u) and lop (M u) through every stencil tile, theta size cycling with the phi size."""
    nt = NTS[NPS.index(np_) % len(NTS)]
    bc = [(0, 0), (1, 1), (0, 1)][NPS.index(np_) % 3]
    mesh, dt, nu_kind, nu = _case(5, nt, np_, uniform, bc, seed=np_)
    oref, gpu = H.both_ops(mesh, dt, nu_kind, nu, bc)
    u = np.random.default_rng(np_).standard_normal(mesh.shape)
    a_ref, l_ref = oref.apply(u), oref.lop(u)
    for tile in range(6):
        gpu.set_option("stencil_tile", tile)
        a = gpu.apply(_t(u)).cpu().numpy().reshape(mesh.shape)
        l = gpu.lop(_t(u)).cpu().numpy().reshape(mesh.shape)
        assert H.apply_gap(a, a_ref, f"edges apply np={np_} tile {tile}") <= H.APPLY_RTOL, (tile, "apply")
        assert H.apply_gap(l, l_ref, f"edges lop np={np_} tile {tile}") <= H.APPLY_RTOL, (tile, "lop")


@pytest.mark.parametrize("uniform", [True, False])
@pytest.mark.parametrize("np_", NPS)
def test_pcg_kernel_families_ragged_phi(np_, uniform):
    """A short solve with every K1 tile, both traffic forms of the iteration (q stored / q recomputed by every
    K2R tile) and the one-kernel path; 12 iterations compared entry by entry."""
    nt = NTS[(NPS.index(np_) + 3) % len(NTS)]
    bc = [(0, 0), (1, 0)][NPS.index(np_) % 2]
    mesh, dt, nu_kind, nu = _case(6, nt, np_, uniform, bc, seed=100 + np_)
    oref, gpu = H.both_ops(mesh, dt, nu_kind, nu, bc)
    rng = np.random.default_rng(np_)
    b, x0 = rng.uniform(-1, 1, mesh.shape), rng.standard_normal(mesh.shape)
    for tile, qrec, k2r_tile, persistent in [(0, 0, 0, 0), (1, 0, 0, 0), (2, 1, 0, 0), (3, 1, 1, 0), (4, 1, 2, 0),
                                             (5, 1, 3, 0), (6, 1, 4, 0), (0, 1, 5, 0), (0, 1, 1, 1)]:
        for name, val in (("persistent", persistent), ("tile", tile), ("qrecompute", qrec), ("k2r_tile", k2r_tile)):
            gpu.set_option(name, val)
        H.check_parity(gpu, oref, b, x0, 0.0, 12, label=f"np={np_} t{tile} q{qrec} k{k2r_tile} p{persistent}")


@pytest.mark.parametrize("nt", NTS)
def test_sts_ragged_theta(nt):
    mesh, dt, nu_kind, nu = _case(4, nt, 130, False, (1, 0), seed=nt)
    oref, gpu = H.both_ops(mesh, 1.0, nu_kind, nu, (1, 0))
    u = np.random.default_rng(nt).standard_normal(mesh.shape)
    tau = 40.0 / gpu.lambda_max()
    s = gpu.sts_stages(tau)
    y_ref = oref.sts(u, tau, s)
    for tile in range(6):
        gpu.set_option("stencil_tile", tile)
        ud = _t(u)
        gpu.sts_advance(ud, tau, s)
        assert np.abs(ud.cpu().numpy().reshape(mesh.shape) - y_ref).max() <= 1e-11 * np.abs(u).max(), tile
