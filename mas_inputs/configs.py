"""The five synthetic workloads of BASELINE.json (`configs[0..4]`), as seeded generators.

They stand in for the paper's production TDm flux-rope run (Sec. 3: ~11 M cells,
"extremely non-uniform grid", large uniform viscosity, ~70 / ~550 PCG iterations per solve),
whose mesh, coefficients and right-hand sides are not available.  Shapes and stiffness follow
it; every array is generated here.

No arithmetic of the method lives here.  The one number that depends on the operator -- the
time step `dt` that realises a requested stiffness `s` -- is read from
`dt_calibration.json`, which `oracle/calibrate_dt.py` writes by calling only `oracle/`.
For a mesh that is not in that file (reduced-size test cases) the caller passes `s1`
(tests obtain it from the oracle).
"""
from __future__ import annotations

import json
import os
from dataclasses import dataclass, field

import numpy as np

from . import grids

_CAL_PATH = os.path.join(os.path.dirname(os.path.abspath(__file__)), "dt_calibration.json")

BC_DIRICHLET = 0
BC_NEUMANN = 1

# (nr, nt, np) of BASELINE.json configs 1..5
FULL_SHAPES = {
    "c1": (32, 32, 64),
    "c2": (64, 96, 128),
    "c3": (128, 192, 256),
    "c4": (256, 256, 512),
    "c5": (192, 256, 384),
}
# stiffness s.  c2 runs at three values.
STIFFNESS = {"c1": 2.0, "c2": (10.0, 100.0, 1000.0), "c3": 1.0e4, "c4": 1.0e4, "c5": 100.0}
RTOL = {"c1": 1e-10, "c2": 1e-10, "c3": 1e-9, "c4": 0.0, "c5": 1e-9}
MAXIT = {"c1": 1000, "c2": 5000, "c3": 5000, "c4": 500, "c5": 2000}
SEED = {"c1": 0, "c2": 1, "c3": 2, "c4": 3, "c5": 4}


@dataclass
class Problem:
    name: str
    mesh: grids.Mesh
    nu_kind: int                 # 0: scalar nu[0]; 1: plane nu[nr, nt]
    nu: np.ndarray
    bc: tuple = (BC_DIRICHLET, BC_DIRICHLET)
    rtol: float = 1e-10
    maxit: int = 1000
    seed: int = 0
    stiffness: tuple = field(default_factory=tuple)

    def key(self) -> str:
        nr, nt, np_ = self.mesh.shape
        return f"{self.name}:{nr}x{nt}x{np_}"

    def s1(self) -> float:
        """max over cells of (d - V)/V at dt = 1 (with this nu), from the calibration file."""
        with open(_CAL_PATH) as f:
            cal = json.load(f)
        if self.key() not in cal["s1"]:
            raise KeyError(f"{self.key()} is not calibrated; pass s1 obtained from the oracle")
        return float(cal["s1"][self.key()])

    def dt_for(self, s: float, s1: float | None = None) -> float:
        return s / (self.s1() if s1 is None else s1)


def nu_profile(mesh: grids.Mesh, nu0: float = 1.0) -> np.ndarray:
    """Config 3: nu(r, theta) = nu0 * (1 + 0.5 tanh((r - 2)/0.3)) at cell centres, stored as
    the [nr][nt] plane although it does not depend on theta (Q17)."""
    prof = nu0 * (1.0 + 0.5 * np.tanh((mesh.r_c - 2.0) / 0.3))
    return np.ascontiguousarray(np.broadcast_to(prof[:, None], (mesh.nr, mesh.nt)))


MESH_KINDS = ("config", "nonuniform", "clustered")


def make(name: str, shape: tuple | None = None, mesh_kind: str = "config") -> Problem:
    """Problem `name` in {"c1".."c5"}; `shape` overrides the grid size (reduced test cases).
    mesh_kind (configs 3-5 only; the problem is then called name + "n" / name + "k"):
      "config"      BASELINE.json's mesh: packed in r, uniform in theta and phi;
      "nonuniform"  the same shape, nu profile, stiffness and right-hand side on grids.random_mesh: r, theta AND phi
                    widths varying by +-30 % ("non-uniform logically-rectangular", "extremely
                    non-uniform grid"): the kernels' general (non-uniform phi) instantiations;
      "clustered"   grids.clustered_mesh: cells packed in r AND theta around an "erupting region" at the inner boundary
                    near the equator, phi uniform, with a large UNIFORM nu: the stiffness then sits
                    in the r / theta couplings, which the phi-line domains of the GPU's PC2 do not contain."""
    nr, nt, np_ = shape if shape is not None else FULL_SHAPES[name]
    if mesh_kind != "config":
        assert name in ("c3", "c4", "c5") and mesh_kind in MESH_KINDS
        if mesh_kind == "nonuniform":
            mesh = grids.random_mesh(nr, nt, np_, seed=100 + SEED[name], amp=0.3)
            nu_kind, nu = 1, nu_profile(mesh)
        else:
            mesh = grids.clustered_mesh(nr, nt, np_)
            nu_kind, nu = 0, np.array([1.0])
        st = STIFFNESS[name]
        return Problem(name=name + {"nonuniform": "n", "clustered": "k"}[mesh_kind], mesh=mesh, nu_kind=nu_kind, nu=nu,
                       rtol=RTOL[name], maxit=MAXIT[name], seed=SEED[name], stiffness=(st,))
    if name in ("c1", "c2"):
        r_f = grids.radial_faces_ratio(nr, 1.02)
    else:
        r_f = grids.radial_faces_pack(nr, 4.0)
    mesh = grids.full_sphere_mesh(r_f, nt, np_)
    if name in ("c1", "c2"):
        nu_kind, nu = 0, np.array([1.0])
    else:
        nu_kind, nu = 1, nu_profile(mesh)
    st = STIFFNESS[name]
    return Problem(name=name, mesh=mesh, nu_kind=nu_kind, nu=nu, rtol=RTOL[name], maxit=MAXIT[name],
                   seed=SEED[name], stiffness=st if isinstance(st, tuple) else (st,))


# ----------------------------------------------------------------------------------------------
# right-hand sides / fields (physical, i.e. NOT volume-scaled)
# ----------------------------------------------------------------------------------------------
def _coords(mesh: grids.Mesh):
    return (mesh.r_c[:, None, None], mesh.th_c[None, :, None], mesh.ph_c[None, None, :])


def rhs_uniform(prob: Problem) -> np.ndarray:
    """Configs 1 and 4: uniform(-1, 1) from the config's seed, one call, C order (Q19)."""
    rng = np.random.default_rng(prob.seed)
    return rng.uniform(-1.0, 1.0, prob.mesh.shape)


def field_manufactured(prob: Problem) -> np.ndarray:
    """Config 2: u = sin(pi (r-1)/29) sin^2(theta) cos(3 phi) + 0.01 N(0,1) from seed 1.
    The right-hand side b = A u is formed by whoever owns an operator (tests: the oracle)."""
    r, th, ph = _coords(prob.mesh)
    rng = np.random.default_rng(prob.seed)
    u = np.sin(np.pi * (r - 1.0) / 29.0) * np.sin(th) ** 2 * np.cos(3.0 * ph)
    return u + 0.01 * rng.standard_normal(prob.mesh.shape)


def blob(mesh: grids.Mesh) -> np.ndarray:
    """Gaussian 'flux-rope-like' blob centred (1.3, pi/2, pi), widths 0.2 (Q18)."""
    r, th, ph = _coords(mesh)
    return np.exp(-0.5 * (((r - 1.3) / 0.2) ** 2 + ((th - 0.5 * np.pi) / 0.2) ** 2
                          + ((ph - np.pi) / 0.2) ** 2))


def rhs_blob(prob: Problem) -> np.ndarray:
    """Config 3: blob + 0.01 N(0,1) from seed 2."""
    rng = np.random.default_rng(prob.seed)
    return blob(prob.mesh) + 0.01 * rng.standard_normal(prob.mesh.shape)


class Chain:
    """Config 5 time-step proxy (Q20): rng(4) draws first uniform(-1,1,nsteps) for
    dt_k = dt0 (1 + 0.2 u_k), then one standard_normal(shape) per step.
    RHS_0 = blob + 0.05 N_0;  RHS_{k+1} = x_k + 0.05 N_{k+1};  x0 = 0 for step 0, x_{k-1} after."""

    def __init__(self, prob: Problem, nsteps: int = 100):
        self.prob = prob
        self.nsteps = nsteps
        self.rng = np.random.default_rng(prob.seed)
        self.dt_factor = 1.0 + 0.2 * self.rng.uniform(-1.0, 1.0, nsteps)
        self.state0 = blob(prob.mesh)

    def noise(self) -> np.ndarray:
        """Next 0.05*N(0,1) array (call once per step, in order)."""
        return 0.05 * self.rng.standard_normal(self.prob.mesh.shape)
