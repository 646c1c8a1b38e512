"""Seeded, synthetic mesh generators shared by the oracle tests and the CUDA tests/bench.

This module holds NO arithmetic of the method (no operator, no diagonal, no PCG):
it only produces the 1-D metric arrays of MAS's "non-uniform logically-rectangular"
spherical (r, theta, phi) mesh (Sec. 2.2) in the layout `include/mas_pcg.h`
documents, i.e. the *inputs* that both sides consume.  numpy only.

Conventions:
  * faces r_f[0..nr], th_f[0..nt]; cell centres are face midpoints;
  * dr_f[i] is the centre-to-centre distance across radial face i, and the
    centre-to-boundary-face distance at i = 0 and i = nr (Dirichlet on the face);
  * sin_f[0] = sin_f[nt] = 0.0 exactly (polar faces have zero area);
  * phi is periodic: dph_f[k] is the distance from centre k to centre (k+1) mod np.
"""
from __future__ import annotations

from dataclasses import dataclass
import numpy as np

R_INNER = 1.0
R_OUTER = 30.0


@dataclass(frozen=True)
class Mesh:
    nr: int
    nt: int
    np_: int
    r_f: np.ndarray      # [nr+1]
    r_c: np.ndarray      # [nr]
    dr_c: np.ndarray     # [nr]
    dr_f: np.ndarray     # [nr+1]
    th_f: np.ndarray     # [nt+1]
    th_c: np.ndarray     # [nt]
    sin_c: np.ndarray    # [nt]
    dth_c: np.ndarray    # [nt]
    sin_f: np.ndarray    # [nt+1]
    dth_f: np.ndarray    # [nt+1]
    ph_c: np.ndarray     # [np]
    dph_c: np.ndarray    # [np]
    dph_f: np.ndarray    # [np]

    @property
    def shape(self):
        return (self.nr, self.nt, self.np_)

    @property
    def ncells(self):
        return self.nr * self.nt * self.np_

    def metric_arrays(self):
        """The ten 1-D arrays of `mas_metric_t`, in declaration order."""
        return (self.r_c, self.dr_c, self.r_f, self.dr_f, self.sin_c, self.dth_c,
                self.sin_f, self.dth_f, self.dph_c, self.dph_f)


def _geometric_faces(n: int, lo: float, hi: float, q: float) -> np.ndarray:
    """Faces lo = f[0] < ... < f[n] = hi with widths w[i] = w0 * q**i (last face forced to hi)."""
    w = q ** np.arange(n, dtype=np.float64)
    w *= (hi - lo) / w.sum()
    f = np.empty(n + 1, dtype=np.float64)
    f[0] = lo
    f[1:] = lo + np.cumsum(w)
    f[n] = hi
    return f


def radial_faces_ratio(nr: int, q: float, lo: float = R_INNER, hi: float = R_OUTER) -> np.ndarray:
    """Configs 1-2: 'geometric stretch ratio 1.02' => dr[i] = dr[0] * 1.02**i (Q16)."""
    return _geometric_faces(nr, lo, hi, q)


def radial_faces_pack(nr: int, pack: float = 4.0, lo: float = R_INNER, hi: float = R_OUTER) -> np.ndarray:
    """Configs 3-5: 'packs 4x more resolution near r=1' => dr[nr-1]/dr[0] = pack (Q15)."""
    q = pack ** (1.0 / (nr - 1)) if nr > 1 else 1.0
    return _geometric_faces(nr, lo, hi, q)


def mesh_from_faces(r_f: np.ndarray, th_f: np.ndarray, ph_f: np.ndarray) -> Mesh:
    """Build all metric arrays from face coordinates.  ph_f has np+1 entries spanning one period."""
    r_f = np.asarray(r_f, dtype=np.float64)
    th_f = np.asarray(th_f, dtype=np.float64)
    ph_f = np.asarray(ph_f, dtype=np.float64)
    nr, nt, np_ = r_f.size - 1, th_f.size - 1, ph_f.size - 1
    period = ph_f[-1] - ph_f[0]

    r_c = 0.5 * (r_f[:-1] + r_f[1:])
    dr_c = r_f[1:] - r_f[:-1]
    dr_f = np.empty(nr + 1)
    dr_f[1:nr] = r_c[1:] - r_c[:-1]
    dr_f[0] = r_c[0] - r_f[0]
    dr_f[nr] = r_f[nr] - r_c[nr - 1]

    th_c = 0.5 * (th_f[:-1] + th_f[1:])
    dth_c = th_f[1:] - th_f[:-1]
    sin_c = np.sin(th_c)
    sin_f = np.sin(th_f)
    dth_f = np.empty(nt + 1)
    dth_f[1:nt] = th_c[1:] - th_c[:-1]
    dth_f[0] = th_c[0] - th_f[0]
    dth_f[nt] = th_f[nt] - th_c[nt - 1]

    ph_c = 0.5 * (ph_f[:-1] + ph_f[1:])
    dph_c = ph_f[1:] - ph_f[:-1]
    dph_f = np.empty(np_)
    dph_f[:-1] = ph_c[1:] - ph_c[:-1]
    dph_f[-1] = ph_c[0] + period - ph_c[-1]

    return Mesh(nr, nt, np_, r_f, r_c, dr_c, dr_f, th_f, th_c, sin_c, dth_c, sin_f, dth_f,
                ph_c, dph_c, dph_f)


def full_sphere_mesh(r_f: np.ndarray, nt: int, np_: int) -> Mesh:
    """theta in (0, pi) uniform cell centres, phi periodic uniform (BASELINE.json config 1).
    Polar faces get sin_f = 0.0 exactly (Q5: set, do not evaluate sin(pi))."""
    th_f = np.pi * np.arange(nt + 1, dtype=np.float64) / nt
    ph_f = 2.0 * np.pi * np.arange(np_ + 1, dtype=np.float64) / np_
    m = mesh_from_faces(r_f, th_f, ph_f)
    m.sin_f[0] = 0.0
    m.sin_f[nt] = 0.0
    # uniform phi: make every width bit-identical (cumulative faces differ in the last ulp)
    m.dph_c[:] = 2.0 * np.pi / np_
    m.dph_f[:] = 2.0 * np.pi / np_
    return m


def wobbly_phi_mesh(r_f: np.ndarray, nt: int, np_: int, seed: int, amp: float = 0.3) -> Mesh:
    """Full sphere with a NON-uniform periodic phi mesh (Q21; the paper's grid is 'extremely
    non-uniform').  Widths are (1 + amp*U(-1,1)) renormalised to 2*pi."""
    rng = np.random.default_rng(seed)
    w = 1.0 + amp * rng.uniform(-1.0, 1.0, np_)
    w *= 2.0 * np.pi / w.sum()
    ph_f = np.concatenate(([0.0], np.cumsum(w)))
    ph_f[-1] = 2.0 * np.pi
    th_f = np.pi * np.arange(nt + 1, dtype=np.float64) / nt
    m = mesh_from_faces(r_f, th_f, ph_f)
    m.sin_f[0] = 0.0
    m.sin_f[nt] = 0.0
    return m


def random_mesh(nr: int, nt: int, np_: int, seed: int, amp: float = 0.3, uniform_phi: bool = False,
                r_lo: float = R_INNER, r_hi: float = R_OUTER, pack: float = 4.0) -> Mesh:
    """Full sphere, NON-uniform in r, theta and (unless uniform_phi) phi: the input class of the paper's mesh
    ("non-uniform logically-rectangular"; "extremely non-uniform grid").  r: the packed
    faces of radial_faces_pack with every width scaled by (1 + amp*U(-1,1)); theta, phi: widths (1 + amp*U(-1,1))
    renormalised to pi and 2*pi.  Polar faces get sin_f = 0.0 exactly.  np_ must be even (mas_grid_t)."""
    rng = np.random.default_rng(seed)
    w_r = np.diff(radial_faces_pack(nr, pack, r_lo, r_hi)) * (1.0 + amp * rng.uniform(-1.0, 1.0, nr))
    w_r *= (r_hi - r_lo) / w_r.sum()
    r_f = r_lo + np.concatenate(([0.0], np.cumsum(w_r)))
    r_f[-1] = r_hi
    w_t = 1.0 + amp * rng.uniform(-1.0, 1.0, nt)
    th_f = np.concatenate(([0.0], np.cumsum(w_t))) * (np.pi / w_t.sum())
    th_f[-1] = np.pi
    if uniform_phi:
        ph_f = 2.0 * np.pi * np.arange(np_ + 1, dtype=np.float64) / np_
    else:
        w_p = 1.0 + amp * rng.uniform(-1.0, 1.0, np_)
        ph_f = np.concatenate(([0.0], np.cumsum(w_p))) * (2.0 * np.pi / w_p.sum())
        ph_f[-1] = 2.0 * np.pi
    m = mesh_from_faces(r_f, th_f, ph_f)
    m.sin_f[0] = 0.0
    m.sin_f[nt] = 0.0
    if uniform_phi:
        m.dph_c[:] = 2.0 * np.pi / np_
        m.dph_f[:] = 2.0 * np.pi / np_
    return m


def clustered_mesh(nr: int, nt: int, np_: int, r_lo: float = 1.0, r_hi: float = 10.0, r_ratio: float = 200.0,
                   th_ratio: float = 20.0, th_width: float = 0.25) -> Mesh:
    """A paper-like mesh (r in [1, 10] solar radii, "extremely non-uniform", cells concentrated on the
    erupting region): geometric radial widths growing by `r_ratio` in total from the inner boundary outwards, theta
    widths `th_ratio` times finer at the equator than at the poles (a smooth Gaussian dip of width `th_width` rad
    around pi/2), phi uniform."""
    q = r_ratio ** (1.0 / max(nr - 1, 1))
    r_f = _geometric_faces(nr, r_lo, r_hi, q)
    xi = (np.arange(nt) + 0.5) / nt * np.pi
    w_t = 1.0 - (1.0 - 1.0 / th_ratio) * np.exp(-0.5 * ((xi - 0.5 * np.pi) / th_width) ** 2)
    th_f = np.concatenate(([0.0], np.cumsum(w_t))) * (np.pi / w_t.sum())
    th_f[-1] = np.pi
    ph_f = 2.0 * np.pi * np.arange(np_ + 1, dtype=np.float64) / np_
    m = mesh_from_faces(r_f, th_f, ph_f)
    m.sin_f[0] = 0.0
    m.sin_f[nt] = 0.0
    m.dph_c[:] = 2.0 * np.pi / np_
    m.dph_f[:] = 2.0 * np.pi / np_
    return m


def shell_wedge_mesh(nr: int, nt: int, np_: int, r_lo=1.0, r_hi=2.0) -> Mesh:
    """Uniform full-sphere mesh on r in [r_lo, r_hi]; used by the continuum-consistency pins."""
    r_f = np.linspace(r_lo, r_hi, nr + 1)
    return full_sphere_mesh(r_f, nt, np_)
