"""Shared test plumbing: build the oracle operator and the CUDA operator from the same inputs,
and the parity gates of BASELINE.json north_star (tolerances stated here, derived in DESIGN.md)."""
from __future__ import annotations

import numpy as np

from mas_inputs import configs, grids
from oracle import ref

# --- the gates (BASELINE.json north_star; readings Q9, Q10 of SURVEY.md 8(c)) ---
HIST_RTOL = 1e-10      # per-iteration relative residual: |h_gpu - h_ref| / h_ref, first 50 iterations
HIST_ITERS = 50
HIST_FLOOR = 1e-15     # absolute slack, applied ONLY to entries h_ref[j] < 1e-4 * h_ref[0]; every entry within four
                       # decades of the initial residual is gated on the raw relative gap (round 3; before, the slack
                       # applied to every entry).  Why not relative everywhere: the recurrence residual carries an
                       # ABSOLUTE rounding error of a few eps * h[0] on either side, which at h[j] = 1e-6 * h[0] already
                       # is 1e-10 relative.  Observed on the B200: 2.0e-10 relative at such an entry of a PC2 solve that
                       # gains two decades per iteration (a threshold of 1e3 * eps * h[0] was tried and fails there),
                       # and <= 1e-12 on every entry above the threshold (R5)
HIST_FLOOR_BELOW = 1e-4
X_RTOL = 1e-9          # final x, relative L2, compared at EQUAL iteration counts
APPLY_RTOL = 1e-14     # single matvec, relative to max |A u| (pure rounding-order difference; SURVEY 7 step 4.
                       # Observed on the B200, round 2: <= 3.7e-16 including config 3 at stiffness 1e4)


# observed GPU-vs-oracle gaps, collected per test and printed by conftest.pytest_terminal_summary
GAPS = []


def record_gap(label, **kw):
    GAPS.append((label, kw))


def apply_gap(y, y_ref, label):
    """max |y - y_ref| / max |y_ref| of a single matvec; recorded, returned for the assertion."""
    g = float(np.abs(y - y_ref).max() / max(np.abs(y_ref).max(), 1e-300))
    record_gap(label, apply=g)
    return g


def hist_gaps(h_g, h_r, m):
    """(gated, raw) largest relative gap over the first m history entries.  `raw` is |h_gpu - h_ref| / h_ref as it
    stands; `gated` is the same except that entries below HIST_FLOOR_BELOW * h_ref[0] get HIST_FLOOR of absolute
    slack (R5) -- it is what the gate tests.  Both are recorded so that the summary shows an observation,
    not the floor (parity hygiene)."""
    h_r = np.asarray(h_r[:m], dtype=np.float64)
    d = np.abs(np.asarray(h_g[:m]) - h_r)
    den = np.maximum(h_r, 1e-300)
    slack = np.where(h_r < HIST_FLOOR_BELOW * h_r[0], HIST_FLOOR, 0.0)
    return float((np.maximum(d - slack, 0.0) / den).max()), float((d / den).max())


def oracle_s1(mesh, nu_kind, nu, bc=(0, 0)) -> float:
    op = ref.RefOperator(mesh, 1.0, nu_kind, nu, bc)
    s1 = op.stiffness_max()
    op.close()
    return s1


def both_ops(mesh, dt, nu_kind, nu, bc=(0, 0)):
    from paper_1811_02605_b200 import MasPcg
    return ref.RefOperator(mesh, dt, nu_kind, nu, bc), MasPcg(mesh, dt, nu_kind, nu, bc)


def general_case(nr=9, nt=11, np_=70, seed=21, s=300.0, bc=(0, 0)):
    """Odd r/theta sizes, phi spanning a ragged second tile, non-uniform phi, nu(r, theta)."""
    mesh = grids.wobbly_phi_mesh(grids.radial_faces_pack(nr, 4.0), nt, np_, seed)
    rng = np.random.default_rng(seed + 1)
    nu = 0.5 + rng.uniform(0.0, 1.0, (nr, nt))
    dt = s / oracle_s1(mesh, 1, nu, bc)
    return mesh, dt, 1, nu


def check_parity(gpu, oref, b, x0, rtol, maxit, *, label=""):
    """Runs both solvers on the same inputs and applies the three gates.  Returns (k_ref, k_gpu)."""
    import torch
    st_r, k_r, x_r, h_r = oref.pcg(b, x0, rtol, maxit)
    bd = torch.from_numpy(np.ascontiguousarray(b)).cuda()
    xd = torch.zeros_like(bd) if x0 is None else torch.from_numpy(np.ascontiguousarray(x0)).cuda()
    st_g, k_g, h_g = gpu.solve(bd, xd, rtol, maxit)
    assert st_g == st_r, f"{label}: status gpu {st_g} vs oracle {st_r}"
    assert abs(k_g - k_r) <= 1, f"{label}: iterations gpu {k_g} vs oracle {k_r}"
    m = min(HIST_ITERS, k_r, k_g) + 1
    hist_gated, hist_raw = hist_gaps(h_g, h_r, m)
    assert hist_gated <= HIST_RTOL, f"{label}: history gap {hist_gated:.3e} (raw {hist_raw:.3e})"
    if k_g != k_r:      # Q10: compare x at equal iteration counts
        xd = torch.zeros_like(bd) if x0 is None else torch.from_numpy(np.ascontiguousarray(x0)).cuda()
        _, k_g2, _ = gpu.solve(bd, xd, 0.0, k_r)
        assert k_g2 == k_r
    xg = xd.cpu().numpy().reshape(x_r.shape)
    err = np.linalg.norm(xg - x_r) / np.linalg.norm(x_r)
    # element-wise: the largest single-cell gap relative to max |x| (a localised error in a few boundary
    # rows would hide under the L2 gate on a large mesh); reported, and gated at 100x the L2 tolerance
    emax = float(np.abs(xg - x_r).max() / np.abs(x_r).max())
    record_gap(label, hist=hist_gated, hist_raw=hist_raw, x_l2=float(err), x_max=emax, k_ref=k_r, k_gpu=k_g)
    assert err <= X_RTOL, f"{label}: x gap {err:.3e}"
    assert emax <= 100 * X_RTOL, f"{label}: element-wise x gap {emax:.3e}"
    return k_r, k_g
