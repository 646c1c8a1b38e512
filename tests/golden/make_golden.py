"""Writes tests/golden/oracle_history_c1.txt and oracle_sts_tiny.txt.  Calls ONLY oracle/ (plus the seeded input
generators in mas_inputs/, which hold no method arithmetic).  Run:  python -m tests.golden.make_golden

The paper prints no worked numeric example for the PCG path, so there is no paper-printed fixture to
store; these files freeze the ORACLE's own output on BASELINE.json config 1 so that a later change to the oracle's
arithmetic cannot go unnoticed (such a change must name, in its commit message, the passage or DESIGN.md reading
that justifies it, and re-run this script).  They are never compared with the CUDA path."""
import os

import numpy as np

from mas_inputs import configs, grids
from oracle import ref

HERE = os.path.dirname(os.path.abspath(__file__))


def main():
    prob = configs.make("c1")
    op = ref.RefOperator(prob.mesh, prob.dt_for(2.0), prob.nu_kind, prob.nu, prob.bc)
    st, k, x, hist = op.pcg(configs.rhs_uniform(prob), None, prob.rtol, prob.maxit)
    with open(os.path.join(HERE, "oracle_history_c1.txt"), "w") as f:
        f.write("# BASELINE.json config 1 (32x32x64, s = 2, rtol 1e-10, RHS uniform(-1,1) seed 0): oracle PCG\n")
        f.write(f"# status {st} iterations {k}; one line per hist[j] = ||r_j|| / ||V.b||, then sum(x), sum(x^2)\n")
        for h in hist:
            f.write(repr(float(h)) + "\n")
        f.write(repr(float(x.sum())) + "\n" + repr(float((x * x).sum())) + "\n")
    m = grids.wobbly_phi_mesh(grids.radial_faces_pack(5, 4.0), 4, 6, 11)
    nu = 0.5 + np.random.default_rng(12).uniform(0, 1, (5, 4))
    op2 = ref.RefOperator(m, 1.0, 1, nu, (0, 1))
    u = np.random.default_rng(13).standard_normal(m.shape)
    y = op2.sts(u, 40.0 / op2.lambda_max_bound(), 7)
    with open(os.path.join(HERE, "oracle_sts_tiny.txt"), "w") as f:
        f.write("# RKL2, 7 stages, tau = 40/lambda_max_bound, 5x4x6 non-uniform mesh (seed 11), nu seed 12, u seed 13\n")
        for v in y.ravel():
            f.write(repr(float(v)) + "\n")


if __name__ == "__main__":
    main()
