"""Basis of the parity tolerances, measured on the ORACLE alone: how far does a
rounding-scale perturbation of the inputs move the residual history over the gated 50 iterations?
GPU and oracle differ only by rounding order, i.e. by perturbations of this size."""
import numpy as np

from mas_inputs import configs
from oracle import ref
from tests import helpers as H


def test_history_sensitivity_to_rounding_scale_perturbations_leaves_slack():
    prob = configs.make("c3", shape=(24, 32, 64))
    op = ref.RefOperator(prob.mesh, 1.0, prob.nu_kind, prob.nu, prob.bc)
    op.set_dt(1.0e4 / op.stiffness_max())                  # the stiffest setting any config uses
    b = configs.rhs_blob(prob)
    _, k0, _, h0 = op.pcg(b, None, 0.0, H.HIST_ITERS)
    rng = np.random.default_rng(17)
    worst = 0.0
    for _ in range(3):
        bp = b * (1.0 + 4.0 * np.finfo(float).eps * rng.uniform(-1, 1, b.shape))   # a few ulps per entry
        _, k1, _, h1 = op.pcg(bp, None, 0.0, H.HIST_ITERS)
        worst = max(worst, float(np.max(np.abs(h1 - h0) / h0)))
    assert k0 == H.HIST_ITERS
    assert worst > 0.0                      # the perturbation is visible ...
    assert worst <= H.HIST_RTOL * 1e-3      # ... and >= 3 digits below the 1e-10 gate
