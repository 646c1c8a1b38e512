"""The oracle reproduces its frozen output (tests/golden/, written by tests/golden/make_golden.py from oracle/
only).  Guards against silent changes to the oracle's arithmetic; never compared with the CUDA path."""
import os

import numpy as np

from mas_inputs import configs, grids
from oracle import ref

G = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden")


def _load(name):
    return np.array([float(l) for l in open(os.path.join(G, name)) if not l.startswith("#")])


def test_config1_history_matches_golden():
    gold = _load("oracle_history_c1.txt")
    prob = configs.make("c1")
    op = ref.RefOperator(prob.mesh, prob.dt_for(2.0), prob.nu_kind, prob.nu, prob.bc)
    st, k, x, hist = op.pcg(configs.rhs_uniform(prob), None, prob.rtol, prob.maxit)
    assert k + 1 == gold.size - 2
    assert np.allclose(hist, gold[:-2], rtol=1e-12, atol=0)
    assert np.allclose([x.sum(), (x * x).sum()], gold[-2:], rtol=1e-11, atol=0)


def test_sts_tiny_matches_golden():
    gold = _load("oracle_sts_tiny.txt")
    m = grids.wobbly_phi_mesh(grids.radial_faces_pack(5, 4.0), 4, 6, 11)
    nu = 0.5 + np.random.default_rng(12).uniform(0, 1, (5, 4))
    op = ref.RefOperator(m, 1.0, 1, nu, (0, 1))
    u = np.random.default_rng(13).standard_normal(m.shape)
    y = op.sts(u, 40.0 / op.lambda_max_bound(), 7)
    assert np.allclose(y.ravel(), gold, rtol=1e-12, atol=1e-14)
