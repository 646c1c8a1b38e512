import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (run on the B200 box)")


def pytest_collection_modifyitems(config, items):
    """GPU tests are skipped (not failed) where no device exists, e.g. a plain `pytest tests/` here."""
    try:
        import torch
        has_gpu = torch.cuda.is_available()
    except Exception:  # pragma: no cover
        has_gpu = False
    if has_gpu:
        return
    skip = pytest.mark.skip(reason="no CUDA device")
    for item in items:
        if "gpu" in item.keywords:
            item.add_marker(skip)


def pytest_terminal_summary(terminalreporter):
    """Observed GPU-vs-oracle gaps (print what is seen, not only that the gate held)."""
    from tests import helpers
    if not helpers.GAPS:
        return
    tr = terminalreporter
    tr.write_sep("-", "observed GPU-vs-oracle gaps")
    worst = {}
    for label, kw in helpers.GAPS:
        for k, v in kw.items():
            if k.startswith("k_"):
                continue
            if k not in worst or v > worst[k][0]:
                worst[k] = (v, label)
    for k, (v, label) in sorted(worst.items()):
        tr.write_line(f"max {k:6s} = {v:.3e}   ({label})")
    big = [(l, kw) for l, kw in helpers.GAPS if any(t in l for t in ("c3", "c4", "c5", "128x192x256"))
           and "x_l2" in kw and "x_max" in kw]
    for label, kw in big:
        raw = f" (raw {kw['hist_raw']:.2e})" if "hist_raw" in kw else ""
        tr.write_line(f"{label}: hist {kw['hist']:.2e}{raw}  x_l2 {kw['x_l2']:.2e}  x_max {kw['x_max']:.2e}  "
                      f"k {kw['k_gpu']}/{kw['k_ref']}")
