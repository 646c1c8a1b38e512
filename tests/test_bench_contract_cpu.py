"""bench.py contract checks that need no GPU: the reference arm (= the oracle on host cores) prints ONE JSON
line with the agreed keys; the workload builder is seeded and rank-offset; helper functions parse their files."""
import json
import os
import subprocess
import sys

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def test_reference_arm_prints_one_json_line_with_contract_keys():
    out = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--workload", "c1",
                          "--steps", "2", "--warmup", "1"], capture_output=True, text=True, cwd=ROOT, timeout=300)
    assert out.returncode == 0, out.stderr
    lines = [l for l in out.stdout.splitlines() if l.strip()]
    assert len(lines) == 1
    d = json.loads(lines[0])
    for key in ("impl", "metric", "value", "unit", "n_gpus", "steps", "warmup", "ms_per_step", "higher_is_better",
                "scaling", "vs_baseline", "dtype", "data", "config", "cpu_baseline", "e2e", "gpu_launches"):
        assert key in d, key
    assert d["impl"] == "reference" and d["dtype"] == "f64" and d["data"] == "synthetic"
    assert d["cpu_baseline"]["kind"] == "oracle" and d["cpu_baseline"]["cores"] == 1
    assert d["e2e"]["h2d_bytes_per_step"] == 0 and d["e2e"]["d2h_bytes_per_step"] == 0
    assert d["value"] > 0 and d["vs_baseline"] is None and d["gpu_launches"] == 0
    assert "workload" in d["config"]


def test_reference_arm_is_silent_on_nonzero_ranks():
    env = dict(os.environ, RANK="1", WORLD_SIZE="2", LOCAL_RANK="1")
    out = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--workload", "c1",
                          "--steps", "1", "--warmup", "0", "--gpus", "2"], capture_output=True, text=True, cwd=ROOT,
                         env=env, timeout=300)
    assert out.returncode == 0 and out.stdout.strip() == ""


def test_workload_is_seeded_and_rank_offset():
    sys.path.insert(0, ROOT)
    import bench
    p0, dt0, b0, rtol, maxit, desc = bench.workload("c1", 0)
    p0b, _, b0b, *_ = bench.workload("c1", 0)
    p1, _, b1, *_ = bench.workload("c1", 1)
    assert np.array_equal(b0, b0b) and not np.array_equal(b0, b1)
    assert (rtol, maxit) == (1e-10, 1000) and "32x32x64" in desc and dt0 > 0
    assert bench.ncu_traffic("k_stencil_sts")[0] > 1e9         # committed ncu summary is readable, with provenance
    assert bench.ncu_traffic("k_stencil_sts")[1]
    peak, src = bench.hbm_peak()
    assert 5000 < peak < 9000 and ("measured" in src or "fallback" in src)
