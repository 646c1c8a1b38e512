"""CPU-side checks of the C-ABI library: it loads, exports every symbol include/mas_pcg.h
declares, validates arguments before touching CUDA, and fails loudly (MAS_ECUDA) without a
device -- there is no CPU fallback.  No compute calls here."""
import ctypes
import os
import re

import numpy as np
import pytest

from mas_inputs import configs
from paper_1811_02605_b200 import binding as B

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def declared_functions():
    src = open(os.path.join(ROOT, "include", "mas_pcg.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(mas_pcg_[a-z_]+)\s*\(", src)))


def test_library_exports_every_declared_symbol():
    names = declared_functions()
    assert {"mas_pcg_create", "mas_pcg_solve", "mas_pcg_destroy", "mas_pcg_apply", "mas_pcg_set_dt",
            "mas_pcg_solve_host", "mas_pcg_solve_multi", "mas_pcg_strerror", "mas_pcg_stats", "mas_pcg_set_option",
            "mas_pcg_slabs_create", "mas_pcg_slabs_solve", "mas_pcg_slabs_destroy"} <= set(names)
    L = ctypes.CDLL(B._build.LIB) if os.path.exists(B._build.LIB) else B.lib()
    for n in names:
        assert hasattr(L, n), f"{n} declared in include/mas_pcg.h but not exported"


def test_measurement_probes_are_not_in_the_product_library():
    """include/mas_pcg_debug.h is a separate library: the product exports none of it."""
    dbg_src = open(os.path.join(ROOT, "include", "mas_pcg_debug.h")).read()
    probes = sorted(set(re.findall(r"\b(mas_pcg_dbg_[a-z_]+)\s*\(", re.sub(r"/\*.*?\*/", "", dbg_src, flags=re.S))))
    assert probes == ["mas_pcg_dbg_mix_probe", "mas_pcg_dbg_profile"]
    B.lib()
    prod, dbg = ctypes.CDLL(B._build.LIB), ctypes.CDLL(B._build.LIB_DBG)
    for n in probes:
        assert not hasattr(prod, n), f"{n} leaked into the product library"
        assert hasattr(dbg, n)
    for n in declared_functions():
        assert hasattr(dbg, n)
    assert not any("dbg" in n or "probe" in n or "profile" in n for n in declared_functions())


def test_python_binding_has_the_same_names():
    for n in declared_functions():
        assert hasattr(B, n), f"binding.{n} missing"


def test_strerror_covers_every_status():
    for st in (0, 1, -1, -2, -3, -4, -5):
        s = B.mas_pcg_strerror(st)
        assert s and s != "unknown status"
    assert B.mas_pcg_strerror(77) == "unknown status"


def _create_status(shape, arrays, dt, nu_kind, nu, bc=(0, 0)):
    try:
        h = B.mas_pcg_create(shape, arrays, dt, nu_kind, nu, bc)
    except B.MasError as e:
        return e.status
    B.mas_pcg_destroy(h)
    return 0


def test_create_validates_before_cuda():
    p = configs.make("c1", shape=(4, 4, 8))
    arrs = list(p.mesh.metric_arrays())
    ok = _create_status(p.mesh.shape, arrs, 1e-3, 0, p.nu)
    assert ok in (B.MAS_OK, B.MAS_ECUDA)            # MAS_ECUDA here: no device, no fallback
    assert _create_status((4, 4, 7), arrs, 1e-3, 0, p.nu) == B.MAS_EINVAL      # odd np
    assert _create_status((0, 4, 8), arrs, 1e-3, 0, p.nu) == B.MAS_EINVAL
    assert _create_status(p.mesh.shape, arrs, -1.0, 0, p.nu) == B.MAS_EINVAL   # dt < 0
    assert _create_status(p.mesh.shape, arrs, 1e-3, 0, np.array([0.0])) == B.MAS_EINVAL   # nu <= 0
    assert _create_status(p.mesh.shape, arrs, 1e-3, 2, p.nu) == B.MAS_EINVAL   # bad nu kind
    assert _create_status(p.mesh.shape, arrs, 1e-3, 0, p.nu, bc=(0, 3)) == B.MAS_EINVAL
    bad = [a.copy() for a in arrs]
    bad[1][2] = -bad[1][2]                                                     # negative dr_c
    assert _create_status(p.mesh.shape, bad, 1e-3, 0, p.nu) == B.MAS_EINVAL
    bad = [a.copy() for a in arrs]
    bad[2][1] = bad[2][3]                                                      # non-monotone r_f
    assert _create_status(p.mesh.shape, bad, 1e-3, 0, p.nu) == B.MAS_EINVAL


def test_null_handle_calls_are_einval_and_destroy_null_is_safe():
    L = B.lib()
    assert L.mas_pcg_solve(None, None, None, 0.0, 1, None, None, None) == B.MAS_EINVAL
    assert L.mas_pcg_apply(None, None, None, None) == B.MAS_EINVAL
    assert L.mas_pcg_set_dt(None, 1.0, None) == B.MAS_EINVAL
    assert L.mas_pcg_stats(None, None) == B.MAS_EINVAL
    assert L.mas_pcg_set_option(None, b"tile", 0) == B.MAS_EINVAL
    assert L.mas_pcg_solve_multi(None, 1, None, None, 0.0, 1, None, None, None, None) == B.MAS_EINVAL
    assert L.mas_pcg_slabs_solve(None, None, None, 0.0, 1, None, None, None) == B.MAS_EINVAL
    assert L.mas_pcg_slabs_set_dt(None, 1.0, None) == B.MAS_EINVAL
    L.mas_pcg_slabs_destroy(None)
    L.mas_pcg_destroy(None)


def test_product_path_does_not_import_the_oracle():
    """The CUDA package must never route through oracle/ (or any CPU fallback)."""
    pkg = os.path.join(ROOT, "paper_1811_02605_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h", ".inc")):
                txt = open(os.path.join(dirpath, f)).read()
                assert not re.search(r"^\s*(from|import)\s+oracle\b", txt, flags=re.M), f
                assert "mas_pcg_ref" not in txt, f
    for f in os.listdir(os.path.join(ROOT, "oracle")):
        if f.endswith((".py", ".c")):
            assert "paper_1811_02605_b200" not in open(os.path.join(ROOT, "oracle", f)).read().replace(
                "(paper_1811_02605_b200/csrc)", ""), f
