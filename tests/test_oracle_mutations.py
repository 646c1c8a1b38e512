"""Mutation check of the oracle's pins (What's weak #3): each single-token mutation of
oracle/mas_pcg_ref.c -- a dropped factor, a wrong index, a sign, a transposed operand -- is built in a temp
directory and the mathematical pin tests are run against it; at least one pin must fail.  The pins are the
ones in tests/test_oracle_pins.py, test_oracle_sts_pins.py, test_oracle_pc2_pins.py and test_oracle_random_pins.py; stored oracle outputs (golden files,
the dt calibration file) do NOT count as pins and are excluded (-k / --deselect below).

One mutation is expected to SURVIVE the mathematical pins and is listed as such: the face-nu mean (reading Q3).
Arithmetic vs harmonic mean of nu on a face are both consistent, symmetric, second-order discretisations, so
no closed form separates them; Q3 is a declared reading and is "parity unpinned".

CPU only.  Each mutation costs one gcc build plus the pin run up to its first failure (-x).
"""
import os
import shutil
import subprocess
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))

# (name, old text, new text, expected to be caught by a mathematical pin)
MUTATIONS = [
    ("phi_face_index", "g[4] = op->gp[(size_t)i * nt + j] / op->dph_f[km];",
     "g[4] = op->gp[(size_t)i * nt + j] / op->dph_f[k];", True),
    ("beta_inverted", "const double beta = rho1 / rho;", "const double beta = rho / rho1;", True),
    ("hist_from_rho", "h = sqrt(rr / bb);\n        if (hist) hist[k] = h;",
     "h = sqrt(rho1 / bb);\n        if (hist) hist[k] = h;", True),
    ("radial_face_rf_times_rc", "double g = nuf * r_f[i] * r_f[i] * sin_c[j] * dth_c[j] / dr_f[i];",
     "double g = nuf * r_f[i] * r_c[i < nr ? i : nr - 1] * sin_c[j] * dth_c[j] / dr_f[i];", True),
    ("boundary_nu_cell", "if (i == 0)        nuf = nu_at(nu_kind, nu, nt, 0, j);",
     "if (i == 0)        nuf = nu_at(nu_kind, nu, nt, nr - 1, j);", True),
    ("z_without_dinv", "else for (size_t c = 0; c < n; c++) z[c] = r[c] / d[c];",
     "else for (size_t c = 0; c < n; c++) z[c] = r[c];", True),
    ("theta_face_sin_c", "g = nuf * dr_c[i] * sin_f[j] / dth_f[j];", "g = nuf * dr_c[i] * sin_c[j] / dth_f[j];", True),
    ("dirichlet_neighbour_not_zero", "const double u_im = i > 0      ? u[c - (size_t)nt * np] : 0.0;\n"
     "                const double u_ip = i < nr - 1 ? u[c + (size_t)nt * np] : 0.0;\n"
     "                const double u_jm = j > 0      ? u[c - np] : 0.0;   /* g[2]",
     "const double u_im = i > 0      ? u[c - (size_t)nt * np] : uc;\n"
     "                const double u_ip = i < nr - 1 ? u[c + (size_t)nt * np] : 0.0;\n"
     "                const double u_jm = j > 0      ? u[c - np] : 0.0;   /* g[2]", True),
    ("rkl2_mu", "const double mu = (2.0 * j - 1.0) / j * bj / bjm1;", "const double mu = (2.0 * j + 1.0) / j * bj / bjm1;",
     True),
    ("rkl2_gamma_tilde", "const double gat = -(1.0 - bjm1) * mut;", "const double gat = -(1.0 - bj) * mut;", True),
    ("float_accumulator", "long double s = 0.0L;\n    for (size_t c = 0; c < n; c++) s += (long double)a[c] * (long double)b[c];",
     "float s = 0.0f;\n    for (size_t c = 0; c < n; c++) s += (float)(a[c] * b[c]);", True),
    ("volume_drops_r", "op->v2[(size_t)i * nt + j] = r_c[i] * r_c[i] * dr_c[i] * sin_c[j] * dth_c[j];",
     "op->v2[(size_t)i * nt + j] = r_c[i] * dr_c[i] * sin_c[j] * dth_c[j];", True),
    ("alpha_sign", "for (size_t c = 0; c < n; c++) r[c] -= alpha * q[c];", "for (size_t c = 0; c < n; c++) r[c] += alpha * q[c];",
     True),
    # PC2 (block-Jacobi ILU(0)); caught by tests/test_oracle_pc2_pins.py
    ("ilu_pivot_division_dropped", "pc->val[e] /= pc->val[pc->diag[k]];", ";", True),
    ("ilu_update_sign", "pc->val[f] -= lik * pc->val[t];", "pc->val[f] += lik * pc->val[t];", True),
    ("ilu_update_wrong_row", "for (size_t t = pc->diag[k] + 1; t < pc->rowptr[k + 1]; t++)",
     "for (size_t t = pc->rowptr[k]; t < pc->diag[k]; t++)", True),
    ("pc2_forward_sign", "for (size_t e = pc->rowptr[i]; e < pc->diag[i]; e++) s -= pc->val[e] * z[pc->col[e]];",
     "for (size_t e = pc->rowptr[i]; e < pc->diag[i]; e++) s += pc->val[e] * z[pc->col[e]];", True),
    ("pc2_backward_without_pivot", "z[i] = s / pc->val[pc->diag[i]];", "z[i] = s;", True),
    ("pc2_box_cut_in_phi_ignored", "if (ii / bi != i / bi || jj / bj != j / bj || kk / bk != k / bk) continue;",
     "if (ii / bi != i / bi || jj / bj != j / bj) continue;", True),
    ("pc2_wrap_coupling_dropped", "const int nb_k[6] = {k, k, k, k, km, kp};",
     "const int nb_k[6] = {k, k, k, k, k > 0 ? km : -1, kp};", True),
    # Q3: a declared reading, not fixed by mathematics -- expected to survive every mathematical pin
    ("face_nu_harmonic_mean_Q3",
     "else               nuf = 0.5 * (nu_at(nu_kind, nu, nt, i - 1, j) + nu_at(nu_kind, nu, nt, i, j));",
     "else               nuf = 2.0 / (1.0 / nu_at(nu_kind, nu, nt, i - 1, j) + 1.0 / nu_at(nu_kind, nu, nt, i, j));", False),
]

# stored oracle outputs are drift guards, not pins
NOT_PINS = ["--deselect", "tests/test_oracle_pins.py::test_calibration_file_matches_oracle"]


def _run_pins(repo, first=None):
    files = ["tests/test_oracle_pins.py", "tests/test_oracle_sts_pins.py", "tests/test_oracle_pc2_pins.py",
             "tests/test_oracle_random_pins.py"]
    if first:
        files = [first] + [f for f in files if f != first]
    cmd = [sys.executable, "-m", "pytest", *files, "-x", "-q",
           "-p", "no:cacheprovider", *NOT_PINS]
    env = dict(os.environ, PYTHONDONTWRITEBYTECODE="1")
    return subprocess.run(cmd, cwd=repo, env=env, capture_output=True, text=True, timeout=900)


@pytest.fixture(scope="module")
def sandbox(tmp_path_factory):
    """A private copy of oracle/, mas_inputs/, the pin tests and their helpers (nothing else)."""
    repo = tmp_path_factory.mktemp("mut")
    for d in ("oracle", "mas_inputs"):
        shutil.copytree(os.path.join(ROOT, d), repo / d, ignore=shutil.ignore_patterns("*.so", "__pycache__", "*.tmp"))
    os.makedirs(repo / "tests")
    for f in ("__init__.py", "helpers.py", "test_oracle_pins.py", "test_oracle_sts_pins.py", "test_oracle_pc2_pins.py",
              "test_oracle_random_pins.py"):
        shutil.copy(os.path.join(ROOT, "tests", f), repo / "tests" / f)
    open(repo / "tests" / "conftest.py", "w").write(
        "import os, sys\nsys.path.insert(0, os.path.dirname(os.path.dirname(os.path.abspath(__file__))))\n")
    shutil.copy(os.path.join(ROOT, "pytest.ini"), repo / "pytest.ini")
    return repo


def test_unmutated_oracle_passes_its_pins(sandbox):
    src = open(os.path.join(ROOT, "oracle", "mas_pcg_ref.c")).read()
    open(sandbox / "oracle" / "mas_pcg_ref.c", "w").write(src)
    so = sandbox / "oracle" / "libmas_pcg_ref.so"
    if so.exists():
        so.unlink()
    res = _run_pins(sandbox)
    assert res.returncode == 0, res.stdout[-2000:]


@pytest.mark.parametrize("name,old,new,caught", MUTATIONS, ids=[m[0] for m in MUTATIONS])
def test_mutation(sandbox, name, old, new, caught):
    src = open(os.path.join(ROOT, "oracle", "mas_pcg_ref.c")).read()
    assert src.count(old) == 1, f"mutation {name}: its anchor text must occur exactly once in the oracle"
    open(sandbox / "oracle" / "mas_pcg_ref.c", "w").write(src.replace(old, new))
    so = sandbox / "oracle" / "libmas_pcg_ref.so"
    if so.exists():
        so.unlink()
    first = ("tests/test_oracle_sts_pins.py" if name.startswith("rkl2") else
             "tests/test_oracle_pc2_pins.py" if name.startswith(("ilu", "pc2")) else None)
    res = _run_pins(sandbox, first=first)
    if caught:
        assert res.returncode != 0, f"mutation {name} survived every mathematical pin"
    else:
        assert res.returncode == 0, (f"mutation {name} is now caught by a pin -- promote it: drop the 'parity unpinned' "
                                     f"note on Q3 in DESIGN.md\n" + res.stdout[-1500:])
