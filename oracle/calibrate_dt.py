"""Writes mas_inputs/dt_calibration.json: for each BASELINE.json config mesh, S1 = max over cells of
(d - V)/V at dt = 1, so that dt = s / S1 realises stiffness s.

Calls only oracle/ (and the mesh generators in mas_inputs/, which hold no method arithmetic).
Run:  python -m oracle.calibrate_dt
"""
import json
import os

from mas_inputs import configs
from oracle import ref


def main():
    out = {"comment": "S1 = max_cells (d - V)/V at dt = 1; written by oracle/calibrate_dt.py (oracle only)",
           "s1": {}}
    cases = [(name, "config") for name in ("c1", "c2", "c3", "c4", "c5")]
    cases += [(name, kind) for kind in ("nonuniform", "clustered") for name in ("c3", "c4", "c5")]
    for name, kind in cases:
        prob = configs.make(name, mesh_kind=kind)
        op = ref.RefOperator(prob.mesh, 1.0, prob.nu_kind, prob.nu, prob.bc)
        out["s1"][prob.key()] = repr(op.stiffness_max())
        op.close()
        print(prob.key(), out["s1"][prob.key()])
    path = os.path.join(os.path.dirname(os.path.abspath(configs.__file__)), "dt_calibration.json")
    with open(path, "w") as f:
        json.dump(out, f, indent=1)
        f.write("\n")


if __name__ == "__main__":
    main()
