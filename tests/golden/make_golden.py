"""Writes tests/golden/config1_sequences.json from the CPU oracle ONLY (never from the CUDA path).

Run:  python tests/golden/make_golden.py
Stored: for BASELINE.json config 1 (seed 1000) and each method, the per-step |I|, the FNV-1a hash of the
packed active set and the oracle's CG iteration counts, plus M-norms of y and u.  The GPU parity tests compare
against the live oracle; this file pins the oracle itself against silent drift (a change to it must be justified
in the commit that regenerates the file).
"""
import json
import os
import sys

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
sys.path.insert(0, ROOT)

from oracle import Oracle, OracleOptions, reference_eigs  # noqa: E402
from workloads import make_config  # noqa: E402


def main():
    w = make_config(1)
    o = Oracle.from_workload(w)
    yd, psi = w.target(0)
    theta, W = reference_eigs(w.rowptr, w.colidx, w.val, w.m, w.alpha, w.k)
    out = {"workload": w.name, "operator_sha256": w.operator_hash(), "theta": [float(t) for t in theta], "methods": {}}
    for name, meth in (("jacobi_cg", 0), ("refdef", 1), ("zeroext", 2)):
        o.reset_sequence()
        r = o.solve_query(meth, yd, psi, W, OracleOptions(pdas_cap=w.pdas_cap))
        out["methods"][name] = {
            "status": r["status"], "n_steps": r["n_steps"],
            "n_inactive": [s["n_inactive"] for s in r["steps"]],
            "active_hash": [f"{s['active_hash']:016x}" for s in r["steps"]],
            "cg_iters": [s["cg_iters"] for s in r["steps"]],
            "y_Mnorm": float(np.sqrt((w.m * r["y"] ** 2).sum())),
            "u_Mnorm": float(np.sqrt((w.m * r["u"] ** 2).sum())),
        }
    with open(os.path.join(os.path.dirname(os.path.abspath(__file__)), "config1_sequences.json"), "w") as f:
        json.dump(out, f, indent=1)


if __name__ == "__main__":
    main()
