"""Writes tests/golden/fullsize_query_c<config>.json / .npz from the CPU oracle ONLY (never from the CUDA path).

Run:  python tests/golden/make_golden_fullsize_query.py [config | config:steps ...]   (no arguments: 3, 78 min of 8-thread oracle time;
      "5:3" = only the first 3 PDAS steps of config 5)

One COMPLETE PDAS query (eq. (7)-(8), Algorithm 1 inside every step) at BASELINE.json's full size: query 0 of the sequence
from the all-active start of PAPER.md:339, RefDef (direct restriction) with the paper's analytical sine reference
(oracle.sine_reference, a deterministic closed form), at the paper's accuracy (verified relative residual
1e-10, recurrence trigger 1e-11) so that the active-set decisions sit above the solver's noise, PDAS cap 400.
Stored per step: FNV-1a hash of the packed active set, |I|, CG iterations, retained rank, status, margin (json); y at 65,536
seeded sample positions with the M-norm of y and u over those positions (npz).  tests/test_gpu_fullsize_query_golden.py runs
the same query through the C ABI and compares.  The oracle is the threaded build of the same source
(oracle.Oracle(..., threaded=True)): sums are taken in another order, nothing else differs.
"""
import json
import os
import sys
import time

import numpy as np

HERE = os.path.dirname(os.path.abspath(__file__))
ROOT = os.path.dirname(os.path.dirname(HERE))
sys.path.insert(0, ROOT)

import oracle  # noqa: E402
from workloads import make_config  # noqa: E402

EPS, EPS_C, PDAS_CAP, N_SAMPLES = 1e-10, 1e-11, 400, 65536


def run(config, first_steps=None):
    """first_steps = None: the complete query.  first_steps = s: only the first s PDAS steps (the query then ends with the
    step-cap status; used where the complete query is out of reach: config 5 needs 95 steps of 12 minutes each), at
    BASELINE.json's accuracy 1e-8 / 1e-8 (cond(H) ~ 1e6 on the 160^3 mesh: 1e-10 is at the limit of double precision)."""
    w = make_config(config)
    assert w.nt == 1
    o = oracle.Oracle.from_workload(w, threaded=True)
    W = np.asfortranarray(oracle.sine_reference(w.dims, w.k)[-1])
    yd, psi = w.target(0)
    t0 = time.time()
    eps, eps_c, cap = (EPS, EPS_C, PDAS_CAP) if first_steps is None else (1e-8, 1e-8, first_steps)
    r = o.solve_query(oracle.REFDEF, yd, psi, W, oracle.OracleOptions(eps=eps, eps_c=eps_c, pdas_cap=cap))
    dt = time.time() - t0
    pos = np.sort(np.random.default_rng(777 + config).choice(w.N, size=min(N_SAMPLES, w.N), replace=False))
    out = {"config": config, "workload": w.name, "N": w.N, "k": w.k, "operator_sha256": w.operator_hash(), "eps": eps, "eps_c": eps_c,
           "pdas_cap": cap, "first_steps_only": first_steps is not None, "method": "refdef, analytical sine reference", "query": 0, "status": r["status"], "n_steps": r["n_steps"],
           "kkt": [float(v) for v in r["kkt"]], "n_inactive": [s["n_inactive"] for s in r["steps"]],
           "active_hash": [f"{s['active_hash']:016x}" for s in r["steps"]], "cg_iters": [s["cg_iters"] for s in r["steps"]],
           "rank_used": [s["rank_used"] for s in r["steps"]], "inner_status": [s["status"] for s in r["steps"]],
           "margin": [float(s["margin"]) for s in r["steps"]], "y_absmax": float(np.abs(r["y"]).max()),
           "y_Mnorm": float(np.sqrt((w.m * r["y"] ** 2).sum())), "u_Mnorm": float(np.sqrt((w.m * r["u"] ** 2).sum())),
           "oracle_seconds": round(dt, 1), "oracle_threads": o.threads}
    tag = f"c{config}" if first_steps is None else f"c{config}_first{first_steps}"
    with open(os.path.join(HERE, f"fullsize_query_{tag}.json"), "w") as f:
        json.dump(out, f)
    np.savez_compressed(os.path.join(HERE, f"fullsize_query_{tag}.npz"), pos=pos, y=r["y"][pos], u=r["u"][pos])
    print("config", config, "status", r["status"], "steps", r["n_steps"], "iters", sum(out["cg_iters"]), f"{dt:.0f} s", flush=True)


if __name__ == "__main__":
    for a in (sys.argv[1:] or ["3"]):  # "3": complete query of config 3; "5:3": the first 3 PDAS steps of config 5
        c, _, fs = a.partition(":")
        run(int(c), int(fs) if fs else None)
