"""Writes tests/golden/fullsize_solve_c<config>.json from the CPU oracle ONLY (never from the CUDA path).

Run:  python tests/golden/make_golden_fullsize_solve.py [config ...]      (no arguments: 2 3 5; config 5 takes the longest)

One COMPLETE Algorithm-1 solve at BASELINE.json's full size per configuration, which the live oracle
is too slow for inside a GPU test (minutes of 8-thread time): the inactive system of the active set
    J = { i : y_d,i > psi_i }        (where the target exceeds the bound: what the first PDAS update leaves active),
    b = (l - H chi_J psi)_I,  l = M y_d,  x0 = 0,
of query 0, solved with direct restriction (eq. (12)) of the paper's analytical sine reference (deterministic closed form,
oracle.sine_reference) at BASELINE.json's accuracy (eps = eps_c = 1e-8).  Stored: the iteration count, retained rank,
status, the verified residual, the M-norm of x and x itself at 4096 seeded sample positions of I.
tests/test_gpu_fullsize_solve_golden.py builds the same system through the C ABI and compares.

The oracle is the threaded build of the same source (oracle.Oracle(..., threaded=True)): sums are taken in another order,
nothing else differs (tests/test_oracle_pins.py::test_threaded_timing_build_matches_the_plain_oracle).
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

N_SAMPLES = 4096
EPS = 1e-8


def system_of(w):
    """(J as bool, idx of I, y_d, psi): pure input construction, shared with the GPU test by restating it there."""
    yd, psi = w.target(0)
    J = yd > psi
    return J, np.flatnonzero(~J).astype(np.int64), yd, psi


def run(config):
    w = make_config(config)
    assert w.nt == 1, "steady configurations only (the sine reference)"
    o = oracle.Oracle.from_workload(w, threaded=True)
    W = np.asfortranarray(oracle.sine_reference(w.dims, w.k)[-1])
    J, idx, yd, psi = system_of(w)
    ell = w.m * yd
    b = (ell - o.apply_H(np.where(J, psi, 0.0)))[idx]
    t0 = time.time()
    x, rep = o.alg1(idx, b, np.zeros(len(idx)), W[idx], eps=EPS, eps_c=EPS)
    dt = time.time() - t0
    rng = np.random.default_rng(4242 + config)
    pos = np.sort(rng.choice(len(idx), size=min(N_SAMPLES, len(idx)), replace=False))
    mI = w.m[idx]
    out = {
        "config": config, "workload": w.name, "N": w.N, "k": w.k, "operator_sha256": w.operator_hash(), "eps": EPS, "eps_c": EPS,
        "n_active": int(J.sum()), "n_inactive": int(len(idx)), "method": "refdef, analytical sine reference",
        "status": rep["status"], "iters": rep["iters"], "rank_used": rep["rank_used"], "restarts": rep.get("restarts"),
        "rel_resid_verified": float(rep["rel_resid_verified"]), "x_Mnorm": float(np.sqrt((mI * x * x).sum())),
        "b_norm": float(np.linalg.norm(b)), "sample_seed": 4242 + config, "sample_positions_in_I": [int(p) for p in pos],
        "x_samples": [float(v) for v in x[pos]], "oracle_seconds": round(dt, 1), "oracle_threads": o.threads,
    }
    with open(os.path.join(HERE, f"fullsize_solve_c{config}.json"), "w") as f:
        json.dump(out, f)
    print("config", config, "n_inactive", len(idx), "of", w.N, "status", rep["status"], "iters", rep["iters"], "rank", rep["rank_used"],
          f"{dt:.0f} s", flush=True)


if __name__ == "__main__":
    for c in ([int(a) for a in sys.argv[1:]] or [2, 3, 5]):
        run(c)
