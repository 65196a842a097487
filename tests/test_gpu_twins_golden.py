"""Complete query sequences on the larger twins of BASELINE.json's configs (N = 16,384 ... 110,592, so that every warp of
the persistent grid owns tiles, warps own several, and the TMA ring wraps inside a CTA) against goldens written by the
CPU oracle alone (tests/golden/make_golden_twins.py; minutes to an hour of oracle time each, hence stored).

Compared per query: the whole active-set sequence (FNV-1a hash of the packed set and |I| at every PDAS step: bit-exact),
status, retained rank and CG iterations per step (5 %), y and u = M^-1 K y to 1e-6 in the M-norm (north_star's bar),
KKT measures.  Both sides run RefDef with the analytical reference at the paper's accuracy, eps = 1e-10 and eps_c = 1e-11
(see the generator's header)."""
import json
import os

import numpy as np
import pytest

pytestmark = pytest.mark.gpu

GOLD = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden")
CASES = ["c3_32", "c2_128", "c4_64x8", "c5_48", "c2_256"]


@pytest.mark.parametrize("case", CASES)
def test_twin_sequence_matches_oracle_golden(oracle_mod, case):
    import torch

    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    jpath, zpath = os.path.join(GOLD, f"twin_{case}.json"), os.path.join(GOLD, f"twin_{case}.npz")
    if not (os.path.exists(jpath) and os.path.exists(zpath)):
        pytest.skip(f"golden for {case} not generated (python tests/golden/make_golden_twins.py {case})")
    import paper_2606_17971_b200 as pkg
    from workloads import make_config

    gold = json.load(open(jpath))
    ys = np.load(zpath)
    w = make_config(**gold["make_config"])
    assert w.operator_hash() == gold["operator_sha256"], "the workload generator changed: regenerate the golden"
    if w.nt > 1:
        W = oracle_mod.spacetime_reference(w.dims, w.nt, 1.0 / w.nt, w.k)[-1]
    else:
        W = oracle_mod.sine_reference(w.dims, w.k)[-1]
    g = pkg.RefDef.from_workload(w, pkg.Options(eps=gold["eps"], eps_c=gold["eps_c"], pdas_cap=gold["pdas_cap"]))
    g.set_reference(np.asfortranarray(W))
    o = oracle_mod.Oracle.from_workload(w)
    nrm = lambda v: float(np.sqrt((w.m * v * v).sum()))
    try:
        for gq in gold["queries"]:
            yd, psi = w.target(gq["query"])
            r = g.solve_query(pkg.REFDEF, yd, psi)
            assert r["status"] == gq["status"] == 0
            hashes = [f"{h:016x}" for h in r["hashes"]]
            n_in = [s["n_inactive"] for s in r["steps"]]
            if hashes != gq["active_hash"]:
                first = next(i for i, (a, b) in enumerate(zip(hashes, gq["active_hash"])) if a != b)
                # A decision of eq. (8) is a threshold on an inexact solve: the two sides may part
                # only where the oracle's own distance to a tie is below the solver's noise, eps * |y|; anything else
                # is a bug.  Both sequences must still end at the unique solution of the QP (checked below).
                noise = 10.0 * gold["eps"] * float(np.abs(ys[f"y{gq['query']}"]).max())
                assert gq["margin"][first - 1] <= noise, (
                    f"{case} query {gq['query']}: active sets differ first at step {first} of {gq['n_steps']} "
                    f"(|I| {n_in[first]} vs {gq['n_inactive'][first]}); oracle margin of the deciding step "
                    f"{gq['margin'][first - 1]:.2e} is not a near-tie (noise level {noise:.1e})")
                y_o = ys[f"y{gq['query']}"]
                assert nrm(r["y"] - y_o) <= 1e-6 * nrm(y_o) and max(r["kkt"]) <= 1e-8
                continue
            assert r["n_steps"] == gq["n_steps"] and n_in == gq["n_inactive"]
            assert r["worst_inner_status"] == 0 and all(s == 0 for s in gq["inner_status"])
            for s, it_o, rk_o in zip(r["steps"], gq["cg_iters"], gq["rank_used"]):
                assert s["rank_used"] <= rk_o
                if s["rank_used"] == rk_o:
                    assert abs(s["cg_iters"] - it_o) <= max(4, 0.05 * it_o), (s["cg_iters"], it_o)
            tot, tot_o = sum(s["cg_iters"] for s in r["steps"]), sum(gq["cg_iters"])
            assert abs(tot - tot_o) <= 0.05 * tot_o
            y_o = ys[f"y{gq['query']}"]
            assert nrm(r["y"] - y_o) <= 1e-6 * nrm(y_o)
            u_o = o.apply_K(y_o) / w.m  # eq. (9) on the oracle's y with the oracle's K
            assert nrm(r["u"] - u_o) <= 1e-6 * nrm(u_o)
            assert max(r["kkt"]) <= 1e-8 and max(gq["kkt"]) <= 1e-8
    finally:
        g.close()
