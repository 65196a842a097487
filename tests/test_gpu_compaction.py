"""S6 compaction (Alg. 2 step 12 "restrict ... on the GPU"): k_alg1_v3 works on the
32-row slices that hold inactive rows (listB) and on those where M^-1 K p can be nonzero (listA) and skips the rest.
Checked here: the lists are what numpy says they are, the solve on clustered active sets (whole slices dead, ragged
tails, fewer live slices than CTAs, nothing live) matches the oracle, and the literal all-rows kernel agrees."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

import oracle  # noqa: E402
import paper_2606_17971_b200 as rd  # noqa: E402
from workloads import make_config, make_steady_2d  # noqa: E402


def expected_lists(w, act):
    N = w.N
    ns = (N + 31) // 32
    inactive = np.zeros(ns * 32, dtype=bool)
    inactive[:N] = act == 0
    liveB = inactive.reshape(ns, 32).any(axis=1)
    K = w.csr()
    hit_rows = np.zeros(ns * 32, dtype=bool)
    Kc = K.tocoo()
    sel = (Kc.data != 0) & (act[Kc.col] == 0)
    hit_rows[np.unique(Kc.row[sel])] = True
    liveA = hit_rows.reshape(ns, 32).any(axis=1) | liveB
    return int(liveA.sum()), int(liveB.sum())


def masks(N, dims):
    rng = np.random.default_rng(3)
    out = {}
    a = np.ones(N, dtype=np.uint8)
    a[N // 3: N // 3 + 700] = 0                      # one contiguous inactive block: most slices dead
    out["block"] = a
    a = np.ones(N, dtype=np.uint8)
    a[rng.choice(N, 40, replace=False)] = 0           # 40 scattered inactive rows: fewer live slices than CTAs
    out["scattered40"] = a
    a = (rng.random(N) < 0.9).astype(np.uint8)        # 90 % active at random: nearly every slice stays live
    out["random90"] = a
    a = np.ones(N, dtype=np.uint8)
    a[-5:] = 0                                        # only the ragged tail slice is live
    out["tail"] = a
    n0 = dims[0]
    a = np.zeros(N, dtype=np.uint8).reshape(-1, n0)
    a[: a.shape[0] // 2] = 1                          # half the grid active (a PDAS front)
    out["half"] = a.reshape(-1)
    return out


@pytest.fixture(scope="module")
def ctx():
    w = make_steady_2d(n=93, channels=[(0.4, 0.6)], vel=20.0, alpha=1e-4, k=12, n_queries=1, n_bumps=3, psi_factor=0.6,
                       pdas_cap=20, config=1, name="n93")  # N = 8649: 271 slices, ragged tail of 9 rows
    o = oracle.Oracle.from_workload(w)
    g = rd.RefDef.from_workload(w, rd.Options(pdas_cap=w.pdas_cap))
    _, W = oracle.reference_eigs(w.rowptr, w.colidx, w.val, w.m, w.alpha, w.k)
    g.set_reference(W)
    yield w, o, g, W
    g.close()


@pytest.mark.parametrize("name", ["block", "scattered40", "random90", "tail", "half"])
@pytest.mark.parametrize("method", [0, 1])
def test_compacted_solve_matches_oracle(ctx, name, method):
    w, o, g, W = ctx
    act = masks(w.N, w.dims)[name]
    idx = np.flatnonzero(act == 0)
    rng = np.random.default_rng(21)
    b = np.where(act == 0, w.m * rng.standard_normal(w.N), 0.0)
    x0 = np.where(act == 0, 0.1 * rng.standard_normal(w.N), 0.0)
    xg, rg = g.solve_inactive(method, act, b, x0)
    nA, nB = expected_lists(w, act)
    assert (rg["live_slices_A"], rg["live_slices_B"]) == (nA, nB)
    assert nB <= nA <= (w.N + 31) // 32
    Zt = o.restrict(method, W, idx) if method else None
    xo, ro = o.alg1(idx, b[idx], x0[idx], Zt)
    assert rg["status"] == ro["status"] == 0
    # The oracle truncates the restricted basis at singular values 1e-12 (QR + SVD), the library at 1e-7
    # (Gram matrix, reading A6): on a few clustered rows the library may keep fewer directions, never more.
    assert rg["rank_used"] <= ro["rank_used"]
    if name in ("random90", "half"):
        assert rg["rank_used"] == ro["rank_used"]
    if rg["rank_used"] == ro["rank_used"]:
        assert abs(rg["iters"] - ro["iters"]) <= max(3, 0.05 * ro["iters"]), (rg["iters"], ro["iters"])
    assert (xg[act == 1] == 0).all()
    assert np.linalg.norm(xg[idx] - xo) <= 1e-6 * np.linalg.norm(xo)
    # the literal kernel (all rows, masked) on the same system
    g.set_options(rd.Options(pdas_cap=w.pdas_cap, alg1_variant=1))
    try:
        xl, rl = g.solve_inactive(method, act, b, x0)
    finally:
        g.set_options(rd.Options(pdas_cap=w.pdas_cap))
    assert rl["status"] == 0 and abs(rl["iters"] - rg["iters"]) <= max(3, 0.05 * rl["iters"])
    assert np.linalg.norm(xl - xg) <= 1e-6 * np.linalg.norm(xg)


def test_nothing_live(ctx):
    w, o, g, W = ctx
    act = np.ones(w.N, dtype=np.uint8)
    x, r = g.solve_inactive(1, act, np.zeros(w.N), np.zeros(w.N))
    assert r["iters"] == 0 and (x == 0).all() and r["live_slices_B"] == 0 and r["live_slices_A"] == 0


def test_compacted_runs_are_bit_identical(ctx):
    w, o, g, W = ctx
    act = masks(w.N, w.dims)["half"]
    rng = np.random.default_rng(5)
    b = np.where(act == 0, w.m * rng.standard_normal(w.N), 0.0)
    runs = [g.solve_inactive(1, act, b, np.zeros(w.N)) for _ in range(3)]
    for x, r in runs[1:]:
        assert np.array_equal(x, runs[0][0]) and r["iters"] == runs[0][1]["iters"]


def test_query_from_the_all_active_start_uses_small_lists():
    """First query of a sequence: every DOF active, then the inactive set grows; the lists follow it."""
    w = make_config(twin="c2_96")
    g = rd.RefDef.from_workload(w, rd.Options(pdas_cap=w.pdas_cap))
    g.build_reference_sine(w.k, w.dims)
    yd, psi = w.target(0)
    o = oracle.Oracle.from_workload(w)
    W = g.get_reference()
    r = g.solve_query(rd.REFDEF, yd, psi)
    ro = o.solve_query(oracle.REFDEF, yd, psi, W, oracle.OracleOptions(pdas_cap=w.pdas_cap))
    assert r["status"] == ro["status"] == 0
    assert np.array_equal(r["J_bits"], ro["J_bits"])
    nrm = lambda v: np.sqrt((w.m * v * v).sum())
    assert nrm(r["y"] - ro["y"]) <= 1e-6 * nrm(ro["y"])
    g.close()
