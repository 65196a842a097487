"""GPU parity: the CUDA path (through the C ABI, paper_2606_17971_b200.RefDef) against the CPU oracle,
element by element on the same seeded inputs (workloads/).  Run on the B200 box with `-m gpu`.

Bars (BASELINE.json north_star): active-set sequences bit-exact; y, u within 1e-6 relative in the M-norm;
every inner solve verified at relative residual 1e-8.  Operator applies are compared at 1e-12 relative
(a different summation order is the only difference).
"""
import numpy as np
import pytest

from workloads import make_config, make_steady_2d

pytestmark = pytest.mark.gpu


def _mnorm(w, v):
    return float(np.sqrt((w.m * v * v).sum()))


def _rel_m(w, a, b):
    nb = _mnorm(w, b)
    return _mnorm(w, a - b) / (nb if nb > 0 else 1.0)


@pytest.fixture(scope="module")
def rd():
    import torch

    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    import paper_2606_17971_b200 as pkg

    pkg.load_library()  # raises if the library was not built: no fallback
    return pkg


WORKLOADS = {
    "config1": lambda: make_config(1),
    "c2_48": lambda: make_config(twin="c2_48"),
    "c3_16": lambda: make_config(twin="c3_16"),
    "c4_32x8": lambda: make_config(twin="c4_32x8"),
    # ragged: N = 37*37 = 1369 is not a multiple of 32 (last ELL slice and last DMMA chunk are partial)
    "ragged37": lambda: make_steady_2d(n=37, channels=[(0.4, 0.6)], vel=20.0, alpha=1e-4, k=5, n_queries=2, n_bumps=3,
                                       psi_factor=0.6, pdas_cap=60, config=1, name="ragged37"),
}


@pytest.fixture(scope="module", params=list(WORKLOADS))
def setup(request, rd, oracle_mod):
    w = WORKLOADS[request.param]()
    o = oracle_mod.Oracle.from_workload(w)
    g = rd.RefDef.from_workload(w, rd.Options(pdas_cap=w.pdas_cap))
    theta, W = oracle_mod.reference_eigs(w.rowptr, w.colidx, w.val, w.m, w.alpha, w.k)
    g.set_reference(W)
    yield w, o, g, W
    g.close()


# ------------------------------------------------------------------ S3: operator
def test_operator_apply_matches_oracle(setup):
    w, o, g, _ = setup
    rng = np.random.default_rng(1)
    v = rng.standard_normal(w.N)
    for name in ("apply_K", "apply_KT", "apply_H"):
        ref = getattr(o, name)(v)
        got = getattr(g, name)(v)
        assert np.abs(got - ref).max() <= 1e-12 * np.abs(ref).max(), name
    assert np.allclose(g.diag_H(), o.diag_H(), rtol=1e-13, atol=0)


def test_masked_apply_matches_oracle(setup):
    w, o, g, _ = setup
    rng = np.random.default_rng(2)
    for frac in (0.0, 0.3, 0.97, 1.0):
        act = (rng.random(w.N) < frac).astype(np.uint8)
        idx = np.flatnonzero(act == 0)
        v = rng.standard_normal(w.N)
        got = g.apply_H(v, active=act)
        ref = np.zeros(w.N)
        if len(idx):
            ref[idx] = o.apply_B(idx, v[idx])
        assert np.abs(got - ref).max() <= 1e-12 * max(np.abs(ref).max(), 1e-300)
        assert (got[act == 1] == 0).all()


def test_device_pointers_give_the_same_result(setup):
    import torch

    w, o, g, _ = setup
    v = np.random.default_rng(3).standard_normal(w.N)
    host = g.apply_H(v)
    dev = g.apply_H(torch.from_numpy(v).cuda())
    assert np.array_equal(dev.cpu().numpy(), host)


# ------------------------------------------------------------------ S1 + S2: restriction and coarse setup
def test_coarse_setup_matches_definition(setup):
    w, o, g, W = setup
    rng = np.random.default_rng(4)
    act = (rng.random(w.N) < 0.35).astype(np.uint8)
    idx = np.flatnonzero(act == 0)
    WI = W[idx]
    HWI = np.column_stack([o.apply_B(idx, WI[:, j]) for j in range(w.k)])
    G, EW = WI.T @ WI, WI.T @ HWI
    cs = g.coarse_setup(1, act)
    assert np.abs(cs["G"] - G).max() <= 1e-12 * np.abs(G).max()
    assert np.abs(cs["EW"] - EW).max() <= 1e-12 * np.abs(EW).max()
    assert cs["rank"] == w.k and cs["fallback"] == 0
    # C = (W_I^T H_II W_I)^{-1} when W_I has full column rank: Q = W_I C W_I^T is the projector of eq. (18)
    Cref = np.linalg.inv(0.5 * (EW + EW.T))
    assert np.abs(cs["C"] - Cref).max() <= 1e-8 * np.abs(Cref).max()
    # cond(E) of the orthonormalised basis: eigenvalues of G^{-1/2} EW G^{-1/2}
    s, V = np.linalg.eigh(0.5 * (G + G.T))
    T = V / np.sqrt(s)
    ev = np.linalg.eigvalsh(T.T @ (0.5 * (EW + EW.T)) @ T)
    assert abs(cs["cond_E"] - ev.max() / ev.min()) <= 1e-6 * ev.max() / ev.min()


def test_coarse_rank_deficient_basis(setup, rd):
    w, o, g, W = setup
    # a reference with a duplicated column: rank k-1 must be detected and C must still be the pseudo-inverse solve
    W2 = W.copy()
    W2[:, -1] = W2[:, 0]
    g.set_reference(W2)
    try:
        act = np.zeros(w.N, dtype=np.uint8)
        cs = g.coarse_setup(1, act)
        assert cs["rank"] == w.k - 1 and cs["fallback"] == 0
        idx = np.arange(w.N)
        rng = np.random.default_rng(5)
        r = rng.standard_normal(w.N)
        HW = np.column_stack([o.apply_H(W2[:, j]) for j in range(w.k)])
        q_gpu = W2 @ (cs["C"] @ (W2.T @ r))
        Z = np.linalg.qr(W2[:, :-1])[0]
        E = Z.T @ np.column_stack([o.apply_H(Z[:, j]) for j in range(w.k - 1)])
        q_ref = Z @ np.linalg.solve(E, Z.T @ r)
        assert np.abs(q_gpu - q_ref).max() <= 1e-8 * np.abs(q_ref).max()
    finally:
        g.set_reference(W)


# ------------------------------------------------------------------ Algorithm 1
@pytest.mark.parametrize("method", [0, 1])
def test_alg1_matches_oracle(setup, method):
    w, o, g, W = setup
    rng = np.random.default_rng(6)
    act = (rng.random(w.N) < 0.25).astype(np.uint8)
    idx = np.flatnonzero(act == 0)
    b = np.zeros(w.N)
    b[idx] = w.m[idx] * rng.standard_normal(len(idx))
    x0 = np.zeros(w.N)
    Zt = W[idx] if method == 1 else None
    xo, ro = o.alg1(idx, b[idx], x0[idx], Zt)
    g.reset_sequence()
    xg, rg = g.solve_inactive(method, act, b, x0)
    assert rg["status"] == 0 and ro["status"] == 0
    assert rg["rel_resid_verified"] <= 1e-8
    assert (xg[act == 1] == 0).all()
    assert rg["rank_used"] == ro["rank_used"]
    # same algorithm, same data, different summation order: iteration counts agree to a few percent
    assert abs(rg["iters"] - ro["iters"]) <= max(3, 0.05 * ro["iters"]), (rg["iters"], ro["iters"])
    # both are 1e-8-residual solutions of the same system: difference bounded by cond * 2e-8; compare to a tight solve
    xt, _ = o.alg1(idx, b[idx], x0[idx], Zt, eps=1e-13)
    ref_err = np.linalg.norm(xo - xt) / np.linalg.norm(xt)
    got_err = np.linalg.norm(xg[idx] - xt) / np.linalg.norm(xt)
    assert got_err <= max(10 * ref_err, 1e-9), (got_err, ref_err)


def test_alg1_rank_zero_is_jacobi_cg_bitwise(setup, rd):
    """rank-zero execution reduces to Jacobi-CG -- same kernel, same bits."""
    w, o, g, W = setup
    rng = np.random.default_rng(7)
    act = (rng.random(w.N) < 0.1).astype(np.uint8)
    b = np.where(act == 0, w.m * rng.standard_normal(w.N), 0.0)
    x0 = np.zeros(w.N)
    xa, ra = g.solve_inactive(0, act, b, x0)
    g.set_reference(np.zeros((w.N, w.k)))  # a zero reference has rank 0
    try:
        xb, rb = g.solve_inactive(1, act, b, x0)
    finally:
        g.set_reference(W)
    assert rb["rank_used"] == 0
    assert ra["iters"] == rb["iters"] and np.array_equal(xa, xb)


def test_alg1_edge_cases(setup):
    w, o, g, W = setup
    # b = 0: immediate return with x = x0-correction = 0
    act = np.zeros(w.N, dtype=np.uint8)
    x, r = g.solve_inactive(1, act, np.zeros(w.N), np.zeros(w.N))
    assert r["status"] == 0 and r["iters"] == 0 and (x == 0).all()
    # a single inactive DOF: 1x1 system
    act = np.ones(w.N, dtype=np.uint8)
    act[w.N // 2] = 0
    b = np.zeros(w.N)
    b[w.N // 2] = 1.0
    for method in (0, 1):
        x, r = g.solve_inactive(method, act, b, np.zeros(w.N))
        assert r["status"] == 0
        assert abs(x[w.N // 2] - 1.0 / o.diag_H()[w.N // 2]) <= 1e-12 / o.diag_H()[w.N // 2]
    # exact start: x0 = solution -> zero iterations
    act = np.zeros(w.N, dtype=np.uint8)
    xs = np.random.default_rng(8).standard_normal(w.N)
    b = o.apply_H(xs)
    x, r = g.solve_inactive(0, act, b, xs)
    assert r["iters"] == 0 and r["status"] == 0
    # iteration cap is a reported soft status
    import paper_2606_17971_b200 as pkg

    g.set_options(pkg.Options(pdas_cap=w.pdas_cap, cg_cap=3))
    try:
        x, r = g.solve_inactive(0, act, w.m * np.random.default_rng(9).standard_normal(w.N), np.zeros(w.N))
        assert r["status"] == -6 and r["iters"] == 3
    finally:
        g.set_options(pkg.Options(pdas_cap=w.pdas_cap))


# ------------------------------------------------------------------ the query (S1-S7)
@pytest.mark.parametrize("method", [0, 1, 2])
def test_query_sequence_parity(setup, oracle_mod, method):
    w, o, g, W = setup
    o.reset_sequence()
    g.reset_sequence()
    nq = min(w.n_queries, 2)
    for q in range(nq):
        yd, psi = w.target(q)
        ro = o.solve_query(method, yd, psi, W, oracle_mod.OracleOptions(pdas_cap=w.pdas_cap))
        rg = g.solve_query(method, yd, psi)
        assert rg["n_steps"] == ro["n_steps"] and rg["status"] == ro["status"]
        margins = [s["margin"] for s in ro["steps"]]
        assert np.array_equal(rg["J_bits"], ro["J_bits"]), f"active sets differ; oracle margins {margins}"
        assert rg["hashes"] == ro["hashes"]
        assert [s["n_inactive"] for s in rg["steps"]] == [s["n_inactive"] for s in ro["steps"]]
        for sg, so in zip(rg["steps"], ro["steps"]):
            assert sg["status"] == so["status"] == 0
            assert sg["rel_resid_verified"] <= 1e-8
            assert sg["rank_used"] == so["rank_used"]
            assert abs(sg["cg_iters"] - so["cg_iters"]) <= max(3, 0.05 * so["cg_iters"])
        assert _rel_m(w, rg["y"], ro["y"]) <= 1e-6
        assert _rel_m(w, rg["u"], ro["u"]) <= 1e-6
        assert np.abs(rg["lam"] - ro["lam"]).max() <= 1e-6 * max(np.abs(ro["lam"]).max(), np.abs(w.m * yd).max())
        for a, b in zip(rg["kkt"], ro["kkt"]):
            assert abs(a - b) <= 1e-8 + 1e-3 * abs(b)


def test_query_unconstrained_limit(setup):
    """psi = +inf: J empty after step 0, one solve H y = l, lambda = 0 (pin P4 on the GPU side)."""
    w, o, g, W = setup
    yd, _ = w.target(0)
    g.reset_sequence()
    r = g.solve_query(1, yd, np.full(w.N, np.inf))
    assert r["n_steps"] == 1 and r["status"] == 0 and r["steps"][0]["n_inactive"] == w.N
    assert (r["lam"] == 0).all()
    res = o.apply_H(r["y"]) - w.m * yd
    assert np.linalg.norm(res) <= 2e-8 * np.linalg.norm(w.m * yd)
    assert _rel_m(w, r["u"], o.apply_K(r["y"]) / w.m) <= 1e-12


def test_query_device_buffers_match_host_buffers(setup):
    import torch

    w, o, g, W = setup
    yd, psi = w.target(0)
    g.reset_sequence()
    rh = g.solve_query(1, yd, psi)
    g.reset_sequence()
    rdv = g.solve_query(1, torch.from_numpy(yd).cuda(), torch.from_numpy(psi).cuda())
    assert np.array_equal(rdv["y"].cpu().numpy(), rh["y"])  # deterministic reductions: same bits
    assert rdv["hashes"] == rh["hashes"]
    assert [s["cg_iters"] for s in rdv["steps"]] == [s["cg_iters"] for s in rh["steps"]]


@pytest.mark.parametrize("method", [0, 1])
def test_alg1_kernel_variants_agree(setup, rd, method):
    """The two persistent kernels (TMA-staged coefficient form over the live slices, literal recurrence over all rows)
    run the same Algorithm 1: same status and rank, iteration counts within a few, solutions equal at the level of the
    1e-8 stop."""
    w, o, g, W = setup
    rng = np.random.default_rng(16)
    act = (rng.random(w.N) < 0.2).astype(np.uint8)
    b = np.where(act == 0, w.m * rng.standard_normal(w.N), 0.0)
    x0 = np.zeros(w.N)
    out = {}
    try:
        for variant in (0, 1):
            g.set_options(rd.Options(pdas_cap=w.pdas_cap, alg1_variant=variant))
            out[variant] = g.solve_inactive(method, act, b, x0)
    finally:
        g.set_options(rd.Options(pdas_cap=w.pdas_cap))
    x_ref, r_ref = out[1]
    for variant in (0,):
        x, r = out[variant]
        assert r["status"] == r_ref["status"] == 0 and r["rank_used"] == r_ref["rank_used"]
        assert r["rel_resid_verified"] <= 1e-8
        assert abs(r["iters"] - r_ref["iters"]) <= max(3, 0.05 * r_ref["iters"]), (variant, r["iters"], r_ref["iters"])
        assert (x[act == 1] == 0).all()
        assert np.linalg.norm(x - x_ref) <= 1e-6 * np.linalg.norm(x_ref)


@pytest.mark.parametrize("k", [1, 9, 17, 24, 33, 41, 57, 64])
def test_alg1_every_tile_width(rd, oracle_mod, k):
    """Every padded rank kp = 8..64 changes the geometry of the TMA ring (tile = 256 kp bytes, min(32, 512/kp) slots,
    one or two columns per lane in the transposed pass): a seeded random reference of k columns, GPU against oracle
    (iterations, rank, solution) and against the literal-recurrence kernel."""
    w = make_steady_2d(n=61, channels=[(0.4, 0.6)], vel=20.0, alpha=1e-4, k=8, n_queries=1, n_bumps=3, psi_factor=0.6,
                       pdas_cap=20, config=1, name="n61")  # N = 3721: 117 slices, ragged tail
    o = oracle_mod.Oracle.from_workload(w)
    rng = np.random.default_rng(1000 + k)
    W = rng.standard_normal((w.N, k))
    act = (rng.random(w.N) < 0.3).astype(np.uint8)
    idx = np.flatnonzero(act == 0)
    b = np.where(act == 0, w.m * rng.standard_normal(w.N), 0.0)
    x0 = np.zeros(w.N)
    g = rd.RefDef.from_workload(w, rd.Options(pdas_cap=w.pdas_cap))
    try:
        g.set_reference(W)
        xg, rg = g.solve_inactive(1, act, b, x0)
        g.set_options(rd.Options(pdas_cap=w.pdas_cap, alg1_variant=1))
        xl, rl = g.solve_inactive(1, act, b, x0)
    finally:
        g.close()
    xo, ro = o.alg1(idx, b[idx], x0[idx], W[idx])
    assert rg["status"] == ro["status"] == rl["status"] == 0
    assert rg["rank_used"] == ro["rank_used"] == k
    assert rg["rel_resid_verified"] <= 1e-8
    assert abs(rg["iters"] - ro["iters"]) <= max(3, 0.05 * ro["iters"]), (rg["iters"], ro["iters"])
    assert (xg[act == 1] == 0).all()
    xt, _ = o.alg1(idx, b[idx], x0[idx], W[idx], eps=1e-13)
    ref_err = np.linalg.norm(xo - xt) / np.linalg.norm(xt)
    got_err = np.linalg.norm(xg[idx] - xt) / np.linalg.norm(xt)
    assert got_err <= max(10 * ref_err, 1e-9), (got_err, ref_err)
    assert np.linalg.norm(xg - xl) <= 1e-6 * np.linalg.norm(xl)


def test_operator_change_keeps_the_reference(rd, oracle_mod):
    """Algorithm 2 steps 6-8: when the flow scale changes the operator is reassembled but the
    reference is kept.  Here: reference built on the nominal operator (velocity 50), injected into a context of the
    off-design operator (velocity 75) through rd_get_reference / rd_set_reference; the query on the new operator
    must match the oracle run with the same retained reference, and deflation must still pay against Jacobi-CG."""
    from workloads.cht import CH2

    mk = lambda vel: make_steady_2d(n=48, channels=CH2, vel=vel, alpha=1e-4, k=16, n_queries=2, n_bumps=5,
                                    psi_factor=0.55, pdas_cap=100, config=2, name=f"c2_48_v{vel:g}")
    w_nom, w_off = mk(50.0), mk(75.0)
    g_nom = rd.RefDef.from_workload(w_nom, rd.Options(pdas_cap=w_nom.pdas_cap))
    g_off = rd.RefDef.from_workload(w_off, rd.Options(pdas_cap=w_off.pdas_cap))
    try:
        _, _, _, st = g_nom.build_reference(w_nom.k, tol=1e-6)
        assert st == 0
        W = g_nom.get_reference()
        g_off.set_reference(W)
        o = oracle_mod.Oracle.from_workload(w_off)
        yd, psi = w_off.target(0)
        ro = o.solve_query(1, yd, psi, W, oracle_mod.OracleOptions(pdas_cap=w_off.pdas_cap))
        rg = g_off.solve_query(1, yd, psi)
        assert rg["status"] == ro["status"] == 0 and rg["n_steps"] == ro["n_steps"]
        assert np.array_equal(rg["J_bits"], ro["J_bits"])
        assert _rel_m(w_off, rg["y"], ro["y"]) <= 1e-6 and _rel_m(w_off, rg["u"], ro["u"]) <= 1e-6
        g_off.reset_sequence()
        rj = g_off.solve_query(0, yd, psi)
        assert rj["status"] == 0 and np.array_equal(rj["J_bits"], rg["J_bits"])
        assert rg["total_cg_iters"] < rj["total_cg_iters"]
    finally:
        g_nom.close()
        g_off.close()


OPTION_SETS = {
    "all_inactive_start": dict(init=2),
    "given_start": dict(init=3),
    "c_is_diag": dict(c_is_diag=1),
    "scheduled_replacement": dict(replace_period=25),
    "no_jacobi": dict(jacobi=0),
    "paper_tolerances": dict(eps=1e-10, eps_c=1e-11),
}


@pytest.mark.parametrize("name", list(OPTION_SETS))
def test_query_parity_under_options(rd, oracle_mod, name):
    """Every rd_options field that changes the path (readings A3, A5, A8, A11 of DESIGN.md; PAPER.md:267, :273, :339,
    :341) against the oracle run with the same option."""
    kw = OPTION_SETS[name]
    w = make_config(twin="c2_48")
    o = oracle_mod.Oracle.from_workload(w)
    _, W = oracle_mod.reference_eigs(w.rowptr, w.colidx, w.val, w.m, w.alpha, w.k)
    g = rd.RefDef.from_workload(w, rd.Options(pdas_cap=w.pdas_cap, **kw))
    try:
        g.set_reference(W)
        yd, psi = w.target(0)
        J0 = None
        if kw.get("init") == 3:
            J0 = (np.random.default_rng(11).random(w.N) < 0.4).astype(np.uint8)
        ro = o.solve_query(1, yd, psi, W, oracle_mod.OracleOptions(pdas_cap=w.pdas_cap, **kw), J0=J0)
        rg = g.solve_query(1, yd, psi, J0=J0)
        assert rg["status"] == ro["status"] and rg["n_steps"] == ro["n_steps"]
        assert np.array_equal(rg["J_bits"], ro["J_bits"]), [s["margin"] for s in ro["steps"]]
        tol = kw.get("eps", 1e-8)
        for sg, so in zip(rg["steps"], ro["steps"]):
            assert sg["status"] == so["status"] == 0 and sg["rel_resid_verified"] <= tol
            assert sg["rank_used"] == so["rank_used"]
            assert abs(sg["cg_iters"] - so["cg_iters"]) <= max(3, 0.05 * so["cg_iters"])
            if kw.get("replace_period"):
                assert sg["replacements"] >= sg["cg_iters"] // kw["replace_period"]
        assert _rel_m(w, rg["y"], ro["y"]) <= 1e-6 and _rel_m(w, rg["u"], ro["u"]) <= 1e-6
    finally:
        g.close()


def test_query_parity_with_sigma_one_over_alpha(rd, oracle_mod):
    """BASELINE.json's literal text H = M + (1/alpha) K^T M^{-1} K (reading A1, sigma_is_alpha = 0): runnable and in
    parity with the oracle given sigma = 1/alpha."""
    w = make_config(1)
    o = oracle_mod.Oracle(w.rowptr, w.colidx, w.val, w.m, 1.0 / w.alpha)
    g = rd.RefDef.from_workload(w, rd.Options(pdas_cap=w.pdas_cap, sigma_is_alpha=0.0))
    try:
        yd, psi = w.target(0)
        ro = o.solve_query(0, yd, psi, None, oracle_mod.OracleOptions(pdas_cap=w.pdas_cap))
        rg = g.solve_query(0, yd, psi)
        # (from the all-active start PDAS may still be releasing DOFs when it reaches config 1's cap of 20 steps:
        # the status, whatever it is, and the whole sequence must agree)
        assert rg["status"] == ro["status"] and rg["n_steps"] == ro["n_steps"]
        assert np.array_equal(rg["J_bits"], ro["J_bits"])
        assert _rel_m(w, rg["y"], ro["y"]) <= 1e-6 and _rel_m(w, rg["u"], ro["u"]) <= 1e-6
    finally:
        g.close()
