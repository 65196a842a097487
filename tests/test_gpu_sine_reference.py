"""GPU parity of the analytical Cartesian reference (NEXT-1; eq. (15), cell-centred form):
rd_build_reference_sine against oracle.sine_reference, and RefDef queries driven by it against the oracle
driven by the same reference."""
import numpy as np
import pytest

from workloads import make_config, make_steady_2d

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def rd():
    import torch

    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    import paper_2606_17971_b200 as pkg

    pkg.load_library()
    return pkg


CASES = {
    "config1": lambda: make_config(1),
    "c2_48": lambda: make_config(twin="c2_48"),
    "c3_16": lambda: make_config(twin="c3_16"),
    # ragged: N = 37^2 is not a multiple of 32
    "ragged37": lambda: make_steady_2d(n=37, channels=[(0.4, 0.6)], vel=20.0, alpha=1e-4, k=5, n_queries=2, n_bumps=3,
                                       psi_factor=0.6, pdas_cap=60, config=1, name="ragged37"),
}


@pytest.mark.parametrize("case", list(CASES))
def test_sine_reference_matches_oracle(rd, oracle_mod, case):
    w = CASES[case]()
    g = rd.RefDef.from_workload(w, rd.Options(pdas_cap=w.pdas_cap))
    try:
        mu, modes = g.build_reference_sine(w.k, w.dims)
        modes_o, mu_o, W_o = oracle_mod.sine_reference(w.dims, w.k)
        assert np.array_equal(modes, modes_o)  # integer work: the same products in the same order
        assert np.allclose(mu, mu_o, rtol=1e-14, atol=0)
        W = g.get_reference()
        assert W.shape == (w.N, w.k)
        assert np.abs(W - W_o).max() <= 1e-14  # entries are O(1/sqrt(N)) products of sines; sinpi vs sin(pi x)
        assert np.allclose(W.T @ W, np.eye(w.k), atol=1e-12)
    finally:
        g.close()


def test_sine_reference_rejects_wrong_grids(rd):
    w = make_config(1)
    g = rd.RefDef.from_workload(w, rd.Options(pdas_cap=w.pdas_cap))
    try:
        with pytest.raises(rd.RefDefError):
            g.build_reference_sine(w.k, (31, 32))  # product != N
        with pytest.raises(rd.RefDefError):
            g.build_reference_sine(w.k, (4, 4, 8, 8))  # more than three axes
    finally:
        g.close()


@pytest.mark.parametrize("case", ["config1", "c2_48", "c3_16"])
def test_query_parity_with_sine_reference(rd, oracle_mod, case):
    """The whole path (S1-S7) with the analytical reference: same active-set sequence, y and u within 1e-6 (M-norm),
    iteration counts within 5 % of the oracle run with oracle.sine_reference."""
    w = CASES[case]()
    o = oracle_mod.Oracle.from_workload(w)
    g = rd.RefDef.from_workload(w, rd.Options(pdas_cap=w.pdas_cap))
    try:
        g.build_reference_sine(w.k, w.dims)
        _, _, W_o = oracle_mod.sine_reference(w.dims, w.k)
        yd, psi = w.target(0)
        ro = o.solve_query(1, yd, psi, W_o, oracle_mod.OracleOptions(pdas_cap=w.pdas_cap))
        rg = g.solve_query(1, yd, psi)
        assert rg["status"] == ro["status"] and rg["n_steps"] == ro["n_steps"]
        assert np.array_equal(rg["J_bits"], ro["J_bits"])
        for sg, so in zip(rg["steps"], ro["steps"]):
            assert sg["status"] == so["status"] == 0 and sg["rel_resid_verified"] <= 1e-8
            assert sg["rank_used"] == so["rank_used"]
            assert abs(sg["cg_iters"] - so["cg_iters"]) <= max(3, 0.05 * so["cg_iters"])

        def rel_m(a, b):
            return float(np.sqrt((w.m * (a - b) ** 2).sum() / (w.m * b * b).sum()))

        assert rel_m(rg["y"], ro["y"]) <= 1e-6 and rel_m(rg["u"], ro["u"]) <= 1e-6
        assert rg["t_reference_ms"] > 0.0  # the build is charged to this first query
    finally:
        g.close()


# ------------------------------------------------------------------ NEXT-2: mode-dependent temporal reference
ST_CASES = {
    "c4_32x8": lambda: make_config(twin="c4_32x8"),
}


def _st_small():
    from workloads import make_spacetime_2d

    # ragged: N = 13 * 13 * 5 = 845 is not a multiple of 32; nt odd (a bye round in the Jacobi ordering)
    return make_spacetime_2d(n=13, nt=5, T=1.0, channels=[(0.4, 0.6)], vel=20.0, alpha=1e-4, k=11, n_queries=1, n_bumps=2,
                             psi_factor=0.6, pdas_cap=40, config=4, name="st13x5")


ST_CASES["st13x5"] = _st_small


@pytest.mark.parametrize("case", list(ST_CASES))
def test_spacetime_reference_matches_oracle(rd, oracle_mod, case):
    w = ST_CASES[case]()
    dt = 1.0 / w.nt
    g = rd.RefDef.from_workload(w, rd.Options(pdas_cap=w.pdas_cap))
    try:
        s, pairs = g.build_reference_spacetime(w.k, w.dims, w.nt, dt)
        pairs_o, s_o, W_o = oracle_mod.spacetime_reference(w.dims, w.nt, dt, w.k)
        assert np.array_equal(pairs, pairs_o)  # the same (spatial mode, temporal index) pairs in the same order
        assert np.allclose(s, s_o, rtol=1e-12, atol=0)
        W = g.get_reference()
        # Jacobi (device) against LAPACK (oracle) eigenvectors of well-separated 5..32-dimensional problems
        assert np.abs(W - W_o).max() <= 1e-11
        assert np.allclose(W.T @ W, np.eye(w.k), atol=1e-11)
    finally:
        g.close()


def test_spacetime_reference_rejects_wrong_sizes(rd):
    w = ST_CASES["st13x5"]()
    g = rd.RefDef.from_workload(w, rd.Options(pdas_cap=w.pdas_cap))
    try:
        with pytest.raises(rd.RefDefError):
            g.build_reference_spacetime(w.k, w.dims, w.nt + 1, 0.2)
        with pytest.raises(rd.RefDefError):
            g.build_reference_spacetime(w.k, w.dims, w.nt, 0.0)
    finally:
        g.close()


@pytest.mark.parametrize("case", list(ST_CASES))
def test_query_parity_with_spacetime_reference(rd, oracle_mod, case):
    w = ST_CASES[case]()
    dt = 1.0 / w.nt
    o = oracle_mod.Oracle.from_workload(w)
    g = rd.RefDef.from_workload(w, rd.Options(pdas_cap=w.pdas_cap))
    try:
        g.build_reference_spacetime(w.k, w.dims, w.nt, dt)
        _, _, W_o = oracle_mod.spacetime_reference(w.dims, w.nt, dt, w.k)
        yd, psi = w.target(0)
        ro = o.solve_query(1, yd, psi, W_o, oracle_mod.OracleOptions(pdas_cap=w.pdas_cap))
        rg = g.solve_query(1, yd, psi)
        assert rg["status"] == ro["status"] and rg["n_steps"] == ro["n_steps"]
        assert np.array_equal(rg["J_bits"], ro["J_bits"])
        for sg, so in zip(rg["steps"], ro["steps"]):
            assert sg["status"] == so["status"] == 0 and sg["rel_resid_verified"] <= 1e-8
            assert sg["rank_used"] == so["rank_used"]
            assert abs(sg["cg_iters"] - so["cg_iters"]) <= max(3, 0.05 * so["cg_iters"])

        def rel_m(a, b):
            return float(np.sqrt((w.m * (a - b) ** 2).sum() / (w.m * b * b).sum()))

        assert rel_m(rg["y"], ro["y"]) <= 1e-6 and rel_m(rg["u"], ro["u"]) <= 1e-6
    finally:
        g.close()


# ------------------------------------------------------------------ NEXT-3: Jacobi-scaled reference
@pytest.mark.parametrize("case", ["config1", "c2_48", "ragged37"])
def test_scaled_reference_matches_oracle(rd, oracle_mod, case):
    w = CASES[case]()
    g = rd.RefDef.from_workload(w, rd.Options(pdas_cap=w.pdas_cap))
    try:
        mu, resid, sweeps, st = g.build_reference_scaled(w.k, tol=1e-7)
        assert st == 0 and resid.max() <= 1e-7
        mu_o, W_o = oracle_mod.reference_eigs_scaled(w.rowptr, w.colidx, w.val, w.m, w.alpha, w.k)
        assert np.allclose(mu, mu_o, rtol=1e-9)
        W = g.get_reference()
        assert np.allclose(np.linalg.norm(W, axis=0), 1.0, atol=1e-12)
        # W is unique only up to rotation inside clusters: compare the subspaces of complete clusters (principal
        # angles), cutting where the spectrum has a relative gap
        cut = w.k
        while cut > 1 and (mu_o[cut - 1] - mu_o[cut - 2]) < 1e-6 * mu_o[cut - 1]:
            cut -= 1
        cut -= 1 if cut == w.k and w.k > 1 else 0  # the last retained pair may share a cluster with the first dropped
        Qa, _ = np.linalg.qr(W[:, :cut])
        Qb, _ = np.linalg.qr(W_o[:, :cut])
        sv = np.linalg.svd(Qa.T @ Qb, compute_uv=False)
        assert sv.min() >= 1.0 - 1e-8
        # generalized residual of every column against the oracle's operator
        o = oracle_mod.Oracle.from_workload(w)
        d = o.diag_H()
        for c in range(w.k):
            r = o.apply_H(W[:, c]) - mu[c] * d * W[:, c]
            assert np.linalg.norm(r) <= 1e-6 * mu[c] * np.linalg.norm(d * W[:, c])
    finally:
        g.close()


def test_query_parity_with_scaled_reference(rd, oracle_mod):
    w = CASES["c2_48"]()
    o = oracle_mod.Oracle.from_workload(w)
    g = rd.RefDef.from_workload(w, rd.Options(pdas_cap=w.pdas_cap))
    try:
        _, _, _, st = g.build_reference_scaled(w.k, tol=1e-6)
        assert st == 0
        W = g.get_reference()
        yd, psi = w.target(0)
        ro = o.solve_query(1, yd, psi, W, oracle_mod.OracleOptions(pdas_cap=w.pdas_cap))
        rg = g.solve_query(1, yd, psi)
        assert rg["status"] == ro["status"] == 0 and rg["n_steps"] == ro["n_steps"]
        assert np.array_equal(rg["J_bits"], ro["J_bits"])
        for sg, so in zip(rg["steps"], ro["steps"]):
            assert sg["rank_used"] == so["rank_used"]
            assert abs(sg["cg_iters"] - so["cg_iters"]) <= max(3, 0.05 * so["cg_iters"])
        rel_m = lambda a, b: float(np.sqrt((w.m * (a - b) ** 2).sum() / (w.m * b * b).sum()))
        assert rel_m(rg["y"], ro["y"]) <= 1e-6 and rel_m(rg["u"], ro["u"]) <= 1e-6
    finally:
        g.close()
