"""GPU parity of the coarse-mesh reference (NEXT-1(ii); section 2.2.2: coarse generalized eigenproblem,
P1 prolongation, Euclidean column normalisation; cell-centred reading A20 of DESIGN.md): rd_build_reference_prolonged
against oracle.prolong_p1, the complete pipeline (coarse context -> rd_build_reference_scaled -> rd_get_reference ->
fine context) against the oracle's, and RefDef queries driven by it against the oracle driven by the same reference."""
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


def _ragged(n, k=5):
    return make_steady_2d(n=n, channels=[(0.4, 0.6)], vel=20.0, alpha=1e-4, k=k, n_queries=2, n_bumps=3,
                          psi_factor=0.6, pdas_cap=60, config=1, name=f"ragged{n}")


# (fine workload, coarse cells per axis): ratio 2 (the usual case), ratio 3, a non-integer ratio on a ragged grid
# (37^2 is not a multiple of 32), 3-D with ratio 2, and the same grid (identity up to the normalisation)
GRIDS = {
    "config1_from16": (lambda: make_config(1), (16, 16)),
    "c2_48_from16": (lambda: make_config(twin="c2_48"), (16, 16)),
    "ragged37_from13x9": (lambda: _ragged(37), (13, 9)),
    "c3_16_from8": (lambda: make_config(twin="c3_16"), (8, 8, 8)),
    "c3_16_from5x8x3": (lambda: make_config(twin="c3_16"), (5, 8, 3)),
    "config1_same": (lambda: make_config(1), (32, 32)),
}


@pytest.mark.parametrize("case", list(GRIDS))
@pytest.mark.parametrize("device_input", [False, True])
def test_prolongation_matches_oracle(rd, oracle_mod, case, device_input):
    """Random coarse vectors (every coarse entry matters, unlike smooth modes): element by element against the oracle."""
    import torch

    mk, dims_c = GRIDS[case]
    w = mk()
    k = 11  # not a multiple of 8: pad columns must stay zero
    rng = np.random.default_rng(5)
    Wc = np.asfortranarray(rng.standard_normal((int(np.prod(dims_c)), k)))
    g = rd.RefDef.from_workload(w, rd.Options(pdas_cap=w.pdas_cap))
    try:
        arg = torch.from_numpy(np.ascontiguousarray(Wc.T)).cuda() if device_input else Wc
        norms = g.build_reference_prolonged(arg, dims_c, w.dims)
        P = oracle_mod.prolong_p1(Wc, dims_c, w.dims)
        nrm_o = np.linalg.norm(P, axis=0)
        assert np.allclose(norms, nrm_o, rtol=1e-13, atol=0)
        W = g.get_reference()
        assert W.shape == (w.N, k)
        assert np.abs(W - P / nrm_o).max() <= 1e-14  # entries are at most 1 in magnitude
        assert np.allclose(np.linalg.norm(W, axis=0), 1.0, atol=1e-13)
    finally:
        g.close()


def test_prolongation_rejects_bad_arguments(rd):
    w = make_config(1)
    g = rd.RefDef.from_workload(w, rd.Options(pdas_cap=w.pdas_cap))
    try:
        Wc = np.ones((16 * 16, 3))
        with pytest.raises(rd.RefDefError):
            g.build_reference_prolonged(Wc, (16, 16), (31, 32))  # product of dims_f != N
        with pytest.raises(ValueError):
            g.build_reference_prolonged(Wc, (16, 8), (32, 32))  # Wc rows != prod(dims_c)
        Wz = np.ones((16 * 16, 3))
        Wz[:, 1] = 0.0
        with pytest.raises(rd.RefDefError):
            g.build_reference_prolonged(Wz, (16, 16), (32, 32))  # a zero column cannot be normalised
        yd, psi = w.target(0)
        with pytest.raises(rd.RefDefError):
            g.solve_query(1, yd, psi)  # and leaves no reference behind
        g.build_reference_prolonged(Wc, (16, 16), (32, 32))
        assert g.solve_query(1, yd, psi)["status"] == 0  # rank-deficient (three equal columns): rank 1 retained
    finally:
        g.close()


PIPE = {
    "config1_from16": (lambda: make_config(1), lambda k: make_config(1, n=16, k=k)),
    "c2_48_from24": (lambda: make_config(twin="c2_48"), lambda k: make_config(2, n=24, k=k)),
    "c3_16_from8": (lambda: make_config(twin="c3_16"), lambda k: make_config(3, n=8, k=k)),
}


@pytest.mark.parametrize("case", list(PIPE))
def test_pipeline_and_query_parity(rd, oracle_mod, case):
    """Coarse eigensolve on the GPU (a second context on the coarse operator), prolongation, then the whole path
    S1-S7: the prolonged subspace agrees with the oracle's pipeline (principal angles; columns are unique only up to
    rotation inside clusters, reading A14), and the query run with the GPU's own W reproduces the oracle run with the
    same W: active sets bit-exact, y and u within 1e-6 (M-norm), iteration counts within 5 %."""
    mk, mkc = PIPE[case]
    w = mk()
    wc = mkc(w.k)
    gc = rd.RefDef.from_workload(wc, rd.Options(pdas_cap=wc.pdas_cap))
    g = rd.RefDef.from_workload(w, rd.Options(pdas_cap=w.pdas_cap))
    try:
        mu, resid, _, st = gc.build_reference_scaled(w.k, tol=1e-8, max_block_iters=400)
        assert st == 0
        Wc = gc.get_reference()
        g.build_reference_prolonged(Wc, wc.dims, w.dims)
        W = g.get_reference()
        mu_o, Wc_o, W_o = oracle_mod.prolonged_reference((wc.rowptr, wc.colidx, wc.val, wc.m, wc.alpha), wc.dims, w.dims, w.k)
        assert np.allclose(mu, mu_o, rtol=1e-8)
        # the same subspace up to the last cluster, which the cut at k may split: compare what is unique
        gap = np.flatnonzero(np.diff(mu_o) > 1e-3 * mu_o[1:])
        kk = int(gap[-1]) + 1 if len(gap) else 0
        if kk:
            Q1, _ = np.linalg.qr(W[:, :kk])
            Q2, _ = np.linalg.qr(W_o[:, :kk])
            assert np.linalg.svd(Q1.T @ Q2, compute_uv=False).min() >= 1 - 1e-8
        o = oracle_mod.Oracle.from_workload(w)
        yd, psi = w.target(0)
        ro = o.solve_query(1, yd, psi, W, oracle_mod.OracleOptions(pdas_cap=w.pdas_cap))
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
        assert rg["t_reference_ms"] > 0.0  # the prolongation is charged to this first query
        # and it deflates: fewer iterations than Jacobi-CG on the same query
        g.reset_sequence()
        rj = g.solve_query(0, yd, psi)
        assert rg["total_cg_iters"] < rj["total_cg_iters"]
    finally:
        g.close()
        gc.close()
