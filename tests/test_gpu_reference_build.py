"""GPU parity of S0, rd_build_reference (the k lowest eigenpairs of H by Chebyshev-filtered subspace iteration),
against the definition evaluated by a library eigensolver in the oracle (oracle.reference_eigs).  W is unique only up
to sign and rotation inside clusters (A14): eigenvalues are compared directly, eigenvectors through the
principal angles of complete clusters and through their residuals against the oracle's operator."""
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
    "c4_32x8": lambda: make_config(twin="c4_32x8"),
    "ragged37": lambda: make_steady_2d(n=37, channels=[(0.4, 0.6)], vel=20.0, alpha=1e-4, k=5, n_queries=2, n_bumps=3,
                                       psi_factor=0.6, pdas_cap=60, config=1, name="ragged37"),
}


def _cluster_cut(theta, k):
    """Largest c <= k such that theta[c-1] and theta[c] are separated (theta has k + 1 entries)."""
    c = k
    while c > 0 and (theta[c] - theta[c - 1]) < 1e-5 * theta[c]:
        c -= 1
    return c


@pytest.mark.parametrize("case", list(CASES))
def test_build_reference_matches_library_eigensolver(rd, oracle_mod, case):
    w = CASES[case]()
    o = oracle_mod.Oracle.from_workload(w)
    g = rd.RefDef.from_workload(w, rd.Options(pdas_cap=w.pdas_cap))
    try:
        theta, resid, sweeps, st = g.build_reference(w.k, tol=1e-7)
        assert st == 0 and resid.max() <= 1e-7 and sweeps >= 1
        th_o, W_o = oracle_mod.reference_eigs(w.rowptr, w.colidx, w.val, w.m, w.alpha, w.k + 1)
        assert np.allclose(theta, th_o[:w.k], rtol=1e-9)
        assert (np.diff(theta) >= 0).all()
        W = g.get_reference()
        assert W.shape == (w.N, w.k)
        assert np.abs(W.T @ W - np.eye(w.k)).max() <= 1e-10
        for c in range(w.k):  # residual of every column against the ORACLE's operator
            r = o.apply_H(W[:, c]) - theta[c] * W[:, c]
            assert np.linalg.norm(r) <= 2e-7 * theta[c]
        cut = _cluster_cut(th_o, w.k)
        if cut > 0:
            sv = np.linalg.svd(W[:, :cut].T @ W_o[:, :cut], compute_uv=False)
            assert sv.min() >= 1.0 - 1e-8
        info = g.reference_info()
        assert info["build_ms"] > 0 and info["total_degree"] > 0 and info["block"] >= w.k + 8
    finally:
        g.close()


def test_build_reference_edge_cases(rd, oracle_mod):
    w = CASES["c2_48"]()
    g = rd.RefDef.from_workload(w, rd.Options(pdas_cap=w.pdas_cap))
    try:
        # k = 1 and the largest k
        th_o, _ = oracle_mod.reference_eigs(w.rowptr, w.colidx, w.val, w.m, w.alpha, 64)
        theta, resid, _, st = g.build_reference(1, tol=1e-6)
        assert st == 0 and abs(theta[0] / th_o[0] - 1) <= 1e-9
        theta, resid, _, st = g.build_reference(64, tol=1e-5)
        assert st == 0 and np.allclose(theta, th_o, rtol=1e-8)
        # a sweep cap that is too small is a soft status: the best block so far is kept as the reference
        theta, resid, sweeps, st = g.build_reference(8, tol=1e-12, max_block_iters=2)
        assert st == -6 and sweeps == 2 and g.get_reference().shape == (w.N, 8)
        r = g.solve_query(1, *w.target(0))
        assert r["status"] == 0  # any full-rank block is a valid reference for Algorithm 1
        # invalid arguments
        with pytest.raises(rd.RefDefError):
            g.build_reference(0)
        with pytest.raises(rd.RefDefError):
            g.build_reference(65)
    finally:
        g.close()


def test_reference_work_accounting_and_tensor_probe(rd):
    """S0's work counters (rd_reference_work) and the FP64 tensor-pipe probe (rd_probe_fp64_tensor_peak): the counters
    exist only after an eigen-build, count whole column applies of the Chebyshev filter (at least one column per
    degree, at most the block), and the bytes per column apply are the DESIGN.md model 3 nnz + 48 N."""
    w = CASES["c2_48"]()
    g = rd.RefDef.from_workload(w, rd.Options(pdas_cap=w.pdas_cap))
    try:
        info0 = g.reference_info()
        assert "filter_GBs" not in info0 and info0["total_degree"] == 0
        theta, resid, sweeps, st = g.build_reference(w.k, tol=1e-5)
        assert st == 0
        info = g.reference_info()
        nnz = len(w.val)
        assert info["filter_bytes_per_column_apply"] == 3 * nnz + 48 * w.N
        # every sweep applies H to at most `block` columns per degree of its filter (locked columns drop out), and once
        # more to the whole block for the Rayleigh-Ritz step
        assert 0 < info["filter_column_applies"] <= info["block"] * (info["total_degree"] + sweeps)
        assert info["filter_column_applies"] >= info["total_degree"] + info["block"] * sweeps
        assert 0 < info["filter_ms"] <= info["build_ms"]
        assert info["filter_GBs"] > 0
        # an analytical reference resets the counters
        g.build_reference_sine(w.k, list(w.dims))
        assert "filter_GBs" not in g.reference_info()
        tf = g.probe_fp64_tensor_peak()
        assert 5.0 < tf < 80.0, tf  # DMMA on B200: tens of TFLOP/s; the FP64 CUDA-core path alone is far below 5
    finally:
        g.close()
