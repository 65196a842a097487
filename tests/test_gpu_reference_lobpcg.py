"""GPU parity of rd_build_reference_lobpcg (S0 by LOBPCG with the sine-transform preconditioner of the homogeneous grid
operator, csrc/lobpcg.cuh) against the same definition as rd_build_reference: the k lowest eigenpairs of H from a
library eigensolver in the oracle (oracle.reference_eigs), residuals against the ORACLE's operator, orthonormality,
principal angles of complete clusters.  The preconditioner cannot change the result, only the number of iterations:
the iteration bounds below are what fails if a transform, an axis stride or the spectral scaling were wrong."""
import numpy as np
import pytest

from workloads import make_config, make_steady_2d, make_steady_3d

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def rd():
    import torch

    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    import paper_2606_17971_b200 as pkg

    pkg.load_library()
    return pkg


@pytest.fixture(scope="module")
def oracle_mod():
    import oracle

    return oracle


CASES = {
    "config1": lambda: make_config(1),                      # 32 x 32, k = 8
    "c2_48": lambda: make_config(twin="c2_48"),             # 48 x 48, k = 16
    "c3_16": lambda: make_config(twin="c3_16"),             # 16^3, k = 16
    "c3_24": lambda: make_config(twin="c3_24"),             # 24^3, k = 24: n not a multiple of 16
    "ragged37": lambda: make_steady_2d(n=37, channels=[(0.4, 0.6)], vel=20.0, alpha=1e-4, k=5, n_queries=2, n_bumps=3,
                                       psi_factor=0.6, pdas_cap=60, config=1, name="ragged37"),  # n odd: ragged tiles
    "ragged3d_13": lambda: make_steady_3d(n=13, bores=[(0.5, 0.5)], R=0.3, vpeak=30.0, alpha=1e-5, k=6, n_queries=1,
                                          n_bumps=4, psi_factor=0.6, pdas_cap=40, config=3, name="ragged3d_13"),
}


def _cluster_cut(theta, k):
    c = k
    while c > 0 and (theta[c] - theta[c - 1]) < 1e-5 * theta[c]:
        c -= 1
    return c


@pytest.mark.parametrize("case", list(CASES))
def test_lobpcg_reference_matches_library_eigensolver(rd, oracle_mod, case):
    w = CASES[case]()
    o = oracle_mod.Oracle.from_workload(w)
    g = rd.RefDef.from_workload(w, rd.Options(pdas_cap=w.pdas_cap))
    try:
        theta, resid, iters, st = g.build_reference_lobpcg(w.k, w.dims, kappa_ref=1.0, tol=1e-7, max_iters=400)
        assert st == 0 and resid.max() <= 1e-7, (st, iters, resid.max())
        assert 1 <= iters <= 250, iters  # a broken preconditioner needs thousands (cond(H) = 1e4 ... 1e7 here)
        th_o, W_o = oracle_mod.reference_eigs(w.rowptr, w.colidx, w.val, w.m, w.alpha, w.k + 1)
        assert np.allclose(theta, th_o[:w.k], rtol=1e-9)
        assert (np.diff(theta) >= 0).all()
        W = g.get_reference()
        assert W.shape == (w.N, w.k)
        assert np.abs(W.T @ W - np.eye(w.k)).max() <= 1e-9
        for c in range(w.k):  # residual of every column against the ORACLE's operator
            r = o.apply_H(W[:, c]) - theta[c] * W[:, c]
            assert np.linalg.norm(r) <= 2e-7 * theta[c]
        cut = _cluster_cut(th_o, w.k)
        if cut > 0:
            sv = np.linalg.svd(W[:, :cut].T @ W_o[:, :cut], compute_uv=False)
            assert sv.min() >= 1.0 - 1e-8
        info = g.reference_info()
        assert info["build_ms"] > 0 and info["block"] >= w.k + 8 and "filter_GBs" not in info
    finally:
        g.close()


def test_lobpcg_reference_serves_a_query_like_the_filter_built_one(rd):
    """The two eigensolvers build the same subspace: a deflated query gives the same active-set sequence with either."""
    import torch

    w = make_config(twin="c2_48")
    yd, psi = w.target(0)
    res = []
    for which in ("filter", "lobpcg"):
        g = rd.RefDef.from_workload(w, rd.Options(pdas_cap=w.pdas_cap))
        try:
            if which == "filter":
                _, _, _, st = g.build_reference(w.k, tol=1e-8)
            else:
                _, _, _, st = g.build_reference_lobpcg(w.k, w.dims, tol=1e-8)
            assert st == 0
            r = g.solve_query(rd.REFDEF, yd, psi)
            assert r["status"] == 0
            res.append(r)
        finally:
            g.close()
    assert res[0]["hashes"] == res[1]["hashes"]
    m = w.m
    assert np.sqrt((m * (res[0]["y"] - res[1]["y"]) ** 2).sum() / (m * res[0]["y"] ** 2).sum()) <= 1e-6


def test_lobpcg_reference_edge_cases(rd, oracle_mod):
    w = make_config(twin="c2_48")
    g = rd.RefDef.from_workload(w, rd.Options(pdas_cap=w.pdas_cap))
    try:
        th_o, _ = oracle_mod.reference_eigs(w.rowptr, w.colidx, w.val, w.m, w.alpha, 64)
        theta, resid, it, st = g.build_reference_lobpcg(1, w.dims, tol=1e-6)
        assert st == 0 and abs(theta[0] / th_o[0] - 1) <= 1e-9
        theta, resid, it, st = g.build_reference_lobpcg(64, w.dims, tol=1e-5)  # 3 b = 240 basis vectors
        assert st == 0 and np.allclose(theta, th_o, rtol=1e-8)
        # a comparison medium that is far off only costs iterations
        theta2, _, it2, st = g.build_reference_lobpcg(64, w.dims, kappa_ref=0.2, tol=1e-5)
        assert st == 0 and np.allclose(theta2, th_o, rtol=1e-8)
        # an iteration cap that is too small is a soft status and leaves a usable reference
        theta, resid, it, st = g.build_reference_lobpcg(8, w.dims, tol=1e-12, max_iters=2)
        assert st == -6 and it == 2 and g.get_reference().shape == (w.N, 8)
        r = g.solve_query(1, *w.target(0))
        assert r["status"] == 0
        for bad in (dict(k=0), dict(k=65), dict(dims=[48, 47]), dict(kappa_ref=0.0), dict(tol=0.0)):
            kw = dict(k=8, dims=list(w.dims), kappa_ref=1.0, tol=1e-3)
            kw.update(bad)
            with pytest.raises(rd.RefDefError):
                g.build_reference_lobpcg(kw["k"], kw["dims"], kappa_ref=kw["kappa_ref"], tol=kw["tol"])
    finally:
        g.close()


def test_lobpcg_work_accounting(rd):
    """rd_reference_lobpcg_work: zeros before / after another construction, a flop count that matches the iteration count."""
    w = make_config(twin="c3_16")
    g = rd.RefDef.from_workload(w)
    try:
        assert "lobpcg_TFLOPs" not in g.reference_info()
        theta, resid, iters, st = g.build_reference_lobpcg(w.k, w.dims, tol=1e-4)
        assert st == 0
        info = g.reference_info()
        b = info["block"]
        assert info["lobpcg_iterations"] == iters and info["lobpcg_loop_ms"] > 0
        # every iteration preconditions and applies H to at most b columns, at least 8; the start adds b applies of each
        assert 8 * iters <= info["lobpcg_t_column_applies"] - b <= b * iters
        assert info["lobpcg_h_column_applies"] >= info["lobpcg_t_column_applies"]
        # lower bound of the tensor work: the sine transforms alone
        assert info["lobpcg_tensor_flop"] >= 4.0 * sum(w.dims) * w.N * info["lobpcg_t_column_applies"]
        g.build_reference_sine(w.k, list(w.dims))
        assert "lobpcg_TFLOPs" not in g.reference_info()
    finally:
        g.close()


def test_lobpcg_eigenvalue_whitening_path(rd, oracle_mod, monkeypatch):
    """The fallback of the Rayleigh-Ritz step (eigen-decomposition of the Gram matrix with dropped directions instead of its
    Cholesky factor) is what runs when the basis [X, W, P] is dependent to working accuracy; RD_LOBPCG_NO_CHOL takes it on
    every iteration.  Same result."""
    w = make_config(twin="c3_16")
    monkeypatch.setenv("RD_LOBPCG_NO_CHOL", "1")
    g = rd.RefDef.from_workload(w)
    try:
        theta, resid, iters, st = g.build_reference_lobpcg(w.k, w.dims, tol=1e-7, max_iters=400)
        assert st == 0 and resid.max() <= 1e-7 and iters <= 250
        th_o, _ = oracle_mod.reference_eigs(w.rowptr, w.colidx, w.val, w.m, w.alpha, w.k)
        assert np.allclose(theta, th_o, rtol=1e-9)
    finally:
        g.close()
