"""Single steps of the path at BASELINE.json's FULL sizes, each against an independent computation that costs seconds:

  S2  rd_coarse_setup: G = W_I^T W_I and E_W = W_I^T H_II W_I at the config's own rank (k = 32, 48, 64, 64) against
      numpy contractions of the oracle's operator applies, C against the definition Q = Z E^-1 Z^T through its action;
  S6  rd_pdas_update: lambda, the new active set, the margin and the counts at N up to 4,096,000 against numpy on the
      oracle's H y (eq. (7)-(8));
  S7  rd_kkt: the five measures of eq. (25) on a perturbed pair at full size against numpy;
  S0  rd_build_reference on config 2 (N = 262,144, k = 32): eigenvalues against the library eigensolver on the assembled H.

The reference used for S2 is the oracle's analytical one (closed form, cheap); the operator applies use the threaded
build of the oracle (bit-identical to the plain build for K, K^T and H, tests/test_oracle_pins.py)."""
import numpy as np
import pytest

from workloads import make_config

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module", params=[2, 3, 4, 5])
def big(request, oracle_mod):
    import torch

    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    import paper_2606_17971_b200 as pkg

    pkg.load_library()
    w = make_config(request.param)
    o = oracle_mod.Oracle.from_workload(w, threaded=True)
    g = pkg.RefDef.from_workload(w, pkg.Options(pdas_cap=w.pdas_cap))
    yield w, o, g, pkg, oracle_mod
    g.close()


def front_mask(w, frac):
    """A PDAS-like active set: everything active except a ball around a hot spot holding `frac` of the DOFs, plus a
    sprinkle of single inactive DOFs (so that slices with one live row exist)."""
    rng = np.random.default_rng(77 + w.config)
    yd = w._target(1000 * w.config)
    thr = np.quantile(yd, 1.0 - frac)
    act = (yd < thr).astype(np.uint8)
    act[rng.choice(w.N, 50, replace=False)] = 0
    return act


def test_fullsize_pdas_update_and_kkt(big):
    w, o, g, pkg, oracle_mod = big
    rng = np.random.default_rng(5 + w.config)
    yd = w._target(1000 * w.config)
    psi = np.full(w.N, 0.6 * yd.max())
    psi[rng.choice(w.N, 1000, replace=False)] = np.inf
    act = front_mask(w, 0.4)
    act[np.isinf(psi)] = 0
    y = np.where(act == 1, np.where(np.isfinite(psi), psi, 0.0), 0.55 * yd.max() + 0.1 * yd.max() * rng.standard_normal(w.N))
    Hy = o.apply_H(y)
    ell = w.m * yd
    lam_ref = np.where(act == 1, ell - Hy, 0.0)
    fin = np.isfinite(psi)
    for c_is_diag in (0, 1):
        g.set_options(pkg.Options(pdas_cap=w.pdas_cap, c_is_diag=c_is_diag))
        c = o.diag_H() if c_is_diag else np.ones(w.N)
        gval = np.where(fin, lam_ref + c * (y - np.where(fin, psi, 0.0)), -1.0)
        new_ref = ((gval > 0) & fin).astype(np.uint8)
        lam, act_new, changed, n_new, margin = g.pdas_update(yd, psi, act, y)
        assert np.abs(lam - lam_ref).max() <= 1e-12 * np.abs(lam_ref).max()
        assert (lam[act == 0] == 0).all()
        # a decision may differ only where |g| is at rounding level of the H y product
        diff = np.flatnonzero(act_new != new_ref)
        assert (np.abs(gval[diff]) <= 1e-12 * np.abs(Hy).max()).all()
        assert abs(changed - int((new_ref != act).sum())) <= len(diff) and abs(n_new - int(new_ref.sum())) <= len(diff)
        assert np.isclose(margin, np.abs(gval[fin]).min(), rtol=1e-6, atol=1e-15 * np.abs(Hy).max())
    g.set_options(pkg.Options(pdas_cap=w.pdas_cap))
    # eq. (25) on the same (infeasible, non-complementary) pair
    lam2 = lam_ref + 0.05 * np.abs(ell).max() * rng.standard_normal(w.N)
    gr = Hy - ell
    s = max(1.0, np.abs(ell).max())
    exp = np.array([np.abs(gr + lam2).max() / s, np.maximum(y[fin] - psi[fin], 0.0).max(), np.maximum(-lam2, 0.0).max() / s,
                    np.abs(lam2[fin] * (psi[fin] - y[fin])).max() / s, np.abs(y - np.minimum(psi, y - gr)).max() / s])
    got = g.kkt(yd, psi, y, lam2)
    assert np.allclose(got, exp, rtol=1e-9, atol=1e-13 * np.abs(Hy).max()), (got, exp)


def test_fullsize_coarse_setup_matches_definition(big):
    w, o, g, pkg, oracle_mod = big
    if w.nt > 1:
        W = oracle_mod.spacetime_reference(w.dims, w.nt, 1.0 / w.nt, w.k)[-1]
    else:
        W = oracle_mod.sine_reference(w.dims, w.k)[-1]
    W = np.asfortranarray(W)
    g.set_reference(W)
    act = front_mask(w, 0.7)
    idx = np.flatnonzero(act == 0)
    cs = g.coarse_setup(pkg.REFDEF, act)
    WI = W[idx]
    G_ref = WI.T @ WI
    HW = np.empty_like(WI)
    for j in range(w.k):
        HW[:, j] = o.apply_B(idx, WI[:, j])
    EW_ref = WI.T @ HW
    assert np.abs(cs["G"] - G_ref).max() <= 1e-11 * np.abs(G_ref).max()
    assert np.abs(cs["EW"] - EW_ref).max() <= 1e-11 * np.abs(EW_ref).max()
    assert cs["rank"] == w.k and cs["fallback"] == 0
    # C is the coarse solve in W_I coordinates: Q = W_I C W_I^T satisfies Q B Q = Q, i.e. C E_W C = C
    C = cs["C"]
    assert np.abs(C @ EW_ref @ C - C).max() <= 1e-7 * np.abs(C).max()
    assert np.abs(C - C.T).max() <= 1e-12 * np.abs(C).max()
    # and the kernel's coarse correction removes the W_I-components of the error: from x0 = 0 the first iterate's
    # residual is B-orthogonal to range(W_I) -- checked through one capped solve
    rng = np.random.default_rng(9)
    b = np.zeros(w.N)
    b[idx] = w.m[idx] * rng.standard_normal(len(idx))
    g.set_options(pkg.Options(pdas_cap=w.pdas_cap, cg_cap=1))
    try:
        x, r = g.solve_inactive(pkg.REFDEF, act, b, np.zeros(w.N))
    finally:
        g.set_options(pkg.Options(pdas_cap=w.pdas_cap))
    res = b[idx] - o.apply_B(idx, x[idx])
    assert np.abs(WI.T @ res).max() <= 1e-8 * np.abs(WI.T @ b[idx]).max()  # Z^T (b - B x) = 0 after line 3 / every step


def test_fullsize_reference_build_config2(oracle_mod):
    import torch

    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    import paper_2606_17971_b200 as pkg

    w = make_config(2)
    g = pkg.RefDef.from_workload(w)
    theta, resid, sweeps, st = g.build_reference(w.k, tol=1e-5, max_block_iters=200)
    assert st == 0 and resid.max() <= 1e-5
    th_ref, W_ref = oracle_mod.reference_eigs(w.rowptr, w.colidx, w.val, w.m, w.alpha, w.k)
    assert np.abs(theta / th_ref - 1.0).max() <= 1e-8  # eigenvalue error ~ residual^2
    # residuals against the ORACLE's operator, and orthonormality
    W = g.get_reference()
    o = oracle_mod.Oracle.from_workload(w, threaded=True)
    for j in (0, w.k // 2, w.k - 1):
        rj = o.apply_H(W[:, j]) - theta[j] * W[:, j]
        assert np.linalg.norm(rj) <= 2e-5 * theta[j]
    assert np.abs(W.T @ W - np.eye(w.k)).max() <= 1e-10
    g.close()


def test_fullsize_lobpcg_reference_config2(oracle_mod):
    """The second eigensolver of S0 (rd_build_reference_lobpcg) at full size: 512 x 512, k = 32, against the library
    eigensolver of the oracle, as for the filter-based one above."""
    import torch

    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    import paper_2606_17971_b200 as pkg

    w = make_config(2)
    g = pkg.RefDef.from_workload(w)
    theta, resid, iters, st = g.build_reference_lobpcg(w.k, w.dims, kappa_ref=1.0, tol=1e-5, max_iters=3000)
    assert st == 0 and resid.max() <= 1e-5, (st, iters, resid.max())
    th_ref, _ = oracle_mod.reference_eigs(w.rowptr, w.colidx, w.val, w.m, w.alpha, w.k)
    assert np.abs(theta / th_ref - 1.0).max() <= 1e-8
    W = g.get_reference()
    o = oracle_mod.Oracle.from_workload(w, threaded=True)
    for j in (0, w.k // 2, w.k - 1):
        rj = o.apply_H(W[:, j]) - theta[j] * W[:, j]
        assert np.linalg.norm(rj) <= 2e-5 * theta[j]
    assert np.abs(W.T @ W - np.eye(w.k)).max() <= 1e-9
    g.close()


def test_fullsize_lobpcg_reference_config3_agrees_with_the_filter(oracle_mod):
    """96^3, k = 48 (the library eigensolver of the oracle does not fit a test at this size): the two eigensolvers of the
    library, which share only the block apply of H, agree on the eigenvalues, and the LOBPCG vectors have small
    residuals against the ORACLE's operator."""
    import torch

    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    import paper_2606_17971_b200 as pkg

    w = make_config(3)
    g = pkg.RefDef.from_workload(w)
    th_f, res_f, _, st_f = g.build_reference(w.k, tol=1e-4, max_block_iters=200)
    th_l, res_l, iters, st_l = g.build_reference_lobpcg(w.k, w.dims, kappa_ref=1.0, tol=1e-4, max_iters=1000)
    assert st_f == 0 and st_l == 0, (st_f, st_l, iters)
    assert np.abs(th_l / th_f - 1.0).max() <= 1e-6, np.abs(th_l / th_f - 1.0).max()
    W = g.get_reference()
    o = oracle_mod.Oracle.from_workload(w, threaded=True)
    for j in (0, w.k // 2, w.k - 1):
        rj = o.apply_H(W[:, j]) - th_l[j] * W[:, j]
        assert np.linalg.norm(rj) <= 2e-4 * th_l[j]
    assert np.abs(W.T @ W - np.eye(w.k)).max() <= 1e-9
    g.close()
