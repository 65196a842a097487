"""Pins of the oracle parts that round 1 left unpinned ("parity unpinned" list):

  K1  the five acceptance measures of eq. (25) on a deliberately perturbed (y, lambda), so that all
      five are non-zero and different, with ||l||_inf > 1 so that the normalisation s = max(1, ||l||_inf) bites, and with
      psi = +inf entries;
  K2  the rank-zero fallback for cond(E) > 1e10: triggered, recorded, and its iterates are Jacobi-CG's;
  K3  the starts of a query (reading A5): a given J0, all inactive, and the inherited (y, J) of the
      previous query, each against dense-direct PDAS from the same start;
  K4  c_i = H_ii in eq. (8) and the reported margin min_i |lambda_i + c_i (y_i - psi_i)| per step.

Every expected value is computed here with numpy from the dense H (an independent route), never by the oracle.
Each pin was checked to FAIL under a plausible mistake (mutations listed in the docstrings; tried by hand on a copy of
oracle/refdef_oracle.c when the pin was written).
"""
import numpy as np
import pytest
import scipy.sparse as sp

import oracle
from workloads import make_steady_2d


def dense_H(K, m, sigma):
    Kd = K.toarray()
    return np.diag(m) + sigma * Kd.T @ np.diag(1.0 / m) @ Kd


def small_problem(n=7, seed=3, mass_scale=1.0):
    """A 2-D CHT operator of workloads/ with a NON-uniform positive lumped mass (so that M, M^-1 and diag(H) cannot be
    confused with multiples of the identity) scaled so that ||l||_inf > 1 when mass_scale is large."""
    w = make_steady_2d(n=n, channels=[(0.4, 0.6)], vel=20.0, alpha=1e-4, k=4, n_queries=2, n_bumps=3, psi_factor=0.4,
                       pdas_cap=60, config=1, name=f"pin_{n}")
    rng = np.random.default_rng(seed)
    m = w.m * mass_scale * rng.uniform(0.5, 2.0, w.N)
    K = sp.csr_matrix((w.val, w.colidx, w.rowptr), shape=(w.N, w.N))
    return w, K, m


def pdas_dense(H, ell, psi, J0, c=None, cap=300):
    """PDAS, eq. (7)-(8), with dense direct solves from the start J0; c = None means c_i = 1.
    Returns y, lam, the list of active sets at the start of each step, and the per-step margins."""
    N = len(ell)
    cvec = np.ones(N) if c is None else c
    J = J0.copy() & np.isfinite(psi)
    sets, margins = [], []
    for _ in range(cap):
        sets.append(J.copy())
        I = ~J
        y = np.where(J, psi, 0.0)
        if I.any():
            y[I] = np.linalg.solve(H[np.ix_(I, I)], ell[I] - H[np.ix_(I, J)] @ psi[J])
        lam = np.where(J, ell - H @ y, 0.0)
        fin = np.isfinite(psi)
        g = np.where(fin, lam + cvec * (y - np.where(fin, psi, 0.0)), -1.0)
        margins.append(np.abs(g[fin]).min() if fin.any() else np.inf)
        Jn = (g > 0) & fin
        if (Jn == J).all():
            return y, lam, sets, margins
        J = Jn
    raise AssertionError("dense PDAS did not converge")


def unpack(Jb, N):
    return np.unpackbits(Jb, bitorder="little")[:N].astype(bool)


# ------------------------------------------------------------------------------------------------------ K1: eq. (25)
@pytest.mark.parametrize("mass_scale", [1.0, 4.0e3])
def test_K1_kkt_measures_on_a_perturbed_pair(mass_scale):
    """Mutations this fails under: s applied to the primal measure, or not applied to one of the other four; s taken as
    ||l||_2 or without the max(1, .); g = l - Hy (sign); [y - psi]_+ taken as |y - psi|; [-lambda]_+ as |lambda|;
    min(psi, y - g) replaced by max or by min(psi, y + g); psi = inf rows contributing to [1] or [3]."""
    w, K, m = small_problem(7, mass_scale=mass_scale)
    N = w.N
    sigma = 1e-4
    H = dense_H(K, m, sigma)
    o = oracle.Oracle(w.rowptr, w.colidx, w.val, m, sigma)
    rng = np.random.default_rng(11)
    yd = rng.uniform(0.2, 1.0, N)
    ell = m * yd
    psi = np.full(N, 0.45)
    psi[rng.choice(N, 6, replace=False)] = np.inf
    # a pair that violates every condition by a different amount
    y = 0.45 + 0.01 * rng.standard_normal(N)          # some y_i > psi_i: primal infeasibility
    lam = 0.3 * ell.max() * rng.standard_normal(N)     # both signs: dual infeasibility, complementarity products
    g = H @ y - ell
    s = max(1.0, np.abs(ell).max())
    if mass_scale > 1:
        assert np.abs(ell).max() > 1.5, "the normalisation must bite in this case"
    else:
        assert np.abs(ell).max() < 1.0
    fin = np.isfinite(psi)
    exp = np.array([
        np.abs(g + lam).max() / s,
        np.maximum(y[fin] - psi[fin], 0.0).max(),
        np.maximum(-lam, 0.0).max() / s,
        np.abs(lam[fin] * (psi[fin] - y[fin])).max() / s,
        np.abs(y - np.minimum(psi, y - g)).max() / s,
    ])
    got = o.kkt(yd, psi, y, lam)
    assert np.allclose(got, exp, rtol=1e-12, atol=0.0), (got, exp)
    assert len(set(np.round(np.log10(exp), 3))) == 5 and (exp > 0).all(), "five different non-zero measures"
    # the projected-gradient measure really sees both branches of the min
    assert (psi < y - g).any() and (psi > y - g)[fin].any()
    # and on an exact KKT point all five vanish
    y_s, lam_s, _, _ = pdas_dense(H, ell, psi, np.ones(N, dtype=bool))
    assert o.kkt(yd, psi, y_s, lam_s).max() <= 1e-12
    assert lam_s.max() > 0, "the bound is active at this optimum"


def test_K1_query_report_uses_the_same_measures():
    w, K, m = small_problem(6)
    o = oracle.Oracle(w.rowptr, w.colidx, w.val, m, 1e-4)
    yd, _ = w.target(0)
    psi = np.full(w.N, 0.4 * yd.max())
    r = o.solve_query(oracle.JACOBI_CG, yd, psi, None, oracle.OracleOptions(eps=1e-9, eps_c=1e-9, pdas_cap=60))
    assert r["status"] == 0
    assert np.array_equal(np.array(r["kkt"]), o.kkt(yd, psi, r["y"], r["lam"]))


# ------------------------------------------------------------------------------------------------------ K2: fallback
def fallback_problem(span):
    """Tiny operator with a lumped mass spanning `span` orders of magnitude and a penalty small enough that
    H_ii = m_i + sigma sum_r K_ri^2 / m_r stays of the size of m_i: H has eigenvalues from ~10^(-span/2) to ~10^(span/2)
    and E = Z^T B Z on Z = [e_first, e_last] has cond ~ 10^span."""
    N = 8
    K = sp.diags([np.full(N, 2.0), np.full(N - 1, -1.0), np.full(N - 1, -0.5)], [0, -1, 1], format="csr")
    m = np.logspace(-span / 2, span / 2, N)
    sigma = 0.05 * m.min() ** 2
    return N, K, m, sigma


@pytest.mark.parametrize("span,expect_fallback", [(12, True), (8, False)])
def test_K2_cond_E_fallback_is_rank_zero_jacobi_cg(span, expect_fallback):
    """"rank-zero fallback if cond(E) > 1e10".  Mutations this fails under: threshold 1e12 or 1e8 (one of
    the two cases flips), fallback recorded but Z still used (iterates differ from Jacobi-CG), rank not reset to 0."""
    N, K, m, sigma = fallback_problem(span)
    H = dense_H(K, m, sigma)
    o = oracle.Oracle(K.indptr.astype(np.int64), K.indices.astype(np.int32), K.data, m, sigma)
    idx = np.arange(N, dtype=np.int64)
    Zt = np.zeros((N, 2))
    Zt[0, 0] = 1.0
    Zt[N - 1, 1] = 1.0
    E = Zt.T @ H @ Zt
    cond = np.linalg.cond(E)
    assert (cond > 1e10) == expect_fallback, cond  # the dense matrix decides which side of the threshold we are on
    rng = np.random.default_rng(5)
    b = H @ rng.standard_normal(N)
    cs = o.coarse(idx, Zt)
    assert cs.fallback == (1 if expect_fallback else 0)
    assert cs.rank == (0 if expect_fallback else 2)
    assert np.isclose(cs.cond_E, cond, rtol=1e-6)
    x_d, r_d = o.alg1(idx, b, np.zeros(N), Zt, eps=1e-10, cap=500)
    x_j, r_j = o.alg1(idx, b, np.zeros(N), None, eps=1e-10, cap=500)
    assert r_d["coarse_fallback"] == (1 if expect_fallback else 0)
    if expect_fallback:
        assert r_d["rank_used"] == 0
        assert np.array_equal(x_d, x_j) and r_d["iters"] == r_j["iters"], "fallback execution must be Jacobi-CG itself"
    else:
        assert r_d["rank_used"] == 2 and not np.array_equal(x_d, x_j)


# ------------------------------------------------------------------------------------------------------ K3: starts
def query_sets(r, N):
    return [unpack(Jb, N) for Jb in r["J_bits"]]


def test_K3_given_and_all_inactive_starts_match_dense_pdas():
    """Mutations this fails under: J0 ignored (start all active), J0 complemented, ALL_INACTIVE starting all active,
    psi = inf entries of J0 kept active."""
    w, K, m = small_problem(8)
    N, sigma = w.N, 1e-4
    H = dense_H(K, m, sigma)
    o = oracle.Oracle(w.rowptr, w.colidx, w.val, m, sigma)
    yd, _ = w.target(0)
    psi = np.full(N, 0.35 * yd.max())
    psi[[3, 17]] = np.inf
    ell = m * yd
    rng = np.random.default_rng(2)
    J0 = rng.random(N) < 0.4
    J0[3] = True  # a psi = inf entry of J0: never active (reading A5)
    for init, start in ((oracle.INIT_GIVEN, J0), (oracle.INIT_ALL_INACTIVE, np.zeros(N, dtype=bool)),
                        (oracle.INIT_ALL_ACTIVE, np.ones(N, dtype=bool))):
        o.reset_sequence()
        y_ref, lam_ref, sets_ref, _ = pdas_dense(H, ell, psi, start)
        opt = oracle.OracleOptions(eps=1e-12, eps_c=1e-12, pdas_cap=80, init=init)
        r = o.solve_query(oracle.JACOBI_CG, yd, psi, None, opt, J0=J0.astype(np.uint8))
        assert r["status"] == 0 and r["n_steps"] == len(sets_ref), (init, r["n_steps"], len(sets_ref))
        for a, b_ in zip(query_sets(r, N), sets_ref):
            assert (a == b_).all()
        assert np.allclose(r["y"], y_ref, rtol=1e-9, atol=1e-12)
    # the three starts give different sequences here (else the pin could not tell them apart)
    lens = {len(pdas_dense(H, ell, psi, s_)[2]) for s_ in (J0, np.zeros(N, dtype=bool), np.ones(N, dtype=bool))}
    first = [pdas_dense(H, ell, psi, s_)[2][0].sum() for s_ in (J0, np.zeros(N, dtype=bool), np.ones(N, dtype=bool))]
    assert len(set(first)) == 3 and len(lens) >= 1


def test_K3_second_query_inherits_state_and_active_set():
    """"Subsequent queries receive the preceding solution and active set".  Mutations this fails under:
    second query restarting all active; inheriting J but not y (the repeated query then needs CG iterations);
    reset_sequence not forgetting the state."""
    w, K, m = small_problem(8)
    N, sigma = w.N, 1e-4
    H = dense_H(K, m, sigma)
    o = oracle.Oracle(w.rowptr, w.colidx, w.val, m, sigma)
    opt = oracle.OracleOptions(eps=1e-12, eps_c=1e-12, pdas_cap=80)  # INIT_PAPER
    yd1, _ = w.target(0)
    yd2, _ = w.target(1)
    psi1 = np.full(N, 0.35 * yd1.max())
    psi2 = np.full(N, 0.30 * yd2.max())
    r1 = o.solve_query(oracle.JACOBI_CG, yd1, psi1, None, opt)
    _, _, sets1, _ = pdas_dense(H, m * yd1, psi1, np.ones(N, dtype=bool))
    assert r1["status"] == 0 and (query_sets(r1, N)[0]).all() and len(sets1) == r1["n_steps"]
    J_final = sets1[-1]
    assert J_final.any()
    # second, different query: dense PDAS started from the inherited set
    r2 = o.solve_query(oracle.JACOBI_CG, yd2, psi2, None, opt)
    y2, _, sets2, _ = pdas_dense(H, m * yd2, psi2, J_final)
    assert r2["status"] == 0 and r2["n_steps"] == len(sets2)
    for a, b_ in zip(query_sets(r2, N), sets2):
        assert (a == b_).all()
    assert np.allclose(r2["y"], y2, rtol=1e-9, atol=1e-12)
    assert len(sets2) != len(pdas_dense(H, m * yd2, psi2, np.ones(N, dtype=bool))[2]) or \
        not (sets2[0] == np.ones(N, dtype=bool)).all()
    # the same query again: the inherited y is already the solution, so the inner solve stops at line 4 of Alg. 1
    r3 = o.solve_query(oracle.JACOBI_CG, yd2, psi2, None, opt)
    assert r3["n_steps"] == 1 and r3["steps"][0]["cg_iters"] == 0
    assert (query_sets(r3, N)[0] == sets2[-1]).all()
    # a new sequence forgets both
    o.reset_sequence()
    r4 = o.solve_query(oracle.JACOBI_CG, yd2, psi2, None, opt)
    assert query_sets(r4, N)[0].all() and r4["steps"][-1]["cg_iters"] > 0


# ------------------------------------------------------------------------------------------------------ K4: c and margin
@pytest.mark.parametrize("c_is_diag", [0, 1])
def test_K4_c_is_diag_and_margin(c_is_diag):
    """eq. (8) with c_i = H_ii or c = 1 (the configs).  With lambda_I = 0 (reading A4) no decision depends
    on c > 0, so what c changes is the reported distance to a tie: margin = min_i |lambda_i + c_i (y_i - psi_i)|.
    Mutations this fails under: c_is_diag ignored, c = 1/H_ii, c = m_i, margin taken over I only or over J only,
    margin without the absolute value."""
    w, K, m = small_problem(8, mass_scale=50.0)
    N, sigma = w.N, 1e-4
    H = dense_H(K, m, sigma)
    d = np.diag(H).copy()
    assert d.max() / d.min() > 3 and not np.allclose(d, 1.0)
    o = oracle.Oracle(w.rowptr, w.colidx, w.val, m, sigma)
    assert np.allclose(o.diag_H(), d, rtol=1e-13)
    yd, _ = w.target(0)
    psi = np.full(N, 0.35 * yd.max())
    ell = m * yd
    opt = oracle.OracleOptions(eps=1e-13, eps_c=1e-13, pdas_cap=80, c_is_diag=c_is_diag)
    r = o.solve_query(oracle.JACOBI_CG, yd, psi, None, opt)
    _, _, sets_ref, margins = pdas_dense(H, ell, psi, np.ones(N, dtype=bool), c=d if c_is_diag else None)
    assert r["status"] == 0 and r["n_steps"] == len(sets_ref)
    for a, b_ in zip(query_sets(r, N), sets_ref):
        assert (a == b_).all()
    got = np.array([s_["margin"] for s_ in r["steps"]])
    assert np.allclose(got, margins, rtol=1e-6, atol=1e-14), (got, margins)
    other = pdas_dense(H, ell, psi, np.ones(N, dtype=bool), c=None if c_is_diag else d)[3]
    assert not np.allclose(margins, other, rtol=1e-3), "the two choices of c must give different margins here"


# ------------------------------------------------------------------------------------------------------ K5: eq. (23)
def test_K5_deflated_spectrum_eq23():
    """eq. (23).  Pins: (a) with Z = the k lowest eigenvectors of the pencil (B, D) the nonzero spectrum
    is exactly the rest of the pencil's spectrum (deflation removes what Z spans and nothing else); (b) rank zero gives
    the whole pencil; (c) for a generic Z the matrix annihilates D^{1/2} Z (r zeros), its nonzero eigenvalues interlace
    the pencil's: mu_j <= lam_j <= mu_{j+r}; (d) Algorithm 1's iteration count obeys the classical CG bound for the
    effective condition number.  Mutations this fails under: D^{-1} in place of D^{-1/2}, Z^T B Z replaced by Z^T Z,
    the r zeros not dropped, B Z taken as Z, D = diag(H) on all N rows instead of diag(B) on I (same here) -- and a
    transposed or unsymmetrised B."""
    import scipy.linalg as sla

    w, K, m = small_problem(9)
    N, sigma = w.N, 1e-4
    H = dense_H(K, m, sigma)
    o = oracle.Oracle(w.rowptr, w.colidx, w.val, m, sigma)
    rng = np.random.default_rng(4)
    idx = np.flatnonzero(rng.random(N) > 0.25).astype(np.int64)
    n = len(idx)
    B = H[np.ix_(idx, idx)]
    D = np.diag(np.diag(B))
    mu, V = sla.eigh(B, D)  # B v = mu D v, ascending
    k = 5
    lam, r = oracle.deflated_spectrum(o, idx, V[:, :k])
    assert r == k and len(lam) == n - k
    assert np.allclose(lam, mu[k:], rtol=1e-9)
    lam0, r0 = oracle.deflated_spectrum(o, idx, None)
    assert r0 == 0 and np.allclose(lam0, mu, rtol=1e-10)
    # generic basis: Cauchy interlacing of the compression to the B-orthogonal complement
    Zt = rng.standard_normal((n, 4))
    lam_g, r_g = oracle.deflated_spectrum(o, idx, Zt)
    assert r_g == 4 and len(lam_g) == n - 4
    assert (lam_g >= mu[: n - 4] * (1 - 1e-9)).all() and (lam_g <= mu[4:] * (1 + 1e-9)).all()
    assert lam_g[0] > 1e-6 * lam_g[-1], "the r zero eigenvalues must have been dropped"
    # independent dense evaluation of the matrix of eq. (23) for the generic basis
    Q, _ = np.linalg.qr(Zt)
    Ssc = np.diag(1.0 / np.sqrt(np.diag(B)))
    A = Ssc @ (B - B @ Q @ np.linalg.solve(Q.T @ B @ Q, Q.T @ B)) @ Ssc
    ref = np.linalg.eigvalsh(0.5 * (A + A.T))[4:]
    assert np.allclose(lam_g, ref, rtol=1e-8)
    # the solver sees this spectrum: iterations <= the CG bound for kappa_eff = lam_max / lam_min
    b = rng.standard_normal(n)
    eps = 1e-10
    _, rep = o.alg1(idx, b, np.zeros(n), Zt, eps=eps)
    kappa = lam_g[-1] / lam_g[0]
    # energy-norm bound 2 ((sqrt(k)-1)/(sqrt(k)+1))^m, converted to the residual with sqrt(kappa(B^)) slack
    bound = np.ceil(0.5 * np.sqrt(kappa) * np.log(2.0 * np.sqrt(mu[-1] / mu[0]) / eps)) + 1
    assert rep["status"] == 0 and rep["iters"] <= bound
    _, rep_j = o.alg1(idx, b, np.zeros(n), None, eps=eps)
    assert rep["iters"] <= rep_j["iters"]
