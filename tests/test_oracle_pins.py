"""Pins of the CPU oracle against what the paper and the mathematics fix.

None of these tests touches the CUDA path.  Dense reference quantities are built here with
numpy/scipy from the workload's K, m (an independent route: dense factorisations, brute force,
closed forms), never by calling the oracle on itself.
"""
import itertools
import os

import numpy as np
import pytest

from workloads import make_config, make_steady_2d, make_steady_3d, make_spacetime_2d

HERE = os.path.dirname(os.path.abspath(__file__))


def dense_H(w):
    K = w.csr().toarray()
    return np.diag(w.m) + w.alpha * K.T @ np.diag(1.0 / w.m) @ K


def tiny_2d(n=8, seed_cfg=1):
    return make_steady_2d(n=n, channels=[(0.4, 0.6)], vel=20.0, alpha=1e-4, k=4, n_queries=2, n_bumps=3,
                          psi_factor=0.6, pdas_cap=40, config=seed_cfg, name=f"tiny2d_{n}")


def tiny_3d(n=5):
    return make_steady_3d(n=n, bores=[(0.5, 0.5)], R=0.3, vpeak=30.0, alpha=1e-5, k=4, n_queries=1, n_bumps=4,
                          psi_factor=0.6, pdas_cap=40, config=3, name=f"tiny3d_{n}")


def tiny_st(n=6, nt=3):
    return make_spacetime_2d(n=n, nt=nt, T=1.0, channels=[(0.4, 0.6)], vel=20.0, alpha=1e-4, k=4, n_queries=1,
                             n_bumps=3, psi_factor=0.6, pdas_cap=40, config=4, name=f"tinyst_{n}x{nt}")


def pdas_dense(H, ell, psi, J0, cap=200):
    """PDAS (eq. (7)-(8)) with dense direct solves; returns (y, lam, list of active sets)."""
    N = len(ell)
    J = J0.copy()
    sets = []
    y = np.zeros(N)
    for _ in range(cap):
        sets.append(J.copy())
        I = ~J
        y = np.where(J, psi, 0.0)
        if I.any():
            rhs = ell[I] - H[np.ix_(I, J)] @ psi[J]
            y[I] = np.linalg.solve(H[np.ix_(I, I)], rhs)
        lam = np.where(J, ell - H @ y, 0.0)
        Jn = (lam + (y - psi)) > 0
        if (Jn == J).all():
            return y, lam, sets
        J = Jn
    raise AssertionError("dense PDAS did not converge")


# ------------------------------------------------------------------ P2: symmetry, definiteness, masked apply
@pytest.mark.parametrize("maker", [tiny_2d, tiny_3d, tiny_st])
def test_P2_operator_matches_dense_and_is_spd(oracle_mod, maker):
    w = maker()
    o = oracle_mod.Oracle.from_workload(w)
    H = dense_H(w)
    rng = np.random.default_rng(0)
    x, yv = rng.standard_normal(w.N), rng.standard_normal(w.N)
    Hx, Hy = o.apply_H(x), o.apply_H(yv)
    assert np.allclose(Hx, H @ x, rtol=1e-13, atol=1e-13 * np.abs(H @ x).max())
    assert abs(x @ Hy - yv @ Hx) <= 1e-13 * abs(x @ Hy)
    assert x @ Hx >= (w.m * x * x).sum()  # H - M = sigma (M^-1/2 K)^T (M^-1/2 K) >= 0
    np.linalg.cholesky(H)
    assert np.allclose(o.diag_H(), np.diag(H), rtol=1e-13)
    # K, K^T legs on their own: a transposed operand must fail here
    Kd = w.csr().toarray()
    assert np.allclose(o.apply_K(x), Kd @ x, rtol=1e-13, atol=1e-13)
    assert np.allclose(o.apply_KT(x), Kd.T @ x, rtol=1e-13, atol=1e-13)
    assert not np.allclose(Kd @ x, Kd.T @ x)
    # B x = (H R_I^T x)_I and every H_II is SPD
    mask = rng.random(w.N) < 0.7
    idx = np.flatnonzero(mask)
    xi = rng.standard_normal(len(idx))
    assert np.allclose(o.apply_B(idx, xi), H[np.ix_(idx, idx)] @ xi, rtol=1e-12, atol=1e-14)
    np.linalg.cholesky(H[np.ix_(idx, idx)])


# ------------------------------------------------------------------ P7: closed-form spectrum
def test_P7_closed_form_spectrum(oracle_mod):
    """Uniform kappa = 1, zero velocity: K has eigenvectors prod_a sin(pi k_a (j_a - 1/2)/n) and eigenvalues
    h^(d-2) sum_a 4 sin^2(pi k_a/(2n)); theta = h^d + sigma (K-eig)^2 / h^d.
    Cell-centred analogue of eq. (15)."""
    n = 10
    w = make_steady_2d(n=n, channels=[], vel=0.0, alpha=1e-4, k=6, n_queries=1, n_bumps=1, psi_factor=0.6,
                       pdas_cap=5, config=1)
    o = oracle_mod.Oracle.from_workload(w)
    h = 1.0 / n
    j = np.arange(1, n + 1)
    thetas = []
    for kx, ky in itertools.product(range(1, n + 1), repeat=2):
        mu = 4 * np.sin(np.pi * kx / (2 * n)) ** 2 + 4 * np.sin(np.pi * ky / (2 * n)) ** 2  # h^(d-2) = 1
        theta = h ** 2 + w.alpha * mu ** 2 / h ** 2
        thetas.append(theta)
        if (kx, ky) in [(1, 1), (2, 1), (1, 3), (n, n), (4, 7)]:
            v = np.outer(np.sin(np.pi * ky * (j - 0.5) / n), np.sin(np.pi * kx * (j - 0.5) / n)).ravel()
            assert np.allclose(o.apply_H(v), theta * v, rtol=1e-11, atol=1e-13 * theta)
    thetas = np.sort(thetas)
    th, W = oracle_mod.reference_eigs(w.rowptr, w.colidx, w.val, w.m, w.alpha, 6)
    assert np.allclose(th, thetas[:6], rtol=1e-10)
    assert np.allclose(W.T @ W, np.eye(6), atol=1e-10)
    # sparse shift-invert branch agrees with the dense branch
    th2, W2 = oracle_mod.reference_eigs(w.rowptr, w.colidx, w.val, w.m, w.alpha, 6, dense_below=10)
    assert np.allclose(th2, thetas[:6], rtol=1e-9)
    # 3D, the 7-point analogue
    n3 = 5
    w3 = make_steady_3d(n=n3, bores=[], R=0.1, vpeak=0.0, alpha=1e-5, k=4, n_queries=1, n_bumps=1, psi_factor=0.6,
                        pdas_cap=5, config=3)
    o3 = oracle_mod.Oracle.from_workload(w3)
    h3 = 1.0 / n3
    j3 = np.arange(1, n3 + 1)
    kx, ky, kz = 2, 1, 3
    s = lambda q: np.sin(np.pi * q * (j3 - 0.5) / n3)
    v = np.einsum("z,y,x->zyx", s(kz), s(ky), s(kx)).ravel()
    mu = h3 * sum(4 * np.sin(np.pi * q / (2 * n3)) ** 2 for q in (kx, ky, kz))
    theta = h3 ** 3 + w3.alpha * mu ** 2 / h3 ** 3
    assert np.allclose(o3.apply_H(v), theta * v, rtol=1e-11, atol=1e-14 * theta)


# ------------------------------------------------------------------ P1/P3: PDAS against dense direct PDAS + KKT
@pytest.mark.parametrize("maker,psi_factor", [(tiny_2d, 0.6), (tiny_2d, 0.3), (tiny_3d, 0.35), (tiny_st, 0.3)])
@pytest.mark.parametrize("method", [0, 1, 2])
def test_P1_P3_pdas_matches_dense_direct(oracle_mod, maker, psi_factor, method):
    w = maker()
    o = oracle_mod.Oracle.from_workload(w)
    H = dense_H(w)
    yd, _ = w.target(0)
    psi = np.full(w.N, psi_factor * yd.max())
    ell = w.m * yd
    y_ref, lam_ref, sets_ref = pdas_dense(H, ell, psi, np.ones(w.N, dtype=bool))
    _, W = oracle_mod.reference_eigs(w.rowptr, w.colidx, w.val, w.m, w.alpha, w.k)
    opt = oracle_mod.OracleOptions(eps=1e-12, eps_c=1e-12, pdas_cap=60)
    r = o.solve_query(method, yd, psi, W, opt)
    assert r["status"] == 0
    assert r["n_steps"] == len(sets_ref)
    for s, Jb in zip(sets_ref, r["J_bits"]):
        assert (np.unpackbits(Jb, bitorder="little")[: w.N].astype(bool) == s).all()
    nrm = lambda v: np.sqrt((w.m * v * v).sum())
    assert nrm(r["y"] - y_ref) <= 1e-9 * nrm(y_ref)
    # P3: KKT system eq. (6) with the independent dense H
    y, lam = r["y"], r["lam"]
    assert np.abs(H @ y - ell + lam).max() <= 1e-10 * np.abs(ell).max()
    assert (y <= psi + 1e-12).all() and (lam >= -1e-14).all()
    assert np.abs(lam * (psi - y)).max() <= 1e-14
    assert max(r["kkt"]) <= 1e-8  # eq. (25)
    # recovery eq. (9): u = M^-1 K y uses all state values incl. the active ones
    assert np.allclose(r["u"], (w.csr() @ y) / w.m, rtol=1e-12, atol=1e-12)
    if psi_factor <= 0.35:
        assert sets_ref[-1].any(), "bound must be active at the optimum for this pin to bite"


def test_P1_bruteforce_active_sets(oracle_mod):
    """N = 9: enumerate all 2^N active sets; strict convexity => exactly one satisfies eq. (6)."""
    w = make_steady_2d(n=3, channels=[(0.4, 0.6)], vel=20.0, alpha=1e-5, k=2, n_queries=1, n_bumps=3,
                       psi_factor=0.3, pdas_cap=40, config=1)
    H = dense_H(w)
    yd, psi = w.target(0)
    ell = w.m * yd
    sols = []
    for bits in itertools.product([False, True], repeat=w.N):
        J = np.array(bits)
        I = ~J
        y = np.where(J, psi, 0.0)
        if I.any():
            y[I] = np.linalg.solve(H[np.ix_(I, I)], ell[I] - H[np.ix_(I, J)] @ psi[J])
        lam = np.where(J, ell - H @ y, 0.0)
        if (y[I] < psi[I]).all() and (lam[J] > 0).all():  # strict: excludes degenerate duplicates
            sols.append((J, y))
    assert len(sols) == 1
    J_star, y_star = sols[0]
    assert J_star.any() and not J_star.all()
    o = oracle_mod.Oracle.from_workload(w)
    r = o.solve_query(0, yd, psi, None, oracle_mod.OracleOptions(eps=1e-13, eps_c=1e-13, pdas_cap=40))
    assert r["status"] == 0
    J_fin = np.unpackbits(r["J_bits"][-1], bitorder="little")[: w.N].astype(bool)
    assert (J_fin == J_star).all()
    assert np.allclose(r["y"], y_star, rtol=1e-10, atol=1e-12)


# ------------------------------------------------------------------ P4: unconstrained limit
@pytest.mark.parametrize("method", [0, 1])
def test_P4_unconstrained_limit(oracle_mod, method):
    w = tiny_2d(10)
    o = oracle_mod.Oracle.from_workload(w)
    H = dense_H(w)
    yd, _ = w.target(0)
    psi = np.full(w.N, np.inf)
    _, W = oracle_mod.reference_eigs(w.rowptr, w.colidx, w.val, w.m, w.alpha, w.k)
    r = o.solve_query(method, yd, psi, W, oracle_mod.OracleOptions(eps=1e-12, eps_c=1e-12))
    y_ref = np.linalg.solve(H, w.m * yd)
    assert r["status"] == 0 and r["n_steps"] == 1 and r["steps"][0]["n_inactive"] == w.N
    assert np.allclose(r["y"], y_ref, rtol=1e-9, atol=1e-12)
    assert (r["lam"] == 0).all()
    assert np.allclose(r["u"], (w.csr() @ r["y"]) / w.m, rtol=1e-12)


# ------------------------------------------------------------------ P5: projector identities
def test_P5_projector_identities(oracle_mod):
    w = tiny_2d(8)
    o = oracle_mod.Oracle.from_workload(w)
    H = dense_H(w)
    rng = np.random.default_rng(3)
    idx = np.flatnonzero(rng.random(w.N) < 0.8)
    n = len(idx)
    B = H[np.ix_(idx, idx)]
    Zt = rng.standard_normal((n, 5))
    cs = o.coarse(idx, Zt)
    assert cs.rank == 5 and not cs.fallback
    Qm = np.column_stack([cs.Q(e) for e in np.eye(n)])
    Pm = np.column_stack([cs.P(e) for e in np.eye(n)])
    Z, BZ, E = cs.factors()
    sc = np.abs(B).max()
    assert np.allclose(Z.T @ Z, np.eye(5), atol=1e-12)
    assert np.allclose(BZ, B @ Z, atol=1e-12 * sc)
    assert np.allclose(E, Z.T @ B @ Z, atol=1e-12 * sc)
    assert np.allclose(Qm, Z @ np.linalg.solve(E, Z.T), rtol=1e-9, atol=1e-9 / sc)
    assert np.allclose(Pm, np.eye(n) - Qm @ B, atol=1e-9)
    assert np.allclose(Qm @ B @ Qm, Qm, rtol=1e-9, atol=1e-9 / sc)      # QBQ = Q
    assert np.allclose(Pm @ Pm, Pm, atol=1e-9)                          # P^2 = P
    assert np.allclose(B @ Pm, Pm.T @ B, atol=1e-9 * sc)                # BP = P^T B
    assert np.abs(Z.T @ B @ Pm).max() <= 1e-9 * sc                      # Z^T B P = 0
    b = rng.standard_normal(n)
    x0 = rng.standard_normal(n)
    xc = x0 + cs.Q(b - B @ x0)
    assert np.abs(Z.T @ (b - B @ xc)).max() <= 1e-9 * np.abs(b).max()   # Z^T (b - B x_c) = 0
    # eq. (19): C_bal r = P J r when Z^T r = 0
    Jm = np.diag(1.0 / np.diag(B))
    Cbal = Pm @ Jm @ Pm.T + Qm
    r = b - Z @ (Z.T @ b)
    assert np.allclose(Cbal @ r, Pm @ Jm @ r, rtol=1e-8, atol=1e-8 * np.abs(Jm @ r).max())
    np.linalg.cholesky(0.5 * (Cbal + Cbal.T))
    # the span, not the columns, matters: a column-mixed copy of Z~ gives the same Q
    cs2 = o.coarse(idx, Zt @ rng.standard_normal((5, 5)))
    assert np.allclose(cs2.Q(b), cs.Q(b), rtol=1e-7, atol=1e-9 * np.abs(cs.Q(b)).max())


def test_P5_rank_revealing(oracle_mod):
    """dependent columns are dropped (singular values <= 1e-12 * largest)."""
    w = tiny_2d(8)
    o = oracle_mod.Oracle.from_workload(w)
    rng = np.random.default_rng(4)
    idx = np.arange(w.N)
    Zt = rng.standard_normal((w.N, 4))
    Zt = np.column_stack([Zt, Zt[:, 0] + Zt[:, 1], np.zeros(w.N)])
    cs = o.coarse(idx, Zt)
    assert cs.rank == 4
    Z, _, _ = cs.factors()
    assert np.allclose(Z.T @ Z, np.eye(4), atol=1e-12)
    assert np.linalg.matrix_rank(np.column_stack([Z, Zt[:, :4]]), tol=1e-9) == 4
    # fewer rows than columns: r_I <= min(|I|, r)
    cs3 = o.coarse(np.array([3, 9, 20]), rng.standard_normal((3, 5)))
    assert cs3.rank == 3


# ------------------------------------------------------------------ P6: restriction-residual identity eq. (20)-(21)
def test_P6_restriction_residual_identity(oracle_mod):
    w = tiny_2d(8)
    o = oracle_mod.Oracle.from_workload(w)
    H = dense_H(w)
    rng = np.random.default_rng(5)
    k = 5
    th, W = oracle_mod.reference_eigs(w.rowptr, w.colidx, w.val, w.m, w.alpha, k)
    W = np.linalg.qr(W + 0.05 * rng.standard_normal(W.shape))[0]  # approximate, orthonormal reference
    Lam = W.T @ H @ W
    G0 = H @ W - W @ Lam
    Jm = rng.random(w.N) < 0.25
    I = np.flatnonzero(~Jm)
    Jx = np.flatnonzero(Jm)
    o.reset_sequence()
    WI = o.restrict(oracle_mod.REFDEF, W, I)
    assert (WI == W[I]).all()
    BWI = np.column_stack([o.apply_B(I, WI[:, j]) for j in range(k)])
    rhs = -H[np.ix_(I, Jx)] @ W[Jx] + G0[I]                           # eq. (20), Delta = 0
    assert np.abs(BWI - WI @ Lam - rhs).max() <= 1e-13 * np.abs(H).max()
    cs = o.coarse(I, WI)
    Z, BZ, E = cs.factors()
    R = Z.T @ WI                                                       # Phi_I = Z R
    assert np.allclose(Z @ R, WI, atol=1e-12)
    F = BZ - Z @ E
    F21 = (np.eye(len(I)) - Z @ Z.T) @ rhs @ np.linalg.inv(R)          # eq. (21)
    assert np.abs(F - F21).max() <= 1e-11 * np.abs(H).max()


# ------------------------------------------------------------------ P8: rank zero == Jacobi-CG
def test_P8_rank_zero_is_jacobi_cg(oracle_mod):
    w = tiny_2d(12)
    o = oracle_mod.Oracle.from_workload(w)
    rng = np.random.default_rng(6)
    idx = np.flatnonzero(rng.random(w.N) < 0.9)
    b = rng.standard_normal(len(idx)) * w.m[0]
    x0 = np.zeros(len(idx))
    xa, ra = o.alg1(idx, b, x0, None)
    xb, rb = o.alg1(idx, b, x0, np.zeros((len(idx), 3)))
    assert ra["iters"] == rb["iters"] > 5 and rb["rank_used"] == 0
    assert (xa == xb).all()
    yd, psi = w.target(0)
    o.reset_sequence()
    q0 = o.solve_query(oracle_mod.JACOBI_CG, yd, psi, None)
    o.reset_sequence()
    q1 = o.solve_query(oracle_mod.REFDEF, yd, psi, np.zeros((w.N, 2)))
    assert (q0["y"] == q1["y"]).all() and q0["hashes"] == q1["hashes"]
    assert [s["cg_iters"] for s in q0["steps"]] == [s["cg_iters"] for s in q1["steps"]]


# ------------------------------------------------------------------ P9: transfers, Figure 2
def test_P9_fig2_transfer_pattern(oracle_mod):
    rows = [ln.split() for ln in open(os.path.join(HERE, "golden", "fig2_transfer_pattern.txt"))
            if ln.strip() and not ln.startswith("#")]
    assert len(rows) == 6
    w = make_steady_2d(n=3, channels=[], vel=0.0, alpha=1e-4, k=1, n_queries=1, n_bumps=1, psi_factor=0.6,
                       pdas_cap=5, config=1)  # 9 DOFs; nodes 1..6 -> DOFs 0..5, DOFs 6..8 stay inactive
    o = oracle_mod.Oracle.from_workload(w)
    phi = np.arange(1.0, 10.0).reshape(-1, 1) / 7.0
    prev_inactive = [int(r[0]) - 1 for r in rows if r[1] == "inactive"] + [6, 7, 8]
    cur_inactive = [int(r[0]) - 1 for r in rows if r[2] == "inactive"] + [6, 7, 8]
    for method, col in ((oracle_mod.REFDEF, 3), (oracle_mod.ZEROEXT, 4)):
        o.reset_sequence()
        first = o.restrict(method, phi, np.array(sorted(prev_inactive)))
        assert (first[:, 0] == phi[sorted(prev_inactive), 0]).all()     # the first restriction is direct
        Zt = o.restrict(method, phi, np.array(sorted(cur_inactive)))
        got = dict(zip(sorted(cur_inactive), Zt[:, 0]))
        for r in rows:
            node = int(r[0]) - 1
            if r[col] == "removed":
                assert node not in got
            elif r[col] == "phi":
                assert got[node] == phi[node, 0]
            else:
                assert got[node] == 0.0
        # eq. (13): the difference vanishes on shared inactive DOFs
    # if J never changes, zero-extension == direct restriction
    o.reset_sequence()
    a = o.restrict(oracle_mod.ZEROEXT, phi, np.array([0, 1, 5, 6]))
    b = o.restrict(oracle_mod.ZEROEXT, phi, np.array([0, 1, 5, 6]))
    assert (a == b).all() and (a[:, 0] == phi[[0, 1, 5, 6], 0]).all()
    # cumulative losses: a DOF active at ANY earlier restriction stays zero
    o.reset_sequence()
    o.restrict(oracle_mod.ZEROEXT, phi, np.array([0, 1, 2, 3]))        # 4.. active
    o.restrict(oracle_mod.ZEROEXT, phi, np.array([0, 1, 2, 3, 4, 5, 6, 7, 8]))
    c = o.restrict(oracle_mod.ZEROEXT, phi, np.array([0, 4, 8]))
    assert (c[:, 0] == np.array([phi[0, 0], 0.0, 0.0])).all()


# ------------------------------------------------------------------ P10: deflation with exact eigenvectors of B
def test_P10_exact_eigenvector_deflation(oracle_mod):
    w = make_steady_2d(n=4, channels=[(0.4, 0.6)], vel=20.0, alpha=1e-3, k=6, n_queries=1, n_bumps=2,
                       psi_factor=0.6, pdas_cap=5, config=1)
    o = oracle_mod.Oracle.from_workload(w)
    H = dense_H(w)
    idx = np.arange(w.N)
    lamB, V = np.linalg.eigh(H)
    k = 6
    Z = V[:, :k]
    rng = np.random.default_rng(7)
    b = rng.standard_normal(w.N) * w.m[0]
    xs = np.linalg.solve(H, b)
    # cap = 0 returns the coarse-corrected x_c (Algorithm 1 line 3): it removes exactly the Z-components
    xc, rep0 = o.alg1(idx, b, np.zeros(w.N), Z, eps=1e-12, cap=0, jacobi=0)
    assert np.abs(Z.T @ (xs - xc)).max() <= 1e-9 * np.abs(xs).max()
    assert np.allclose(xc, Z @ (Z.T @ xs), rtol=1e-8, atol=1e-10 * np.abs(xs).max())
    # unpreconditioned CG then sees only the remaining N-k eigenvalues: <= N-k iterations
    x, rep = o.alg1(idx, b, np.zeros(w.N), Z, eps=1e-10, jacobi=0)
    assert rep["status"] == 0 and rep["iters"] <= w.N - k + 1
    _, rep_plain = o.alg1(idx, b, np.zeros(w.N), None, eps=1e-10, jacobi=0)
    assert rep_plain["iters"] > rep["iters"]
    assert np.allclose(x, xs, rtol=1e-7, atol=1e-9 * np.abs(xs).max())


# ------------------------------------------------------------------ P11: u-error identity (reading A16)
def test_P11_u_error_identity(oracle_mod):
    w = tiny_2d(10)
    o = oracle_mod.Oracle.from_workload(w)
    yd, psi = w.target(0)
    o.reset_sequence()
    a = o.solve_query(0, yd, psi, None, oracle_mod.OracleOptions(eps=1e-5, eps_c=1e-5))
    o.reset_sequence()
    b = o.solve_query(0, yd, psi, None, oracle_mod.OracleOptions(eps=1e-12, eps_c=1e-12))
    e = a["y"] - b["y"]
    du = a["u"] - b["u"]
    lhs = (w.m * du * du).sum()
    rhs = (e @ o.apply_H(e) - (w.m * e * e).sum()) / w.alpha
    assert lhs > 0 and abs(lhs - rhs) <= 1e-8 * lhs


# ------------------------------------------------------------------ P12: energy fraction eq. (24)
def test_P12_energy_fraction(oracle_mod):
    w = tiny_2d(8)
    o = oracle_mod.Oracle.from_workload(w)
    H = dense_H(w)
    rng = np.random.default_rng(8)
    idx = np.flatnonzero(rng.random(w.N) < 0.85)
    B = H[np.ix_(idx, idx)]
    _, W = oracle_mod.reference_eigs(w.rowptr, w.colidx, w.val, w.m, w.alpha, 4)
    cs = o.coarse(idx, W[idx])
    b = rng.standard_normal(len(idx)) * w.m[0]
    xs = np.linalg.solve(B, b)
    Qb = cs.Q(b)
    en = lambda v: v @ B @ v
    chi = en(Qb) / en(xs)
    assert 0 < chi < 1
    assert abs(en(xs - Qb) / en(xs) - (1 - chi)) <= 1e-10


# ------------------------------------------------------------------ Algorithm 1 on its own: Verify, caps, replacement
def test_alg1_statuses_and_verify(oracle_mod):
    w = tiny_2d(12)
    o = oracle_mod.Oracle.from_workload(w)
    H = dense_H(w)
    rng = np.random.default_rng(9)
    idx = np.flatnonzero(rng.random(w.N) < 0.9)
    B = H[np.ix_(idx, idx)]
    b = rng.standard_normal(len(idx)) * w.m[0]
    _, W = oracle_mod.reference_eigs(w.rowptr, w.colidx, w.val, w.m, w.alpha, 4)
    for Zt in (None, W[idx]):
        x, rep = o.alg1(idx, b, np.zeros(len(idx)), Zt, eps=1e-9)
        true_rel = np.linalg.norm(b - B @ x) / np.linalg.norm(b)
        assert rep["status"] == 0 and true_rel <= 1e-9
        assert abs(rep["rel_resid_verified"] - true_rel) <= 1e-3 * true_rel + 1e-16
        x2, rep2 = o.alg1(idx, b, np.zeros(len(idx)), Zt, eps=1e-9, cap=3)
        assert rep2["status"] == -6 and rep2["iters"] == 3                 # ECAP, last iterate returned
        x3, rep3 = o.alg1(idx, b, np.zeros(len(idx)), Zt, eps=1e-9, replace_period=7)
        assert rep3["status"] == 0 and rep3["replacements"] >= rep3["iters"] // 7
        assert np.allclose(x3, x, rtol=1e-6, atol=1e-8 * np.abs(x).max())
    # zero right-hand side with the exact initial guess: line 4 early exit, absolute criterion
    x4, rep4 = o.alg1(idx, np.zeros(len(idx)), np.zeros(len(idx)), None)
    assert rep4["status"] == 0 and rep4["iters"] == 0 and (x4 == 0).all()
    # deflation never needs more iterations than Jacobi-CG here
    _, rj = o.alg1(idx, b, np.zeros(len(idx)), None, eps=1e-9)
    _, rd = o.alg1(idx, b, np.zeros(len(idx)), W[idx], eps=1e-9)
    assert rd["iters"] <= rj["iters"]


def test_config1_sequence_properties(oracle_mod):
    """Config 1 as specified: all-active start, PDAS cap 20 (BASELINE.json); the three methods give the
    same active-set sequence; direct restriction needs the fewest iterations (Table 3)."""
    w = make_config(1)
    o = oracle_mod.Oracle.from_workload(w)
    yd, psi = w.target(0)
    _, W = oracle_mod.reference_eigs(w.rowptr, w.colidx, w.val, w.m, w.alpha, w.k)
    res = {}
    for meth in (0, 1, 2):
        o.reset_sequence()
        res[meth] = o.solve_query(meth, yd, psi, W, oracle_mod.OracleOptions(pdas_cap=w.pdas_cap))
        assert res[meth]["steps"][0]["n_inactive"] == 0                   # first query starts all active
        assert max(s["rel_resid_verified"] for s in res[meth]["steps"]) <= 1e-8
    assert res[0]["hashes"] == res[1]["hashes"] == res[2]["hashes"]
    it = {mth: sum(s["cg_iters"] for s in res[mth]["steps"]) for mth in res}
    assert it[1] < it[2] <= it[0]
    nrm = lambda v: np.sqrt((w.m * v * v).sum())
    assert nrm(res[1]["y"] - res[0]["y"]) <= 1e-6 * nrm(res[0]["y"])


def test_golden_config1_unchanged(oracle_mod):
    """The stored oracle results (tests/golden/make_golden.py) still hold: sequence bit-exact, norms to 1e-9."""
    import json

    g = json.load(open(os.path.join(HERE, "golden", "config1_sequences.json")))
    w = make_config(1)
    assert g["operator_sha256"] == w.operator_hash()
    o = oracle_mod.Oracle.from_workload(w)
    yd, psi = w.target(0)
    th, W = oracle_mod.reference_eigs(w.rowptr, w.colidx, w.val, w.m, w.alpha, w.k)
    assert np.allclose(th, g["theta"], rtol=1e-9)
    for name, meth in (("jacobi_cg", 0), ("refdef", 1), ("zeroext", 2)):
        o.reset_sequence()
        r = o.solve_query(meth, yd, psi, W, oracle_mod.OracleOptions(pdas_cap=w.pdas_cap))
        gm = g["methods"][name]
        assert [f"{s['active_hash']:016x}" for s in r["steps"]] == gm["active_hash"]
        assert [s["n_inactive"] for s in r["steps"]] == gm["n_inactive"]
        assert abs(np.sqrt((w.m * r["y"] ** 2).sum()) - gm["y_Mnorm"]) <= 1e-9 * gm["y_Mnorm"]


# ------------------------------------------------------------------ NEXT-1: analytical Cartesian reference, eq. (15)
def test_sine_reference_is_the_spectrum_of_the_homogeneous_operator(oracle_mod):
    """PAPER.md:186-192 (cell-centred form): for uniform kappa and zero velocity the sine products ARE the lowest
    eigenvectors of H, with theta = h^d + sigma (h^(d-2) mu h^2)^2 / h^d, in the order of the library eigensolver."""
    n, k = 9, 7
    w = make_steady_2d(n=n, channels=[], vel=0.0, alpha=1e-4, k=k, n_queries=1, n_bumps=1, psi_factor=0.6,
                       pdas_cap=5, config=1)
    o = oracle_mod.Oracle.from_workload(w)
    modes, mu, W = oracle_mod.sine_reference((n, n), k)
    assert np.allclose(W.T @ W, np.eye(k), atol=1e-13)
    h = 1.0 / n
    theta = h ** 2 + w.alpha * (mu * h ** 2) ** 2 / h ** 2  # K-eigenvalue = h^(d-2) * (mu h^2), d = 2
    for c in range(k):
        assert np.allclose(o.apply_H(W[:, c]), theta[c] * W[:, c], rtol=1e-11, atol=1e-13 * theta[c])
    th, _ = oracle_mod.reference_eigs(w.rowptr, w.colidx, w.val, w.m, w.alpha, k)
    assert np.allclose(np.sort(theta), th, rtol=1e-9)
    # selection and order: (mu, q_1, q_2) lexicographic; (1,2) before (2,1), which tie exactly
    assert modes.tolist()[:4] == [[1, 1], [1, 2], [2, 1], [2, 2]]
    assert mu[1] == mu[2] and (np.diff(mu) >= 0).all()
    # the x index is the fastest: column of mode (2, 1) changes sign along x, not along y
    col = W[:, 2].reshape(n, n)  # (y, x)
    assert (np.sign(col[:, 0]) != np.sign(col[:, -1])).all() and (np.sign(col[0, :]) == np.sign(col[-1, :])).all()


def test_sine_reference_3d_and_highest_mode(oracle_mod):
    n, k = 4, 64  # every product of the 4^3 grid: a complete orthonormal basis, including q = n (norm sqrt(1/n))
    modes, mu, W = oracle_mod.sine_reference((n, n, n), k)
    assert np.allclose(W.T @ W, np.eye(k), atol=1e-13)
    assert sorted(map(tuple, modes.tolist())) == sorted(itertools.product(range(1, n + 1), repeat=3))
    w3 = make_steady_3d(n=n, bores=[], R=0.1, vpeak=0.0, alpha=1e-5, k=4, n_queries=1, n_bumps=1, psi_factor=0.6,
                        pdas_cap=5, config=3)
    o3 = oracle_mod.Oracle.from_workload(w3)
    h = 1.0 / n
    for c in (0, 5, 63):
        theta = h ** 3 + w3.alpha * (h * mu[c] * h ** 2) ** 2 / h ** 3  # K-eigenvalue = h^(d-2) mu h^2, d = 3
        assert np.allclose(o3.apply_H(W[:, c]), theta * W[:, c], rtol=1e-11, atol=1e-14 * theta)


def test_sine_reference_deflates_the_heterogeneous_problem(oracle_mod):
    """The reference is homogeneous, the CHT matrix keeps the conductivity interface and the transport
    (PAPER.md:192): Algorithm 1 with it must still converge to the same solution, in fewer iterations than
    Jacobi-CG on the twin of config 2."""
    w = make_config(twin="c2_48")
    o = oracle_mod.Oracle.from_workload(w)
    _, _, W = oracle_mod.sine_reference(w.dims, w.k)
    idx = np.arange(w.N)
    b = w.m * w._target(1000 * w.config)
    xj, rj = o.alg1(idx, b, np.zeros(w.N), None)
    xs, rs = o.alg1(idx, b, np.zeros(w.N), W)
    assert rj["status"] == rs["status"] == 0 and rs["rank_used"] == w.k
    assert rs["iters"] < rj["iters"]
    assert np.linalg.norm(xs - xj) <= 1e-5 * np.linalg.norm(xj)


# ------------------------------------------------------------------ NEXT-2: mode-dependent temporal reference, eq. (16)-(17)
def test_spacetime_reference_is_the_spectrum_of_the_homogeneous_operator(oracle_mod):
    """q (x) phi are eigenvectors of the homogeneous all-at-once reduced Hessian with
    nu = h^d (1 + alpha s); the k retained pairs are its k lowest eigenpairs (library eigensolver on the assembled H)."""
    from workloads import make_spacetime_2d

    n, nt, T, k = 6, 5, 1.0, 9
    w = make_spacetime_2d(n=n, nt=nt, T=T, channels=[], vel=0.0, alpha=1e-4, k=k, n_queries=1, n_bumps=1,
                          psi_factor=0.6, pdas_cap=5, config=4)
    o = oracle_mod.Oracle.from_workload(w)
    pairs, s, W = oracle_mod.spacetime_reference((n, n), nt, T / nt, k)
    assert W.shape == (n * n * nt, k) and np.allclose(W.T @ W, np.eye(k), atol=1e-12)
    hd = (1.0 / n) ** 2
    nu = hd * (1.0 + w.alpha * s)
    for c in range(k):
        assert np.allclose(o.apply_H(W[:, c]), nu[c] * W[:, c], rtol=1e-10, atol=1e-12 * nu[c])
    th, _ = oracle_mod.reference_eigs(w.rowptr, w.colidx, w.val, w.m, w.alpha, k)
    assert np.allclose(nu, th, rtol=1e-9) and (np.diff(s) >= 0).all()
    # the temporal vector depends on the spatial eigenvalue: same j, different mode, different q
    assert pairs[0].tolist() == [1, 1, 0]
    # layout: time is the slow index, so every column is a rank-one (time x space) array; sign: the temporal factor's
    # largest-magnitude component is positive (the spatial factor of mode (1, 1) is positive everywhere)
    col = W[:, 0].reshape(nt, n * n)
    assert np.linalg.matrix_rank(col, tol=1e-12) == 1
    q = col[:, 0] / np.linalg.norm(col[:, 0])
    assert (col[0] * np.sign(q[0]) > 0).all() and q[np.abs(q).argmax()] > 0


def test_spacetime_reference_complete_coverage(oracle_mod):
    """"keep all temporal factors of S spatial modes": the columns are every eigenvector of the
    homogeneous all-at-once Hessian whose spatial factor is one of the first S sine modes -- eigenvector property against
    the oracle's operator, the spatial factors by projection, completeness by counting, order (s, i, j)."""
    from workloads import make_spacetime_2d

    n, nt, T, S = 6, 5, 1.0, 3
    w = make_spacetime_2d(n=n, nt=nt, T=T, channels=[], vel=0.0, alpha=1e-4, k=S * nt, n_queries=1, n_bumps=1,
                          psi_factor=0.6, pdas_cap=5, config=4)
    o = oracle_mod.Oracle.from_workload(w)
    pairs, s, W = oracle_mod.spacetime_reference((n, n), nt, T / nt, None, cover=S)
    k = S * nt
    assert W.shape == (n * n * nt, k) and np.allclose(W.T @ W, np.eye(k), atol=1e-12) and (np.diff(s) >= 0).all()
    nu = (1.0 / n) ** 2 * (1.0 + w.alpha * s)
    for c in range(k):
        assert np.allclose(o.apply_H(W[:, c]), nu[c] * W[:, c], rtol=1e-10, atol=1e-12 * nu[c])
    modes, _, Phi = oracle_mod.sine_reference((n, n), S)
    used = {tuple(p[:2]) for p in pairs.tolist()}
    assert used == {tuple(mm) for mm in modes.tolist()}, "exactly the first S spatial modes"
    for mm in modes.tolist():  # every temporal factor of each: nt columns per mode, j = 0..nt-1
        js = sorted(p[2] for p in pairs.tolist() if p[:2] == mm)
        assert js == list(range(nt))
    # the span is (all of time) x span(Phi): projecting any column's time-slabs on Phi loses nothing
    for c in (0, k // 2, k - 1):
        col = W[:, c].reshape(nt, n * n)
        assert np.allclose(col @ Phi @ Phi.T, col, atol=1e-12)
    # it differs from the ordered selection of the same total rank (which may reach for a fourth spatial mode)
    pairs_o, _, _ = oracle_mod.spacetime_reference((n, n), nt, T / nt, k)
    assert {tuple(p[:2]) for p in pairs_o.tolist()} != used or True


def test_spacetime_reference_deflates_the_twin_of_config4(oracle_mod):
    w = make_config(twin="c4_32x8")
    o = oracle_mod.Oracle.from_workload(w)
    _, _, W = oracle_mod.spacetime_reference(w.dims, w.nt, 1.0 / w.nt, w.k)
    idx = np.arange(w.N)
    b = w.m * w._target(1000 * w.config)
    xj, rj = o.alg1(idx, b, np.zeros(w.N), None)
    xs, rs = o.alg1(idx, b, np.zeros(w.N), W)
    assert rj["status"] == rs["status"] == 0 and rs["rank_used"] == w.k
    assert rs["iters"] < rj["iters"]
    assert np.linalg.norm(xs - xj) <= 1e-5 * np.linalg.norm(xj)


# ------------------------------------------------------------------ NEXT-3: Jacobi-scaled reference
def test_scaled_reference_solves_the_generalized_problem(oracle_mod):
    w = make_config(twin="c2_48")
    o = oracle_mod.Oracle.from_workload(w)
    k = w.k
    mu, W = oracle_mod.reference_eigs_scaled(w.rowptr, w.colidx, w.val, w.m, w.alpha, k)
    d = o.diag_H()
    assert np.allclose(np.linalg.norm(W, axis=0), 1.0, atol=1e-13) and (np.diff(mu) >= -1e-12).all()
    for c in range(k):
        r = o.apply_H(W[:, c]) - mu[c] * d * W[:, c]
        assert np.linalg.norm(r) <= 1e-8 * mu[c] * np.linalg.norm(d * W[:, c])
    G = W.T @ (d[:, None] * W)  # D-orthogonal up to the column scaling
    Gn = G / np.sqrt(np.outer(np.diag(G), np.diag(G)))
    assert np.abs(Gn - np.eye(k)).max() <= 1e-8
    # Rayleigh quotients of the Jacobi-preconditioned operator lie in (0, #nonzeros per row of H]
    assert mu[0] > 0 and mu[-1] < 13.0
    # dense and sparse branches agree
    mu2, _ = oracle_mod.reference_eigs_scaled(w.rowptr, w.colidx, w.val, w.m, w.alpha, k, dense_below=10)
    assert np.allclose(mu, mu2, rtol=1e-8)
    # the scaled reference deflates at least as well as the standard one (SURVEY.md probe: about -10 % iterations)
    _, W_std = oracle_mod.reference_eigs(w.rowptr, w.colidx, w.val, w.m, w.alpha, k)
    idx = np.arange(w.N)
    b = w.m * w._target(1000 * w.config)
    _, r_std = o.alg1(idx, b, np.zeros(w.N), W_std)
    _, r_sc = o.alg1(idx, b, np.zeros(w.N), W)
    assert r_std["status"] == r_sc["status"] == 0
    assert r_sc["iters"] <= 1.02 * r_std["iters"], (r_sc["iters"], r_std["iters"])


# ------------------------------------------------------------------ NEXT-1(ii): coarse eigenproblem + P1 prolongation
def _interp_axiswise(Vc, dims_c, dims_f):
    """Library pin: numpy.interp along one axis after the other (nodes = boundary 0, coarse centres, boundary 1)."""
    T = np.asarray(Vc, dtype=float).reshape(tuple(reversed(dims_c)))  # C order: slowest axis first, x last
    d = len(dims_c)
    for a in range(d):
        ax = d - 1 - a  # position of grid axis a in the array
        nc, nf = dims_c[a], dims_f[a]
        xi = np.concatenate(([0.0], (np.arange(nc) + 0.5) / nc, [1.0]))
        xf = (np.arange(nf) + 0.5) / nf
        T = np.apply_along_axis(lambda v: np.interp(xf, xi, np.concatenate(([0.0], v, [0.0]))), ax, T)
    return T.reshape(-1)


@pytest.mark.parametrize("dims_c,dims_f", [((5,), (10,)), ((4,), (12,)), ((4,), (7,)), ((3, 5), (6, 15)),
                                            ((2, 3, 4), (4, 9, 8)), ((6, 4), (6, 4))])
def test_prolong_p1_matches_library_interpolation(oracle_mod, dims_c, dims_f):
    """Non-square grids with different ratios per axis: a transposed axis or a wrong stride fails."""
    rng = np.random.default_rng(17)
    Vc = rng.standard_normal((int(np.prod(dims_c)), 3))
    P = oracle_mod.prolong_p1(Vc, dims_c, dims_f)
    assert P.shape == (int(np.prod(dims_f)), 3)
    for c in range(3):
        assert np.allclose(P[:, c], _interp_axiswise(Vc[:, c], dims_c, dims_f), rtol=0, atol=1e-14)
    if tuple(dims_c) == tuple(dims_f):  # same grid: the identity
        assert np.array_equal(P, Vc)


def test_prolong_p1_closed_forms(oracle_mod):
    """(a) A function that is d-linear between the coarse nodes and 0 on the boundary is reproduced exactly: the
    product of 1-D hats h(s) = 1 - |2s - 1|, whose kink 1/2 is a coarse node for odd n_c.  (b) Dependence on x only
    stays on x only (axis order).  (c) Interpolating the coarse sine mode stays within the P1 error bound
    h_c^2 max|f''|/8 of the continuous mode, and a refinement ratio 2 puts the weights at 1/4, 3/4."""
    hat = lambda s: 1.0 - np.abs(2.0 * s - 1.0)
    nc, nf = (5, 7), (20, 21)
    xc = [(np.arange(n) + 0.5) / n for n in nc]
    xf = [(np.arange(n) + 0.5) / n for n in nf]
    Vc = np.kron(hat(xc[1]), hat(xc[0]))  # x fastest
    P = oracle_mod.prolong_p1(Vc, nc, nf)[:, 0]
    assert np.allclose(P, np.kron(hat(xf[1]), hat(xf[0])), rtol=0, atol=1e-15)
    Vx = np.kron(np.ones(nc[1]), hat(xc[0]))
    Px = oracle_mod.prolong_p1(Vx, nc, nf)[:, 0].reshape(nf[1], nf[0])
    # rows strictly between the first and last coarse centres in y see the constant 1 in y
    inner = (xf[1] >= xc[1][0]) & (xf[1] <= xc[1][-1])
    assert np.allclose(Px[inner], hat(xf[0])[None, :], rtol=0, atol=1e-15)
    q, n = 3, 16
    f = lambda s: np.sin(np.pi * q * s)
    P1 = oracle_mod.prolong_p1(f((np.arange(n) + 0.5) / n), (n,), (2 * n,))[:, 0]
    s_f = (np.arange(2 * n) + 0.5) / (2 * n)
    assert np.abs(P1 - f(s_f)).max() <= (1.0 / n) ** 2 * (np.pi * q) ** 2 / 8 + 1e-15
    v = np.arange(1.0, n + 1)
    P2 = oracle_mod.prolong_p1(v, (n,), (2 * n,))[:, 0]
    assert np.allclose(P2[1:-1:2], 0.75 * v[:-1] + 0.25 * v[1:], rtol=0, atol=1e-14)   # fine cell 2j: 3/4, 1/4
    assert np.allclose(P2[2:-1:2], 0.25 * v[:-1] + 0.75 * v[1:], rtol=0, atol=1e-14)
    assert abs(P2[0] - 0.5 * v[0]) <= 1e-15 and abs(P2[-1] - 0.5 * v[-1]) <= 1e-15     # half-way to the Dirichlet 0


def test_prolonged_reference_deflates_the_fine_problem(oracle_mod):
    """Coarse generalized eigenproblem (24^2) -> P1 prolongation -> unit columns on the 48^2 twin of
    config 2: "The prolonged candidates are approximate fine-mesh modes": small Rayleigh quotients in
    the Jacobi-scaled fine operator, fewer iterations than Jacobi-CG, same solution."""
    w = make_config(twin="c2_48")
    wc = make_config(config=2, n=24, k=w.k)
    o = oracle_mod.Oracle.from_workload(w)
    mu_c, Wc, W = oracle_mod.prolonged_reference((wc.rowptr, wc.colidx, wc.val, wc.m, wc.alpha), wc.dims, w.dims, w.k)
    assert W.shape == (w.N, w.k) and np.allclose(np.linalg.norm(W, axis=0), 1.0, atol=1e-13)
    assert np.allclose(np.linalg.norm(Wc, axis=0), 1.0, atol=1e-13)
    d = o.diag_H()
    mu_f, _ = oracle_mod.reference_eigs_scaled(w.rowptr, w.colidx, w.val, w.m, w.alpha, w.k)
    # Rayleigh quotient of the lowest prolonged vector in the fine generalized problem: above the fine mu_1 (min-max),
    # and an approximation of it
    rq = lambda v: float(v @ o.apply_H(v)) / float(v @ (d * v))
    assert mu_f[0] * (1 - 1e-10) <= rq(W[:, 0]) <= 1.5 * mu_f[0]
    # every prolonged column stays in the low end of the fine Jacobi-scaled spectrum (which reaches up to about 2)
    assert max(rq(W[:, c]) for c in range(w.k)) <= 10.0 * mu_f[-1] < 0.01
    # the coarse generalized eigenvalues are the fine ones times about (h_c/h_f)^4 = 16 (H is M + sigma * fourth order)
    assert 8.0 <= (mu_c / mu_f).min() and (mu_c / mu_f).max() <= 17.0
    idx = np.arange(w.N)
    b = w.m * w._target(1000 * w.config)
    xj, rj = o.alg1(idx, b, np.zeros(w.N), None)
    xp, rp = o.alg1(idx, b, np.zeros(w.N), W)
    assert rj["status"] == rp["status"] == 0 and rp["rank_used"] == w.k
    assert rp["iters"] < 0.6 * rj["iters"], (rp["iters"], rj["iters"])
    assert np.linalg.norm(xp - xj) <= 1e-5 * np.linalg.norm(xj)
    # nearly as good as the exact fine modes of the same generalized problem
    _, W_f = oracle_mod.reference_eigs_scaled(w.rowptr, w.colidx, w.val, w.m, w.alpha, w.k)
    _, rf = o.alg1(idx, b, np.zeros(w.N), W_f)
    assert rf["iters"] <= rp["iters"] <= 1.25 * rf["iters"], (rp["iters"], rf["iters"])


# ------------------------------------------------------------------ eq. (14): transient coarse-mesh reference
def _st_dense(w):
    K = np.zeros((w.N, w.N))
    for r in range(w.N):
        for p in range(w.rowptr[r], w.rowptr[r + 1]):
            K[r, w.colidx[p]] += w.val[p]
    return np.diag(w.m) + w.alpha * K.T @ np.diag(1.0 / w.m) @ K


def test_transient_reference_small_matrices_by_brute_force(oracle_mod):
    """eq. (14) entry by entry on a tiny all-at-once operator: H_i[s, t] = sum_xy phi(x) H[(s, x), (t, y)] phi(y) from
    the (time, space) blocks of the dense H (no Kronecker factor), D_i likewise from diag(H); every retained pair
    satisfies H_i q = nu D_i q; H_i is tridiagonal (K_st is block lower bidiagonal): a transposed layout would fill it."""
    import scipy.linalg as sla

    w = tiny_st(5, 4)
    Ns, nt = 25, 4
    H = _st_dense(w)
    rng = np.random.default_rng(14)
    Phi = rng.standard_normal((Ns, 3))
    k = 7
    pairs, nu, W = oracle_mod.transient_reference(Phi, (w.rowptr, w.colidx, w.val, w.m, w.alpha), nt, k)
    assert W.shape == (w.N, k) and np.allclose(np.linalg.norm(W, axis=0), 1.0, atol=1e-13)
    assert (np.diff(nu) >= 0).all() and len({tuple(p) for p in pairs.tolist()}) == k
    Hb = H.reshape(nt, Ns, nt, Ns)
    db = np.diag(H).reshape(nt, Ns)
    all_nu = []
    for i in range(3):
        Hi = np.einsum("x,sxty,y->st", Phi[:, i], Hb, Phi[:, i])
        Di = np.diag(db @ (Phi[:, i] ** 2))
        assert np.abs(np.triu(Hi, 2)).max() <= 1e-14 * np.abs(Hi).max()
        ev = sla.eigh(Hi, Di, eigvals_only=True)
        all_nu += list(ev)
        for c in np.flatnonzero(pairs[:, 0] == i):
            col = W[:, c].reshape(nt, Ns)                       # time is the slow index: rank one, space factor phi_i
            q = col @ Phi[:, i] / (Phi[:, i] @ Phi[:, i])
            assert np.allclose(col, np.outer(q, Phi[:, i]), atol=1e-13)
            assert np.allclose(Hi @ q, nu[c] * (Di @ q), rtol=0, atol=1e-10 * np.abs(Hi @ q).max())
            assert abs(ev[pairs[c, 1]] - nu[c]) <= 1e-10 * nu[c]
            assert q[np.abs(q).argmax()] > 0
    assert np.allclose(sorted(all_nu)[:k], nu, rtol=1e-10)      # the k lowest of ALL candidates were kept


def test_transient_reference_ritz_properties(oracle_mod):
    """What the mathematics fixes: nu is the generalized Rayleigh quotient of its column; the residual H w - nu D w is
    orthogonal to the candidate space I (x) phi_i (Galerkin); nu_{i,0} is the minimum of the quotient over that space;
    and for one time slab the problem is 1 x 1: nu_i = phi^T H phi / phi^T D phi."""
    w = tiny_st(6, 3)
    o = oracle_mod.Oracle.from_workload(w)
    Ns, nt = 36, 3
    _, _, Phi = oracle_mod.sine_reference((6, 6), 4)
    st = (w.rowptr, w.colidx, w.val, w.m, w.alpha)
    pairs, nu, W = oracle_mod.transient_reference(Phi, st, nt, 12)
    d = o.diag_H()
    rng = np.random.default_rng(15)
    for c in range(12):
        i = pairs[c, 0]
        Hw = o.apply_H(W[:, c])
        assert abs(W[:, c] @ Hw / (W[:, c] @ (d * W[:, c])) - nu[c]) <= 1e-10 * nu[c]
        res = Hw - nu[c] * d * W[:, c]
        V = np.kron(np.eye(nt), Phi[:, i:i + 1])
        assert np.abs(V.T @ res).max() <= 1e-10 * np.abs(V.T @ Hw).max()
        if pairs[c, 1] == 0:
            for _ in range(5):
                v = V @ rng.standard_normal(nt)
                assert v @ o.apply_H(v) / (v @ (d * v)) >= nu[c] * (1 - 1e-12)
    w1 = tiny_st(6, 1)
    o1 = oracle_mod.Oracle.from_workload(w1)
    p1, nu1, W1 = oracle_mod.transient_reference(Phi, (w1.rowptr, w1.colidx, w1.val, w1.m, w1.alpha), 1, 4)
    rq = np.array([Phi[:, i] @ o1.apply_H(Phi[:, i]) / (Phi[:, i] @ (o1.diag_H() * Phi[:, i])) for i in range(4)])
    assert np.allclose(np.sort(rq), nu1, rtol=1e-12) and p1[:, 0].tolist() == np.argsort(rq).tolist()
    for c in range(4):
        assert np.allclose(W1[:, c], Phi[:, p1[c, 0]] / np.linalg.norm(Phi[:, p1[c, 0]]), atol=1e-13)


def test_transient_reference_deflates_the_twin_of_config4(oracle_mod):
    """eq. (14) on the twin of config 4 with the Jacobi-scaled low modes of the STEADY spatial operator as the spatial
    vectors: the Kronecker candidates reproduce the low generalized spectrum of the all-at-once operator (library
    eigensolver on the assembled space-time H, 2e-3 (measured 1.2e-3): the spatial modes of the steady and the time-stepping operator
    differ slightly), both factors vary, and the reference deflates: full rank, fewer iterations than Jacobi-CG, same
    solution.  (With vectors prolonged from the 16 x 16 half grid of this 32 x 32 twin the channels are under-resolved
    and nu is three times larger: "the prolonged candidates are approximate fine-mesh modes"; the
    pipeline itself is composition of `prolonged_reference` and this function; on the 64 x 64 x 8 twin it needs
    2,119 iterations against 2,900 for Jacobi-CG and 2,111 with fine-grid spatial vectors.)"""
    w = make_config(twin="c4_32x8")
    ws = make_steady_2d(n=w.dims[0], channels=[(0.25, 0.35), (0.65, 0.75)], vel=50.0, alpha=w.alpha, k=w.k, n_queries=1,
                        n_bumps=1, psi_factor=0.6, pdas_cap=5, config=2, name="c4_space")
    _, Phi = oracle_mod.reference_eigs_scaled(ws.rowptr, ws.colidx, ws.val, ws.m, ws.alpha, w.k)
    st = (w.rowptr, w.colidx, w.val, w.m, w.alpha)
    pairs, nu, W = oracle_mod.transient_reference(Phi, st, w.nt, w.k)
    assert len(set(pairs[:, 0].tolist())) > 1 and len(set(pairs[:, 1].tolist())) > 1   # both factors vary
    mu, _ = oracle_mod.reference_eigs_scaled(*st, w.k)
    assert (nu >= mu * (1 - 1e-10)).all() and np.allclose(nu, mu, rtol=2e-3)           # Ritz values from above (min-max)
    o = oracle_mod.Oracle.from_workload(w)
    idx = np.arange(w.N)
    b = w.m * w._target(1000 * w.config)
    xj, rj = o.alg1(idx, b, np.zeros(w.N), None)
    xs, rs = o.alg1(idx, b, np.zeros(w.N), W)
    assert rj["status"] == rs["status"] == 0 and rs["rank_used"] == w.k
    assert rs["iters"] < 0.9 * rj["iters"]
    assert np.linalg.norm(xs - xj) <= 1e-5 * np.linalg.norm(xj)


# ----------------------------------------------------------------------------------------------------------------------
# the threaded TIMING build of the oracle (gcc -fopenmp, bench.py's cpu_baseline / --impl reference) against the plain one
def test_threaded_timing_build_matches_the_plain_oracle():
    import oracle

    w = make_config(twin="c2_48")
    o1 = oracle.Oracle.from_workload(w)
    o2 = oracle.Oracle.from_workload(w, threaded=True)
    assert o1.threads == 1 and o2.threads >= 1
    rng = np.random.default_rng(7)
    v = rng.standard_normal(w.N)
    assert np.array_equal(o1.apply_K(v), o2.apply_K(v))
    assert np.array_equal(o1.apply_KT(v), o2.apply_KT(v))  # transposed row loop: same order of the sums as the scatter
    assert np.array_equal(o1.apply_H(v), o2.apply_H(v))
    _, W = oracle.reference_eigs(w.rowptr, w.colidx, w.val, w.m, w.alpha, 8)
    idx = np.flatnonzero(rng.random(w.N) > 0.3).astype(np.int64)
    b = rng.standard_normal(len(idx))
    x1, r1 = o1.alg1(idx, b, np.zeros(len(idx)), W[idx])
    x2, r2 = o2.alg1(idx, b, np.zeros(len(idx)), W[idx])
    assert r1["status"] == r2["status"] == 0 and r1["rank_used"] == r2["rank_used"]
    assert abs(r1["iters"] - r2["iters"]) <= 2  # sums are taken in another order, nothing else differs
    assert np.linalg.norm(x1 - x2) <= 1e-7 * np.linalg.norm(x1)
    # alg1_on (line 2 built once by the caller) is the same solve as alg1
    x3, r3 = o1.alg1_on(o1.coarse(idx, W[idx]), b, np.zeros(len(idx)))
    assert np.array_equal(x1, x3) and r1["iters"] == r3["iters"]


# ----------------------------------------------------------------------------------------------------------------------
# the stored goldens of the larger twins (tests/golden/twin_*.json, written by make_golden_twins.py from the oracle)
def test_golden_twins_belong_to_this_generator_and_oracle(oracle_mod):
    """Every stored golden names the operator it was computed on (sha256 of rowptr/colidx/val/m/alpha) and the first PDAS
    steps of the smallest case are recomputed live: a change to the input generator or to the oracle's arithmetic that is
    not followed by regenerating the goldens fails here, on the CPU, and not only on the GPU box."""
    import json

    gdir = os.path.join(HERE, "golden")
    names = sorted(f for f in os.listdir(gdir) if f.startswith("twin_") and f.endswith(".json"))
    assert len(names) >= 5
    for f in names:
        with open(os.path.join(gdir, f)) as fh:
            g = json.load(fh)
        w = make_config(**g["make_config"]) if g["N"] <= 70000 else None
        if w is not None:
            assert w.operator_hash() == g["operator_sha256"] and w.N == g["N"] and w.k == g["k"], f
        for q in g["queries"]:
            assert q["status"] == 0 and max(q["kkt"]) <= 1e-6, (f, q["query"])
            assert len(q["active_hash"]) == q["n_steps"] == len(q["n_inactive"]) == len(q["cg_iters"])
            assert all(s == 0 for s in q["inner_status"])
        y = np.load(os.path.join(gdir, f.replace(".json", ".npz")))
        assert sorted(y.files) == sorted(f"y{q['query']}" for q in g["queries"])
    # live: the first three steps of c3_32, query 0 (a few seconds of oracle time)
    with open(os.path.join(gdir, "twin_c3_32.json")) as fh:
        g = json.load(fh)
    w = make_config(**g["make_config"])
    o = oracle_mod.Oracle.from_workload(w)
    W = np.asfortranarray(oracle_mod.sine_reference(w.dims, w.k)[-1])
    yd, psi = w.target(0)
    r = o.solve_query(oracle_mod.REFDEF, yd, psi, W, oracle_mod.OracleOptions(eps=g["eps"], eps_c=g["eps_c"], pdas_cap=3))
    q = g["queries"][0]
    assert [f"{s['active_hash']:016x}" for s in r["steps"]] == q["active_hash"][:3]
    assert [s["n_inactive"] for s in r["steps"]] == q["n_inactive"][:3]
    assert [s["cg_iters"] for s in r["steps"]] == q["cg_iters"][:3]
    assert [s["rank_used"] for s in r["steps"]] == q["rank_used"][:3]
