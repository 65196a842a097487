"""GPU side of the pins added in round 2: the kernels that share a formula with the oracle are compared on inputs where a
shared misreading could not hide (the oracle itself is pinned to numpy on the same inputs, tests/test_oracle_pins_kkt_init.py).

  k_kkt (eq. (25)) on a perturbed (y, lambda) with ||l||_inf > 1 and psi = inf entries, against numpy
  the cond(E) > 1e10 rank-zero fallback: triggered on the device, execution bit-identical to Jacobi-CG
  the sequence state: single-step entry points between two queries do not disturb what the next inherits
"""
import numpy as np
import pytest
import scipy.sparse as sp

pytestmark = pytest.mark.gpu

import oracle  # noqa: E402
import paper_2606_17971_b200 as rd  # noqa: E402
from test_oracle_pins_kkt_init import dense_H, fallback_problem, small_problem  # noqa: E402
from workloads import make_config  # noqa: E402


@pytest.mark.parametrize("mass_scale", [1.0, 4.0e3])
@pytest.mark.parametrize("host", [True, False])
def test_kkt_kernel_on_a_perturbed_pair(mass_scale, host):
    import torch

    w, K, m = small_problem(7, mass_scale=mass_scale)
    N, sigma = w.N, 1e-4
    H = dense_H(K, m, sigma)
    g = rd.RefDef(w.rowptr, w.colidx, w.val, m, sigma)
    rng = np.random.default_rng(11)
    yd = rng.uniform(0.2, 1.0, N)
    ell = m * yd
    psi = np.full(N, 0.45)
    psi[rng.choice(N, 6, replace=False)] = np.inf
    y = 0.45 + 0.01 * rng.standard_normal(N)
    lam = 0.3 * ell.max() * rng.standard_normal(N)
    gr = H @ y - ell
    s = max(1.0, np.abs(ell).max())
    fin = np.isfinite(psi)
    exp = np.array([np.abs(gr + lam).max() / s, np.maximum(y[fin] - psi[fin], 0.0).max(), np.maximum(-lam, 0.0).max() / s,
                    np.abs(lam[fin] * (psi[fin] - y[fin])).max() / s, np.abs(y - np.minimum(psi, y - gr)).max() / s])
    conv = (lambda a: a) if host else (lambda a: torch.from_numpy(a).cuda())
    got = g.kkt(conv(yd), conv(psi), conv(y), conv(lam))
    assert np.allclose(got, exp, rtol=1e-11, atol=0.0), (got, exp)
    o = oracle.Oracle(w.rowptr, w.colidx, w.val, m, sigma)
    assert np.allclose(got, o.kkt(yd, psi, y, lam), rtol=1e-11, atol=0.0)
    g.close()


@pytest.mark.parametrize("span,expect_fallback", [(12, True), (8, False)])
def test_cond_E_fallback_on_the_device(span, expect_fallback):
    N, K, m, sigma = fallback_problem(span)
    H = dense_H(K, m, sigma)
    g = rd.RefDef(K.indptr.astype(np.int64), K.indices.astype(np.int32), K.data, m, sigma, rd.Options(eps=1e-10, eps_c=1e-10, cg_cap=500))
    W = np.zeros((N, 2))
    W[0, 0] = 1.0
    W[N - 1, 1] = 1.0
    g.set_reference(W)
    act = np.zeros(N, dtype=np.uint8)
    cond = np.linalg.cond(W.T @ H @ W)
    cs = g.coarse_setup(rd.REFDEF, act)
    assert cs["fallback"] == (1 if expect_fallback else 0) and cs["rank"] == (0 if expect_fallback else 2)
    assert np.isclose(cs["cond_E"], cond, rtol=1e-6)
    rng = np.random.default_rng(5)
    b = H @ rng.standard_normal(N)
    x_d, r_d = g.solve_inactive(rd.REFDEF, act, b, np.zeros(N))
    x_j, r_j = g.solve_inactive(rd.JACOBI_CG, act, b, np.zeros(N))
    assert r_d["coarse_fallback"] == (1 if expect_fallback else 0)
    # the oracle takes the same decision on the same system
    o = oracle.Oracle(K.indptr.astype(np.int64), K.indices.astype(np.int32), K.data, m, sigma)
    _, r_o = o.alg1(np.arange(N, dtype=np.int64), b, np.zeros(N), W, eps=1e-10, cap=500)
    assert r_o["coarse_fallback"] == r_d["coarse_fallback"] and r_o["rank_used"] == r_d["rank_used"]
    if expect_fallback:
        assert r_d["rank_used"] == 0 and r_d["iters"] == r_j["iters"]
        assert np.array_equal(x_d, x_j), "fallback execution must be Jacobi-CG itself (PAPER.md:265)"
    else:
        assert r_d["rank_used"] == 2 and not np.array_equal(x_d, x_j)
    assert r_d["status"] == 0 and np.linalg.norm(H @ x_d - b) <= 1e-9 * np.linalg.norm(b)
    g.close()


def test_single_steps_do_not_disturb_the_sequence_state():
    """query 1; then rd_coarse_setup / rd_energy_fraction / rd_solve_inactive with ANOTHER active set; then query 2 must
    start from the set query 1 ended with and reproduce an undisturbed sequence bit for bit."""
    w = make_config(twin="c2_48")
    yd1, psi1 = w.target(0)
    yd2, psi2 = w.target(1)
    psi1 = np.full(w.N, 0.3 * yd1.max())
    psi2 = np.full(w.N, 0.3 * yd2.max())

    def run(disturb):
        g = rd.RefDef.from_workload(w, rd.Options(pdas_cap=w.pdas_cap))
        g.build_reference_sine(w.k, w.dims)
        r1 = g.solve_query(rd.JACOBI_CG, yd1, psi1)
        if disturb:
            rng = np.random.default_rng(0)
            other = (rng.random(w.N) < 0.5).astype(np.uint8)
            g.coarse_setup(rd.REFDEF, other)
            g.energy_fraction(rd.REFDEF, other, rng.standard_normal(w.N), rng.standard_normal(w.N))
            g.solve_inactive(rd.JACOBI_CG, other, rng.standard_normal(w.N), np.zeros(w.N))
        r2 = g.solve_query(rd.JACOBI_CG, yd2, psi2)
        g.close()
        return r1, r2

    (a1, a2), (b1, b2) = run(False), run(True)
    assert a1["status"] == 0 and a2["status"] == 0
    last1 = a1["J_bits"][a1["n_steps"] - 1]
    assert np.unpackbits(last1).any(), "query 1 must end with a non-empty active set for this test to bite"
    assert np.array_equal(a2["J_bits"][0], last1)
    assert np.array_equal(b2["J_bits"], a2["J_bits"]) and np.array_equal(b2["y"], a2["y"])
    assert [s["cg_iters"] for s in b2["steps"]] == [s["cg_iters"] for s in a2["steps"]]


def test_query_report_carries_inner_statuses():
    w = make_config(1)
    g = rd.RefDef.from_workload(w, rd.Options(pdas_cap=w.pdas_cap, cg_cap=5))  # every inner solve ends at the cap
    yd, psi = w.target(0)
    r = g.solve_query(rd.JACOBI_CG, yd, psi)
    assert r["worst_inner_status"] == -6 and r["n_inner_failed"] >= 1 and r["n_fallbacks"] == 0
    assert r["n_inner_failed"] == sum(1 for s in r["steps"] if s["status"] != 0)
    g.set_options(rd.Options(pdas_cap=w.pdas_cap))
    g.reset_sequence()
    r = g.solve_query(rd.JACOBI_CG, yd, psi)
    assert r["status"] == 0 and r["worst_inner_status"] == 0 and r["n_inner_failed"] == 0
    g.close()
