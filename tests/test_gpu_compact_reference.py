"""NEXT-2 of SURVEY.md 8(f): the space-time references are stored compactly ("the reference stores
N_s r_s + N_t r floating-point values and r spatial-column indices.  Restriction evaluates a selected product at its
inactive space-time entries") and the complete-coverage selection ("all temporal factors of S spatial modes") exists.

Checked: storage counts; the dense block the library forms on request equals the oracle's W; the restricted basis
formed from the factors equals the restriction of the dense block (Gram matrices and a whole query, bit for bit, against a
context that holds the same reference densely); complete coverage against the oracle; the transient (eq. (14)) variant."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

import oracle  # noqa: E402
import paper_2606_17971_b200 as rd  # noqa: E402
from workloads import make_config  # noqa: E402


@pytest.fixture(scope="module")
def twin():
    return make_config(twin="c4_32x8")  # 32 x 32 x 8 slabs, k = 16


def subspace_gap(A, B):
    Qa, _ = np.linalg.qr(A)
    Qb, _ = np.linalg.qr(B)
    s = np.linalg.svd(Qa.T @ Qb, compute_uv=False)
    return float(np.sqrt(max(0.0, 1.0 - s.min() ** 2)))


def test_compact_storage_counts_and_dense_block(twin):
    w = twin
    Ns = w.dims[0] * w.dims[1]
    g = rd.RefDef.from_workload(w, rd.Options(pdas_cap=w.pdas_cap))
    assert g.reference_storage()[0] == -1
    s, pairs = g.build_reference_spacetime(w.k, w.dims, w.nt, 1.0 / w.nt)
    kind, nv, ni = g.reference_storage()
    rs_used = len({tuple(p[:2]) for p in pairs.tolist()})
    assert kind == 1 and nv == Ns * rs_used + w.nt * w.k and ni == w.k
    assert nv < 0.2 * w.N * w.k, "the compact form is far smaller than the dense block"
    po, so, Wo = oracle.spacetime_reference(w.dims, w.nt, 1.0 / w.nt, w.k)
    assert np.array_equal(pairs, po) and np.allclose(s, so, rtol=1e-12)
    W = g.get_reference()
    assert np.abs(W - Wo).max() <= 1e-11
    # a dense reference reports itself as such
    g.set_reference(Wo)
    assert g.reference_storage() == (0, w.N * w.k, 0)
    g.close()


@pytest.mark.parametrize("method", [1, 2])
def test_restriction_from_factors_equals_restriction_of_the_dense_block(twin, method):
    w = twin
    gc = rd.RefDef.from_workload(w, rd.Options(pdas_cap=w.pdas_cap))
    gd = rd.RefDef.from_workload(w, rd.Options(pdas_cap=w.pdas_cap))
    gc.build_reference_spacetime(w.k, w.dims, w.nt, 1.0 / w.nt)
    gd.set_reference(gc.get_reference())  # the same numbers, held densely
    rng = np.random.default_rng(8)
    act = (rng.random(w.N) < 0.4).astype(np.uint8)
    a, b = gc.coarse_setup(method, act), gd.coarse_setup(method, act)
    assert np.array_equal(a["G"], b["G"]) and np.array_equal(a["EW"], b["EW"]) and a["rank"] == b["rank"]
    yd, psi = w.target(0)
    psi = np.full(w.N, 0.4 * yd.max())
    rc, rdn = gc.solve_query(method, yd, psi), gd.solve_query(method, yd, psi)
    assert rc["status"] == rdn["status"] == 0
    assert np.array_equal(rc["J_bits"], rdn["J_bits"]) and np.array_equal(rc["y"], rdn["y"])
    assert [s["cg_iters"] for s in rc["steps"]] == [s["cg_iters"] for s in rdn["steps"]]
    gc.close()
    gd.close()


def test_complete_temporal_coverage_matches_oracle(twin):
    w = twin
    S = 2  # 2 spatial modes x 8 slabs = rank 16
    g = rd.RefDef.from_workload(w, rd.Options(pdas_cap=w.pdas_cap))
    s, pairs = g.build_reference_spacetime_cover(S, w.dims, w.nt, 1.0 / w.nt)
    po, so, Wo = oracle.spacetime_reference(w.dims, w.nt, 1.0 / w.nt, None, cover=S)
    assert np.array_equal(pairs, po) and np.allclose(s, so, rtol=1e-12)
    W = g.get_reference()
    assert W.shape == (w.N, S * w.nt) and np.abs(W - Wo).max() <= 1e-11
    kind, nv, ni = g.reference_storage()
    assert kind == 1 and nv == w.dims[0] * w.dims[1] * S + w.nt * S * w.nt and ni == S * w.nt
    # every slab of each retained spatial mode is covered: for any time level t, e_t (x) phi_i lies in the span
    _, _, Phi = oracle.sine_reference(w.dims, S)
    probe = np.kron(np.eye(w.nt)[:, 3], Phi[:, 1])
    assert np.linalg.norm(probe - W @ (W.T @ probe)) <= 1e-10
    # query parity against the oracle with the same reference
    yd, psi = w.target(0)
    o = oracle.Oracle.from_workload(w)
    r = g.solve_query(rd.REFDEF, yd, psi)
    ro = o.solve_query(oracle.REFDEF, yd, psi, Wo, oracle.OracleOptions(pdas_cap=w.pdas_cap))
    assert r["status"] == ro["status"] == 0 and np.array_equal(r["J_bits"], ro["J_bits"])
    nrm = lambda v: np.sqrt((w.m * v * v).sum())
    assert nrm(r["y"] - ro["y"]) <= 1e-6 * nrm(ro["y"])
    with pytest.raises(rd.RefDefError):
        g.build_reference_spacetime_cover(9, w.dims, w.nt, 1.0 / w.nt)  # 9 x 8 > 64
    g.close()


def test_transient_reference_is_stored_compactly(twin):
    w = twin
    Ns = w.dims[0] * w.dims[1]
    _, _, Phi = oracle.sine_reference(w.dims, 6)
    Phi = np.asfortranarray(Phi * np.linspace(1.0, 2.0, 6))  # non-unit spatial vectors: the normalisation must bite
    g = rd.RefDef.from_workload(w, rd.Options(pdas_cap=w.pdas_cap))
    pairs, nu = g.build_reference_transient(w.k, Phi, w.nt)
    kind, nv, ni = g.reference_storage()
    rs_used = len(set(pairs[:, 0].tolist()))
    assert kind == 1 and nv == Ns * rs_used + w.nt * w.k and ni == w.k
    po, nuo, Wo = oracle.transient_reference(Phi, (w.rowptr, w.colidx, w.val, w.m, w.alpha), w.nt, w.k)
    W = g.get_reference()
    assert np.array_equal(pairs, po) and np.allclose(nu, nuo, rtol=1e-9)
    assert np.abs(W - Wo).max() <= 1e-8 and np.allclose(np.linalg.norm(W, axis=0), 1.0, atol=1e-12)
    g.close()
