"""GPU parity for the transient coarse-mesh reference of eq. (14), rd_build_reference_transient,
against the oracle (oracle.transient_reference, pinned in tests/test_oracle_pins.py) on the same seeded inputs.

Bars: selected pairs (i, j) identical (integer work; the candidates' nu are separated by far more than rounding on
these inputs -- checked); nu to 1e-9 relative (Jacobi against LAPACK on nt x nt problems whose entries are sums of N_s
products); W to 1e-8 in the max norm of unit columns (an eigenvector moves by rounding / gap, gaps >= 1e-4 relative
here); query parity through the installed reference: identical active sets, states 1e-6 in the M-norm."""
import numpy as np
import pytest

from workloads import make_config, make_spacetime_2d, make_steady_2d

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def rd():
    import torch

    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    import paper_2606_17971_b200 as pkg

    pkg.load_library()
    return pkg


def _spatial_vectors(oracle_mod, w, rs, coarse):
    n = w.dims[0]
    ws = make_steady_2d(n=n // 2 if coarse else n, channels=[(0.25, 0.35), (0.65, 0.75)], vel=50.0, alpha=w.alpha, k=rs,
                        n_queries=1, n_bumps=1, psi_factor=0.6, pdas_cap=5, config=2, name="space")
    op = (ws.rowptr, ws.colidx, ws.val, ws.m, ws.alpha)
    if coarse:
        return oracle_mod.prolonged_reference(op, ws.dims, w.dims, rs)[2]
    return oracle_mod.reference_eigs_scaled(*op, rs)[1]


CASES = {
    # (workload, number of spatial vectors, k, prolonged from the half grid?)
    "c4_32x8_fine": (lambda: make_config(twin="c4_32x8"), 16, 16, False),
    "c4_32x8_prolonged": (lambda: make_config(twin="c4_32x8"), 6, 24, True),
    # ragged: N_s = 19 * 19 and nt = 5 (neither a multiple of 8 or 32)
    "ragged19x5": (lambda: make_spacetime_2d(n=19, nt=5, T=1.0, channels=[(0.4, 0.6)], vel=20.0, alpha=1e-4, k=7, n_queries=1,
                                             n_bumps=3, psi_factor=0.6, pdas_cap=40, config=4, name="ragged19x5"), 3, 7, None),
}


@pytest.mark.parametrize("case", list(CASES))
def test_transient_reference_matches_oracle(rd, oracle_mod, case):
    import torch

    mk, rs, k, coarse = CASES[case]
    w = mk()
    if coarse is None:
        Phi = np.random.default_rng(14).standard_normal((w.N // w.nt, rs))
    else:
        Phi = _spatial_vectors(oracle_mod, w, rs, coarse)
    pairs_o, nu_o, W_o = oracle_mod.transient_reference(Phi, (w.rowptr, w.colidx, w.val, w.m, w.alpha), w.nt, k)
    assert np.diff(nu_o).min() > 1e-7 * nu_o[0]                 # the order is decided far above rounding
    g = rd.RefDef.from_workload(w, rd.Options(pdas_cap=w.pdas_cap))
    try:
        pairs, nu = g.build_reference_transient(k, Phi, w.nt)
        assert pairs.tolist() == pairs_o.tolist()
        assert np.abs(nu - nu_o).max() <= 1e-9 * nu_o.max()
        W = g.get_reference()
        assert W.shape == W_o.shape
        assert np.abs(W - W_o).max() <= 1e-8
        assert np.allclose(np.linalg.norm(W, axis=0), 1.0, atol=1e-13)
        # device input (column-major = a (rs, N_s) row-major tensor): bit-identical
        pairs_d, nu_d = g.build_reference_transient(k, torch.from_numpy(np.ascontiguousarray(Phi.T)).cuda(), w.nt)
        assert pairs_d.tolist() == pairs.tolist() and (nu_d == nu).all() and (g.get_reference() == W).all()
    finally:
        g.close()


def test_transient_reference_query_parity(rd, oracle_mod):
    w = make_config(twin="c4_32x8")
    Phi = _spatial_vectors(oracle_mod, w, w.k, False)
    _, _, W_o = oracle_mod.transient_reference(Phi, (w.rowptr, w.colidx, w.val, w.m, w.alpha), w.nt, w.k)
    o = oracle_mod.Oracle.from_workload(w)
    g = rd.RefDef.from_workload(w, rd.Options(pdas_cap=w.pdas_cap))
    try:
        g.build_reference_transient(w.k, Phi, w.nt)
        yd, psi = w.target(0)
        ro = o.solve_query(1, yd, psi, W_o, oracle_mod.OracleOptions(pdas_cap=w.pdas_cap))
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


def test_transient_reference_invalid_arguments(rd):
    w = make_config(twin="c4_32x8")
    g = rd.RefDef.from_workload(w)
    try:
        Phi = np.ones((w.N // w.nt, 2))
        with pytest.raises(rd.RefDefError):
            g.build_reference_transient(2 * w.nt + 1, Phi, w.nt)          # more than rs * nt candidates
        with pytest.raises(rd.RefDefError):
            g.build_reference_transient(2, np.zeros((w.N // w.nt, 2)), w.nt)   # zero vector: D_i = 0
    finally:
        g.close()
