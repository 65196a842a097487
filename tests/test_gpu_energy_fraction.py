"""GPU parity for the energy fraction of eq. (24), rd_energy_fraction:
chi = ||Qb||_B^2 / ||x_*||_B^2 with B = H_II, Q = Z E^{-1} Z^T, against the oracle's definition written out
(oracle CoarseSpace.Q, oracle apply_H; pinned by P12 in tests/test_oracle_pins.py), on the same seeded inputs.

Bars: chi and both energies to 1e-9 relative (sums of ~N products in a different order; the coarse solve is
k x k with cond(E) <= 1e10 guarded, on these workloads <= 1e4); 1 - chi equals the complementary fraction
||x_* - Qb||_B^2 / ||x_*||_B^2 when x_* solves the system (1e-6: x_* is a 1e-10 solve); rank zero gives 0."""
import numpy as np
import pytest

from workloads import make_config, make_steady_2d

pytestmark = pytest.mark.gpu

WORKLOADS = {
    "config1": lambda: make_config(1),
    "c3_16": lambda: make_config(twin="c3_16"),
    "ragged37": lambda: make_steady_2d(n=37, channels=[(0.4, 0.6)], vel=20.0, alpha=1e-4, k=5, n_queries=2, n_bumps=3,
                                       psi_factor=0.6, pdas_cap=60, config=1, name="ragged37"),
}


@pytest.fixture(scope="module", params=list(WORKLOADS))
def setup(request, oracle_mod):
    import torch

    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    import paper_2606_17971_b200 as rd

    rd.load_library()
    w = WORKLOADS[request.param]()
    o = oracle_mod.Oracle.from_workload(w)
    g = rd.RefDef.from_workload(w, rd.Options(pdas_cap=w.pdas_cap))
    _, W = oracle_mod.reference_eigs(w.rowptr, w.colidx, w.val, w.m, w.alpha, w.k)
    g.set_reference(W)
    yield rd, w, o, g, W
    g.close()


def _oracle_chi(o, w, idx, Zt, b_I, xs_I):
    """eq. (24) written out with the oracle's operator and coarse space."""
    def energy(v_I):
        v = np.zeros(w.N)
        v[idx] = v_I
        return float(v_I @ o.apply_H(v)[idx])
    Qb = o.coarse(idx, Zt).Q(b_I)
    return energy(Qb) / energy(xs_I), energy(Qb), energy(xs_I), energy(xs_I - Qb)


@pytest.mark.parametrize("frac_active", [0.0, 0.15, 0.6])
def test_energy_fraction_matches_definition(setup, frac_active):
    rd, w, o, g, W = setup
    rng = np.random.default_rng(24)
    active = (rng.random(w.N) < frac_active).astype(np.uint8)
    idx = np.flatnonzero(active == 0)
    b = rng.standard_normal(w.N) * w.m
    xs_I, rep = o.alg1(idx, b[idx], np.zeros(len(idx)), W[idx], eps=1e-10)
    assert rep["status"] == 0
    xs = rng.standard_normal(w.N)          # entries on J are garbage on purpose: they must be ignored
    xs[idx] = xs_I
    chi_o, qb_o, en_o, comp_o = _oracle_chi(o, w, idx, W[idx], b[idx], xs_I)
    chi, qb, en = g.energy_fraction(rd.REFDEF, active, b, xs)
    assert 0.0 < chi < 1.0
    assert abs(qb - qb_o) <= 1e-9 * qb_o
    assert abs(en - en_o) <= 1e-9 * en_o
    assert abs(chi - chi_o) <= 1e-9 * chi_o
    assert abs((1.0 - chi) - comp_o / en_o) <= 1e-6


def test_energy_fraction_device_pointers_and_rank_zero(setup):
    import torch

    rd, w, o, g, W = setup
    rng = np.random.default_rng(25)
    active = (rng.random(w.N) < 0.3).astype(np.uint8)
    b = rng.standard_normal(w.N) * w.m
    xs = rng.standard_normal(w.N)          # any vector: the two energies are defined for every x_*
    host = g.energy_fraction(rd.REFDEF, active, b, xs)
    dev = g.energy_fraction(rd.REFDEF, torch.from_numpy(active).cuda(), torch.from_numpy(b).cuda(), torch.from_numpy(xs).cuda())
    assert host == dev                     # same kernels, fixed summation order: bit-identical
    again = g.energy_fraction(rd.REFDEF, active, b, xs)
    assert again == host
    chi0, qb0, en0 = g.energy_fraction(rd.JACOBI_CG, active, b, xs)
    assert chi0 == 0.0 and qb0 == 0.0 and en0 == host[2]
    # all DOFs active: empty inactive system
    chi_e, qb_e, en_e = g.energy_fraction(rd.REFDEF, np.ones(w.N, np.uint8), b, xs)
    assert (chi_e, qb_e, en_e) == (0.0, 0.0, 0.0)


def test_energy_fraction_zero_extension_uses_history(setup):
    """Zero-extension (eq. (13)) zeroes the rows that were active at an earlier restriction of the
    sequence.  With an empty history its basis is the directly restricted one, so chi is bit-identical; and the
    diagnostic reads the history without advancing it."""
    rd, w, o, g, W = setup
    rng = np.random.default_rng(26)
    active = (rng.random(w.N) < 0.2).astype(np.uint8)
    b = rng.standard_normal(w.N) * w.m
    xs = rng.standard_normal(w.N)
    g.reset_sequence()
    a = g.energy_fraction(rd.REFDEF, active, b, xs)
    z = g.energy_fraction(rd.ZEROEXT, active, b, xs)
    assert z == a
    z2 = g.energy_fraction(rd.ZEROEXT, active, b, xs)      # the call does not advance the history
    assert z2 == a
