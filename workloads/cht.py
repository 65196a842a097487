"""Conjugate-heat-transfer (CHT) workload generator.

One specification for the oracle and the CUDA harness (reading A15;
BASELINE.json `configs`).  Host numpy/scipy, deterministic, seeded.  Nothing here
belongs to the method of the paper (§2.1-2.3): the generator only assembles
the *inputs* the C-ABI takes -- the state operator K in integrated finite-volume form
(CSR), the lumped mass diagonal m, the target y_d and the bound psi.

Discretisation (cell-centred finite volumes on the unit square/cube, n cells per side,
h = 1/n, cell centres (i+1/2)h, index id = ix + n*(iy + n*iz), x fastest;
space-time id = s + N_s*t, "ordered by time level, then by spatial node"):

* material by cell centre, closed intervals: fluid where y_c in [a,b] (2D channels) or
  (y_c-c_y)^2 + (z_c-c_z)^2 < R^2 (bores along x); kappa = 1 solid, 0.1 fluid;
* diffusion, integrated form: interior face coefficient kappa_f h^(d-2) with the HARMONIC
  mean kappa_f = 2 k1 k2/(k1+k2); zero-Dirichlet boundary face:
  2 kappa_cell h^(d-2) on the diagonal (half-cell distance);
* convection, first-order upwind, velocity (v,0[,0]), v >= 0 a function of the transverse
  coordinates only: K_ii += v_i h^(d-1), K_{i,west(i)} -= v_i h^(d-1) when the west
  neighbour exists (inflow value 0 at x = 0);
* lumped mass m_i = h^d;
* space-time (eq. (2)-(3)): K_st = I (x) K_s + L (x) M_s with
  L_nn = 1/dt, L_{n,n-1} = -1/dt, capacity 1, y^0 = 0, f = 0, uniform dt = T/N_t;
  M_st = I (x) M_s (W_t = I for uniform steps).

Targets: y_d(x) = sum_b a_b exp(-|x-c_b|^2/(2*0.08^2)), rng = default_rng(1000*config+query);
per bump draw the d centre coordinates U[0.2,0.8] then the amplitude U[0.5,1.0].
Space-time: per bump draw start point, end point and amplitude; the centre at time level
n is p0 + (p1-p0)*n*dt, n = 1..N_t.  psi = factor*max(y_d) (scalar broadcast).
"""
from __future__ import annotations

import hashlib
from dataclasses import dataclass, field
from typing import Callable, Dict, List, Optional, Sequence, Tuple

import numpy as np
import scipy.sparse as sp

BUMP_WIDTH = 0.08
KAPPA_SOLID = 1.0
KAPPA_FLUID = 0.1


# --------------------------------------------------------------------------------------
# operator assembly
# --------------------------------------------------------------------------------------
def _assemble_grid_operator(dims: Tuple[int, ...], kappa: np.ndarray, vel: np.ndarray) -> sp.csr_matrix:
    """K (integrated FV form) on a Cartesian grid.

    dims = (nx, ny) or (nx, ny, nz) with nx == ny (== nz) = n; kappa, vel are per-cell arrays
    of shape dims[::-1] (z, y, x order so that x is the fastest index)."""
    d = len(dims)
    n = dims[0]
    assert all(q == n for q in dims)
    h = 1.0 / n
    N = n ** d
    ids = np.arange(N, dtype=np.int64).reshape(dims[::-1])
    face_scale = h ** (d - 2)
    rows: List[np.ndarray] = []
    cols: List[np.ndarray] = []
    vals: List[np.ndarray] = []

    def add(r, c, v):
        rows.append(np.asarray(r, dtype=np.int64).ravel())
        cols.append(np.asarray(c, dtype=np.int64).ravel())
        vals.append(np.asarray(v, dtype=np.float64).ravel())

    for axis in range(d):  # numpy axis: 0 is the slowest coordinate
        lo = [slice(None)] * d
        hi = [slice(None)] * d
        lo[axis] = slice(0, n - 1)
        hi[axis] = slice(1, n)
        lo_t, hi_t = tuple(lo), tuple(hi)
        k1 = kappa[lo_t]
        k2 = kappa[hi_t]
        coef = 2.0 * k1 * k2 / (k1 + k2) * face_scale
        i = ids[lo_t]
        j = ids[hi_t]
        add(i, i, coef)
        add(j, j, coef)
        add(i, j, -coef)
        add(j, i, -coef)
        # zero-Dirichlet boundary faces on both ends of this axis
        for end in (0, n - 1):
            b = [slice(None)] * d
            b[axis] = end
            b_t = tuple(b)
            add(ids[b_t], ids[b_t], 2.0 * kappa[b_t] * face_scale)

    # first-order upwind convection in +x (the last numpy axis)
    flux = vel * h ** (d - 1)
    add(ids, ids, flux)
    west = [slice(None)] * d
    here = [slice(None)] * d
    west[-1] = slice(0, n - 1)
    here[-1] = slice(1, n)
    add(ids[tuple(here)], ids[tuple(west)], -flux[tuple(here)])

    K = sp.coo_matrix((np.concatenate(vals), (np.concatenate(rows), np.concatenate(cols))), shape=(N, N)).tocsr()
    K.sum_duplicates()
    K.sort_indices()
    return K


def _centres(n: int) -> np.ndarray:
    return (np.arange(n, dtype=np.float64) + 0.5) / n


def _channel_fields_2d(n: int, channels: Sequence[Tuple[float, float]], v: float):
    yc = _centres(n)
    fluid_y = np.zeros(n, dtype=bool)
    for a, b in channels:
        fluid_y |= (yc >= a) & (yc <= b)
    fluid = np.repeat(fluid_y[:, None], n, axis=1)  # shape (ny, nx)
    kappa = np.where(fluid, KAPPA_FLUID, KAPPA_SOLID)
    vel = np.where(fluid, float(v), 0.0)
    return kappa, vel


def _bore_fields_3d(n: int, bores: Sequence[Tuple[float, float]], R: float, vpeak: float):
    c = _centres(n)
    zc, yc = np.meshgrid(c, c, indexing="ij")  # shape (nz, ny)
    vel2 = np.zeros((n, n))
    fluid2 = np.zeros((n, n), dtype=bool)
    for cy, cz in bores:
        r2 = (yc - cy) ** 2 + (zc - cz) ** 2
        inside = r2 < R * R
        fluid2 |= inside
        vel2 = np.where(inside, vpeak * (1.0 - r2 / (R * R)), vel2)
    fluid = np.repeat(fluid2[:, :, None], n, axis=2)  # (nz, ny, nx)
    vel = np.repeat(vel2[:, :, None], n, axis=2)
    kappa = np.where(fluid, KAPPA_FLUID, KAPPA_SOLID)
    return kappa, vel


# --------------------------------------------------------------------------------------
# targets
# --------------------------------------------------------------------------------------
def gaussian_targets(dims: Tuple[int, ...], n_bumps: int, seed: int) -> np.ndarray:
    """Steady target: sum of Gaussian bumps; draws per bump: d centre coords then amplitude."""
    d = len(dims)
    n = dims[0]
    rng = np.random.default_rng(seed)
    c = _centres(n)
    yd = np.zeros(dims[::-1], dtype=np.float64)
    grids = np.meshgrid(*([c] * d), indexing="ij")  # slowest .. fastest == (z,) y, x
    for _ in range(n_bumps):
        centre = rng.uniform(0.2, 0.8, size=d)  # (x, y[, z])
        amp = rng.uniform(0.5, 1.0)
        r2 = np.zeros_like(yd)
        for a in range(d):
            # coordinate a (x=0) lives on numpy axis d-1-a
            r2 += (grids[d - 1 - a] - centre[a]) ** 2
        yd += amp * np.exp(-r2 / (2.0 * BUMP_WIDTH ** 2))
    return yd.ravel()


def spacetime_targets(n: int, nt: int, T: float, n_bumps: int, seed: int) -> np.ndarray:
    """Moving bumps on seeded linear paths (config 4); id = s + N_s*t, time levels n = 1..nt."""
    rng = np.random.default_rng(seed)
    c = _centres(n)
    yy, xx = np.meshgrid(c, c, indexing="ij")
    dt = T / nt
    yd = np.zeros((nt, n, n), dtype=np.float64)
    for _ in range(n_bumps):
        p0 = rng.uniform(0.2, 0.8, size=2)
        p1 = rng.uniform(0.2, 0.8, size=2)
        amp = rng.uniform(0.5, 1.0)
        for lvl in range(1, nt + 1):
            ctr = p0 + (p1 - p0) * (lvl * dt)
            r2 = (xx - ctr[0]) ** 2 + (yy - ctr[1]) ** 2
            yd[lvl - 1] += amp * np.exp(-r2 / (2.0 * BUMP_WIDTH ** 2))
    return yd.ravel()


def sha_arrays(*arrays: np.ndarray) -> str:
    """Hash of inputs, as the paper does for targets and matrices."""
    hsh = hashlib.sha256()
    for a in arrays:
        a = np.ascontiguousarray(a)
        hsh.update(str(a.dtype).encode())
        hsh.update(str(a.shape).encode())
        hsh.update(a.tobytes())
    return hsh.hexdigest()


# --------------------------------------------------------------------------------------
# workload container
# --------------------------------------------------------------------------------------
@dataclass
class Workload:
    name: str
    config: int
    kind: str  # "2d", "3d", "st2d"
    dims: Tuple[int, ...]  # spatial grid
    nt: int  # 1 for steady
    N: int
    rowptr: np.ndarray  # int64, N+1
    colidx: np.ndarray  # int32, nnz
    val: np.ndarray  # float64, nnz
    m: np.ndarray  # float64, N (lumped mass, > 0)
    alpha: float
    k: int
    pdas_cap: int
    psi_factor: float
    n_bumps: int
    query_order: List[int]
    _target: Callable[[int], np.ndarray] = field(repr=False, default=None)

    @property
    def nnz(self) -> int:
        return int(self.rowptr[-1])

    @property
    def n_queries(self) -> int:
        return len(self.query_order)

    def csr(self) -> sp.csr_matrix:
        return sp.csr_matrix((self.val, self.colidx, self.rowptr), shape=(self.N, self.N))

    def target(self, q: int) -> Tuple[np.ndarray, np.ndarray]:
        """(y_d, psi) of the q-th query IN SEQUENCE ORDER (query_order[q] picks the seed)."""
        qid = self.query_order[q]
        yd = self._target(1000 * self.config + qid)
        psi = np.full(self.N, self.psi_factor * float(yd.max()), dtype=np.float64)
        return yd, psi

    def operator_hash(self) -> str:
        return sha_arrays(self.rowptr, self.colidx, self.val, self.m)


def _finish(name, config, kind, dims, nt, K, m, alpha, k, pdas_cap, psi_factor, n_bumps, order, target):
    K = K.tocsr()
    K.sort_indices()
    return Workload(
        name=name, config=config, kind=kind, dims=tuple(dims), nt=nt, N=K.shape[0],
        rowptr=K.indptr.astype(np.int64), colidx=K.indices.astype(np.int32),
        val=K.data.astype(np.float64), m=np.ascontiguousarray(m, dtype=np.float64),
        alpha=float(alpha), k=int(k), pdas_cap=int(pdas_cap), psi_factor=float(psi_factor),
        n_bumps=int(n_bumps), query_order=list(order), _target=target)


def make_steady_2d(n, channels, vel, alpha, k, n_queries, n_bumps, psi_factor, pdas_cap, config, name=None,
                   order=None) -> Workload:
    kappa, v = _channel_fields_2d(n, channels, vel)
    K = _assemble_grid_operator((n, n), kappa, v)
    m = np.full(n * n, (1.0 / n) ** 2)
    order = list(range(n_queries)) if order is None else order
    return _finish(name or f"cht2d_{n}", config, "2d", (n, n), 1, K, m, alpha, k, pdas_cap, psi_factor, n_bumps,
                   order, lambda seed: gaussian_targets((n, n), n_bumps, seed))


def make_steady_3d(n, bores, R, vpeak, alpha, k, n_queries, n_bumps, psi_factor, pdas_cap, config, name=None,
                   order=None) -> Workload:
    kappa, v = _bore_fields_3d(n, bores, R, vpeak)
    K = _assemble_grid_operator((n, n, n), kappa, v)
    m = np.full(n ** 3, (1.0 / n) ** 3)
    order = list(range(n_queries)) if order is None else order
    return _finish(name or f"cht3d_{n}", config, "3d", (n, n, n), 1, K, m, alpha, k, pdas_cap, psi_factor, n_bumps,
                   order, lambda seed: gaussian_targets((n, n, n), n_bumps, seed))


def make_spacetime_2d(n, nt, T, channels, vel, alpha, k, n_queries, n_bumps, psi_factor, pdas_cap, config,
                      name=None, order=None) -> Workload:
    kappa, v = _channel_fields_2d(n, channels, vel)
    Ks = _assemble_grid_operator((n, n), kappa, v)
    Ns = n * n
    ms = np.full(Ns, (1.0 / n) ** 2)
    dt = T / nt
    L = sp.diags([np.full(nt, 1.0 / dt), np.full(nt - 1, -1.0 / dt)], [0, -1], format="csr")
    K = (sp.kron(sp.identity(nt, format="csr"), Ks, format="csr") + sp.kron(L, sp.diags(ms), format="csr")).tocsr()
    K.sum_duplicates()
    m = np.tile(ms, nt)
    order = list(range(n_queries)) if order is None else order
    return _finish(name or f"cht2d_{n}x{nt}", config, "st2d", (n, n), nt, K, m, alpha, k, pdas_cap, psi_factor,
                   n_bumps, order, lambda seed: spacetime_targets(n, nt, T, n_bumps, seed))


# --------------------------------------------------------------------------------------
# BASELINE.json configs (1-based) and their scaled-down twins
# --------------------------------------------------------------------------------------
CH2 = [(0.25, 0.35), (0.65, 0.75)]
BORES4 = [(0.3, 0.3), (0.7, 0.3), (0.3, 0.7), (0.7, 0.7)]

CONFIGS: Dict[int, dict] = {
    1: dict(kind="2d", n=32, channels=[(0.4, 0.6)], vel=20.0, alpha=1e-4, k=8, n_queries=1, n_bumps=3,
            psi_factor=0.6, pdas_cap=20),
    2: dict(kind="2d", n=512, channels=CH2, vel=50.0, alpha=1e-4, k=32, n_queries=8, n_bumps=5,
            psi_factor=0.55, pdas_cap=100),
    3: dict(kind="3d", n=96, bores=[(0.5, 0.5)], R=0.15, vpeak=30.0, alpha=1e-5, k=48, n_queries=6, n_bumps=4,
            psi_factor=0.6, pdas_cap=100),
    4: dict(kind="st2d", n=256, nt=32, T=1.0, channels=CH2, vel=50.0, alpha=1e-4, k=64, n_queries=1, n_bumps=3,
            psi_factor=0.6, pdas_cap=100),
    5: dict(kind="3d", n=160, bores=BORES4, R=0.15, vpeak=30.0, alpha=1e-5, k=64, n_queries=10, n_bumps=4,
            psi_factor=0.6, pdas_cap=100, shuffled=True),
}

# scaled-down twins for full-sequence oracle parity (same generator, same seeds)
TWINS: Dict[str, dict] = {
    "c2_48": dict(config=2, n=48, k=16),
    "c2_96": dict(config=2, n=96, k=32),
    "c2_128": dict(config=2, n=128, k=32),
    "c3_16": dict(config=3, n=16, k=16),
    "c3_24": dict(config=3, n=24, k=24),
    "c3_32": dict(config=3, n=32, k=48),
    "c4_32x8": dict(config=4, n=32, nt=8, k=16),
    "c4_64x8": dict(config=4, n=64, nt=8, k=32),
    "c5_24": dict(config=5, n=24, k=24),
    "c5_48": dict(config=5, n=48, k=64),
}


def make_config(config: Optional[int] = None, n: Optional[int] = None, nt: Optional[int] = None, k: Optional[int] = None,
                n_queries: Optional[int] = None, twin: Optional[str] = None) -> Workload:
    """Workload of BASELINE.json config `config` (1..5); n / nt / k override the size for twins."""
    if twin is not None:
        t = dict(TWINS[twin])
        config = t.pop("config")
        n = t.get("n", n)
        nt = t.get("nt", nt)
        k = t.get("k", k)
    p = dict(CONFIGS[config])
    kind = p.pop("kind")
    shuffled = p.pop("shuffled", False)
    if n is not None:
        p["n"] = n
    if k is not None:
        p["k"] = k
    if n_queries is not None:
        p["n_queries"] = n_queries
    order = None
    if shuffled:
        # config 5: shuffled query order (Table 6 "Shuffled order")
        order = [int(x) for x in np.random.default_rng(5999).permutation(10)][: p["n_queries"]]
    name = twin or f"config{config}" + ("" if n is None else f"_n{p['n']}")
    if kind == "2d":
        return make_steady_2d(config=config, name=name, order=order, **p)
    if kind == "3d":
        return make_steady_3d(config=config, name=name, order=order, **p)
    if kind == "st2d":
        if nt is not None:
            p["nt"] = nt
        return make_spacetime_2d(config=config, name=name, order=order, **p)
    raise ValueError(kind)
