"""ctypes front end of the CPU oracle (oracle/refdef_oracle.c) -- TEST INFRASTRUCTURE.

The arithmetic lives in the C file, written from PAPER.md step by step; this module only
builds it (gcc -O2), marshals numpy arrays, and provides `reference_eigs`, the plain
definition of what `build_reference` must produce: the k lowest eigenpairs of the full
H = M + sigma K^T M^{-1} K (BASELINE.json north_star; nearest paper text Alg. 2 step 2,
PAPER.md:382), computed with a library eigensolver on the assembled matrix.
"""
from __future__ import annotations

import ctypes as C
import itertools
import os
import subprocess
from dataclasses import dataclass
from typing import List, Optional

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "refdef_oracle.c")
_LIB = os.path.join(_HERE, "librefdef_oracle.so")
_LIB_OMP = os.path.join(_HERE, "librefdef_oracle_omp.so")

JACOBI_CG, REFDEF, ZEROEXT = 0, 1, 2
INIT_PAPER, INIT_ALL_ACTIVE, INIT_ALL_INACTIVE, INIT_GIVEN = 0, 1, 2, 3
STATUS_NAMES = {0: "ok", -1: "einval", -2: "enomem", -5: "enotspd", -6: "ecap", -7: "esteps", -8: "ecycle",
                -9: "eresid"}


def build_oracle(force: bool = False, threaded: bool = False) -> str:
    """Compile the oracle with gcc (plain -O2, no fast-math).  threaded = False: the single-thread build every parity
    test uses.  threaded = True: the same file with -fopenmp (row loops split over the host cores), for the TIMING
    legs of bench.py only."""
    lib = _LIB_OMP if threaded else _LIB
    if force or not os.path.exists(lib) or os.path.getmtime(lib) < os.path.getmtime(_SRC):
        subprocess.check_call(["gcc", "-O2", "-std=c99"] + (["-fopenmp"] if threaded else []) +
                              ["-fPIC", "-shared", "-o", lib, _SRC, "-lm"])
    return lib


class _StepReport(C.Structure):
    _fields_ = [("n_inactive", C.c_int32), ("cg_iters", C.c_int32), ("rank_used", C.c_int32),
                ("coarse_fallback", C.c_int32), ("replacements", C.c_int32), ("status", C.c_int32),
                ("rel_resid_verified", C.c_double), ("cond_E", C.c_double), ("margin", C.c_double),
                ("active_hash", C.c_uint64)]


class _QueryReport(C.Structure):
    _fields_ = [("n_steps", C.c_int32), ("status", C.c_int32), ("kkt", C.c_double * 5)]


class _Options(C.Structure):
    _fields_ = [("eps", C.c_double), ("eps_c", C.c_double), ("cg_cap", C.c_int32), ("pdas_cap", C.c_int32),
                ("replace_period", C.c_int32), ("jacobi", C.c_int32), ("c_is_diag", C.c_int32),
                ("init", C.c_int32)]


class _SolveReport(C.Structure):
    _fields_ = [("iters", C.c_int32), ("rank_used", C.c_int32), ("coarse_fallback", C.c_int32),
                ("replacements", C.c_int32), ("status", C.c_int32), ("rel_resid_verified", C.c_double),
                ("cond_E", C.c_double)]


@dataclass
class OracleOptions:
    eps: float = 1e-8          # Verify tolerance (reading A11; the paper's own is 1e-10)
    eps_c: float = 1e-8        # recurrence trigger
    cg_cap: int = 500000       # reading A12
    pdas_cap: int = 100
    replace_period: int = 0    # reading A8
    jacobi: int = 1
    c_is_diag: int = 0         # reading A3: c = 1 (configs) or d_i (eq. (8))
    init: int = INIT_PAPER

    def c_struct(self) -> _Options:
        return _Options(self.eps, self.eps_c, self.cg_cap, self.pdas_cap, self.replace_period, self.jacobi,
                        self.c_is_diag, self.init)


def _dp(a):
    return a.ctypes.data_as(C.POINTER(C.c_double))


def _load(threaded: bool = False):
    lib = C.CDLL(build_oracle(threaded=threaded))
    lib.orc_threads.restype = C.c_int
    lib.orc_create.restype = C.c_void_p
    lib.orc_create.argtypes = [C.c_int64, C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p, C.c_double]
    lib.orc_destroy.argtypes = [C.c_void_p]
    lib.orc_reset_sequence.argtypes = [C.c_void_p]
    for f in ("orc_apply_K", "orc_apply_KT", "orc_apply_H"):
        getattr(lib, f).argtypes = [C.c_void_p, C.c_void_p, C.c_void_p]
    lib.orc_diag_H.argtypes = [C.c_void_p, C.c_void_p]
    lib.orc_apply_B.argtypes = [C.c_void_p, C.c_void_p, C.c_int64, C.c_void_p, C.c_void_p]
    lib.orc_coarse_build.restype = C.c_void_p
    lib.orc_coarse_build.argtypes = [C.c_void_p, C.c_void_p, C.c_int64, C.c_void_p, C.c_int]
    lib.orc_coarse_free.argtypes = [C.c_void_p]
    lib.orc_coarse_Q.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p]
    lib.orc_coarse_P.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p]
    lib.orc_coarse_rank.argtypes = [C.c_void_p]
    lib.orc_coarse_fallback.argtypes = [C.c_void_p]
    lib.orc_coarse_cond.restype = C.c_double
    lib.orc_coarse_cond.argtypes = [C.c_void_p]
    lib.orc_coarse_get.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p]
    lib.orc_alg1.argtypes = [C.c_void_p, C.c_void_p, C.c_int64, C.c_void_p, C.c_void_p, C.c_void_p, C.c_int,
                             C.c_double, C.c_double, C.c_int, C.c_int, C.c_int, C.POINTER(_SolveReport)]
    lib.orc_alg1_cs.argtypes = [C.c_void_p, C.c_void_p, C.c_int64, C.c_void_p, C.c_void_p, C.c_void_p,
                                C.c_double, C.c_double, C.c_int, C.c_int, C.c_int, C.POINTER(_SolveReport)]
    lib.orc_solve_query.argtypes = [C.c_void_p, C.c_int, C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p, C.c_int,
                                    C.POINTER(_Options), C.c_void_p, C.c_void_p, C.c_void_p,
                                    C.POINTER(_StepReport), C.c_void_p, C.POINTER(_QueryReport)]
    lib.orc_kkt.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p]
    lib.orc_restrict.argtypes = [C.c_void_p, C.c_int, C.c_void_p, C.c_int, C.c_void_p, C.c_int64, C.c_void_p]
    lib.orc_get_state.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p]
    return lib


_libs = {}


def _get_lib(threaded: bool = False):
    if threaded not in _libs:
        _libs[threaded] = _load(threaded)
    return _libs[threaded]


class CoarseSpace:
    """Handle on the oracle's coarse space of one inactive system (eq. (18))."""

    def __init__(self, orc: "Oracle", idx: np.ndarray, Zt: np.ndarray):
        self._lib = orc._lib  # the build (plain or threaded) of the context it belongs to
        self._orc = orc
        self.idx = np.ascontiguousarray(idx, dtype=np.int64)
        self.n = len(self.idx)
        Zt = np.asfortranarray(Zt, dtype=np.float64)
        k = Zt.shape[1] if Zt.ndim == 2 else 0
        self._h = self._lib.orc_coarse_build(orc._h, self.idx.ctypes.data, self.n, Zt.ctypes.data, k)
        self.rank = self._lib.orc_coarse_rank(self._h)
        self.fallback = self._lib.orc_coarse_fallback(self._h)
        self.cond_E = self._lib.orc_coarse_cond(self._h)

    def Q(self, v):
        v = np.ascontiguousarray(v, dtype=np.float64)
        out = np.empty(self.n)
        self._lib.orc_coarse_Q(self._h, v.ctypes.data, out.ctypes.data)
        return out

    def P(self, v):
        v = np.ascontiguousarray(v, dtype=np.float64)
        out = np.empty(self.n)
        self._lib.orc_coarse_P(self._h, v.ctypes.data, out.ctypes.data)
        return out

    def factors(self):
        Z = np.empty((self.n, self.rank), order="F")
        BZ = np.empty((self.n, self.rank), order="F")
        E = np.empty((self.rank, self.rank), order="F")
        if self.rank:
            self._lib.orc_coarse_get(self._h, Z.ctypes.data, BZ.ctypes.data, E.ctypes.data)
        return Z, BZ, E

    def __del__(self):
        try:
            self._lib.orc_coarse_free(self._h)
        except Exception:
            pass


class Oracle:
    """One operator = one context (host arrays).  sigma = alpha (reading A1)."""

    def __init__(self, rowptr, colidx, val, m, sigma, threaded: bool = False):
        self._lib = _get_lib(threaded)
        self.threads = int(self._lib.orc_threads())
        self.N = len(m)
        self._rowptr = np.ascontiguousarray(rowptr, dtype=np.int64)
        self._colidx = np.ascontiguousarray(colidx, dtype=np.int32)
        self._val = np.ascontiguousarray(val, dtype=np.float64)
        self._m = np.ascontiguousarray(m, dtype=np.float64)
        self.sigma = float(sigma)
        self._h = self._lib.orc_create(self.N, self._rowptr.ctypes.data, self._colidx.ctypes.data,
                                       self._val.ctypes.data, self._m.ctypes.data, self.sigma)
        if not self._h:
            raise ValueError("orc_create failed (N <= 0 or m_i <= 0)")

    @classmethod
    def from_workload(cls, w, threaded: bool = False):
        return cls(w.rowptr, w.colidx, w.val, w.m, w.alpha, threaded=threaded)

    def __del__(self):
        try:
            if self._h:
                self._lib.orc_destroy(self._h)
        except Exception:
            pass

    def reset_sequence(self):
        self._lib.orc_reset_sequence(self._h)

    def _apply(self, name, v):
        v = np.ascontiguousarray(v, dtype=np.float64)
        out = np.empty(self.N)
        getattr(self._lib, name)(self._h, v.ctypes.data, out.ctypes.data)
        return out

    def apply_K(self, v):
        return self._apply("orc_apply_K", v)

    def apply_KT(self, v):
        return self._apply("orc_apply_KT", v)

    def apply_H(self, v):
        return self._apply("orc_apply_H", v)

    def diag_H(self):
        d = np.empty(self.N)
        self._lib.orc_diag_H(self._h, d.ctypes.data)
        return d

    def apply_B(self, idx, x):
        idx = np.ascontiguousarray(idx, dtype=np.int64)
        x = np.ascontiguousarray(x, dtype=np.float64)
        out = np.empty(len(idx))
        self._lib.orc_apply_B(self._h, idx.ctypes.data, len(idx), x.ctypes.data, out.ctypes.data)
        return out

    def restrict(self, method, W, idx):
        """Restricted candidate basis Z~ (O3a) of the inactive set idx; updates the zero-extension history."""
        idx = np.ascontiguousarray(idx, dtype=np.int64)
        W = np.asfortranarray(W, dtype=np.float64)
        k = W.shape[1]
        Zt = np.zeros((len(idx), k), order="F")
        self._lib.orc_restrict(self._h, method, W.ctypes.data, k, idx.ctypes.data, len(idx), Zt.ctypes.data)
        return Zt

    def coarse(self, idx, Zt) -> CoarseSpace:
        return CoarseSpace(self, idx, Zt)

    def alg1(self, idx, b, x0, Zt=None, eps=1e-8, eps_c=None, cap=500000, replace_period=0, jacobi=1):
        """Algorithm 1 on the inactive system (idx ascending).  Returns (x, report dict)."""
        idx = np.ascontiguousarray(idx, dtype=np.int64)
        b = np.ascontiguousarray(b, dtype=np.float64)
        x = np.array(x0, dtype=np.float64, copy=True)
        k = 0
        zp = None
        if Zt is not None and Zt.size:
            Zt = np.asfortranarray(Zt, dtype=np.float64)
            k = Zt.shape[1]
            zp = Zt.ctypes.data
        rep = _SolveReport()
        self._lib.orc_alg1(self._h, idx.ctypes.data, len(idx), b.ctypes.data, x.ctypes.data, zp, k, eps,
                           eps if eps_c is None else eps_c, cap, replace_period, jacobi, C.byref(rep))
        return x, {f: getattr(rep, f) for f, _ in _SolveReport._fields_}

    def kkt(self, y_d, psi, y, lam):
        """The five measures of eq. (25) for any (y, lambda); l = M y_d."""
        ell = np.ascontiguousarray(self._m * np.asarray(y_d, dtype=np.float64))
        psi = np.ascontiguousarray(psi, dtype=np.float64)
        y = np.ascontiguousarray(y, dtype=np.float64)
        lam = np.ascontiguousarray(lam, dtype=np.float64)
        out = np.zeros(5)
        self._lib.orc_kkt(self._h, ell.ctypes.data, psi.ctypes.data, y.ctypes.data, lam.ctypes.data, out.ctypes.data)
        return out

    def alg1_on(self, cs: "CoarseSpace", b, x0, eps=1e-8, eps_c=None, cap=500000, replace_period=0, jacobi=1):
        """Algorithm 1 on a coarse space that line 2 has already built (self.coarse(idx, Zt)): the same solve as alg1
        without repeating the setup.  Returns (x, report dict)."""
        b = np.ascontiguousarray(b, dtype=np.float64)
        x = np.array(x0, dtype=np.float64, copy=True)
        rep = _SolveReport()
        self._lib.orc_alg1_cs(self._h, cs.idx.ctypes.data, cs.n, b.ctypes.data, x.ctypes.data, cs._h, eps,
                              eps if eps_c is None else eps_c, cap, replace_period, jacobi, C.byref(rep))
        return x, {f: getattr(rep, f) for f, _ in _SolveReport._fields_}

    def solve_query(self, method, y_d, psi, W=None, opt: Optional[OracleOptions] = None, J0=None,
                    want_sets: bool = True):
        """PDAS query (O2).  W: N x k (any order; copied column-major).  Returns a dict."""
        opt = opt or OracleOptions()
        N = self.N
        y_d = np.ascontiguousarray(y_d, dtype=np.float64)
        psi = np.ascontiguousarray(psi, dtype=np.float64)
        k = 0
        wp = None
        if W is not None and method != JACOBI_CG:
            W = np.asfortranarray(W, dtype=np.float64)
            k = W.shape[1]
            wp = W.ctypes.data
        j0p = None
        if J0 is not None:
            J0 = np.ascontiguousarray(J0, dtype=np.uint8)
            j0p = J0.ctypes.data
        y = np.empty(N)
        u = np.empty(N)
        lam = np.empty(N)
        steps = (_StepReport * opt.pdas_cap)()
        nbytes = (N + 7) // 8
        Jb = np.zeros((opt.pdas_cap, nbytes), dtype=np.uint8) if want_sets else None
        rep = _QueryReport()
        o = opt.c_struct()
        st = self._lib.orc_solve_query(self._h, method, y_d.ctypes.data, psi.ctypes.data, j0p, wp, k, C.byref(o),
                                       y.ctypes.data, u.ctypes.data, lam.ctypes.data, steps,
                                       Jb.ctypes.data if want_sets else None, C.byref(rep))
        ns = rep.n_steps
        step_list: List[dict] = [{f: getattr(steps[i], f) for f, _ in _StepReport._fields_} for i in range(ns)]
        return dict(status=st, n_steps=ns, kkt=[rep.kkt[i] for i in range(5)], y=y, u=u, lam=lam, steps=step_list,
                    J_bits=(Jb[:ns] if want_sets else None),
                    hashes=[s["active_hash"] for s in step_list])

    def state(self):
        y = np.empty(self.N)
        J = np.empty(self.N, dtype=np.uint8)
        A = np.empty(self.N, dtype=np.uint8)
        self._lib.orc_get_state(self._h, y.ctypes.data, J.ctypes.data, A.ctypes.data)
        return y, J, A


def reference_eigs(rowptr, colidx, val, m, sigma, k, dense_below: int = 1500):
    """The definition `build_reference` must reach: the k lowest eigenpairs (theta, W) of
    H = M + sigma K^T M^{-1} K, W with orthonormal columns (N x k, column-major).

    A library eigensolver on the assembled matrix (dense eigh for small N, shift-invert
    Lanczos otherwise).  W is unique only up to sign / rotation inside clusters (reading A14)."""
    import scipy.sparse as sp
    import scipy.sparse.linalg as spla

    N = len(m)
    K = sp.csr_matrix((val, colidx, rowptr), shape=(N, N))
    H = (sp.diags(m) + sigma * (K.T @ sp.diags(1.0 / np.asarray(m)) @ K)).tocsc()
    H = 0.5 * (H + H.T)
    if N <= dense_below:
        th, V = np.linalg.eigh(H.toarray())
        return th[:k].copy(), np.asfortranarray(V[:, :k])
    scale = float(np.mean(m))  # keep the shift-invert factorisation well scaled
    th, V = spla.eigsh((H / scale).tocsc(), k=k, sigma=0.0, which="LM", tol=1e-12)
    order = np.argsort(th)
    return th[order] * scale, np.asfortranarray(V[:, order])


def sine_reference(dims, k):
    """Analytical Cartesian spatial reference (NEXT-1 of SURVEY.md 8(f)): section 2.2.3, eq. (15),
    restated for the cell-centred grids of workloads/ (the paper's grid is node-centred; pin P7 fixes the
    cell-centred form against the assembled operator).

    For axis a with n_a cells, the 1-D factors and Laplacian eigenvalues (h_a = 1/n_a) are
        v_q(j) = sqrt(2/n_a) sin(pi q (j - 1/2)/n_a)   (sqrt(1/n_a) for q = n_a),     j, q = 1..n_a
        mu_q   = 4 n_a^2 sin^2(pi q / (2 n_a)).
    A product phi = v_{q_1} (x) ... (x) v_{q_d} (x fastest) has Laplacian eigenvalue mu = sum_a mu_{q_a}.  "We retain
    the r lowest products.  Lexicographic ordering fixes the choice within repeated eigenvalues":
    sorted by (mu, q_1, ..., q_d), where mu is summed over the per-axis terms in ascending order of the terms so that
    permuted index tuples tie exactly (reading A18).

    Returns (modes, mu, W): modes int (k, d), mu (k,), W (N, k) column-major with orthonormal columns."""
    dims = [int(n) for n in dims]
    d = len(dims)
    N = int(np.prod(dims))
    if not (1 <= k <= N):
        raise ValueError("k out of range")
    terms = [4.0 * n * n * np.sin(np.pi * np.arange(1, min(n, k) + 1) / (2.0 * n)) ** 2 for n in dims]
    cand = []
    for q in itertools.product(*[range(1, len(t) + 1) for t in terms]):  # q = (q_1, ..., q_d), q_1 = x index
        parts = sorted(terms[a][q[a] - 1] for a in range(d))
        mu = 0.0
        for p in parts:
            mu += p
        cand.append((mu, q))
    cand.sort()
    cand = cand[:k]
    modes = np.array([q for _, q in cand], dtype=np.int32).reshape(k, d)
    mu = np.array([m for m, _ in cand])
    W = np.empty((N, k), order="F")
    for c in range(k):
        col = np.ones(1)
        for a in range(d):  # x fastest: kron(v_{q_d}, ..., v_{q_1})
            n, q = dims[a], int(modes[c, a])
            j = np.arange(1, n + 1)
            v = np.sqrt((1.0 if q == n else 2.0) / n) * np.sin(np.pi * q * (j - 0.5) / n)
            col = np.kron(v, col)
        W[:, c] = col
    return modes, mu, W


def temporal_sign(q):
    """Fixed sign of a temporal eigenvector: the component of largest magnitude (lowest index on ties) is positive."""
    j = int(np.argmax(np.abs(q)))
    return q if q[j] > 0 else -q


def spacetime_reference(dims, nt, dt, k, cover=None):
    """Mode-dependent temporal reference (NEXT-2 of SURVEY.md 8(f)): section 2.2.4, eq. (16)-(17),
    for the backward-Euler all-at-once operator of workloads/ (K_st = I (x) K_s + L (x) M_s, L lower bidiagonal with
    1/dt and -1/dt, capacity c_0 = 1, W_t = I).

    Homogeneous reference operator: A_0 = I (x) L_s + L (x) I with L_s the constant-coefficient Dirichlet Laplacian
    (eq. (16)); for a spatial sine mode phi_i with Laplacian eigenvalue mu_i (sine_reference), eq. (17) reads
        H_i = W_t + alpha (mu_i I + L)^T W_t (mu_i I + L),   H_i q_{i,j} = nu_{i,j} q_{i,j},
    and q_{i,j} (x) phi_i is an eigenvector of eq. (16).  H_i and S_i = (mu_i I + L)^T (mu_i I + L) share eigenvectors
    and nu = h^d (1 + alpha s) is increasing in s, so candidates are ordered by s (no alpha needed).  "The
    construction considers the first min(r, N_s) spatial modes ... We order the candidate pairs by nu and retain a
    total space-time rank r.  A fixed ordering resolves repeated eigenvalues": sorted by
    (s, i, j), i the position of the spatial mode in sine_reference's order, j the index of s within S_i ascending.

    cover = S (k is then ignored and set to S nt): complete temporal coverage, "The timed Cartesian
    trajectories keep all temporal factors of S spatial modes (Table 1), which pairs each retained mode with every time
    level": every pair (i, j) with i < S, in the same (s, i, j) order.

    Layout id = space + N_s * t: column = kron(q, phi).  Returns (pairs, s, W): pairs int (k, d + 1) = (q_1..q_d, j),
    s (k,), W (N_s nt, k) column-major, orthonormal columns."""
    dims = [int(n) for n in dims]
    Ns = int(np.prod(dims))
    if cover is not None:
        rs = int(cover)
        k = rs * nt
    else:
        rs = min(k, Ns)
    modes, mu, Phi = sine_reference(dims, rs)
    L = (np.eye(nt) - np.eye(nt, k=-1)) / dt
    cand = []
    Q = []
    for i in range(rs):
        B = mu[i] * np.eye(nt) + L
        s, V = np.linalg.eigh(B.T @ B)
        Q.append(V)
        for j in range(nt):
            cand.append((s[j], i, j))
    cand.sort()
    cand = cand[:k]
    d = len(dims)
    pairs = np.zeros((k, d + 1), dtype=np.int32)
    svals = np.zeros(k)
    W = np.empty((Ns * nt, k), order="F")
    for c, (s, i, j) in enumerate(cand):
        pairs[c, :d] = modes[i]
        pairs[c, d] = j
        svals[c] = s
        W[:, c] = np.kron(temporal_sign(Q[i][:, j]), Phi[:, i])
    return pairs, svals, W


def reference_eigs_scaled(rowptr, colidx, val, m, sigma, k, dense_below: int = 1500):
    """Jacobi-scaled reference (NEXT-3 of SURVEY.md 8(f)): the k lowest pairs of the generalized problem
    H w = mu D w, D = diag(H) -- the paper's "M_c phi_j = mu_j D_c phi_j supplies low modes in Jacobi-scaled
    coordinates", each column then "normalized in the Euclidean norm", here on the fine operator (A13).

    Returns (mu, W): mu ascending, W (N x k, column-major) with unit columns (not orthogonal: they are D-orthogonal
    before the normalisation).  A library eigensolver on the assembled matrices."""
    import scipy.linalg as sla
    import scipy.sparse as sp
    import scipy.sparse.linalg as spla

    N = len(m)
    K = sp.csr_matrix((val, colidx, rowptr), shape=(N, N))
    H = (sp.diags(m) + sigma * (K.T @ sp.diags(1.0 / np.asarray(m)) @ K)).tocsc()
    H = 0.5 * (H + H.T)
    d = H.diagonal()
    if N <= dense_below:
        mu, V = sla.eigh(H.toarray(), np.diag(d))
        mu, V = mu[:k], V[:, :k]
    else:
        s = 1.0 / np.sqrt(d)
        Hs = (sp.diags(s) @ H @ sp.diags(s)).tocsc()
        mu, Vs = spla.eigsh(Hs, k=k, sigma=0.0, which="LM", tol=1e-12)
        order = np.argsort(mu)
        mu, V = mu[order], s[:, None] * Vs[:, order]
    V = V / np.linalg.norm(V, axis=0)
    return mu.copy(), np.asfortranarray(V)


def prolong_p1(Vc, dims_c, dims_f):
    """P1 prolongation of coarse vectors to the fine grid (NEXT-1(ii) of SURVEY.md 8(f)): "P1 prolongation maps these
    vectors to the full fine mesh" (section 2.2.2), restated for the cell-centred Cartesian grids of
    workloads/ (reading A20): the continuous d-linear interpolant of the coarse cell-centre values, extended
    by the homogeneous Dirichlet value 0 on the boundary of the unit box, evaluated at the fine cell centres.

    Per axis with n_c coarse and n_f fine cells the interpolation nodes are xi_0 = 0, xi_j = (j - 1/2)/n_c (j = 1..n_c),
    xi_{n_c+1} = 1 with nodal values (0, v_1, ..., v_{n_c}, 0); the fine centre x_i = (i - 1/2)/n_f lies in one interval
    [xi_j, xi_{j+1}] and takes (1 - t) v_j + t v_{j+1}, t = (x_i - xi_j)/(xi_{j+1} - xi_j).  In d dimensions the value at
    a fine cell is the sum over the 2^d corners of the enclosing box of the product of the per-axis weights times the
    corner value (x fastest ordering on both grids).  No normalisation here.

    Vc: (N_c, k).  Returns (N_f, k) column-major.  Plain loops: small cases only."""
    dims_c = [int(n) for n in dims_c]
    dims_f = [int(n) for n in dims_f]
    d = len(dims_c)
    assert d == len(dims_f) and 1 <= d <= 3
    Vc = np.asarray(Vc, dtype=np.float64)
    if Vc.ndim == 1:
        Vc = Vc[:, None]
    Nc, Nf = int(np.prod(dims_c)), int(np.prod(dims_f))
    assert Vc.shape[0] == Nc
    k = Vc.shape[1]
    # per axis: for each fine index the two node numbers (0 and n_c + 1 are the boundary nodes) and the weight t
    axis = []
    for a in range(d):
        nc, nf = dims_c[a], dims_f[a]
        xi = np.concatenate(([0.0], (np.arange(1, nc + 1) - 0.5) / nc, [1.0]))
        ent = []
        for i in range(1, nf + 1):
            x = (i - 0.5) / nf
            j = 0
            while j + 1 <= nc and xi[j + 1] <= x:  # last node not to the right of x
                j += 1
            t = (x - xi[j]) / (xi[j + 1] - xi[j])
            ent.append((j, t))
        axis.append(ent)
    strides_c = [int(np.prod(dims_c[:a])) for a in range(d)]
    out = np.zeros((Nf, k), order="F")
    for fi, idx in enumerate(itertools.product(*[range(n) for n in reversed(dims_f)])):
        idx = idx[::-1]  # (i_x, i_y, i_z) with x fastest in fi
        acc = np.zeros(k)
        for corner in itertools.product((0, 1), repeat=d):
            wgt, cid, inside = 1.0, 0, True
            for a in range(d):
                j, t = axis[a][idx[a]]
                node = j + corner[a]
                wgt *= t if corner[a] else (1.0 - t)
                if node == 0 or node == dims_c[a] + 1:
                    inside = False  # boundary node: value 0
                else:
                    cid += (node - 1) * strides_c[a]
            if inside:
                acc += wgt * Vc[cid]
        out[fi] = acc
    return out


def prolonged_reference(coarse, dims_c, dims_f, k):
    """The paper's coarse-mesh reference: the k lowest pairs of the coarse generalized problem
    H_c phi = mu D_c phi (`reference_eigs_scaled` on the coarse operator `coarse` = (rowptr, colidx, val, m, sigma)),
    P1-prolonged to the fine grid, "each column is normalized in the Euclidean norm".
    Returns (mu, Wc, W): Wc the coarse vectors (unit columns), W (N_f, k) column-major with unit columns."""
    mu, Wc = reference_eigs_scaled(*coarse, k)
    W = prolong_p1(Wc, dims_c, dims_f)
    W = np.asfortranarray(W / np.linalg.norm(W, axis=0))
    return mu, Wc, W


def transient_reference(Phi, st, nt, k):
    """Transient variant of the coarse-mesh reference, eq. (14) (section 2.2.2): every spatial
    vector phi_i (column of Phi, N_s x r_s: "each prolonged vector") defines the small temporal matrices
        H_i = (I (x) phi_i)^T H (I (x) phi_i),   D_i = (I (x) phi_i)^T diag(H) (I (x) phi_i),   H_i q = nu D_i q,
    with H the all-at-once reduced Hessian `st` = (rowptr, colidx, val, m, sigma) of N_s nt DOFs in the layout
    id = space + N_s * t (so I (x) phi_i has the nt columns e_t (x) phi_i).  "The construction selects the requested
    total rank from these spatial-temporal candidates" (:182): reading A21 of DESIGN.md -- all r_s nt pairs ordered
    by (nu, i, j), j the index of nu within its own problem ascending; column = kron(q, phi_i) with the sign of
    `temporal_sign`, normalised in the Euclidean norm like the steady columns (:176).

    Written as the definition: H assembled by the library's sparse products, the Kronecker factor formed explicitly,
    a library generalized symmetric eigensolver per i.  Returns (pairs, nu, W): pairs int (k, 2) = (i, j), nu (k,),
    W (N_s nt, k) column-major with unit columns."""
    import scipy.linalg as sla
    import scipy.sparse as sp

    rowptr, colidx, val, m, sigma = st
    N = len(m)
    Phi = np.asarray(Phi, dtype=np.float64)
    Ns, rs = Phi.shape
    if Ns * nt != N:
        raise ValueError("Phi has %d rows, the operator %d = N_s * %d DOFs expected" % (Ns, N, nt))
    if k > rs * nt:
        raise ValueError("rank %d exceeds the %d candidates" % (k, rs * nt))
    K = sp.csr_matrix((val, colidx, rowptr), shape=(N, N))
    H = (sp.diags(m) + sigma * (K.T @ sp.diags(1.0 / np.asarray(m)) @ K)).tocsr()
    d = H.diagonal()
    cand = []
    Q = []
    for i in range(rs):
        V = np.kron(np.eye(nt), Phi[:, i:i + 1])          # I (x) phi_i : (N_s nt) x nt
        Hi = V.T @ (H @ V)
        Hi = 0.5 * (Hi + Hi.T)
        Di = V.T @ (d[:, None] * V)
        nu, Qi = sla.eigh(Hi, Di)
        Q.append(Qi)
        for j in range(nt):
            cand.append((nu[j], i, j))
    cand.sort()
    cand = cand[:k]
    pairs = np.zeros((k, 2), dtype=np.int32)
    nus = np.zeros(k)
    W = np.empty((N, k), order="F")
    for c, (nu, i, j) in enumerate(cand):
        pairs[c] = (i, j)
        nus[c] = nu
        col = np.kron(temporal_sign(Q[i][:, j]), Phi[:, i])
        W[:, c] = col / np.linalg.norm(col)
    return pairs, nus, W


def deflated_spectrum(orc: "Oracle", idx, Zt, jacobi: bool = True):
    """Jacobi-scaled diagnostic of the paper (NEXT-3 of SURVEY.md 8(f)): eq. (23).  "For
    Jacobi-preconditioned CG, the relevant matrix is B^ = D^{-1/2} B D^{-1/2} and the relevant coarse space is
    range(D^{1/2} Z) ... We measure the nonzero spectrum of
        B^ - D^{-1/2} B Z (Z^T B Z)^{-1} Z^T B D^{-1/2}
    on the small replay systems."  Written out densely: B = H_II from n operator applies on unit vectors, D = diag(B),
    Z, BZ, E = the factors of the coarse space the oracle builds from the restricted candidate basis Zt (QR + SVD,
    threshold 1e-12, cond(E) guard), the symmetric n x n matrix above, a library eigensolver.  The
    matrix has exactly r = rank(Z) zero eigenvalues (it annihilates D^{1/2} Z); they are dropped.

    Returns (lam, r): the n - r nonzero eigenvalues ascending, and r.  The effective condition number that the
    deflated, Jacobi-preconditioned CG of Algorithm 1 sees is lam[-1] / lam[0].  jacobi = False: D = I.
    Small systems only (dense n x n)."""
    idx = np.ascontiguousarray(idx, dtype=np.int64)
    n = len(idx)
    B = np.empty((n, n))
    e = np.zeros(n)
    for j in range(n):
        e[j] = 1.0
        B[:, j] = orc.apply_B(idx, e)
        e[j] = 0.0
    B = 0.5 * (B + B.T)
    cs = orc.coarse(idx, Zt if Zt is not None else np.zeros((n, 0)))
    r = cs.rank
    A = B.copy()
    if r:
        Z, BZ, E = cs.factors()
        A -= BZ @ np.linalg.solve(E, BZ.T)
    if jacobi:
        s = 1.0 / np.sqrt(np.diag(B))
        A = A * s[:, None] * s[None, :]
    lam = np.linalg.eigvalsh(0.5 * (A + A.T))
    return lam[r:].copy(), r
