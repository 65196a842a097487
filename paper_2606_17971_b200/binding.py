"""ctypes binding of include/refdef.h -- argument marshalling only; every step runs in the CUDA library.

Arrays may be numpy arrays (host pointers) or torch CUDA tensors (device pointers); the library tells
them apart itself (cudaPointerGetAttributes).  Names mirror the C entry points.
"""
from __future__ import annotations

import ctypes as C
import os
from dataclasses import dataclass
from typing import Optional

import numpy as np

HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(HERE, "librefdef_b200.so")

JACOBI_CG, REFDEF, ZEROEXT = 0, 1, 2
INIT_PAPER, INIT_ALL_ACTIVE, INIT_ALL_INACTIVE, INIT_GIVEN = 0, 1, 2, 3
STATUS_NAMES = {0: "ok", -1: "einval", -2: "enomem", -3: "ecuda", -4: "enoref", -5: "enotspd", -6: "ecap",
                -7: "esteps", -8: "ecycle", -9: "eresid"}
SOFT = (-5, -6, -7, -8, -9)

EXPORTS = ["rd_default_options", "rd_create", "rd_destroy", "rd_last_error", "rd_kernel_launches", "rd_set_options",
           "rd_build_reference", "rd_build_reference_scaled", "rd_build_reference_lobpcg", "rd_reference_lobpcg_work", "rd_build_reference_sine", "rd_build_reference_spacetime", "rd_build_reference_spacetime_cover", "rd_reference_storage", "rd_build_reference_prolonged", "rd_build_reference_transient", "rd_reference_info", "rd_reference_work", "rd_probe_fp64_tensor_peak", "rd_set_reference", "rd_get_reference", "rd_solve_query", "rd_reset_sequence",
           "rd_apply_K", "rd_apply_KT", "rd_apply_H", "rd_apply_H_noalloc", "rd_diag_H", "rd_solve_inactive", "rd_coarse_setup", "rd_energy_fraction", "rd_kkt", "rd_pdas_update"]


NOALLOC_MAX_N = 1 << 20  # RD_NOALLOC_MAX_N of include/refdef.h


class RefDefError(RuntimeError):
    pass


class _Options(C.Structure):
    _fields_ = [("sigma_is_alpha", C.c_double), ("eps", C.c_double), ("eps_c", C.c_double), ("cg_cap", C.c_int32),
                ("pdas_cap", C.c_int32), ("replace_period", C.c_int32), ("jacobi", C.c_int32),
                ("c_is_diag", C.c_int32), ("init", C.c_int32), ("alg1_variant", C.c_int32)]


class _StepReport(C.Structure):
    _fields_ = [("n_inactive", C.c_int32), ("cg_iters", C.c_int32), ("rank_used", C.c_int32),
                ("coarse_fallback", C.c_int32), ("replacements", C.c_int32), ("status", C.c_int32),
                ("rel_resid_verified", C.c_double), ("cond_E", C.c_double), ("margin", C.c_double),
                ("active_hash", C.c_uint64), ("t_restrict", C.c_double), ("t_coarse", C.c_double),
                ("t_iter", C.c_double), ("t_update", C.c_double)]


class _QueryReport(C.Structure):
    _fields_ = [("n_steps", C.c_int32), ("status", C.c_int32), ("kkt", C.c_double * 5), ("t_total", C.c_double),
                ("t_reference_charged", C.c_double), ("total_cg_iters", C.c_int64), ("worst_inner_status", C.c_int32),
                ("n_inner_failed", C.c_int32), ("n_fallbacks", C.c_int32), ("reserved", C.c_int32)]


class _SolveReport(C.Structure):
    _fields_ = [("iters", C.c_int32), ("rank_used", C.c_int32), ("coarse_fallback", C.c_int32),
                ("replacements", C.c_int32), ("status", C.c_int32), ("rel_resid_verified", C.c_double),
                ("cond_E", C.c_double), ("t_iter_ms", C.c_double), ("bytes_per_iter", C.c_double),
                ("t_stage_us", C.c_double * 8), ("ritz_min", C.c_double), ("ritz_max", C.c_double), ("ritz_count", C.c_int32),
                ("live_slices_A", C.c_int32), ("live_slices_B", C.c_int32), ("reserved", C.c_int32)]


@dataclass
class Options:
    sigma_is_alpha: float = 1.0
    eps: float = 1e-8
    eps_c: float = 1e-8
    cg_cap: int = 500000
    pdas_cap: int = 100
    replace_period: int = 0
    jacobi: int = 1
    c_is_diag: int = 0
    init: int = INIT_PAPER
    alg1_variant: int = 0

    def c_struct(self) -> _Options:
        return _Options(self.sigma_is_alpha, self.eps, self.eps_c, self.cg_cap, self.pdas_cap, self.replace_period,
                        self.jacobi, self.c_is_diag, self.init, self.alg1_variant)


_lib = None


def load_library(path: Optional[str] = None):
    """dlopen the CUDA library; raises RefDefError if it has not been built (no fallback of any kind)."""
    global _lib
    if _lib is not None and path is None:
        return _lib
    path = path or LIB_PATH
    if not os.path.exists(path):
        raise RefDefError(f"{path} is missing: build it with `python -m paper_2606_17971_b200.build` "
                          "(nvcc, sm_100a); there is no CPU fallback")
    lib = C.CDLL(path)
    vp, i32, i64, dbl = C.c_void_p, C.c_int32, C.c_int64, C.c_double
    lib.rd_default_options.argtypes = [C.POINTER(_Options)]
    lib.rd_default_options.restype = None
    lib.rd_create.argtypes = [C.POINTER(vp), i64, vp, vp, vp, vp, dbl, C.POINTER(_Options), vp]
    lib.rd_destroy.argtypes = [vp]
    lib.rd_destroy.restype = None
    lib.rd_last_error.argtypes = [vp]
    lib.rd_last_error.restype = C.c_char_p
    lib.rd_kernel_launches.argtypes = [vp]
    lib.rd_kernel_launches.restype = i64
    lib.rd_set_options.argtypes = [vp, C.POINTER(_Options)]
    lib.rd_build_reference.argtypes = [vp, i32, dbl, i32, vp, vp, C.POINTER(i32)]
    lib.rd_build_reference_scaled.argtypes = [vp, i32, dbl, i32, vp, vp, C.POINTER(i32)]
    lib.rd_reference_lobpcg_work.argtypes = [vp, vp, vp, vp, vp]
    lib.rd_build_reference_lobpcg.argtypes = [vp, i32, dbl, i32, i32, vp, dbl, vp, vp, C.POINTER(i32)]
    lib.rd_build_reference_sine.argtypes = [vp, i32, i32, vp, vp, vp]
    lib.rd_build_reference_spacetime.argtypes = [vp, i32, i32, vp, i32, dbl, vp, vp]
    lib.rd_build_reference_spacetime_cover.argtypes = [vp, i32, i32, vp, i32, dbl, vp, vp]
    lib.rd_reference_storage.argtypes = [vp, C.POINTER(i32), C.POINTER(i64), C.POINTER(i64)]
    lib.rd_build_reference_prolonged.argtypes = [vp, i32, i32, vp, vp, vp, vp]
    lib.rd_build_reference_transient.argtypes = [vp, i32, i32, i32, vp, vp, vp]
    lib.rd_reference_info.argtypes = [vp, C.POINTER(i32), C.POINTER(i64), C.POINTER(dbl)]
    lib.rd_probe_fp64_tensor_peak.argtypes = [vp, C.POINTER(dbl)]
    lib.rd_reference_work.argtypes = [vp, C.POINTER(i64), C.POINTER(dbl), C.POINTER(dbl)]
    lib.rd_set_reference.argtypes = [vp, i32, vp]
    lib.rd_get_reference.argtypes = [vp, vp, C.POINTER(i32)]
    lib.rd_solve_query.argtypes = [vp, i32, vp, vp, vp, vp, vp, vp, C.POINTER(_StepReport), vp, C.POINTER(_QueryReport)]
    lib.rd_reset_sequence.argtypes = [vp]
    lib.rd_apply_K.argtypes = [vp, vp, vp]
    lib.rd_apply_KT.argtypes = [vp, vp, vp]
    lib.rd_apply_H.argtypes = [vp, vp, vp, vp]
    lib.rd_apply_H_noalloc.argtypes = [vp, vp, vp, vp]
    lib.rd_diag_H.argtypes = [vp, vp]
    lib.rd_solve_inactive.argtypes = [vp, i32, vp, vp, vp, C.POINTER(_SolveReport)]
    lib.rd_coarse_setup.argtypes = [vp, i32, vp, vp, vp, vp, C.POINTER(i32), C.POINTER(dbl), C.POINTER(i32)]
    lib.rd_energy_fraction.argtypes = [vp, i32, vp, vp, vp, C.POINTER(dbl), C.POINTER(dbl), C.POINTER(dbl)]
    lib.rd_kkt.argtypes = [vp, vp, vp, vp, vp, vp]
    lib.rd_pdas_update.argtypes = [vp, vp, vp, vp, vp, vp, vp, C.POINTER(i64), C.POINTER(i64), C.POINTER(dbl)]
    _lib = lib
    return lib


def exported_symbols(path: Optional[str] = None):
    """Names from EXPORTS that the built library really exports (a CPU-side check; no CUDA call is made)."""
    lib = C.CDLL(path or LIB_PATH)
    return [s for s in EXPORTS if hasattr(lib, s)]


def declared_in_header(path: Optional[str] = None):
    """Names of the functions include/refdef.h declares (parsed from the header text)."""
    import re

    path = path or os.path.join(os.path.dirname(HERE), "include", "refdef.h")
    text = re.sub(r"/\*.*?\*/", "", open(path).read(), flags=re.S)
    return sorted(set(re.findall(r"\b(rd_[a-z_A-Z0-9]+)\s*\(", text)))


def _ptr(a):
    """Raw pointer of a numpy array (host) or a torch tensor (host or device); None -> NULL."""
    if a is None:
        return None
    if isinstance(a, np.ndarray):
        if not a.flags["C_CONTIGUOUS"] and not a.flags["F_CONTIGUOUS"]:
            raise ValueError("array must be contiguous")
        return a.ctypes.data
    if hasattr(a, "data_ptr"):
        if not a.is_contiguous():
            raise ValueError("tensor must be contiguous")
        return a.data_ptr()
    raise TypeError(type(a))


def _np(a, dtype):
    return np.ascontiguousarray(a, dtype=dtype)


class RefDef:
    """One context = one operator (K, m, alpha) = one reference.  Mirrors rd_* one to one."""

    def __init__(self, rowptr, colidx, val, m, alpha, opt: Optional[Options] = None, stream: int = 0):
        self._lib = load_library()
        self._h = C.c_void_p()
        self.N = int(len(m))
        self.opt = opt or Options()
        o = self.opt.c_struct()
        rp, ci, va, mm = _np(rowptr, np.int64), _np(colidx, np.int32), _np(val, np.float64), _np(m, np.float64)
        st = self._lib.rd_create(C.byref(self._h), self.N, rp.ctypes.data, ci.ctypes.data, va.ctypes.data,
                                 mm.ctypes.data, float(alpha), C.byref(o), C.c_void_p(stream or None))
        if st != 0:
            msg = self._lib.rd_last_error(self._h).decode() if self._h else ""
            if self._h:
                self._lib.rd_destroy(self._h)
                self._h = C.c_void_p()
            raise RefDefError(f"rd_create: {STATUS_NAMES.get(st, st)} {msg}")
        self.k = 0

    @classmethod
    def from_workload(cls, w, opt: Optional[Options] = None, stream: int = 0):
        return cls(w.rowptr, w.colidx, w.val, w.m, w.alpha, opt, stream)

    def close(self):
        if getattr(self, "_h", None):
            self._lib.rd_destroy(self._h)
            self._h = C.c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def _check(self, st, what, soft_ok=False):
        if st == 0 or (soft_ok and st in SOFT):
            return st
        raise RefDefError(f"{what}: {STATUS_NAMES.get(st, st)} {self._lib.rd_last_error(self._h).decode()}")

    # ---- plumbing
    def kernel_launches(self) -> int:
        return int(self._lib.rd_kernel_launches(self._h))

    def set_options(self, opt: Options):
        o = opt.c_struct()
        self._check(self._lib.rd_set_options(self._h, C.byref(o)), "rd_set_options")
        self.opt = opt

    def reset_sequence(self):
        self._check(self._lib.rd_reset_sequence(self._h), "rd_reset_sequence")

    # ---- reference
    def build_reference(self, k, tol=1e-3, max_block_iters=200):
        """Returns (theta, relative residuals, sweeps, status); status -6 = not converged within the sweeps."""
        theta = np.zeros(k)
        resid = np.zeros(k)
        it = C.c_int32(0)
        st = self._check(self._lib.rd_build_reference(self._h, k, tol, max_block_iters, theta.ctypes.data,
                                                      resid.ctypes.data, C.byref(it)), "rd_build_reference", soft_ok=True)
        self.k = k
        return theta, resid, it.value, st

    def build_reference_scaled(self, k, tol=1e-3, max_block_iters=200):
        """Jacobi-scaled reference H w = mu D w.  Returns (mu, relative residuals, sweeps, status)."""
        mu = np.zeros(k)
        resid = np.zeros(k)
        it = C.c_int32(0)
        st = self._check(self._lib.rd_build_reference_scaled(self._h, k, tol, max_block_iters, mu.ctypes.data,
                                                             resid.ctypes.data, C.byref(it)), "rd_build_reference_scaled",
                         soft_ok=True)
        self.k = k
        return mu, resid, it.value, st

    def build_reference_lobpcg(self, k, dims, kappa_ref=1.0, tol=1e-3, max_iters=500):
        """k lowest eigenvectors of H by LOBPCG with the sine-transform preconditioner of the homogeneous grid operator.
        Returns (theta, relative residuals, iterations, status); status -6 = not converged within max_iters."""
        dims = np.ascontiguousarray(dims, dtype=np.int64)
        theta = np.zeros(k)
        resid = np.zeros(k)
        it = C.c_int32(0)
        st = self._check(self._lib.rd_build_reference_lobpcg(self._h, k, tol, max_iters, len(dims), dims.ctypes.data,
                                                             float(kappa_ref), theta.ctypes.data, resid.ctypes.data,
                                                             C.byref(it)), "rd_build_reference_lobpcg", soft_ok=True)
        self.k = k
        return theta, resid, it.value, st

    def build_reference_sine(self, k, dims):
        """Analytical Cartesian reference: dims = cells per axis, x first.  Returns (mu, modes)."""
        dims = np.ascontiguousarray(dims, dtype=np.int64)
        mu = np.zeros(k)
        modes = np.zeros((k, len(dims)), dtype=np.int32)
        self._check(self._lib.rd_build_reference_sine(self._h, k, len(dims), dims.ctypes.data, mu.ctypes.data,
                                                      modes.ctypes.data), "rd_build_reference_sine")
        self.k = k
        return mu, modes

    def build_reference_spacetime(self, k, dims, nt, dt):
        """Mode-dependent temporal reference.  Returns (s, pairs): pairs k x (d + 1) = (q_1..q_d, j)."""
        dims = np.ascontiguousarray(dims, dtype=np.int64)
        s = np.zeros(k)
        pairs = np.zeros((k, len(dims) + 1), dtype=np.int32)
        self._check(self._lib.rd_build_reference_spacetime(self._h, k, len(dims), dims.ctypes.data, nt, dt, s.ctypes.data,
                                                           pairs.ctypes.data), "rd_build_reference_spacetime")
        self.k = k
        return s, pairs

    def build_reference_spacetime_cover(self, S, dims, nt, dt):
        """Complete temporal coverage: all nt temporal factors of the first S spatial modes, k = S nt."""
        dims = np.ascontiguousarray(dims, dtype=np.int64)
        k = S * nt
        s = np.zeros(k)
        pairs = np.zeros((k, len(dims) + 1), dtype=np.int32)
        self._check(self._lib.rd_build_reference_spacetime_cover(self._h, S, len(dims), dims.ctypes.data, nt, dt, s.ctypes.data,
                                                                 pairs.ctypes.data), "rd_build_reference_spacetime_cover")
        self.k = k
        return s, pairs

    def reference_storage(self):
        """(kind, doubles stored, int32 stored): kind -1 none, 0 dense, 1 compact space-time factors."""
        kind, nv, ni = C.c_int32(0), C.c_int64(0), C.c_int64(0)
        self._check(self._lib.rd_reference_storage(self._h, C.byref(kind), C.byref(nv), C.byref(ni)), "rd_reference_storage")
        return kind.value, nv.value, ni.value

    def build_reference_prolonged(self, Wc, dims_c, dims_f):
        """Coarse-mesh reference: P1 prolongation of Wc (N_c x k numpy, or a column-major device tensor of
        shape (k, N_c)) from the grid dims_c to the grid dims_f, unit columns.  Returns the norms before normalisation."""
        dims_c = np.ascontiguousarray(dims_c, dtype=np.int64)
        dims_f = np.ascontiguousarray(dims_f, dtype=np.int64)
        if len(dims_c) != len(dims_f):
            raise ValueError("dims_c and dims_f differ in length")
        if isinstance(Wc, np.ndarray):
            Wc = np.asfortranarray(Wc, dtype=np.float64)
            nc, k = Wc.shape
        else:
            k, nc = Wc.shape
        if nc != int(np.prod(dims_c)):
            raise ValueError("Wc does not have prod(dims_c) rows")
        norms = np.zeros(k)
        self._check(self._lib.rd_build_reference_prolonged(self._h, k, len(dims_c), dims_c.ctypes.data, dims_f.ctypes.data,
                                                           _ptr(Wc), norms.ctypes.data), "rd_build_reference_prolonged")
        self.k = k
        return norms

    def build_reference_transient(self, k, Phi, nt):
        """Transient coarse-mesh reference, eq. (14): Phi = N_s x rs spatial vectors (numpy, or a
        column-major device tensor of shape (rs, N_s)).  Returns (pairs (k, 2) = (i, j), nu (k,))."""
        if isinstance(Phi, np.ndarray):
            Phi = np.asfortranarray(Phi, dtype=np.float64)
            ns, rs = Phi.shape
        else:
            rs, ns = Phi.shape
        if ns * nt != self.N:
            raise ValueError("Phi does not have N / nt rows")
        nu = np.zeros(k)
        pairs = np.zeros((k, 2), dtype=np.int32)
        self._check(self._lib.rd_build_reference_transient(self._h, k, rs, nt, _ptr(Phi), nu.ctypes.data, pairs.ctypes.data),
                    "rd_build_reference_transient")
        self.k = k
        return pairs, nu

    def reference_info(self):
        b, deg, ms = C.c_int32(0), C.c_int64(0), C.c_double(0)
        self._check(self._lib.rd_reference_info(self._h, C.byref(b), C.byref(deg), C.byref(ms)), "rd_reference_info")
        ca, fms, bpc = C.c_int64(0), C.c_double(0), C.c_double(0)
        self._check(self._lib.rd_reference_work(self._h, C.byref(ca), C.byref(fms), C.byref(bpc)), "rd_reference_work")
        d = dict(block=b.value, total_degree=deg.value, build_ms=ms.value)
        fl, lms, ha, ta = C.c_double(0), C.c_double(0), C.c_int64(0), C.c_int64(0)
        self._check(self._lib.rd_reference_lobpcg_work(self._h, C.byref(fl), C.byref(lms), C.byref(ha), C.byref(ta)),
                    "rd_reference_lobpcg_work")
        if fl.value > 0 and lms.value > 0:
            # S0 by LOBPCG: FP64 tensor-core flop of the whole iteration loop over its CUDA-event time
            d.update(lobpcg_iterations=deg.value, lobpcg_tensor_flop=fl.value, lobpcg_loop_ms=lms.value,
                     lobpcg_TFLOPs=fl.value / (lms.value * 1e-3) / 1e12, lobpcg_h_column_applies=ha.value,
                     lobpcg_t_column_applies=ta.value)
        if ca.value > 0 and fms.value > 0:
            # S0's Chebyshev filter: algorithmic bytes (3 nnz + 48 N per column and degree) over its CUDA-event time
            d.update(filter_column_applies=ca.value, filter_ms=fms.value, filter_bytes_per_column_apply=bpc.value,
                     filter_GBs=ca.value * bpc.value / (fms.value * 1e-3) / 1e9)
        return d

    def probe_fp64_tensor_peak(self):
        t = C.c_double(0)
        self._check(self._lib.rd_probe_fp64_tensor_peak(self._h, C.byref(t)), "rd_probe_fp64_tensor_peak")
        return t.value

    def set_reference(self, W):
        """W: N x k, numpy (any order; copied column-major) or a column-major device tensor of shape (k, N)."""
        if isinstance(W, np.ndarray):
            W = np.asfortranarray(W, dtype=np.float64)
            k = W.shape[1]
        else:
            k = W.shape[0]
        self._check(self._lib.rd_set_reference(self._h, k, _ptr(W)), "rd_set_reference")
        self.k = k

    def get_reference(self):
        k = C.c_int32(0)
        self._check(self._lib.rd_get_reference(self._h, None, C.byref(k)), "rd_get_reference")
        W = np.zeros((self.N, k.value), order="F")
        if k.value:
            self._check(self._lib.rd_get_reference(self._h, W.ctypes.data, C.byref(k)), "rd_get_reference")
        return W

    # ---- single steps
    def _apply(self, fn, v, out=None, *extra):
        if out is None:
            out = np.empty(self.N) if isinstance(v, np.ndarray) else v.new_empty(v.shape)
        self._check(fn(self._h, _ptr(v), *extra, _ptr(out)), fn.__name__)
        return out

    def apply_K(self, v, out=None):
        return self._apply(self._lib.rd_apply_K, v, out)

    def apply_KT(self, v, out=None):
        return self._apply(self._lib.rd_apply_KT, v, out)

    def apply_H(self, v, active=None, out=None):
        return self._apply(self._lib.rd_apply_H, v, out, _ptr(active))

    def apply_H_noalloc(self, v, active, out):
        """rd_apply_H_noalloc: device tensors only, `out` given by the caller, nothing allocated, NOT synchronised
        (N <= NOALLOC_MAX_N; the scratch is a static device array shared by every call on the device)."""
        self._check(self._lib.rd_apply_H_noalloc(self._h, _ptr(v), _ptr(active), _ptr(out)), "rd_apply_H_noalloc")
        return out

    def diag_H(self):
        d = np.empty(self.N)
        self._check(self._lib.rd_diag_H(self._h, d.ctypes.data), "rd_diag_H")
        return d

    def solve_inactive(self, method, active, b, x0):
        """Algorithm 1 on the inactive system of `active` (N bytes).  Returns (x, report dict)."""
        if isinstance(x0, np.ndarray):
            x = np.array(x0, dtype=np.float64, copy=True)
        else:
            x = x0.clone()
        rep = _SolveReport()
        self._check(self._lib.rd_solve_inactive(self._h, method, _ptr(active), _ptr(b), _ptr(x), C.byref(rep)),
                    "rd_solve_inactive", soft_ok=True)
        d = {f: getattr(rep, f) for f, _ in _SolveReport._fields_}
        d["t_stage_us"] = list(rep.t_stage_us)
        return x, d

    def coarse_setup(self, method, active):
        k = self.k
        G, EW, Cm = np.zeros((k, k), order="F"), np.zeros((k, k), order="F"), np.zeros((k, k), order="F")
        rank, fb, cond = C.c_int32(0), C.c_int32(0), C.c_double(0)
        self._check(self._lib.rd_coarse_setup(self._h, method, _ptr(active), G.ctypes.data, EW.ctypes.data,
                                              Cm.ctypes.data, C.byref(rank), C.byref(cond), C.byref(fb)), "rd_coarse_setup")
        return dict(G=G, EW=EW, C=Cm, rank=rank.value, cond_E=cond.value, fallback=fb.value)

    def energy_fraction(self, method, active, b, x_star):
        """eq. (24): chi = ||Qb||_B^2 / ||x_*||_B^2 on the inactive system of `active`.  Returns (chi, ||Qb||_B^2, ||x_*||_B^2)."""
        chi, qb, xs = C.c_double(0), C.c_double(0), C.c_double(0)
        self._check(self._lib.rd_energy_fraction(self._h, method, _ptr(active), _ptr(b), _ptr(x_star), C.byref(chi),
                                                 C.byref(qb), C.byref(xs)), "rd_energy_fraction")
        return chi.value, qb.value, xs.value

    def kkt(self, y_d, psi, y, lam):
        """The five measures of eq. (25) for any (y, lambda)."""
        out = (C.c_double * 5)()
        self._check(self._lib.rd_kkt(self._h, _ptr(y_d), _ptr(psi), _ptr(y), _ptr(lam), out), "rd_kkt")
        return np.array(list(out))

    def pdas_update(self, y_d, psi, active, y):
        """One multiplier / active-set update (eq. (7)-(8)): returns (lambda, active_new, changed, n_active_new, margin)."""
        host = isinstance(y, np.ndarray)
        lam = np.empty(self.N) if host else y.new_empty(self.N)
        if host:
            act_new = np.empty(self.N, dtype=np.uint8)
        else:
            import torch

            act_new = torch.empty(self.N, dtype=torch.uint8, device=y.device)
        ch, na, mg = C.c_int64(0), C.c_int64(0), C.c_double(0)
        self._check(self._lib.rd_pdas_update(self._h, _ptr(y_d), _ptr(psi), _ptr(active), _ptr(y), _ptr(lam), _ptr(act_new),
                                             C.byref(ch), C.byref(na), C.byref(mg)), "rd_pdas_update")
        return lam, act_new, ch.value, na.value, mg.value

    # ---- the query
    def solve_query(self, method, y_d, psi, J0=None, y=None, u=None, lam=None, want_sets=True):
        """PDAS query.  Host (numpy) or device (torch) y_d / psi; outputs allocated to match unless given."""
        N = self.N
        host = isinstance(y_d, np.ndarray)
        if y is None:
            y = np.empty(N) if host else y_d.new_empty(N)
        if u is None:
            u = np.empty(N) if host else y_d.new_empty(N)
        if lam is None:
            lam = np.empty(N) if host else y_d.new_empty(N)
        cap = self.opt.pdas_cap
        steps = (_StepReport * cap)()
        nbytes = (N + 7) // 8
        Jb = np.zeros((cap, nbytes), dtype=np.uint8) if want_sets else None
        rep = _QueryReport()
        st = self._lib.rd_solve_query(self._h, method, _ptr(y_d), _ptr(psi), _ptr(J0), _ptr(y), _ptr(u), _ptr(lam), steps,
                                      Jb.ctypes.data if want_sets else None, C.byref(rep))
        self._check(st, "rd_solve_query", soft_ok=True)
        ns = rep.n_steps
        step_list = [{f: getattr(steps[i], f) for f, _ in _StepReport._fields_} for i in range(ns)]
        return dict(status=st, n_steps=ns, kkt=[rep.kkt[i] for i in range(5)], y=y, u=u, lam=lam, steps=step_list,
                    J_bits=(Jb[:ns] if want_sets else None), hashes=[s["active_hash"] for s in step_list],
                    t_total_ms=rep.t_total, t_reference_ms=rep.t_reference_charged, total_cg_iters=rep.total_cg_iters,
                    worst_inner_status=rep.worst_inner_status, n_inner_failed=rep.n_inner_failed, n_fallbacks=rep.n_fallbacks)
