// cg.cuh -- Algorithm 1 of the paper: coarse-corrected, projected-direction,
// Jacobi-preconditioned CG on B = H_II, as ONE persistent cooperative kernel per solve.
//
//   S3  masked operator apply      stage_K / stage_KT            (operator.cuh)
//   S4  tall-skinny projections    c = (HW_I)^T (J r),  z = J r - W_I (C c)
//   S5  CG vector updates + dots   fused into the stages below
//
// All vectors are full-domain (length N) and identically zero on the active set J, so no index list is
// needed: B v = chi_I H (chi_I v).  One CTA of 1024 threads per SM owns a contiguous range of 32-row slices
// for the whole solve.  Grid-wide reductions are two-phase and deterministic: every CTA writes one partial
// per quantity, a grid barrier follows, every CTA then sums all partials in the same fixed order, so all
// CTAs take identical branches without any host round trip.
//
// Basis: Z spans range(W_I) without being orthogonalised: with C = T E^{-1} T^T (coarse.cuh, k x k),
// Q v = W_I C W_I^T v and P v = v - W_I C (H_II W_I)^T v are the operators of eq. (18)
// for the orthonormal basis Z = W_I T; (BZ)^T J r = T^T (HW_I)^T J r uses the cached product.
#pragma once
#include "operator.cuh"

namespace rd {

enum { RD_ENOTSPD_DEV = -5, RD_ECAP_DEV = -6, RD_ERESID_DEV = -9 };  // rd_status values (refdef.h)
enum { SL_BB = 0, SL_DOT = 1, SL_RR = 2, SL_RHO = 3, SL_NSCAL = 4, SL_NSLOT = SL_NSCAL + RD_MAX_K };

struct CgDevReport {
    int32_t iters, replacements, status, pad;
    double rel_resid_verified, bnorm, rr_last;
    double t_stage_us[8];  // CTA 0's time per phase (k_alg1_v3): A, bar, B, bar, small dense, C, bar, outside the loop
};

struct CgParams {
    int64_t N, ldw;
    int32_t kp;          // columns of Wm / HWm / C (k rounded up to a multiple of 8)
    int32_t use_coarse;  // 0: rank-zero execution = Jacobi-CG
    Ell K, KT;
    const double *m, *minv, *dinv;  // dinv = 1/diag(H) (Jacobi) or all ones
    double sigma;
    const uint8_t* act;  // 1 = active (J)
    const double* b;     // rhs, 0 on J
    double *x, *r, *p0, *p1, *z, *w, *t;
    const double *Wm, *HWm;  // the basis of eq. (18) and its cached product, N x kp column-major (ld = ldw): since round 2 the
                             // explicit Z = W_I T and H_II Z (coarse.cuh), so that C = E^{-1}; any full-rank basis with its C works
    const double* HWt;       // HWm tile-major: (i, j) at (i / 32) * 32 kp + 32 j + i % 32 (k_alg1_v3)
    const double* Wt;        // Wm (= Z) tile-major, same layout (k_alg1_v3: coarse corrections outside the loop)
    const int32_t *listA, *listB;  // S6 compaction: live 32-row slices of the current active set (pdas.cuh k_slice_lists)
    const int32_t* live_counts;    // [0] = |listA|, [1] = |listB|
    const double* C;         // kp x kp column-major, symmetric: the coarse solve in the coordinates of Wm
    const double* EW;        // Wm^T HWm, kp x kp column-major (k_alg1_v3: curvature in coefficient form)
    double eps, eps_c;
    int32_t cap, replace_period;
    double* partial;  // [2][SL_NSLOT][gridDim.x]
    GridBarrier* bar;
    double2* coef;        // NULL or coef_cap entries: (a_it, beta_it) of every loop iteration (CG-Lanczos coefficients; eq. (23) diagnostic)
    int32_t coef_cap;
    int32_t hw_res_tiles; // tiles per CTA of the H_II W_I stream requested with L2 evict_last (kept resident)
    CgDevReport* rep;
};

struct CgShared {
    double C[RD_MAX_K * RD_MAX_K];
    double s[RD_CG_THREADS];
    double c[RD_MAX_K];
    double mu[RD_MAX_K];
    double scal[SL_NSCAL];
    double red[32];
};

struct CgCta {
    const CgParams& P;
    CgShared& sh;
    int64_t s0, s1, row0, row1;
    unsigned int nbar;  // barriers passed so far (same on every CTA)
    int G;

    __device__ CgCta(const CgParams& p, CgShared& s) : P(p), sh(s), nbar(0)
    {
        G = gridDim.x;
        const int64_t per = (P.K.nslices + G - 1) / G;
        s0 = min((int64_t)blockIdx.x * per, P.K.nslices);
        s1 = min(s0 + per, P.K.nslices);
        row0 = s0 * RD_SLICE;
        row1 = min(P.N, s1 * RD_SLICE);
    }
    __device__ double* slot(int sl) const { return P.partial + ((size_t)(nbar & 1u) * SL_NSLOT + sl) * G; }
    __device__ void put(int sl, double v) const
    {
        if (threadIdx.x == 0) slot(sl)[blockIdx.x] = v;
    }

    // Grid barrier, then every CTA reduces the partials of the set written before it: the four scalars
    // always, the kp projection coefficients when want_c.  Fixed order => identical on all CTAs and runs.
    __device__ void sync_fetch(bool want_c)
    {
        const double* base = P.partial + (size_t)(nbar & 1u) * SL_NSLOT * G;
        grid_barrier(P.bar, G);
        nbar++;
        const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5, nw = blockDim.x >> 5;
        const int nsl = want_c ? SL_NSCAL + P.kp : SL_NSCAL;
        for (int sl = warp; sl < nsl; sl += nw) {
            const double* q = base + (size_t)sl * G;
            double a = 0.0;
            for (int i = lane; i < G; i += 32) a += __ldcg(q + i);
            a = warp_sum(a);
            if (lane == 0) {
                if (sl < SL_NSCAL) sh.scal[sl] = a; else sh.c[sl - SL_NSCAL] = a;
            }
        }
        __syncthreads();
    }

    // mu = C c  (the r x r coarse solve of eq. (18) in W_I coordinates)
    __device__ void coarse_solve()
    {
        const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5, nw = blockDim.x >> 5;
        const int kp = P.kp;
        for (int i = warp; i < kp; i += nw) {
            double a = 0.0;
            for (int j = lane; j < kp; j += 32) a = fma(sh.C[i + j * kp], sh.c[j], a);
            a = warp_sum(a);
            if (lane == 0) sh.mu[i] = a;
        }
        __syncthreads();
    }

    // S5 + first half of S4.  RECOMPUTE = false: x += a p, r -= a w (Alg. 1 line 10).  true: r = b - w
    // (lines 3, 12, 16).  Then rr = ||r||^2 and, with a coarse space, c = M^T s with s = dinv.*r (M = HW_I,
    // for P) or s = r (M = W_I, for Q).
    template <bool RECOMPUTE>
    __device__ void stage_update(double a, const double* p, const double* M, bool scale)
    {
        const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5, nw = blockDim.x >> 5;
        const int kp = (P.use_coarse && M) ? P.kp : 0;  // M == NULL: no projection wanted (Verify)
        double rr = 0.0;
        double acc[(RD_MAX_K + 31) / 32];
#pragma unroll
        for (int q = 0; q < (RD_MAX_K + 31) / 32; ++q) acc[q] = 0.0;
        __syncthreads();  // w of this CTA's rows was written by other threads of the CTA
        for (int64_t tile = row0; tile < row1; tile += blockDim.x) {
            const int64_t i = tile + threadIdx.x;
            double s = 0.0;
            if (i < row1) {
                double ri;
                if (RECOMPUTE) {
                    ri = P.b[i] - P.w[i];
                } else {
                    P.x[i] = fma(a, p[i], P.x[i]);
                    ri = fma(-a, P.w[i], P.r[i]);
                }
                P.r[i] = ri;
                rr = fma(ri, ri, rr);
                s = scale ? ri * ldg_f64(P.dinv + i) : ri;
            }
            if (kp) {
                sh.s[threadIdx.x] = s;
                __syncthreads();
                const int64_t rows_here = min((int64_t)blockDim.x, row1 - tile);
                const int ngroups = (int)((rows_here + 31) >> 5);
#pragma unroll
                for (int q = 0; q < (RD_MAX_K + 31) / 32; ++q) {
                    const int j = warp + q * nw;
                    if (j < kp) {
                        const double* col = M + (size_t)j * P.ldw + tile + lane;
                        double a0 = 0.0, a1 = 0.0, a2 = 0.0, a3 = 0.0;
                        int g = 0;
                        for (; g + 4 <= ngroups; g += 4) {  // full groups except possibly the last one
                            const bool last_ok = (int64_t)(g + 3) * 32 + lane < rows_here;
                            double m0 = ldg_f64(col + (g + 0) * 32), m1 = ldg_f64(col + (g + 1) * 32);
                            double m2 = ldg_f64(col + (g + 2) * 32);
                            double m3 = last_ok ? ldg_f64(col + (g + 3) * 32) : 0.0;
                            a0 = fma(m0, sh.s[(g + 0) * 32 + lane], a0);
                            a1 = fma(m1, sh.s[(g + 1) * 32 + lane], a1);
                            a2 = fma(m2, sh.s[(g + 2) * 32 + lane], a2);
                            a3 = fma(m3, sh.s[(g + 3) * 32 + lane], a3);
                        }
                        for (; g < ngroups; ++g)
                            if ((int64_t)g * 32 + lane < rows_here) a0 = fma(ldg_f64(col + g * 32), sh.s[g * 32 + lane], a0);
                        acc[q] += (a0 + a1) + (a2 + a3);
                    }
                }
                __syncthreads();
            }
        }
        if (kp) {
#pragma unroll
            for (int q = 0; q < (RD_MAX_K + 31) / 32; ++q) {
                const int j = warp + q * nw;
                if (j < kp) {
                    const double v = warp_sum(acc[q]);
                    if (lane == 0) slot(SL_NSCAL + j)[blockIdx.x] = v;
                }
            }
        }
        rr = block_sum(rr, sh.red);
        put(SL_RR, rr);
    }

    // Second half of S4: z = dinv.*r - W_I mu,  rho = r^T z   (Alg. 1 lines 7, 20, 22)
    __device__ void stage_project()
    {
        const int kp = P.use_coarse ? P.kp : 0;
        double rho = 0.0;
        for (int64_t i = row0 + threadIdx.x; i < row1; i += blockDim.x) {
            const double ri = P.r[i];
            double zi = ri * ldg_f64(P.dinv + i);
            if (kp) {
                const double* wrow = P.Wm + i;
                double a0 = 0.0, a1 = 0.0, a2 = 0.0, a3 = 0.0;
                for (int j = 0; j < kp; j += 8) {  // kp is a multiple of 8
                    double w0 = ldg_f64(wrow + (size_t)(j + 0) * P.ldw), w1 = ldg_f64(wrow + (size_t)(j + 1) * P.ldw);
                    double w2 = ldg_f64(wrow + (size_t)(j + 2) * P.ldw), w3 = ldg_f64(wrow + (size_t)(j + 3) * P.ldw);
                    double w4 = ldg_f64(wrow + (size_t)(j + 4) * P.ldw), w5 = ldg_f64(wrow + (size_t)(j + 5) * P.ldw);
                    double w6 = ldg_f64(wrow + (size_t)(j + 6) * P.ldw), w7 = ldg_f64(wrow + (size_t)(j + 7) * P.ldw);
                    a0 = fma(w0, sh.mu[j + 0], a0); a1 = fma(w1, sh.mu[j + 1], a1);
                    a2 = fma(w2, sh.mu[j + 2], a2); a3 = fma(w3, sh.mu[j + 3], a3);
                    a0 = fma(w4, sh.mu[j + 4], a0); a1 = fma(w5, sh.mu[j + 5], a1);
                    a2 = fma(w6, sh.mu[j + 6], a2); a3 = fma(w7, sh.mu[j + 7], a3);
                }
                zi -= (a0 + a1) + (a2 + a3);
            }
            P.z[i] = zi;
            rho = fma(ri, zi, rho);
        }
        rho = block_sum(rho, sh.red);
        put(SL_RHO, rho);
    }

    // x += W_I mu   (coarse correction x + Q r, Alg. 1 lines 3 and 16)
    __device__ void stage_coarse_correct()
    {
        const int kp = P.kp;
        for (int64_t i = row0 + threadIdx.x; i < row1; i += blockDim.x) {
            const double* wrow = P.Wm + i;
            double a0 = 0.0, a1 = 0.0;
            for (int j = 0; j < kp; j += 2) {
                a0 = fma(ldg_f64(wrow + (size_t)j * P.ldw), sh.mu[j], a0);
                a1 = fma(ldg_f64(wrow + (size_t)(j + 1) * P.ldw), sh.mu[j + 1], a1);
            }
            P.x[i] += a0 + a1;
        }
    }

    // w = B v (both SpMVs with the barrier between them); returns nothing, v^T w goes to SL_DOT.
    __device__ void apply_B_plain(const double* v)
    {
        stage_K<false>(P.K, P.N, s0, s1, P.minv, v, nullptr, 0.0, nullptr, P.t);
        sync_fetch(false);
        double d = stage_KT(P.KT, P.N, s0, s1, P.m, P.sigma, P.act, v, P.t, P.w);
        d = block_sum(d, sh.red);
        put(SL_DOT, d);
    }
};

__global__ void __launch_bounds__(RD_CG_THREADS, 1) k_alg1(const CgParams P)
{
    __shared__ CgShared sh;
    CgCta cta(P, sh);
    const bool coarse = P.use_coarse != 0;
    if (coarse)
        for (int q = threadIdx.x; q < P.kp * P.kp; q += blockDim.x) sh.C[q] = P.C[q];

    // line 1: tau = eps_c ||b||_2
    {
        double bb = 0.0;
        for (int64_t i = cta.row0 + threadIdx.x; i < cta.row1; i += blockDim.x) bb = fma(P.b[i], P.b[i], bb);
        bb = block_sum(bb, sh.red);
        cta.put(SL_BB, bb);  // stays in set 0 until the first fetch: read right after the first barrier below
    }
    // BB is fetched at the first sync_fetch (set 0); keep it in a register afterwards.
    // line 3: x <- x0 + Q (b - B x0);  r <- b - B x
    // the first apply's barrier carries BB
    stage_K<false>(P.K, P.N, cta.s0, cta.s1, P.minv, P.x, nullptr, 0.0, nullptr, P.t);
    cta.sync_fetch(false);
    const double bnorm = sqrt(sh.scal[SL_BB]);
    const double tau = (bnorm > 0.0) ? P.eps_c * bnorm : P.eps_c;
    __syncthreads();  // everyone has read scal[BB] before a later fetch overwrites it
    {
        double d = stage_KT(P.KT, P.N, cta.s0, cta.s1, P.m, P.sigma, P.act, P.x, P.t, P.w);
        (void)d;
    }
    int status = RD_ECAP_DEV;
    int iters = 0, replacements = 0;
    bool done = false;
    double rho = 0.0, beta = 0.0;
    int cur = 0;  // p_old = cur ? p1 : p0

    if (coarse) {
        cta.stage_update<true>(0.0, nullptr, P.Wm, false);  // r = b - B x0, c = W_I^T r
        cta.sync_fetch(true);
        cta.coarse_solve();
        cta.stage_coarse_correct();  // x += W_I C W_I^T r
        cta.sync_fetch(false);
        cta.apply_B_plain(P.x);
    }
    cta.stage_update<true>(0.0, nullptr, P.HWm, true);  // r = b - B x, rr, c = (HW_I)^T J r
    cta.sync_fetch(coarse);
    // lines 4-6
    if (sqrt(sh.scal[SL_RR]) <= tau) { status = 0; done = true; }
    if (!done) {
        // line 7: z <- P J r; p <- z (beta = 0 in the fused update); rho <- r^T z
        if (coarse) cta.coarse_solve();
        cta.stage_project();
        cta.sync_fetch(false);
        rho = sh.scal[SL_RHO];
        beta = 0.0;
    }
    // line 8
    while (!done && iters < P.cap) {
        // line 23 (deferred) + line 9: p <- z + beta p ; w <- B p
        double* pold = cur ? P.p1 : P.p0;
        double* pnew = cur ? P.p0 : P.p1;
        stage_K<true>(P.K, P.N, cta.s0, cta.s1, P.minv, P.z, pold, beta, pnew, P.t);
        cur ^= 1;
        cta.sync_fetch(false);
        {
            double d = stage_KT(P.KT, P.N, cta.s0, cta.s1, P.m, P.sigma, P.act, pnew, P.t, P.w);
            d = block_sum(d, sh.red);
            cta.put(SL_DOT, d);
        }
        cta.sync_fetch(false);
        iters++;
        const double pw = sh.scal[SL_DOT];
        if (!(pw > 0.0) || !(rho > 0.0)) { status = RD_ENOTSPD_DEV; break; }
        // line 10
        const double a = rho / pw;
        cta.stage_update<false>(a, pnew, P.HWm, true);
        cta.sync_fetch(coarse);
        // line 11
        const bool scheduled = P.replace_period > 0 && (iters % P.replace_period) == 0;
        if (sqrt(sh.scal[SL_RR]) <= tau || scheduled) {
            replacements++;
            // line 12: recompute r = b - B x
            cta.apply_B_plain(P.x);
            cta.stage_update<true>(0.0, nullptr, coarse ? P.Wm : P.HWm, !coarse);
            cta.sync_fetch(coarse);
            if (sqrt(sh.scal[SL_RR]) <= tau) { status = 0; break; }  // lines 13-15
            if (coarse) {
                // line 16: x <- x + Q r; r <- b - B x
                cta.coarse_solve();
                cta.stage_coarse_correct();
                cta.sync_fetch(false);
                cta.apply_B_plain(P.x);
                cta.stage_update<true>(0.0, nullptr, P.HWm, true);
                cta.sync_fetch(true);
                if (sqrt(sh.scal[SL_RR]) <= tau) { status = 0; break; }  // lines 17-19
                cta.coarse_solve();
            }
            // line 20: restart
            cta.stage_project();
            cta.sync_fetch(false);
            rho = sh.scal[SL_RHO];
            beta = 0.0;
        } else {
            // line 22
            if (coarse) cta.coarse_solve();
            cta.stage_project();
            cta.sync_fetch(false);
            const double rho_new = sh.scal[SL_RHO];
            // line 23 (the direction update itself is fused into the next stage_K)
            beta = rho_new / rho;
            rho = rho_new;
        }
    }
    // line 26: Verify(x, eps): ||b - B x||/||b|| from a fresh apply
    const double rr_last = sh.scal[SL_RR];
    __syncthreads();
    cta.apply_B_plain(P.x);
    cta.stage_update<true>(0.0, nullptr, nullptr, false);  // r = b - B x, rr (c partials are unused)
    cta.sync_fetch(false);
    if (blockIdx.x == 0 && threadIdx.x == 0) {
        const double rn = sqrt(sh.scal[SL_RR]);
        const double rel = (bnorm > 0.0) ? rn / bnorm : rn;
        if (status == 0 && !(rel <= P.eps)) status = RD_ERESID_DEV;
        P.rep->iters = iters;
        P.rep->replacements = replacements;
        P.rep->status = status;
        P.rep->rel_resid_verified = rel;
        P.rep->bnorm = bnorm;
        P.rep->rr_last = rr_last;
    }
}

}  // namespace rd
