// cg2.cuh -- Algorithm 1 with the projection carried in coefficient form: the default
// persistent kernel of the library.  Same method as cg.cuh (k_alg1, the literal two-pass recurrence, kept as
// rd_options.alg1_variant = 1), same results up to rounding, but ONE pass over the cached product HW_I per
// iteration instead of a pass over HW_I and a pass over W_I, and three grid barriers instead of four.
//
// Write the search direction and the iterate of Alg. 1 as   p = p~ - W_I nu,   x = x~ - W_I xi   with k-vectors
// nu, xi kept (replicated, bit-identical) in the shared memory of every CTA.  With z~ = J r (never projected):
//   line 22  z = P J r = z~ - W_I mu,  mu = C c,  c = (HW_I)^T z~                       (eq. (18))
//   line 23  p = z + beta p      <=>  p~ = z~ + beta p~,   nu = mu + beta nu
//   line  9  w = B p = w~ - HW_I nu  with w~ = B p~  (the two SpMVs act on p~ only)
//            p^T w = p~^T w~ - 2 nu^T g + nu^T E_W nu,   g = (HW_I)^T p~ = c + beta g,   E_W = W_I^T HW_I
//   line 10  x~ += a p~, xi += a nu;   r = r - a w~ + HW_I (a nu)
//   line 22  rho = r^T z = r^T z~ - s^T mu,   s = W_I^T r = s - a (g - E_W nu)   (zero in exact arithmetic,
//            Z^T(b - B x_c) = 0 and Z^T B P = 0; the recurrence carries its rounding-level drift)
// One pass over a 32-row tile of HW_I does both  q_i = sum_j HW_ij (a nu_j)  (needed for r_i) and
// c_j += HW_ij z~_i  (from the values still in registers).  x is made explicit (x = x~ - W_I xi, one pass over
// W_I) only where Alg. 1 recomputes the residual (lines 12, 16, Verify).
//
// Stages of one iteration (grid barrier after each):
//   A  p~ = z~ + beta p~ (fused into the gather),  t = M^{-1} K p~                        S3
//   B  w~ = chi_I (m.p~ + sigma K^T t),  p~^T w~                                           S3
//   C  x~, r, z~ updates, ||r||^2, r^T z~, c = (HW_I)^T z~   (one pass over HW_I)           S4 + S5
#pragma once
#include "cg.cuh"

namespace rd {

struct Cg2Shared {
    double C[RD_MAX_K * RD_MAX_K];
    double EW[RD_MAX_K * RD_MAX_K];
    double s[RD_CG_THREADS];              // transposition buffer of the two-phase update (outside the loop)
    double qpart[2][4][8][32];            // stage C: partial row dots, [buffer][warp group][column group][lane]
    double cpart[4][RD_MAX_K];            // stage C: c partials of the four warp groups
    double c[RD_MAX_K], mu[RD_MAX_K], nu[RD_MAX_K], g[RD_MAX_K], sv[RD_MAX_K], xi[RD_MAX_K], anu[RD_MAX_K], e[RD_MAX_K];
    double scal[SL_NSCAL];
    double small[4];
    double red[32];
};

__device__ __forceinline__ void named_bar_sync(int id, int nthreads)
{
    asm volatile("bar.sync %0, %1;" ::"r"(id), "r"(nthreads) : "memory");
}

template <class SH>
struct Cg2CtaT {
    const CgParams& P;
    SH& sh;
    int64_t s0, s1, row0, row1;
    unsigned int nbar;
    int G;

    __device__ Cg2CtaT(const CgParams& p, SH& s) : P(p), sh(s), nbar(0)
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
    // Grid barrier, then every CTA sums the partials written before it, in the same fixed order.
    __device__ void sync_fetch(bool want_scal, bool want_c)
    {
        const double* base = P.partial + (size_t)(nbar & 1u) * SL_NSLOT * G;
        grid_barrier(P.bar, G);
        nbar++;
        if (!want_scal) return;
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
    // out = M v  (kp x kp column-major in shared memory), one warp per row
    __device__ void small_matvec(const double* M, const double* v, double* out)
    {
        const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5, nw = blockDim.x >> 5;
        const int kp = P.kp;
        for (int i = warp; i < kp; i += nw) {
            double a = 0.0;
            for (int j = lane; j < kp; j += 32) a = fma(M[i + j * kp], v[j], a);
            a = warp_sum(a);
            if (lane == 0) out[i] = a;
        }
        __syncthreads();
    }
    // sh.small[slot] = u^T v  (every thread reads it after the call)
    __device__ void small_dot2(const double* u0, const double* v0, const double* u1, const double* v1)
    {
        if (threadIdx.x < 32) {
            double a = 0.0, b = 0.0;
            for (int j = threadIdx.x; j < P.kp; j += 32) { a = fma(u0[j], v0[j], a); b = fma(u1[j], v1[j], b); }
            a = warp_sum(a); b = warp_sum(b);
            if (threadIdx.x == 0) { sh.small[0] = a; sh.small[1] = b; }
        }
        __syncthreads();
    }

    // Outside the loop (Alg. 1 lines 3, 12, 16, Verify): r = b - w, z~ = J r, ||r||^2, r^T z~ and, with a coarse
    // space and M != NULL, c = M^T s with s = z~ (M = HW_I) or s = r (M = W_I, scale = false).
    __device__ void stage_recompute(const double* M, bool scale)
    {
        const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5, nw = blockDim.x >> 5;
        const int kp = (P.use_coarse && M) ? P.kp : 0;
        double rr = 0.0, rho = 0.0;
        double acc[(RD_MAX_K + 31) / 32];
#pragma unroll
        for (int q = 0; q < (RD_MAX_K + 31) / 32; ++q) acc[q] = 0.0;
        __syncthreads();  // w of this CTA's rows was written by other threads of the CTA
        for (int64_t tile = row0; tile < row1; tile += blockDim.x) {
            const int64_t i = tile + threadIdx.x;
            double s = 0.0;
            if (i < row1) {
                const double ri = P.b[i] - P.w[i];
                const double zi = ri * ldg_f64(P.dinv + i);
                P.r[i] = ri;
                P.z[i] = zi;
                rr = fma(ri, ri, rr);
                rho = fma(ri, zi, rho);
                s = scale ? zi : ri;
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
                        double a0 = 0.0, a1 = 0.0;
                        for (int g = 0; g < ngroups; ++g)
                            if ((int64_t)g * 32 + lane < rows_here) {
                                if (g & 1) a1 = fma(ldg_f64(col + g * 32), sh.s[g * 32 + lane], a1);
                                else a0 = fma(ldg_f64(col + g * 32), sh.s[g * 32 + lane], a0);
                            }
                        acc[q] += a0 + a1;
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
        rho = block_sum(rho, sh.red);
        put(SL_RR, rr);
        put(SL_RHO, rho);
    }

    // Stage C without a coarse space (rank-zero execution = Jacobi-CG)
    __device__ void stage_update_plain(double a, const double* p)
    {
        double rr = 0.0, rho = 0.0;
        __syncthreads();
        for (int64_t i = row0 + threadIdx.x; i < row1; i += blockDim.x) {
            const double rn = fma(-a, P.w[i], P.r[i]);
            const double zn = rn * ldg_f64(P.dinv + i);
            P.x[i] = fma(a, p[i], P.x[i]);
            P.r[i] = rn;
            P.z[i] = zn;
            rr = fma(rn, rn, rr);
            rho = fma(rn, zn, rho);
        }
        rr = block_sum(rr, sh.red);
        rho = block_sum(rho, sh.red);
        put(SL_RR, rr);
        put(SL_RHO, rho);
    }

    // Stage C with a coarse space: one pass over HW_I.  Four groups of eight warps; a group owns 32-row tiles
    // (lane = row), warp cg of the group owns the kp/8 columns [cg kp/8, (cg+1) kp/8).  Per tile: partial row dots
    // q_i of HW_I (a nu) exchanged through shared memory (one named barrier per tile, double buffered), then
    // r_i, x~_i, z~_i and the column dots c_j += HW_ij z~_i from the HW values still in registers.
    __device__ void stage_update_coarse(double a, const double* p)
    {
        const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
        const int gi = warp >> 3, cg = warp & 7;
        const int cpw = P.kp >> 3;  // 1..8 columns per warp
        const double* HWc = P.HWm + (size_t)(cg * cpw) * P.ldw;
        const double* anu = sh.anu + cg * cpw;  // warp-uniform shared-memory reads (entries past kp are zero)
        double acc[8];
#pragma unroll
        for (int jj = 0; jj < 8; ++jj) acc[jj] = 0.0;
        double rr = 0.0, rho = 0.0;
        int buf = 0;
        __syncthreads();  // w~ of this CTA's rows was written by other threads of the CTA
        for (int64_t tile = row0 + 32 * gi; tile < row1; tile += 128, buf ^= 1) {
            const int64_t i = tile + lane;
            const bool in = i < row1;
            double hw[8];
#pragma unroll
            for (int jj = 0; jj < 8; ++jj) hw[jj] = (jj < cpw && in) ? ldg_f64(HWc + i + (size_t)jj * P.ldw) : 0.0;
            double ri = 0.0, wi = 0.0, pi = 0.0, xi = 0.0, di = 0.0;
            if (in) { ri = P.r[i]; wi = P.w[i]; di = ldg_f64(P.dinv + i); if (cg == 0) { pi = p[i]; xi = P.x[i]; } }
            double q0 = 0.0, q1 = 0.0;
#pragma unroll
            for (int jj = 0; jj < 8; jj += 2) { q0 = fma(hw[jj], anu[jj], q0); q1 = fma(hw[jj + 1], anu[jj + 1], q1); }
            sh.qpart[buf][gi][cg][lane] = q0 + q1;
            named_bar_sync(1 + gi, 256);
            double qs = 0.0;
#pragma unroll
            for (int c8 = 0; c8 < 8; ++c8) qs += sh.qpart[buf][gi][c8][lane];
            const double rn = fma(-a, wi, ri) + qs;
            const double zn = rn * di;
            if (cg == 0 && in) {
                P.r[i] = rn;
                P.x[i] = fma(a, pi, xi);
                P.z[i] = zn;
                rr = fma(rn, rn, rr);
                rho = fma(rn, zn, rho);
            }
#pragma unroll
            for (int jj = 0; jj < 8; ++jj) acc[jj] = fma(hw[jj], zn, acc[jj]);
        }
        // c: lanes -> warp, then the four groups through shared memory (fixed order)
#pragma unroll
        for (int jj = 0; jj < 8; ++jj) {
            const double v = warp_sum(acc[jj]);
            if (lane == 0 && jj < cpw) sh.cpart[gi][cg * cpw + jj] = v;
        }
        __syncthreads();
        if ((int)threadIdx.x < P.kp)
            slot(SL_NSCAL + threadIdx.x)[blockIdx.x] =
                (sh.cpart[0][threadIdx.x] + sh.cpart[1][threadIdx.x]) + (sh.cpart[2][threadIdx.x] + sh.cpart[3][threadIdx.x]);
        rr = block_sum(rr, sh.red);
        rho = block_sum(rho, sh.red);
        put(SL_RR, rr);
        put(SL_RHO, rho);
    }

    // x += sign * W_I v   (v = sh.mu: coarse correction x + Q r of lines 3 / 16;  v = sh.xi, sign = -1: x = x~ - W_I xi)
    __device__ void stage_add_W(const double* v, double sign)
    {
        const int kp = P.kp;
        for (int64_t i = row0 + threadIdx.x; i < row1; i += blockDim.x) {
            const double* wrow = P.Wm + i;
            double a0 = 0.0, a1 = 0.0;
            for (int j = 0; j < kp; j += 2) {
                a0 = fma(ldg_f64(wrow + (size_t)j * P.ldw), v[j], a0);
                a1 = fma(ldg_f64(wrow + (size_t)(j + 1) * P.ldw), v[j + 1], a1);
            }
            P.x[i] = fma(sign, a0 + a1, P.x[i]);
        }
    }

    // ---- the k x k coefficient recurrences of the header comment (replicated in every CTA)
    // lines 7 / 20 / 22-23: mu = C c, rho = r^T z~ - s^T mu, beta, nu = mu + beta nu, g = c + beta g
    __device__ void coef_direction(bool restart, double rho_prime, double& rho, double& beta)
    {
        const int kp = P.kp;
        small_matvec(sh.C, sh.c, sh.mu);
        if (restart) {
            if ((int)threadIdx.x < kp) { sh.sv[threadIdx.x] = 0.0; }
            __syncthreads();
        }
        small_dot2(sh.sv, sh.mu, sh.sv, sh.mu);
        const double rho_new = rho_prime - sh.small[0];
        beta = restart ? 0.0 : rho_new / rho;
        rho = rho_new;
        __syncthreads();
        if ((int)threadIdx.x < kp) {
            sh.nu[threadIdx.x] = fma(beta, sh.nu[threadIdx.x], sh.mu[threadIdx.x]);
            sh.g[threadIdx.x] = fma(beta, sh.g[threadIdx.x], sh.c[threadIdx.x]);
        }
        __syncthreads();
    }
    // line 9: p^T B p = p~^T w~ - 2 nu^T g + nu^T E_W nu
    __device__ double coef_curvature(double pw)
    {
        small_matvec(sh.EW, sh.nu, sh.e);
        small_dot2(sh.nu, sh.g, sh.nu, sh.e);
        return pw - 2.0 * sh.small[0] + sh.small[1];
    }
    // line 10 in coefficients: s = W_I^T r, a nu, xi
    __device__ void coef_step(double a)
    {
        __syncthreads();
        if ((int)threadIdx.x < P.kp) {
            const int j = threadIdx.x;
            sh.sv[j] = fma(-a, sh.g[j] - sh.e[j], sh.sv[j]);
            sh.anu[j] = a * sh.nu[j];
            sh.xi[j] = fma(a, sh.nu[j], sh.xi[j]);
        }
        __syncthreads();
    }

    // the two SpMVs of S3 over this CTA's slices (operator.cuh)
    template <bool COMBINE>
    __device__ void opK(const double* v0, const double* v1, double beta, double* pnew)
    {
        stage_K<COMBINE>(P.K, P.N, s0, s1, P.minv, v0, v1, beta, pnew, P.t);
    }
    __device__ double opKT(const double* v) { return stage_KT(P.KT, P.N, s0, s1, P.m, P.sigma, P.act, v, P.t, P.w); }
    __device__ void tick(int) {}
    __device__ void finish(CgDevReport*) {}
};

// w = B v (both SpMVs with the barrier between them); v^T w goes to SL_DOT.
template <class CTA>
__device__ __forceinline__ void apply_B_plain(CTA& cta, const double* v)
{
    cta.template opK<false>(v, nullptr, 0.0, nullptr);
    cta.sync_fetch(false, false);
    double d = cta.opKT(v);
    d = block_sum(d, cta.sh.red);
    cta.put(SL_DOT, d);
}

using Cg2Cta = Cg2CtaT<Cg2Shared>;

// Algorithm 1, the whole solve; CTA supplies the stages (Cg2Cta here, Cg3Cta in cg3.cuh).
template <class CTA, class SH>
__device__ __forceinline__ void alg1_coeff_body(const CgParams& P, SH& sh, CTA& cta)
{
    const bool coarse = P.use_coarse != 0;
    const int kp = P.kp;
    if (coarse)
        for (int q = threadIdx.x; q < kp * kp; q += blockDim.x) { sh.C[q] = P.C[q]; sh.EW[q] = P.EW[q]; }
    if (threadIdx.x < RD_MAX_K) { sh.xi[threadIdx.x] = 0.0; sh.nu[threadIdx.x] = 0.0; sh.g[threadIdx.x] = 0.0; sh.sv[threadIdx.x] = 0.0; sh.anu[threadIdx.x] = 0.0; }

    // line 1: tau = eps_c ||b||_2
    {
        double bb = 0.0;
        for (int64_t i = cta.row0 + threadIdx.x; i < cta.row1; i += blockDim.x) bb = fma(P.b[i], P.b[i], bb);
        bb = block_sum(bb, sh.red);
        cta.put(SL_BB, bb);
    }
    // line 3: x <- x0 + Q (b - B x0);  r <- b - B x
    cta.template opK<false>(P.x, nullptr, 0.0, nullptr);
    cta.sync_fetch(true, false);
    const double bnorm = sqrt(sh.scal[SL_BB]);
    const double tau = (bnorm > 0.0) ? P.eps_c * bnorm : P.eps_c;
    __syncthreads();
    (void)cta.opKT(P.x);
    int status = RD_ECAP_DEV;
    int iters = 0, replacements = 0;
    bool done = false;
    bool x_split = false;  // x = x~ - W_I xi with xi != 0
    double rho = 0.0, beta = 0.0;
    int cur = 0;

    if (coarse) {
        cta.stage_recompute(P.Wm, false);  // r = b - B x0, c = W_I^T r
        cta.sync_fetch(true, true);
        cta.small_matvec(sh.C, sh.c, sh.mu);
        cta.stage_add_W(sh.mu, 1.0);  // x += W_I C W_I^T r
        cta.sync_fetch(false, false);
        apply_B_plain(cta, P.x);
    }
    cta.stage_recompute(P.HWm, true);  // r = b - B x, z~ = J r, ||r||^2, r^T z~, c = (HW_I)^T z~
    cta.sync_fetch(true, coarse);
    // lines 4-6
    if (sqrt(sh.scal[SL_RR]) <= tau) { status = 0; done = true; }
    bool restart = true;  // line 7 / line 20: p <- z, i.e. p~ = z~, nu = mu, g = c, s = 0
    double rho_prime = sh.scal[SL_RHO];
    // line 8
    cta.tick(7);
    while (!done && iters < P.cap) {
        // ---- coefficient part of lines 7 / 20 / 22-23
        if (coarse) {
            cta.coef_direction(restart, rho_prime, rho, beta);
        } else {
            beta = restart ? 0.0 : rho_prime / rho;
            rho = rho_prime;
        }
        restart = false;
        cta.tick(4);
        // ---- stage A: line 23 fused into line 9's first product
        double* pold = cur ? P.p1 : P.p0;
        double* pnew = cur ? P.p0 : P.p1;
        cta.template opK<true>(P.z, pold, beta, pnew);
        cur ^= 1;
        cta.tick(0);
        cta.sync_fetch(false, false);
        cta.tick(1);
        // ---- stage B
        {
            double d = cta.opKT(pnew);
            d = block_sum(d, sh.red);
            cta.put(SL_DOT, d);
        }
        cta.tick(2);
        cta.sync_fetch(true, false);
        cta.tick(3);
        iters++;
        double pw = sh.scal[SL_DOT];
        if (coarse) pw = cta.coef_curvature(pw);  // p^T B p
        if (!(pw > 0.0) || !(rho > 0.0)) { status = RD_ENOTSPD_DEV; break; }
        // line 10
        const double a = rho / pw;
        if (coarse) {
            cta.coef_step(a);
            x_split = true;
            cta.tick(4);
            cta.stage_update_coarse(a, pnew);
        } else {
            cta.tick(4);
            cta.stage_update_plain(a, pnew);
        }
        cta.tick(5);
        cta.sync_fetch(true, coarse);
        cta.tick(6);
        rho_prime = sh.scal[SL_RHO];
        // line 11
        const bool scheduled = P.replace_period > 0 && (iters % P.replace_period) == 0;
        if (sqrt(sh.scal[SL_RR]) <= tau || scheduled) {
            replacements++;
            if (x_split) {  // x = x~ - W_I xi
                cta.stage_add_W(sh.xi, -1.0);
                __syncthreads();
                if (threadIdx.x < RD_MAX_K) sh.xi[threadIdx.x] = 0.0;
                x_split = false;
                cta.sync_fetch(false, false);
            }
            // line 12: recompute r = b - B x
            apply_B_plain(cta, P.x);
            cta.stage_recompute(coarse ? P.Wm : P.HWm, !coarse);
            cta.sync_fetch(true, coarse);
            if (sqrt(sh.scal[SL_RR]) <= tau) { status = 0; break; }  // lines 13-15
            if (coarse) {
                // line 16: x <- x + Q r; r <- b - B x
                cta.small_matvec(sh.C, sh.c, sh.mu);
                cta.stage_add_W(sh.mu, 1.0);
                cta.sync_fetch(false, false);
                apply_B_plain(cta, P.x);
                cta.stage_recompute(P.HWm, true);
                cta.sync_fetch(true, true);
                if (sqrt(sh.scal[SL_RR]) <= tau) { status = 0; break; }  // lines 17-19
            }
            rho_prime = sh.scal[SL_RHO];
            restart = true;  // line 20
        }
    }
    // line 26: Verify(x, eps) from a fresh apply on the explicit x
    const double rr_last = sh.scal[SL_RR];
    __syncthreads();
    if (x_split) {
        cta.stage_add_W(sh.xi, -1.0);
        cta.sync_fetch(false, false);
    }
    apply_B_plain(cta, P.x);
    cta.stage_recompute(nullptr, false);
    cta.sync_fetch(true, false);
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
        cta.tick(7);
        cta.finish(P.rep);
    }
}

__global__ void __launch_bounds__(RD_CG_THREADS, 1) k_alg1_v2(const CgParams P)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    Cg2Shared& sh = *reinterpret_cast<Cg2Shared*>(smem_raw);
    Cg2Cta cta(P, sh);
    alg1_coeff_body(P, sh, cta);
}

}  // namespace rd
