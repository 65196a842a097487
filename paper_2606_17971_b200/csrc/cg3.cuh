// cg3.cuh -- k_alg1_v3: Algorithm 1 in the coefficient form of cg2.cuh, with every streamed
// operand staged through shared memory by 1-D TMA bulk copies (cp.async.bulk + mbarrier, async.cuh) instead of
// register loads.  Default kernel of the library (rd_options.alg1_variant = 0).
//
// Why: the loop is HBM-bound (DESIGN.md bytes model) and a register-staged kernel at 64 registers per thread
// cannot keep enough bytes in flight: every 32-row tile of the HW_I pass waited on its own loads.  Here
//   stage C  the n x kp block HW_I streams through a ring of NST = min(32, 512/kp) tiles of 32 rows x kp columns
//            (256 kp bytes each, 128 KB in total); consumer warp cw owns ring slot cw and its mbarrier, processes
//            tiles cw, cw + NST, ... and refills its slot as soon as its lanes have read it.  A tile is consumed
//            by ONE warp in two passes over shared memory: lane = row for q_i = sum_j HW_ij (a nu_j) and the
//            row updates, then lane = column for c_j += sum_i HW_ij z~_i, rows visited in a skewed order
//            (i + lane) mod 32 so that the transposed reads are bank-conflict free.  No cross-warp exchange.
//   stage A/B the sliced-ELL streams of K and K^T: every warp prefetches the values and column indices of its
//            next 32-row slice into its own 4 KB slot while it gathers for the current one.
// The arithmetic per row and all reduction orders are fixed, so results are bit-reproducible run to run.
#pragma once
#include "async.cuh"
#include "cg2.cuh"

namespace rd {

#define RD_RING_BYTES (128 * 1024)
#define RD_SPMV_WD 8             // ELL entries per row that the staged SpMV path holds (wider slices: direct loads)
#define RD_SPMV_SLOT_BYTES 4096  // per warp: values 8 x 256 B, then indices 8 x 128 B

struct __align__(128) Cg3Shared {
    double C[RD_MAX_K * RD_MAX_K];
    double EW[RD_MAX_K * RD_MAX_K];
    double s[RD_CG_THREADS];  // transposition buffer of stage_recompute (outside the loop)
    double zb[32][32];        // stage C: z~ of the warp's tile, for the transposed pass
    double cpart[512];        // stage C: c partials of the consumer warps, NST x kp <= 512
    double c[RD_MAX_K], mu[RD_MAX_K], nu[RD_MAX_K], g[RD_MAX_K], sv[RD_MAX_K], xi[RD_MAX_K], anu[RD_MAX_K], e[RD_MAX_K];
    double scal[SL_NSCAL];
    double small[4];
    double red[32];
    uint64_t full[32];  // one mbarrier per warp
    uint64_t tacc[8];
    uint64_t tlast;
    __align__(128) unsigned char ring[RD_RING_BYTES];  // written by the async proxy only
};


struct Cg3Cta : Cg2CtaT<Cg3Shared> {
    using Base = Cg2CtaT<Cg3Shared>;
    uint32_t ph;  // phase parity of this warp's mbarrier (uniform in the warp)

    __device__ Cg3Cta(const CgParams& p, Cg3Shared& s) : Base(p, s), ph(0)
    {
        if (threadIdx.x == 0) {
            for (int w = 0; w < 32; ++w) mbar_init(&sh.full[w], 1);
            mbar_fence_init();
            for (int q = 0; q < 8; ++q) sh.tacc[q] = 0;
            sh.tlast = global_timer_ns();
        }
        __syncthreads();
    }

    __device__ void tick(int slot)
    {
        if (blockIdx.x == 0 && threadIdx.x == 0) {
            const uint64_t t = global_timer_ns();
            sh.tacc[slot] += t - sh.tlast;
            sh.tlast = t;
        }
    }
    __device__ void finish(CgDevReport* rep)
    {
        for (int q = 0; q < 8; ++q) rep->t_stage_us[q] = 1e-3 * (double)sh.tacc[q];
    }

    // ---- grid barrier + all-reduce.  Every CTA has written one partial per reduced quantity; the barrier is the
    // single-hop counter barrier of common.cuh (arrival = release reduction on one monotone counter, everybody polls
    // that counter); then every CTA sums all partials in the same fixed order (deterministic, identical branches).
    __device__ void sync_fetch(bool want_scal, bool want_c)
    {
        const double* base = P.partial + (size_t)(nbar & 1u) * SL_NSLOT * G;
        nbar++;
        const unsigned int gen = nbar;
        grid_barrier_counter(reinterpret_cast<unsigned long long*>(P.bar), G, gen);
        if (!want_scal) return;
        // all slots in one round: 8 lanes per slot (128 slot groups >= 4 + kp), fixed order => identical on all CTAs
        const int nsl = want_c ? SL_NSCAL + P.kp : SL_NSCAL;
        const int sl = threadIdx.x >> 3, sub = threadIdx.x & 7;
        if ((sl & ~3) < nsl) {  // warp-uniform: some slot of this warp is live
            double a0 = 0.0, a1 = 0.0;
            if (sl < nsl) {
                const double* q = base + (size_t)sl * G;
#pragma unroll 4
                for (int i = sub; i < G; i += 16) {
                    a0 += __ldcg(q + i);
                    if (i + 8 < G) a1 += __ldcg(q + i + 8);
                }
            }
            double a = a0 + a1;
            a += __shfl_xor_sync(0xffffffffu, a, 4);
            a += __shfl_xor_sync(0xffffffffu, a, 2);
            a += __shfl_xor_sync(0xffffffffu, a, 1);
            if (sub == 0 && sl < nsl) {
                if (sl < SL_NSCAL) sh.scal[sl] = a; else sh.c[sl - SL_NSCAL] = a;
            }
        }
        __syncthreads();
    }

    // ---- k x k coefficient recurrences (cg2.cuh header), done by warp 0 alone: lane owns rows lane and lane + 32
    // of the kp x kp matrices (column-major: conflict-free), vectors are broadcast reads.  One __syncthreads.
    __device__ __forceinline__ void matvec_w0(const double* M, const double* v, int kp, int lane, double& o0, double& o1)
    {
        double a0 = 0.0, a1 = 0.0, b0 = 0.0, b1 = 0.0;
        const bool r0 = lane < kp, r1 = lane + 32 < kp;
        const double* m0 = M + (r0 ? lane : 0);
        const double* m1 = M + (r1 ? lane + 32 : 0);
        for (int j = 0; j < kp; j += 2) {
            const double v0 = v[j], v1 = v[j + 1];
            a0 = fma(m0[(size_t)j * kp], v0, a0);
            b0 = fma(m0[(size_t)(j + 1) * kp], v1, b0);
            a1 = fma(m1[(size_t)j * kp], v0, a1);
            b1 = fma(m1[(size_t)(j + 1) * kp], v1, b1);
        }
        o0 = r0 ? a0 + b0 : 0.0;
        o1 = r1 ? a1 + b1 : 0.0;
    }
    // lines 7 / 20 / 22-23 and the curvature terms of line 9 that do not need p~^T w~:
    //   mu = C c, rho = r^T z~ - s^T mu, beta, nu = mu + beta nu, g = c + beta g, e = E_W nu, nu^T g, nu^T e
    __device__ void coef_direction(bool restart, double rho_prime, double& rho, double& beta)
    {
        const int kp = P.kp;
        if (threadIdx.x < 32) {
            const int lane = threadIdx.x;
            const bool r0 = lane < kp, r1 = lane + 32 < kp;
            double mu0, mu1;
            matvec_w0(sh.C, sh.c, kp, lane, mu0, mu1);
            const double s0_ = (restart || !r0) ? 0.0 : sh.sv[lane], s1_ = (restart || !r1) ? 0.0 : sh.sv[lane + 32];
            const double smu = warp_sum(fma(s0_, mu0, s1_ * mu1));
            const double rho_new = rho_prime - smu;
            const double bt = restart ? 0.0 : rho_new / rho;
            double nu0 = 0.0, nu1 = 0.0, g0 = 0.0, g1 = 0.0;
            if (r0) { nu0 = fma(bt, sh.nu[lane], mu0); g0 = fma(bt, sh.g[lane], sh.c[lane]); sh.nu[lane] = nu0; sh.g[lane] = g0; sh.mu[lane] = mu0; if (restart) sh.sv[lane] = 0.0; }
            if (r1) { nu1 = fma(bt, sh.nu[lane + 32], mu1); g1 = fma(bt, sh.g[lane + 32], sh.c[lane + 32]); sh.nu[lane + 32] = nu1; sh.g[lane + 32] = g1; sh.mu[lane + 32] = mu1; if (restart) sh.sv[lane + 32] = 0.0; }
            __syncwarp();
            double e0, e1;
            matvec_w0(sh.EW, sh.nu, kp, lane, e0, e1);
            if (r0) sh.e[lane] = e0;
            if (r1) sh.e[lane + 32] = e1;
            const double ng = warp_sum(fma(nu0, g0, nu1 * g1));
            const double ne = warp_sum(fma(nu0, e0, nu1 * e1));
            if (lane == 0) { sh.small[0] = rho_new; sh.small[1] = bt; sh.small[2] = ng; sh.small[3] = ne; }
        }
        __syncthreads();
        rho = sh.small[0];
        beta = sh.small[1];
    }
    __device__ double coef_curvature(double pw) { return pw - 2.0 * sh.small[2] + sh.small[3]; }
    // line 10 in coefficients; the __syncthreads that opens stage_update_coarse publishes anu
    __device__ void coef_step(double a)
    {
        if ((int)threadIdx.x < P.kp) {
            const int j = threadIdx.x;
            sh.sv[j] = fma(-a, sh.g[j] - sh.e[j], sh.sv[j]);
            sh.anu[j] = a * sh.nu[j];
            sh.xi[j] = fma(a, sh.nu[j], sh.xi[j]);
        }
    }

    // values and column indices of one 32-row slice (wd entries per row) into this warp's slot
    __device__ __forceinline__ void issue_slice(const Ell& A, int64_t o, int wd)
    {
        if ((threadIdx.x & 31) == 0) {
            unsigned char* slot_ = sh.ring + (threadIdx.x >> 5) * RD_SPMV_SLOT_BYTES;
            uint64_t* bar = &sh.full[threadIdx.x >> 5];
            mbar_arrive_expect_tx(bar, (uint32_t)wd * 384u);
            if (wd > 0) {
                {
                    bulk_g2s(slot_, A.val + o, (uint32_t)wd * 256u, bar);
                    bulk_g2s(slot_ + RD_SPMV_WD * 256, A.col + o, (uint32_t)wd * 128u, bar);
                }
            }
        }
    }
    // sum_e A[row,e] vin[col_e] for this lane's row of the slice staged in (sval, scol); WDC = register budget
    // (entries per row).  All gathers are issued before the first use; `next` refills the slot in between.
    template <bool COMBINE, int WDC, class Next>
    __device__ __forceinline__ double staged_row_dot(const double* sval, const int32_t* scol, int wd, int lane,
                                                     const double* v0, const double* v1, double beta, Next next)
    {
        int cc[WDC];
        double aa[WDC], xx[WDC], yy[WDC];
#pragma unroll
        for (int q = 0; q < WDC; ++q) {
            const bool ok = q < wd;
            cc[q] = ok ? scol[q * 32 + lane] : 0;
            aa[q] = ok ? sval[q * 32 + lane] : 0.0;
        }
        // The refill below is an async-proxy write into the slot just read through the generic proxy (a bulk copy
        // issued right after the loads can otherwise land before they have executed: seen on config 5 in round 1).
        // refill_fence = __syncwarp + fence.proxy.async.shared::cta orders the two (async.cuh).
        refill_fence();
        next();
#pragma unroll
        for (int q = 0; q < WDC; ++q) xx[q] = (q < wd) ? v0[cc[q]] : 0.0;
        if (COMBINE) {
#pragma unroll
            for (int q = 0; q < WDC; ++q) yy[q] = (q < wd) ? v1[cc[q]] : 0.0;
#pragma unroll
            for (int q = 0; q < WDC; ++q) xx[q] = fma(beta, yy[q], xx[q]);
        }
        double acc = 0.0;
#pragma unroll
        for (int q = 0; q < WDC; ++q) acc = fma(aa[q], xx[q], acc);
        return acc;
    }

    // ---- staged sliced-ELL product over this CTA's slices.  pre(row) loads what the epilogue needs of the row
    // (issued before the wait on the slice, so it never adds a round trip); epi(row, acc, pre(row)) consumes
    // sum_e A[row,e] vin[col_e].  A matrix of uniform slice width needs no extent lookups (Ell::uwd).
    template <bool COMBINE, class Pre, class Epi>
    __device__ __forceinline__ void spmv_staged(const Ell& A, const double* v0, const double* v1, double beta, Pre pre, Epi epi)
    {
        const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
        unsigned char* slot_ = sh.ring + warp * RD_SPMV_SLOT_BYTES;
        const double* sval = reinterpret_cast<const double*>(slot_);
        const int32_t* scol = reinterpret_cast<const int32_t*>(slot_ + RD_SPMV_WD * 256);
        uint64_t* bar = &sh.full[warp];
        const int uwd = A.uwd;
        auto extent = [&](int64_t s, int64_t& o, int& wd) {
            if (uwd >= 0) { o = s * 32 * uwd; wd = uwd; }
            else { o = A.off[s]; wd = (int)((A.off[s + 1] - o) >> 5); }
        };
        int64_t s = s0 + warp;
        int wd = 0;
        refill_fence();  // the ring was last read (generic proxy) by the previous stage, possibly by another warp, before a CTA barrier
        if (s < s1) {
            int64_t o;
            extent(s, o, wd);
            if (wd <= RD_SPMV_WD) issue_slice(A, o, wd);
        }
        for (; s < s1; s += 32) {
            const int64_t sn = s + 32;
            int64_t on = 0;
            int wdn = 0;
            if (sn < s1) extent(sn, on, wdn);
            const int64_t row = s * RD_SLICE + lane;
            auto rowdata = pre(row);
            auto next = [&]() { if (sn < s1 && wdn <= RD_SPMV_WD) issue_slice(A, on, wdn); };
            double acc;
            if (wd <= RD_SPMV_WD) {
                mbar_wait(bar, ph);
                ph ^= 1u;
                if (wd <= 5) acc = staged_row_dot<COMBINE, 5>(sval, scol, wd, lane, v0, v1, beta, next);
                else if (wd <= 7) acc = staged_row_dot<COMBINE, 7>(sval, scol, wd, lane, v0, v1, beta, next);
                else acc = staged_row_dot<COMBINE, RD_SPMV_WD>(sval, scol, wd, lane, v0, v1, beta, next);
            } else {
                next();
                acc = ell_row_dot<COMBINE>(A, s, lane, v0, v1, beta);
            }
            epi(row, acc, rowdata);
            wd = wdn;
        }
    }

    struct RowK { double minv, x; };
    struct RowKT { double v, m; bool act; };

    // stage A: t = M^{-1} K (v0 + beta v1), pnew = v0 + beta v1 on this CTA's rows  (Alg. 1 lines 23 + 9)
    template <bool COMBINE>
    __device__ void opK(const double* v0, const double* v1, double beta, double* pnew)
    {
        const int64_t N = P.N;
        const double* minv = P.minv;
        double* t = P.t;
        spmv_staged<COMBINE>(
            P.K, v0, v1, beta,
            [&](int64_t row) {
                RowK r{0.0, 0.0};
                if (row < N) {
                    r.minv = ldg_f64(minv + row);
                    if (pnew) {
                        r.x = v0[row];
                        if (COMBINE) r.x = fma(beta, v1[row], r.x);
                    }
                }
                return r;
            },
            [&](int64_t row, double acc, const RowK& r) {
                if (row < N) {
                    t[row] = acc * r.minv;
                    if (pnew) pnew[row] = r.x;
                }
            });
    }
    // stage B: w = chi_I (m.v + sigma K^T t); returns this thread's partial of v^T w  (Alg. 1 line 9)
    __device__ double opKT(const double* v)
    {
        const int64_t N = P.N;
        const double* m = P.m;
        const uint8_t* act = P.act;
        const double sigma = P.sigma;
        double* w = P.w;
        double dot = 0.0;
        spmv_staged<false>(
            P.KT, P.t, nullptr, 0.0,
            [&](int64_t row) {
                RowKT r{0.0, 0.0, false};
                if (row < N) {
                    r.v = v[row];
                    r.m = ldg_f64(m + row);
                    r.act = act && act[row];
                }
                return r;
            },
            [&](int64_t row, double acc, const RowKT& r) {
                if (row < N) {
                    double wi = fma(sigma, acc, r.m * r.v);
                    if (r.act) wi = 0.0;
                    w[row] = wi;
                    dot = fma(r.v, wi, dot);
                }
            });
        return dot;
    }

    // Stage C without a coarse space (rank-zero execution = Jacobi-CG): two rows per thread in flight
    __device__ void stage_update_plain(double a, const double* p)
    {
        double rr = 0.0, rho = 0.0;
        __syncthreads();
        const int64_t step = 2 * (int64_t)blockDim.x;
        for (int64_t i0 = row0 + threadIdx.x; i0 < row1; i0 += step) {
            const int64_t i1 = i0 + blockDim.x;
            const bool in1 = i1 < row1;
            const double w0 = P.w[i0], r0 = P.r[i0], d0 = ldg_f64(P.dinv + i0), p0 = p[i0], x0 = P.x[i0];
            double w1 = 0.0, r1 = 0.0, d1 = 0.0, p1 = 0.0, x1 = 0.0;
            if (in1) { w1 = P.w[i1]; r1 = P.r[i1]; d1 = ldg_f64(P.dinv + i1); p1 = p[i1]; x1 = P.x[i1]; }
            const double rn0 = fma(-a, w0, r0), zn0 = rn0 * d0;
            P.x[i0] = fma(a, p0, x0);
            P.r[i0] = rn0;
            P.z[i0] = zn0;
            rr = fma(rn0, rn0, rr);
            rho = fma(rn0, zn0, rho);
            if (in1) {
                const double rn1 = fma(-a, w1, r1), zn1 = rn1 * d1;
                P.x[i1] = fma(a, p1, x1);
                P.r[i1] = rn1;
                P.z[i1] = zn1;
                rr = fma(rn1, rn1, rr);
                rho = fma(rn1, zn1, rho);
            }
        }
        rr = block_sum(rr, sh.red);
        rho = block_sum(rho, sh.red);
        put(SL_RR, rr);
        put(SL_RHO, rho);
    }

    // one 32-row x kp tile of the tile-major copy of HW_I (contiguous 256 kp bytes) into this consumer warp's slot
    __device__ __forceinline__ void issue_tile(int64_t t)
    {
        if ((threadIdx.x & 31) == 0) {
            const int warp = threadIdx.x >> 5;
            const uint32_t tile_bytes = 256u * (uint32_t)P.kp;
            void* tile = sh.ring + (size_t)warp * tile_bytes;
            uint64_t* bar = &sh.full[warp];
            mbar_arrive_expect_tx(bar, tile_bytes);
            const double* src = P.HWt + ((size_t)(row0 >> 5) + t) * 32 * P.kp;
            // no reuse before the next iteration: evict_first keeps the gathered vectors and K in L2; when the working
            // set nearly fits the L2 the first hw_res_tiles tiles of every CTA are kept instead (evict_last)
            bulk_g2s_hint(tile, src, tile_bytes, bar, t < P.hw_res_tiles ? l2_policy_evict_last() : l2_policy_evict_first());
        }
    }
    // Stage C with a coarse space: one pass over HW_I through the shared-memory ring (header comment).
    //   r_i  <- r_i - a w~_i + sum_j HW_ij (a nu_j)      x~_i <- x~_i + a p~_i      z~_i <- r_i / d_i
    //   ||r||^2, r^T z~,  c_j = sum_i HW_ij z~_i                                      (eq. (18))
    __device__ void stage_update_coarse(double a, const double* p)
    {
        const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
        const int kp = P.kp;
        const uint32_t tile_bytes = 256u * (uint32_t)kp;
        const int nst = min(32, (int)(RD_RING_BYTES / tile_bytes));
        const int64_t ntiles = (row1 - row0 + 31) >> 5;
        double rr = 0.0, rho = 0.0;
        double acc[(RD_MAX_K + 31) / 32];
#pragma unroll
        for (int q = 0; q < (RD_MAX_K + 31) / 32; ++q) acc[q] = 0.0;
        __syncthreads();  // w~ of this CTA's rows was written by other threads of the CTA; anu is in place
        if (warp < nst) {
            double* tile = reinterpret_cast<double*>(sh.ring + (size_t)warp * tile_bytes);
            uint64_t* bar = &sh.full[warp];
            double* zbw = sh.zb[warp];
            const double* anu = sh.anu;
            auto issue = [&](int64_t t) { issue_tile(t); };
            int64_t t = warp;
            double ri = 0.0, wi = 0.0, di = 0.0, pi = 0.0, xi = 0.0;
            refill_fence();  // as in spmv_staged: previous stage's generic reads of these bytes precede the CTA barrier above
            if (t < ntiles) {
                issue(t);
                const int64_t i = row0 + 32 * t + lane;
                if (i < row1) { ri = P.r[i]; wi = P.w[i]; di = ldg_f64(P.dinv + i); pi = p[i]; xi = P.x[i]; }
            }
            for (; t < ntiles; t += nst) {
                const int64_t i = row0 + 32 * t + lane;
                const bool in = i < row1;
                // next tile's row data: in flight while this tile is processed
                const int64_t tn = t + nst;
                const int64_t inx = row0 + 32 * tn + lane;
                double rin = 0.0, win = 0.0, din = 0.0, pin = 0.0, xin = 0.0;
                if (tn < ntiles && inx < row1) { rin = P.r[inx]; win = P.w[inx]; din = ldg_f64(P.dinv + inx); pin = p[inx]; xin = P.x[inx]; }
                mbar_wait(bar, ph);
                ph ^= 1u;
                // pass 1: lane = row
                double q0 = 0.0, q1 = 0.0, q2 = 0.0, q3 = 0.0;
                const double* trow = tile + lane;
#pragma unroll 2
                for (int j = 0; j < kp; j += 4) {
                    q0 = fma(trow[(j + 0) * 32], anu[j + 0], q0);
                    q1 = fma(trow[(j + 1) * 32], anu[j + 1], q1);
                    q2 = fma(trow[(j + 2) * 32], anu[j + 2], q2);
                    q3 = fma(trow[(j + 3) * 32], anu[j + 3], q3);
                }
                const double rn = fma(-a, wi, ri) + ((q0 + q1) + (q2 + q3));
                const double zn = in ? rn * di : 0.0;
                if (in) {
                    P.r[i] = rn;
                    P.x[i] = fma(a, pi, xi);
                    P.z[i] = zn;
                    rr = fma(rn, rn, rr);
                    rho = fma(rn, zn, rho);
                }
                zbw[lane] = zn;
                __syncwarp();
                // pass 2: lane = column(s) lane and lane + 32, rows in the skewed order (ii + lane) mod 32
                if (lane < kp) {
                    const double* t0 = tile + lane * 32;
                    double a0 = 0.0, a1 = 0.0, b0 = 0.0, b1 = 0.0;
                    if (lane + 32 < kp) {
                        const double* t1 = t0 + 32 * 32;
#pragma unroll 8
                        for (int ii = 0; ii < 32; ii += 2) {
                            const int r0 = (ii + lane) & 31, r1 = (ii + 1 + lane) & 31;
                            const double z0 = zbw[r0], z1 = zbw[r1];
                            a0 = fma(t0[r0], z0, a0);
                            a1 = fma(t0[r1], z1, a1);
                            b0 = fma(t1[r0], z0, b0);
                            b1 = fma(t1[r1], z1, b1);
                        }
                    } else {
#pragma unroll 8
                        for (int ii = 0; ii < 32; ii += 2) {
                            const int r0 = (ii + lane) & 31, r1 = (ii + 1 + lane) & 31;
                            a0 = fma(t0[r0], zbw[r0], a0);
                            a1 = fma(t0[r1], zbw[r1], a1);
                        }
                    }
                    acc[0] += a0 + a1;
                    acc[1] += b0 + b1;
                }
                refill_fence();  // every lane has read the tile and zb; generic reads ordered before the async refill
                if (tn < ntiles) issue(tn);
                ri = rin; wi = win; di = din; pi = pin; xi = xin;
            }
#pragma unroll
            for (int q = 0; q < (RD_MAX_K + 31) / 32; ++q) {
                const int j = lane + 32 * q;
                if (j < kp) sh.cpart[warp * kp + j] = acc[q];
            }
        }
        __syncthreads();
        if ((int)threadIdx.x < kp) {
            double v = 0.0;
            for (int cw = 0; cw < nst; ++cw) v += sh.cpart[cw * kp + threadIdx.x];
            slot(SL_NSCAL + threadIdx.x)[blockIdx.x] = v;
        }
        rr = block_sum(rr, sh.red);
        rho = block_sum(rho, sh.red);
        put(SL_RR, rr);
        put(SL_RHO, rho);
    }
};

__global__ void __launch_bounds__(RD_CG_THREADS, 1) k_alg1_v3(const CgParams P)
{
    extern __shared__ __align__(128) unsigned char smem_raw[];
    Cg3Shared& sh = *reinterpret_cast<Cg3Shared*>(smem_raw);
    Cg3Cta cta(P, sh);
    alg1_coeff_body(P, sh, cta);
}

}  // namespace rd
