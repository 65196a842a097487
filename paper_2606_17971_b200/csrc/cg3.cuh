// cg3.cuh -- k_alg1_v3: Algorithm 1 with the projection carried in coefficient form, every
// streamed operand staged through shared memory by 1-D TMA bulk copies (cp.async.bulk + mbarrier, async.cuh), and all
// work restricted to the live 32-row slices of the current active set (S6 compaction, pdas.cuh).  Default kernel of the
// library (rd_options.alg1_variant = 0); cg.cuh keeps the literal two-pass recurrence as variant 1.
//
// (W_I below stands for the basis handed to the kernel, HW_I for its cached product and C for the coarse solve in its
// coordinates; since round 2 that basis is the explicit Z = W_I T of coarse.cuh, so HW_I = H_II Z, E_W = E, C = E^{-1}.)
//
// ---- coefficient form.  Write the search direction and the iterate of Alg. 1 as  p = p~ - W_I nu,  x = x~ - W_I xi  with
// k-vectors nu, xi kept (replicated, bit-identical) in the shared memory of every CTA.  With z~ = J r (never projected):
//   line 22  z = P J r = z~ - W_I mu,  mu = C c,  c = (HW_I)^T z~                       (eq. (18))
//   line 23  p = z + beta p      <=>  p~ = z~ + beta p~,   nu = mu + beta nu
//   line  9  w = B p = w~ - HW_I nu  with w~ = B p~  (the two SpMVs act on p~ only)
//            p^T w = p~^T w~ - 2 nu^T g + nu^T E_W nu,   g = (HW_I)^T p~ = c + beta g,   E_W = W_I^T HW_I
//   line 10  x~ += a p~, xi += a nu;   r = r - a w~ + HW_I (a nu)
//   line 22  rho = r^T z = r^T z~ - s^T mu,   s = W_I^T r = s - a (g - E_W nu)   (zero in exact arithmetic,
//            Z^T(b - B x_c) = 0 and Z^T B P = 0; the recurrence carries its rounding-level drift)
// One pass over a 32-row tile of HW_I does both  q_i = sum_j HW_ij (a nu_j)  (needed for r_i) and
// c_j += HW_ij z~_i.  x is made explicit (x = x~ - W_I xi, one pass over W_I) only where Alg. 1 recomputes the
// residual (lines 12, 16, Verify).  ONE pass over the cached product HW_I per iteration instead of a pass over HW_I
// and a pass over W_I.
//
// ---- stages of one iteration (grid barrier after each):
//   A  p~ = z~ + beta p~ (fused into the gather),  t = M^{-1} K p~           over listA, this CTA's share    S3
//   B  w~ = chi_I (m.p~ + sigma K^T t),  p~^T w~                             over listB, this CTA's share    S3
//   C  x~, r, z~ updates, ||r||^2, r^T z~, c = (HW_I)^T z~   (one pass over HW_I, tile-major, through the ring)  S4 + S5
// Each stage splits ITS list evenly over the CTAs (listA and listB differ only near the boundary of the inactive
// set), so a PDAS step with |I| << N streams |I|-proportional bytes and stays balanced.  The k x k recurrences
// between C and A run on two warps (one thread per matrix row, no shuffles in the products).
//
// ---- staging.  Stage C: the n x kp block streams through a ring of NST = min(32, 512/kp) tiles of 32 rows x kp
// columns (256 kp bytes each, 128 KB in total); consumer warp cw owns ring slot cw and its mbarrier, processes the
// tiles cw, cw + NST, ... of this CTA's share and refills its slot as soon as its lanes have read it.  A tile is
// consumed by ONE warp in two passes over shared memory: lane = row for q_i and the row updates, then lane = column
// for c_j, rows visited in the skewed order (i + lane) mod 32 so that the transposed reads are bank-conflict free.
// Stages A/B: every warp prefetches the values and column indices of its next slice into its own 4 KB slot while it
// gathers for the current one.  Write-after-read on a slot (generic-proxy loads, then an async-proxy refill) is
// ordered by refill_fence() (async.cuh).  The arithmetic per row and all reduction orders are fixed by the lists and
// the grid size, so results are bit-reproducible run to run.
#pragma once
#include "async.cuh"
#include "cg.cuh"

namespace rd {

#define RD_RING_BYTES (128 * 1024)
#define RD_SPMV_WD 8             // ELL entries per row that the staged SpMV path holds (wider slices: direct loads)
#define RD_SPMV_SLOT_BYTES 4096  // per warp: values 8 x 256 B, then indices 8 x 128 B

struct __align__(128) Cg3Shared {
    double C[RD_MAX_K * RD_MAX_K];   // E^{-1} (coordinates of the explicit basis Z), symmetric
    double EW[RD_MAX_K * RD_MAX_K];  // E = Z^T H_II Z, symmetrised on load
    double zb[32][32];               // tile streams: the per-row multiplier of the warp's tile, for the transposed pass
    double cpart[512];               // tile streams: c partials of the consumer warps, NST x kp <= 512
    double c[RD_MAX_K], mu[RD_MAX_K], nu[2][RD_MAX_K], g[2][RD_MAX_K], sv[RD_MAX_K], xi[RD_MAX_K], anu[RD_MAX_K], e[RD_MAX_K];
    double scal[SL_NSCAL];
    double small[4];                 // rho, beta, nu^T g, nu^T E_W nu of the current direction
    double red[32];
    uint64_t full[32];  // one mbarrier per warp
    uint64_t tacc[8];   // SM clock cycles per phase (CTA 0 only)
    uint64_t tlast;     // clock64 at the last tick
    uint64_t t0_ns;     // %globaltimer at kernel start: cycles are scaled to microseconds with it at the end
    uint64_t c0;        // clock64 at kernel start
    __align__(128) unsigned char ring[RD_RING_BYTES];  // written by the async proxy only
};

enum { TS_UPDATE = 0, TS_RECOMP_Z = 1, TS_RECOMP_R = 2, TS_ADDW = 3 };

__device__ __forceinline__ void named_bar_sync(int id, int nthreads)
{
    asm volatile("bar.sync %0, %1;" ::"r"(id), "r"(nthreads) : "memory");
}

// entry i of a live-slice list; DENSE: the list is the identity (entry 2 i + 1 with SHIFT = 1: flag set)
template <bool DENSE, int SHIFT>
__device__ __forceinline__ int32_t list_entry(const int32_t* list, int64_t i)
{
    return DENSE ? (int32_t)((i << SHIFT) | SHIFT) : __ldg(list + i);
}

struct Cg3Cta {
    const CgParams& P;
    Cg3Shared& sh;
    int64_t a0, a1, b0, b1;  // this CTA's shares of listA / listB (index ranges)
    bool dense;              // every slice is live (the lists are the identity): the loop stages index directly
    unsigned int nbar;
    int G;
    uint32_t ph;    // phase parity of this warp's mbarrier (uniform in the warp)
    int par;        // which copy of nu / g is current
    double ng, ne;  // nu^T g, nu^T E_W nu of the current direction (every thread holds them)

    __device__ Cg3Cta(const CgParams& p, Cg3Shared& s) : P(p), sh(s), nbar(0), ph(0), par(0), ng(0.0), ne(0.0)
    {
        G = gridDim.x;
        const int64_t nA = P.live_counts[0], nB = P.live_counts[1];
        a0 = (int64_t)blockIdx.x * nA / G;
        a1 = (int64_t)(blockIdx.x + 1) * nA / G;
        b0 = (int64_t)blockIdx.x * nB / G;
        b1 = (int64_t)(blockIdx.x + 1) * nB / G;
        dense = (nB == P.K.nslices);  // listA contains listB
        if (threadIdx.x == 0) {
            for (int w = 0; w < 32; ++w) mbar_init(&sh.full[w], 1);
            mbar_fence_init();
            for (int q = 0; q < 8; ++q) sh.tacc[q] = 0;
            sh.t0_ns = global_timer_ns();
            sh.c0 = sh.tlast = (uint64_t)clock64();
        }
        __syncthreads();
    }

    __device__ double* slot(int sl) const { return P.partial + ((size_t)(nbar & 1u) * SL_NSLOT + sl) * G; }
    __device__ void put(int sl, double v) const
    {
        if (threadIdx.x == 0) slot(sl)[blockIdx.x] = v;
    }
    __device__ void tick(int slot_)
    {
        // the SM's own cycle counter (a %globaltimer read per phase would slow CTA 0, and every barrier waits for it)
        if (blockIdx.x == 0 && threadIdx.x == 0) {
            const uint64_t t = (uint64_t)clock64();
            sh.tacc[slot_] += t - sh.tlast;
            sh.tlast = t;
        }
    }
    __device__ void finish(CgDevReport* rep)
    {
        const double ns = (double)(global_timer_ns() - sh.t0_ns), cyc = (double)((uint64_t)clock64() - sh.c0);
        const double us_per_cycle = cyc > 0.0 ? 1e-3 * ns / cyc : 0.0;
        for (int q = 0; q < 8; ++q) rep->t_stage_us[q] = us_per_cycle * (double)sh.tacc[q];
    }

    // (Round 2 also tried per-CTA flags instead of the grid barrier between stages A and B -- a CTA's K^T rows gather t only
    // from a few neighbouring shares on these banded operators; commit d22bb87, RD_NEIGHBOUR_SYNC.  Config 5: 566.3 against
    // 567.0 us per iteration (the wait moves to the next barrier), config 4 293.8 against 289.1, config 2 35.6 against 32.7:
    // removed.)
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
            double a0_ = 0.0, a1_ = 0.0;
            if (sl < nsl) {
                const double* q = base + (size_t)sl * G;
#pragma unroll 4
                for (int i = sub; i < G; i += 16) {
                    a0_ += __ldcg(q + i);
                    if (i + 8 < G) a1_ += __ldcg(q + i + 8);
                }
            }
            double a = a0_ + a1_;
            a += __shfl_xor_sync(0xffffffffu, a, 4);
            a += __shfl_xor_sync(0xffffffffu, a, 2);
            a += __shfl_xor_sync(0xffffffffu, a, 1);
            if (sub == 0 && sl < nsl) {
                if (sl < SL_NSCAL) sh.scal[sl] = a; else sh.c[sl - SL_NSCAL] = a;
            }
        }
        __syncthreads();
    }

    // ---- k x k part.  Matrices are symmetric and column-major.  Two warps (64 threads, one per row: M[i + j kp] is
    // conflict-free across a warp and the vector entry is a broadcast) form the matrix-vector products with serial FMA
    // chains and no shuffles; warp 0 alone takes the k-long dots; named barrier 1 (64 threads) separates the steps and
    // one block barrier publishes the scalars.  The chain c -> mu -> beta -> nu -> e -> nu^T e is sequential by nature.
    __device__ __forceinline__ double row_matvec(const double* M, const double* v, int i, int kp)
    {
        const double* m = M + i;
        double a0 = 0.0, a1 = 0.0, a2 = 0.0, a3 = 0.0;
#pragma unroll 2
        for (int j = 0; j < kp; j += 4) {  // kp is a multiple of 8
            a0 = fma(m[(size_t)(j + 0) * kp], v[j + 0], a0);
            a1 = fma(m[(size_t)(j + 1) * kp], v[j + 1], a1);
            a2 = fma(m[(size_t)(j + 2) * kp], v[j + 2], a2);
            a3 = fma(m[(size_t)(j + 3) * kp], v[j + 3], a3);
        }
        return (a0 + a1) + (a2 + a3);
    }
    // mu = C c  (the coarse solve of eq. (18) in W_I coordinates; lines 3 and 16)
    __device__ void coarse_solve()
    {
        const int kp = P.kp;
        if ((int)threadIdx.x < kp) sh.mu[threadIdx.x] = row_matvec(sh.C, sh.c, threadIdx.x, kp);
        __syncthreads();
    }
    // lines 7 / 20 / 22-23 in coefficients and the curvature terms of line 9 that do not need p~^T w~:
    //   mu = C c, rho = r^T z~ - s^T mu, beta, nu = mu + beta nu, g = c + beta g, e = E_W nu, nu^T g, nu^T e
    __device__ void coef_direction(bool restart, double rho_prime, double& rho, double& beta)
    {
        const int kp = P.kp, tid = threadIdx.x;
        if (tid < 64) {
            const int lane = tid & 31;
            const bool row = tid < kp;
            const bool r0 = lane < kp, r1 = lane + 32 < kp;
            const double* nu_o = sh.nu[par];
            const double* g_o = sh.g[par];
            double* nu_n = sh.nu[par ^ 1];
            double* g_n = sh.g[par ^ 1];
            if (row) sh.mu[tid] = row_matvec(sh.C, sh.c, tid, kp);
            named_bar_sync(1, 64);
            if (tid < 32) {  // lane j owns entries j and j + 32
                const double mu0 = r0 ? sh.mu[lane] : 0.0, mu1 = r1 ? sh.mu[lane + 32] : 0.0;
                const double s0_ = (restart || !r0) ? 0.0 : sh.sv[lane], s1_ = (restart || !r1) ? 0.0 : sh.sv[lane + 32];
                const double smu = warp_sum(fma(s0_, mu0, s1_ * mu1));
                const double rho_new = rho_prime - smu;
                const double bt = restart ? 0.0 : rho_new / rho;
                if (r0) { nu_n[lane] = fma(bt, nu_o[lane], mu0); g_n[lane] = fma(bt, g_o[lane], sh.c[lane]); if (restart) sh.sv[lane] = 0.0; }
                if (r1) { nu_n[lane + 32] = fma(bt, nu_o[lane + 32], mu1); g_n[lane + 32] = fma(bt, g_o[lane + 32], sh.c[lane + 32]); if (restart) sh.sv[lane + 32] = 0.0; }
                if (lane == 0) { sh.small[0] = rho_new; sh.small[1] = bt; }
            }
            named_bar_sync(1, 64);
            if (row) sh.e[tid] = row_matvec(sh.EW, nu_n, tid, kp);
            named_bar_sync(1, 64);
            if (tid < 32) {
                const double nu0 = r0 ? nu_n[lane] : 0.0, nu1 = r1 ? nu_n[lane + 32] : 0.0;
                const double g0 = r0 ? g_n[lane] : 0.0, g1 = r1 ? g_n[lane + 32] : 0.0;
                const double e0 = r0 ? sh.e[lane] : 0.0, e1 = r1 ? sh.e[lane + 32] : 0.0;
                double x = fma(nu0, g0, nu1 * g1), y = fma(nu0, e0, nu1 * e1);
#pragma unroll
                for (int o = 16; o > 0; o >>= 1) {  // the two sums interleaved
                    x += __shfl_xor_sync(0xffffffffu, x, o);
                    y += __shfl_xor_sync(0xffffffffu, y, o);
                }
                if (lane == 0) { sh.small[2] = x; sh.small[3] = y; }
            }
        }
        __syncthreads();
        par ^= 1;
        rho = sh.small[0];
        beta = sh.small[1];
        ng = sh.small[2];
        ne = sh.small[3];
    }
    __device__ double coef_curvature(double pw) const { return pw - 2.0 * ng + ne; }  // p^T B p
    // line 10 in coefficients; the __syncthreads that opens the tile stream publishes anu
    __device__ void coef_step(double a)
    {
        if ((int)threadIdx.x < P.kp) {
            const int j = threadIdx.x;
            const double nuj = sh.nu[par][j];
            sh.sv[j] = fma(-a, sh.g[par][j] - sh.e[j], sh.sv[j]);
            sh.anu[j] = a * nuj;
            sh.xi[j] = fma(a, nuj, sh.xi[j]);
        }
    }

    // ================================================================== stages A / B: staged sliced-ELL products
    // values and column indices of one 32-row slice (wd entries per row) into this warp's slot
    __device__ __forceinline__ void issue_slice(const Ell& A, int64_t o, int wd)
    {
        if ((threadIdx.x & 31) == 0) {
            unsigned char* slot_ = sh.ring + (threadIdx.x >> 5) * RD_SPMV_SLOT_BYTES;
            uint64_t* bar = &sh.full[threadIdx.x >> 5];
            mbar_arrive_expect_tx(bar, (uint32_t)wd * 384u);
            if (wd > 0) {
                bulk_g2s(slot_, A.val + o, (uint32_t)wd * 256u, bar);
                bulk_g2s(slot_ + RD_SPMV_WD * 256, A.col + o, (uint32_t)wd * 128u, bar);
            }
        }
    }
    // sum_e A[row,e] vin[col_e] for this lane's row of the slice staged in (sval, scol); WDC = register budget
    // (entries per row).  The slot is read into registers, then refilled (`next`), then the gathers go out.
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
        // The refill is an async-proxy write into the slot just read through the generic proxy (a bulk copy issued
        // right after the loads can otherwise land before they have executed: seen on config 5 in round 1).
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

    // Staged product over the list entries [i0, i1) of `list` (SHIFT = 1: entries carry a flag in bit 0).
    // pre(row, flag) loads what the epilogue needs of the row (issued before the wait on the slice, so it never adds a
    // round trip); epi(row, flag, acc, pre(row)) consumes sum_e A[row,e] vin[col_e].
    template <bool COMBINE, int SHIFT, bool DENSE, class Pre, class Epi>
    __device__ __forceinline__ void spmv_staged(const Ell& A, const int32_t* list, int64_t i0, int64_t i1, const double* v0,
                                                const double* v1, double beta, Pre pre, Epi epi)
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
        int64_t i = i0 + warp;
        int32_t ecur = (i < i1) ? list_entry<DENSE, SHIFT>(list, i) : 0;
        int32_t enxt = (i + 32 < i1) ? list_entry<DENSE, SHIFT>(list, i + 32) : 0;
        int wd = 0;
        refill_fence();  // the ring was last read (generic proxy) by the previous stage, before a CTA barrier
        if (i < i1) {
            int64_t o;
            extent((int64_t)(ecur >> SHIFT), o, wd);
            if (wd <= RD_SPMV_WD) issue_slice(A, o, wd);
        }
        for (; i < i1; i += 32) {
            const int64_t in = i + 32;
            const int32_t enn = (in + 32 < i1) ? list_entry<DENSE, SHIFT>(list, in + 32) : 0;  // two ahead: its latency hides behind this slice
            const int64_t s = (int64_t)(ecur >> SHIFT), sn = (int64_t)(enxt >> SHIFT);
            const int flag = SHIFT ? (ecur & 1) : 1;
            int64_t on = 0;
            int wdn = 0;
            if (in < i1) extent(sn, on, wdn);
            const int64_t row = s * RD_SLICE + lane;
            auto rowdata = pre(row, flag);
            auto next = [&]() { if (in < i1 && wdn <= RD_SPMV_WD) issue_slice(A, on, wdn); };
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
            epi(row, flag, acc, rowdata);
            wd = wdn;
            ecur = enxt;
            enxt = enn;
        }
    }

    struct RowK { double minv, x; };
    struct RowKT { double v, m; bool act; };

    // stage A: t = M^{-1} K (v0 + beta v1) on the rows of listA; pnew = v0 + beta v1 on those that hold inactive rows
    // (elsewhere p~ is identically zero and stays so)                                       (Alg. 1 lines 23 + 9)
    template <bool COMBINE, bool DENSE>
    __device__ void opK(const double* v0, const double* v1, double beta, double* pnew)
    {
        const int64_t N = P.N;
        const double* minv = P.minv;
        double* t = P.t;
        spmv_staged<COMBINE, 1, DENSE>(
            P.K, P.listA, a0, a1, v0, v1, beta,
            [&](int64_t row, int flag) {
                RowK r{0.0, 0.0};
                if (row < N) {
                    r.minv = ldg_f64(minv + row);
                    if (pnew && flag) {
                        r.x = v0[row];
                        if (COMBINE) r.x = fma(beta, v1[row], r.x);
                    }
                }
                return r;
            },
            [&](int64_t row, int flag, double acc, const RowK& r) {
                if (row < N) {
                    t[row] = acc * r.minv;
                    if (pnew && flag) pnew[row] = r.x;
                }
            });
    }
    // stage B: w = chi_I (m.v + sigma K^T t) on the rows of listB; returns this thread's partial of v^T w  (line 9)
    template <bool DENSE>
    __device__ double opKT(const double* v)
    {
        const int64_t N = P.N;
        const double* m = P.m;
        const uint8_t* act = P.act;
        const double sigma = P.sigma;
        double* w = P.w;
        double dot = 0.0;
        spmv_staged<false, 0, DENSE>(
            P.KT, P.listB, b0, b1, P.t, nullptr, 0.0,
            [&](int64_t row, int) {
                RowKT r{0.0, 0.0, false};
                if (row < N) {
                    r.v = v[row];
                    r.m = ldg_f64(m + row);
                    r.act = act && act[row];
                }
                return r;
            },
            [&](int64_t row, int, double acc, const RowKT& r) {
                if (row < N) {
                    double wi = fma(sigma, acc, r.m * r.v);
                    if (r.act) wi = 0.0;
                    w[row] = wi;
                    dot = fma(r.v, wi, dot);
                }
            });
        return dot;
    }

    // ================================================================== row stages without a tall-skinny block
    // ||b||^2 over this CTA's share (b is zero outside listB's rows)
    __device__ double bnorm2_part()
    {
        const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
        double bb = 0.0;
        for (int64_t t = b0 + warp; t < b1; t += 32) {
            const int64_t i = (int64_t)__ldg(P.listB + t) * 32 + lane;
            if (i < P.N) { const double v = P.b[i]; bb = fma(v, v, bb); }
        }
        return block_sum(bb, sh.red);
    }
    // UPDATE = true: x += a p, r -= a w (line 10, rank zero = Jacobi-CG).  false: r = b - w (lines 3, 12,
    // 16, Verify).  Then z~ = J r, ||r||^2, r^T z~.  Two slices per warp in flight.
    template <bool UPDATE, bool DENSE>
    __device__ void stage_rows_plain(double a, const double* p)
    {
        const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
        double rr = 0.0, rho = 0.0;
        __syncthreads();  // w of this CTA's rows was written by other threads of the CTA
        for (int64_t t = b0 + warp; t < b1; t += 64) {
            const int64_t i0 = (int64_t)list_entry<DENSE, 0>(P.listB, t) * 32 + lane;
            const bool two = t + 32 < b1;
            const int64_t i1 = two ? (int64_t)list_entry<DENSE, 0>(P.listB, t + 32) * 32 + lane : 0;
            const bool in0 = i0 < P.N, in1 = two && i1 < P.N;
            double w0 = 0.0, r0 = 0.0, d0 = 0.0, p0 = 0.0, x0 = 0.0, w1 = 0.0, r1 = 0.0, d1 = 0.0, p1 = 0.0, x1 = 0.0;
            if (in0) { w0 = P.w[i0]; d0 = ldg_f64(P.dinv + i0); if (UPDATE) { r0 = P.r[i0]; p0 = p[i0]; x0 = P.x[i0]; } else r0 = P.b[i0]; }
            if (in1) { w1 = P.w[i1]; d1 = ldg_f64(P.dinv + i1); if (UPDATE) { r1 = P.r[i1]; p1 = p[i1]; x1 = P.x[i1]; } else r1 = P.b[i1]; }
            if (in0) {
                const double rn = UPDATE ? fma(-a, w0, r0) : r0 - w0, zn = rn * d0;
                if (UPDATE) P.x[i0] = fma(a, p0, x0);
                P.r[i0] = rn;
                P.z[i0] = zn;
                rr = fma(rn, rn, rr);
                rho = fma(rn, zn, rho);
            }
            if (in1) {
                const double rn = UPDATE ? fma(-a, w1, r1) : r1 - w1, zn = rn * d1;
                if (UPDATE) P.x[i1] = fma(a, p1, x1);
                P.r[i1] = rn;
                P.z[i1] = zn;
                rr = fma(rn, rn, rr);
                rho = fma(rn, zn, rho);
            }
        }
        rr = block_sum(rr, sh.red);
        rho = block_sum(rho, sh.red);
        put(SL_RR, rr);
        put(SL_RHO, rho);
    }

    // ================================================================== tile streams over a tile-major n x kp block
    // one 32-row x kp tile (contiguous 256 kp bytes) of slice s into this consumer warp's slot
    __device__ __forceinline__ void issue_tile(const double* Mt, int64_t s, bool keep)
    {
        if ((threadIdx.x & 31) == 0) {
            const int warp = threadIdx.x >> 5;
            const uint32_t tile_bytes = 256u * (uint32_t)P.kp;
            void* tile = sh.ring + (size_t)warp * tile_bytes;
            uint64_t* bar = &sh.full[warp];
            mbar_arrive_expect_tx(bar, tile_bytes);
            // no reuse before the next iteration: evict_first keeps the gathered vectors and K in L2; when the working
            // set nearly fits the L2 the first hw_res_tiles tiles of every CTA are kept instead (evict_last)
            bulk_g2s_hint(tile, Mt + (size_t)s * 32 * P.kp, tile_bytes, bar, keep ? l2_policy_evict_last() : l2_policy_evict_first());
        }
    }
    // MODE (Mt = the tile-major copy of HW_I or of W_I):
    //   TS_UPDATE    r_i <- r_i - a w~_i + sum_j HW_ij (a nu_j), x~_i <- x~_i + a p~_i, z~_i <- r_i / d_i,
    //                ||r||^2, r^T z~, c_j = sum_i HW_ij z~_i                                  (line 10 + line 22; eq. (18))
    //   TS_RECOMP_Z  r = b - w, z~ = J r, ||r||^2, r^T z~, c = HW_I^T z~                      (after lines 3, 16)
    //   TS_RECOMP_R  r = b - w, z~ = J r, ||r||^2, r^T z~, c = W_I^T r                        (lines 3, 12: Q r needs Z^T r)
    //   TS_ADDW      x_i <- x_i + sign sum_j W_ij v_j     (x + Q r of lines 3 / 16 with v = mu; x = x~ - W_I xi with v = xi)
    template <int MODE, bool DENSE>
    __device__ void stage_tiles(const double* Mt, double a, const double* p, const double* v, double sign)
    {
        constexpr bool PASS1 = (MODE == TS_UPDATE || MODE == TS_ADDW);
        constexpr bool PASS2 = (MODE != TS_ADDW);
        const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
        const int kp = P.kp;
        const uint32_t tile_bytes = 256u * (uint32_t)kp;
        const int nst = min(32, (int)(RD_RING_BYTES / tile_bytes));
        const int64_t ntiles = b1 - b0;
        const int64_t N = P.N;
        double rr = 0.0, rho = 0.0;
        double acc[(RD_MAX_K + 31) / 32];
#pragma unroll
        for (int q = 0; q < (RD_MAX_K + 31) / 32; ++q) acc[q] = 0.0;
        __syncthreads();  // w~ of this CTA's rows was written by other threads of the CTA; v / anu are in place
        if (warp < nst) {
            double* tile = reinterpret_cast<double*>(sh.ring + (size_t)warp * tile_bytes);
            uint64_t* bar = &sh.full[warp];
            double* zbw = sh.zb[warp];
            int64_t t = warp;
            int32_t s = (t < ntiles) ? list_entry<DENSE, 0>(P.listB, b0 + t) : 0;
            int32_t sn = (t + nst < ntiles) ? list_entry<DENSE, 0>(P.listB, b0 + t + nst) : 0;
            double ri = 0.0, wi = 0.0, di = 0.0, pi = 0.0, xi_ = 0.0;
            auto load_rows = [&](int64_t i, double& r_, double& w_, double& d_, double& p_, double& x_) {
                r_ = w_ = d_ = p_ = x_ = 0.0;
                if (i < N) {
                    if (MODE == TS_UPDATE) { r_ = P.r[i]; w_ = P.w[i]; d_ = ldg_f64(P.dinv + i); p_ = p[i]; x_ = P.x[i]; }
                    else if (MODE == TS_ADDW) { x_ = P.x[i]; }
                    else { r_ = P.b[i]; w_ = P.w[i]; d_ = ldg_f64(P.dinv + i); }
                }
            };
            refill_fence();  // previous stage's generic reads of these bytes precede the CTA barrier above
            if (t < ntiles) {
                issue_tile(Mt, s, MODE == TS_UPDATE && t < P.hw_res_tiles);
                load_rows((int64_t)s * 32 + lane, ri, wi, di, pi, xi_);
            }
            for (; t < ntiles; t += nst) {
                const int64_t i = (int64_t)s * 32 + lane;
                const bool in = i < N;
                const int64_t tn = t + nst;
                const int32_t snn = (tn + nst < ntiles) ? list_entry<DENSE, 0>(P.listB, b0 + tn + nst) : 0;
                // next tile's row data: in flight while this tile is processed
                double rin = 0.0, win = 0.0, din = 0.0, pin = 0.0, xin = 0.0;
                if (tn < ntiles) load_rows((int64_t)sn * 32 + lane, rin, win, din, pin, xin);
                mbar_wait(bar, ph);
                ph ^= 1u;
                double q = 0.0;
                if (PASS1) {  // lane = row
                    double q0 = 0.0, q1 = 0.0, q2 = 0.0, q3 = 0.0;
                    const double* trow = tile + lane;
#pragma unroll 2
                    for (int j = 0; j < kp; j += 4) {
                        q0 = fma(trow[(j + 0) * 32], v[j + 0], q0);
                        q1 = fma(trow[(j + 1) * 32], v[j + 1], q1);
                        q2 = fma(trow[(j + 2) * 32], v[j + 2], q2);
                        q3 = fma(trow[(j + 3) * 32], v[j + 3], q3);
                    }
                    q = (q0 + q1) + (q2 + q3);
                }
                if (MODE == TS_ADDW) {
                    if (in) P.x[i] = fma(sign, q, xi_);
                } else {
                    const double rn = (MODE == TS_UPDATE) ? fma(-a, wi, ri) + q : ri - wi;
                    const double zn = in ? rn * di : 0.0;
                    if (in) {
                        P.r[i] = rn;
                        if (MODE == TS_UPDATE) P.x[i] = fma(a, pi, xi_);
                        P.z[i] = zn;
                        rr = fma(rn, rn, rr);
                        rho = fma(rn, zn, rho);
                    }
                    zbw[lane] = (MODE == TS_RECOMP_R) ? (in ? rn : 0.0) : zn;
                    __syncwarp();
                }
                if (PASS2) {  // lane = column(s) lane and lane + 32, rows in the skewed order (ii + lane) mod 32
                    if (lane < kp) {
                        const double* t0 = tile + lane * 32;
                        double a0_ = 0.0, a1_ = 0.0, b0_ = 0.0, b1_ = 0.0;
                        if (lane + 32 < kp) {
                            const double* t1 = t0 + 32 * 32;
#pragma unroll 8
                            for (int ii = 0; ii < 32; ii += 2) {
                                const int r0 = (ii + lane) & 31, r1 = (ii + 1 + lane) & 31;
                                const double z0 = zbw[r0], z1 = zbw[r1];
                                a0_ = fma(t0[r0], z0, a0_);
                                a1_ = fma(t0[r1], z1, a1_);
                                b0_ = fma(t1[r0], z0, b0_);
                                b1_ = fma(t1[r1], z1, b1_);
                            }
                        } else {
#pragma unroll 8
                            for (int ii = 0; ii < 32; ii += 2) {
                                const int r0 = (ii + lane) & 31, r1 = (ii + 1 + lane) & 31;
                                a0_ = fma(t0[r0], zbw[r0], a0_);
                                a1_ = fma(t0[r1], zbw[r1], a1_);
                            }
                        }
                        acc[0] += a0_ + a1_;
                        acc[1] += b0_ + b1_;
                    }
                }
                refill_fence();  // every lane has read the tile and zb: generic reads ordered before the async refill
                if (tn < ntiles) issue_tile(Mt, sn, MODE == TS_UPDATE && tn < P.hw_res_tiles);
                ri = rin; wi = win; di = din; pi = pin; xi_ = xin;
                s = sn;
                sn = snn;
            }
            if (PASS2) {
#pragma unroll
                for (int q_ = 0; q_ < (RD_MAX_K + 31) / 32; ++q_) {
                    const int j = lane + 32 * q_;
                    if (j < kp) sh.cpart[warp * kp + j] = acc[q_];
                }
            }
        }
        if (!PASS2) return;
        __syncthreads();
        if ((int)threadIdx.x < kp) {
            double vsum = 0.0;
            for (int cw = 0; cw < nst; ++cw) vsum += sh.cpart[cw * kp + threadIdx.x];
            slot(SL_NSCAL + threadIdx.x)[blockIdx.x] = vsum;
        }
        rr = block_sum(rr, sh.red);
        rho = block_sum(rho, sh.red);
        put(SL_RR, rr);
        put(SL_RHO, rho);
    }
};

// w = B v (both SpMVs with the barrier between them); v^T w goes to SL_DOT.
__device__ __forceinline__ void apply_B_plain(Cg3Cta& cta, const double* v)
{
    cta.opK<false, false>(v, nullptr, 0.0, nullptr);
    cta.sync_fetch(false, false);
    double d = cta.opKT<false>(v);
    d = block_sum(d, cta.sh.red);
    cta.put(SL_DOT, d);
}

// Algorithm 1, the whole solve (line numbers of SURVEY.md 8(c) O3).
__global__ void __launch_bounds__(RD_CG_THREADS, 1) k_alg1_v3(const CgParams P)
{
    extern __shared__ __align__(128) unsigned char smem_raw[];
    Cg3Shared& sh = *reinterpret_cast<Cg3Shared*>(smem_raw);
    Cg3Cta cta(P, sh);
    const bool coarse = P.use_coarse != 0;
    const int kp = P.kp;
    if (coarse)
        for (int q = threadIdx.x; q < kp * kp; q += blockDim.x) {
            const int i = q % kp, j = q / kp;
            sh.C[q] = P.C[q];
            sh.EW[q] = 0.5 * (P.EW[q] + P.EW[j + (size_t)i * kp]);
        }
    if (threadIdx.x < RD_MAX_K) {
        const int j = threadIdx.x;
        sh.xi[j] = 0.0; sh.nu[0][j] = 0.0; sh.nu[1][j] = 0.0; sh.g[0][j] = 0.0; sh.g[1][j] = 0.0; sh.sv[j] = 0.0; sh.anu[j] = 0.0;
        sh.e[j] = 0.0; sh.mu[j] = 0.0; sh.c[j] = 0.0;
    }
    // line 1: tau = eps_c ||b||_2
    {
        const double bb = cta.bnorm2_part();
        cta.put(SL_BB, bb);
    }
    // line 3: x <- x0 + Q (b - B x0);  r <- b - B x
    cta.opK<false, false>(P.x, nullptr, 0.0, nullptr);
    cta.sync_fetch(true, false);
    const double bnorm = sqrt(sh.scal[SL_BB]);
    const double tau = (bnorm > 0.0) ? P.eps_c * bnorm : P.eps_c;
    // ||r||_2 <= tau is tested as ||r||^2 <= tau^2 (no square root on the loop's critical path) unless tau^2 underflows
    const double tau2 = tau * tau;
    auto below_tau = [&](double rr) { return tau2 > 0.0 ? rr <= tau2 : sqrt(rr) <= tau; };
    __syncthreads();
    (void)cta.opKT<false>(P.x);
    int status = RD_ECAP_DEV;
    int iters = 0, replacements = 0;
    bool done = false;
    bool x_split = false;  // x = x~ - W_I xi with xi != 0
    double rho = 0.0, beta = 0.0;
    int cur = 0;

    if (coarse) {
        cta.stage_tiles<TS_RECOMP_R, false>(P.Wt, 0.0, nullptr, nullptr, 0.0);  // r = b - B x0, c = W_I^T r
        cta.sync_fetch(true, true);
        cta.coarse_solve();
        cta.stage_tiles<TS_ADDW, false>(P.Wt, 0.0, nullptr, sh.mu, 1.0);  // x += W_I C W_I^T r
        cta.sync_fetch(false, false);
        apply_B_plain(cta, P.x);
        cta.stage_tiles<TS_RECOMP_Z, false>(P.HWt, 0.0, nullptr, nullptr, 0.0);  // r = b - B x, z~ = J r, c = (HW_I)^T z~
    } else {
        cta.stage_rows_plain<false, false>(0.0, nullptr);
    }
    cta.sync_fetch(true, coarse);
    // lines 4-6
    if (below_tau(sh.scal[SL_RR])) { status = 0; done = true; }
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
        if (cta.dense) cta.opK<true, true>(P.z, pold, beta, pnew);
        else cta.opK<true, false>(P.z, pold, beta, pnew);
        cur ^= 1;
        cta.tick(0);
        cta.sync_fetch(false, false);
        cta.tick(1);
        // ---- stage B
        {
            double d = cta.dense ? cta.opKT<true>(pnew) : cta.opKT<false>(pnew);
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
        if (P.coef && blockIdx.x == 0 && threadIdx.x == 0 && iters <= P.coef_cap) P.coef[iters - 1] = make_double2(a, beta);
        if (coarse) {
            cta.coef_step(a);
            x_split = true;
            cta.tick(4);
            if (cta.dense) cta.stage_tiles<TS_UPDATE, true>(P.HWt, a, pnew, sh.anu, 0.0);
            else cta.stage_tiles<TS_UPDATE, false>(P.HWt, a, pnew, sh.anu, 0.0);
        } else {
            cta.tick(4);
            if (cta.dense) cta.stage_rows_plain<true, true>(a, pnew);
            else cta.stage_rows_plain<true, false>(a, pnew);
        }
        cta.tick(5);
        cta.sync_fetch(true, coarse);
        cta.tick(6);
        rho_prime = sh.scal[SL_RHO];
        // line 11
        const bool scheduled = P.replace_period > 0 && (iters % P.replace_period) == 0;
        if (below_tau(sh.scal[SL_RR]) || scheduled) {
            replacements++;
            if (x_split) {  // x = x~ - W_I xi
                cta.stage_tiles<TS_ADDW, false>(P.Wt, 0.0, nullptr, sh.xi, -1.0);
                __syncthreads();
                if (threadIdx.x < RD_MAX_K) sh.xi[threadIdx.x] = 0.0;
                x_split = false;
                cta.sync_fetch(false, false);
            }
            // line 12: recompute r = b - B x
            apply_B_plain(cta, P.x);
            if (coarse) cta.stage_tiles<TS_RECOMP_R, false>(P.Wt, 0.0, nullptr, nullptr, 0.0);
            else cta.stage_rows_plain<false, false>(0.0, nullptr);
            cta.sync_fetch(true, coarse);
            if (below_tau(sh.scal[SL_RR])) { status = 0; break; }  // lines 13-15
            if (coarse) {
                // line 16: x <- x + Q r; r <- b - B x
                cta.coarse_solve();
                cta.stage_tiles<TS_ADDW, false>(P.Wt, 0.0, nullptr, sh.mu, 1.0);
                cta.sync_fetch(false, false);
                apply_B_plain(cta, P.x);
                cta.stage_tiles<TS_RECOMP_Z, false>(P.HWt, 0.0, nullptr, nullptr, 0.0);
                cta.sync_fetch(true, true);
                if (below_tau(sh.scal[SL_RR])) { status = 0; break; }  // lines 17-19
            }
            rho_prime = sh.scal[SL_RHO];
            restart = true;  // line 20
        }
    }
    // line 26: Verify(x, eps) from a fresh apply on the explicit x
    const double rr_last = sh.scal[SL_RR];
    __syncthreads();
    if (x_split) {
        cta.stage_tiles<TS_ADDW, false>(P.Wt, 0.0, nullptr, sh.xi, -1.0);
        cta.sync_fetch(false, false);
    }
    apply_B_plain(cta, P.x);
    cta.stage_rows_plain<false, false>(0.0, nullptr);
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

}  // namespace rd
