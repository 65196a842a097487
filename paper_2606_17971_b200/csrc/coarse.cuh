// coarse.cuh -- S1 (restriction of the reference) and S2 (coarse setup) of every PDAS step.
//
//   S1  Wm = chi_I W               direct restriction, eq. (12); for the zero-extension
//                                  comparator rows whose DOF was active at an earlier restriction of the
//                                  sequence are zero as well, eq. (13) PAPER.md:158-162.
//   S2  HWm = chi_I H Wm           k masked operator applies as a blocked SpMM (cached "BZ")
//       G = Wm^T Wm, EW = Wm^T HWm two N x k by k contractions on the FP64 tensor cores (mma.sync DMMA)
//       rank-revealing T from G, E = T^T EW T, cond(E) guard, Cholesky, C = T E^{-1} T^T
#pragma once
#include "dense.cuh"
#include "operator.cuh"

namespace rd {

// ---------------------------------------------------------------- S1
// Wt (may be NULL): the same block written tile-major for k_alg1_v3's ring, element (i, j) at
// (i / 32) * 32 kp + 32 j + i % 32 (one 32-row x kp tile = one contiguous 256 kp bytes), like HWt below.
__global__ void k_restrict(int64_t N, int64_t ldw, int k, int kp, const double* W, const uint8_t* act,
                           const uint8_t* hist, int zeroext, double* Wm, double* Wt)
{
    for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < N; i += (int64_t)gridDim.x * blockDim.x) {
        const bool keep = !act[i] && !(zeroext && hist[i]);
        double* wt = Wt ? Wt + (size_t)(i >> 5) * 32 * kp + (i & 31) : nullptr;
        for (int j = 0; j < kp; ++j) {
            const double v = (keep && j < k) ? ldg_f64(W + i + (size_t)j * ldw) : 0.0;
            Wm[i + (size_t)j * ldw] = v;
            if (wt) wt[(size_t)j * 32] = v;
        }
    }
}
// zero-extension history: A <- A u J after every restriction (reading A9 in DESIGN.md)
__global__ void k_hist_update(int64_t N, const uint8_t* act, uint8_t* hist)
{
    for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < N; i += (int64_t)gridDim.x * blockDim.x)
        if (act[i]) hist[i] = 1;
}

// ---------------------------------------------------------------- S2: blocked SpMM, CB columns per pass
template <int CB>
__global__ void k_spmm_K(Ell K, int64_t N, int64_t ldv, const double* minv, const double* V, int64_t ldt, double* T)
{
    const int lane = threadIdx.x & 31;
    const int64_t gw = ((int64_t)blockIdx.x * blockDim.x + threadIdx.x) >> 5;
    const int64_t nwt = ((int64_t)gridDim.x * blockDim.x) >> 5;
    for (int64_t s = gw; s < K.nslices; s += nwt) {
        const int64_t row = s * RD_SLICE + lane;
        const int64_t o = K.off[s];
        const int wd = (int)((K.off[s + 1] - o) >> 5);
        double acc[CB];
#pragma unroll
        for (int q = 0; q < CB; ++q) acc[q] = 0.0;
        for (int e = 0; e < wd; ++e) {
            const int c = ldg_i32(K.col + o + e * 32 + lane);
            const double a = ldg_f64(K.val + o + e * 32 + lane);
#pragma unroll
            for (int q = 0; q < CB; ++q) acc[q] = fma(a, V[c + (size_t)q * ldv], acc[q]);
        }
        if (row < N) {
            const double mi = minv ? minv[row] : 1.0;
#pragma unroll
            for (int q = 0; q < CB; ++q) T[row + (size_t)q * ldt] = acc[q] * mi;
        }
    }
}

template <int CB>
__global__ void k_spmm_KT(Ell KT, int64_t N, int64_t ldv, const double* m, double sigma, const uint8_t* act,
                          const double* V, int64_t ldt, const double* T, int64_t ldo, double* OUT, double* OUTT, int kp,
                          int jbase)
{
    // OUTT (may be NULL): the same block written tile-major for k_alg1_v3's ring, element (i, j) of the N x kp
    // matrix at (i / 32) * 32 kp + 32 j + i % 32, so that a 32-row x kp tile is one contiguous 256 kp bytes.
    const int lane = threadIdx.x & 31;
    const int64_t gw = ((int64_t)blockIdx.x * blockDim.x + threadIdx.x) >> 5;
    const int64_t nwt = ((int64_t)gridDim.x * blockDim.x) >> 5;
    for (int64_t s = gw; s < KT.nslices; s += nwt) {
        const int64_t row = s * RD_SLICE + lane;
        const int64_t o = KT.off[s];
        const int wd = (int)((KT.off[s + 1] - o) >> 5);
        double acc[CB];
#pragma unroll
        for (int q = 0; q < CB; ++q) acc[q] = 0.0;
        for (int e = 0; e < wd; ++e) {
            const int c = ldg_i32(KT.col + o + e * 32 + lane);
            const double a = ldg_f64(KT.val + o + e * 32 + lane);
#pragma unroll
            for (int q = 0; q < CB; ++q) acc[q] = fma(a, T[c + (size_t)q * ldt], acc[q]);
        }
        if (row < N) {
            const double mi = m[row];
            const bool zero = act && act[row];
            double* ot = OUTT ? OUTT + (size_t)s * 32 * kp + (size_t)jbase * 32 + lane : nullptr;
#pragma unroll
            for (int q = 0; q < CB; ++q) {
                const double o_ = zero ? 0.0 : fma(sigma, acc[q], mi * V[row + (size_t)q * ldv]);
                OUT[row + (size_t)q * ldo] = o_;
                if (ot) ot[q * 32] = o_;
            }
        }
    }
}

// ---------------------------------------------------------------- S2: Gram products on FP64 tensor cores
// Cpart[blockIdx.x] (p x q, column-major, ld = p) = A[rows of this CTA, :]^T B[rows of this CTA, :]
// A: N x p, B: N x q column-major, p and q multiples of 8.  grid = (row chunks, ceil(p/64), ceil(q/64)),
// 256 threads: warp w owns the 8 A-columns [64 by + 8w, +8) against up to 64 B-columns, i.e. eight
// m8n8k4 DMMA accumulator tiles; 32 rows are staged per step in shared memory.
#define RD_GRAM_R 32
#define RD_GRAM_LD (RD_GRAM_R + 4)

__device__ __forceinline__ void dmma_m8n8k4(double& d0, double& d1, double a, double b)
{
    asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};"
                 : "+d"(d0), "+d"(d1)
                 : "d"(a), "d"(b));
}

__global__ void __launch_bounds__(256) k_gram_dmma(int64_t N, int p, int q, const double* A, int64_t lda,
                                                   const double* B, int64_t ldb, double* Cpart)
{
    __shared__ double sA[64 * RD_GRAM_LD];
    __shared__ double sB[64 * RD_GRAM_LD];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int i0 = blockIdx.y * 64, j0 = blockIdx.z * 64;
    const int pa = min(64, p - i0), qb = min(64, q - j0);
    const int64_t nchunks = (N + RD_GRAM_R - 1) / RD_GRAM_R;
    const int64_t per = (nchunks + gridDim.x - 1) / gridDim.x;
    const int64_t c0 = min((int64_t)blockIdx.x * per, nchunks), c1 = min(c0 + per, nchunks);
    double acc[8][2];
#pragma unroll
    for (int t = 0; t < 8; ++t) acc[t][0] = acc[t][1] = 0.0;
    const int am = lane >> 2, ak = lane & 3;
    for (int64_t ch = c0; ch < c1; ++ch) {
        const int64_t r0 = ch * RD_GRAM_R;
        __syncthreads();
        for (int cidx = warp; cidx < 64; cidx += 8) {
            const int64_t row = r0 + lane;
            sA[cidx * RD_GRAM_LD + lane] = (cidx < pa && row < N) ? ldg_f64(A + row + (size_t)(i0 + cidx) * lda) : 0.0;
            sB[cidx * RD_GRAM_LD + lane] = (cidx < qb && row < N) ? ldg_f64(B + row + (size_t)(j0 + cidx) * ldb) : 0.0;
        }
        __syncthreads();
        if (warp * 8 < pa) {
#pragma unroll
            for (int kk = 0; kk < RD_GRAM_R; kk += 4) {
                const double a = sA[(warp * 8 + am) * RD_GRAM_LD + kk + ak];
#pragma unroll
                for (int t = 0; t < 8; ++t) {
                    if (t * 8 < qb) {
                        const double b = sB[(t * 8 + am) * RD_GRAM_LD + kk + ak];
                        dmma_m8n8k4(acc[t][0], acc[t][1], a, b);
                    }
                }
            }
        }
    }
    if (warp * 8 < pa) {
        double* Cp = Cpart + (size_t)blockIdx.x * p * q;
#pragma unroll
        for (int t = 0; t < 8; ++t) {
            if (t * 8 < qb) {
                const int gi = i0 + warp * 8 + am, gj = j0 + t * 8 + 2 * ak;
                Cp[gi + (size_t)gj * p] = acc[t][0];
                Cp[gi + (size_t)(gj + 1) * p] = acc[t][1];
            }
        }
    }
}

// out[e] = sum over parts of part[part][e], fixed order (deterministic)
__global__ void k_reduce_parts(int nparts, int64_t len, const double* parts, double* out)
{
    for (int64_t e = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; e < len; e += (int64_t)gridDim.x * blockDim.x) {
        double a = 0.0;
        for (int pI = 0; pI < nparts; ++pI) a += parts[(size_t)pI * len + e];
        out[e] = a;
    }
}

// ---------------------------------------------------------------- S2: the k x k part, one CTA
struct CoarseInfo {
    int32_t rank, fallback;
    double cond_E;
};

// In:  G, EW (kp x kp, column-major, ld kp).  Work: 6 kp x kp scratch matrices.  Out: C = T E^{-1} T^T
// (kp x kp), info.  Reading A6 of DESIGN.md: G = V S V^T (Jacobi), keep S_j > 1e-14 S_max (singular
// values of W_I above 1e-7 relative; the paper's QR + SVD threshold is 1e-12),
// T = V_r S_r^{-1/2}, so Z = W_I T has orthonormal columns; E = T^T EW T = Z^T B Z (eq. (18));
// cond_2(E) from a Jacobi eigensolve, rank-zero fallback above 1e10.
__global__ void __launch_bounds__(1024) k_coarse_small(int kp, const double* G, const double* EW, double* work,
                                                       double* C, CoarseInfo* info)
{
    __shared__ DenseShared ds;
    __shared__ int sel[RD_MAX_K];
    __shared__ int s_rank;
    __shared__ double s_lmin, s_lmax;
    const int n = kp;
    const size_t nn = (size_t)n * n;
    double* A1 = work;            // G -> eigenvalues on the diagonal; later copy of E for cond; later L^{-1}
    double* V = work + nn;        // eigenvectors -> T (in place)
    double* A3 = work + 2 * nn;   // EW symmetrised; later E^{-1}
    double* A4 = work + 3 * nn;   // EW T ; later L (Cholesky of E); later T E^{-1}
    double* E = work + 4 * nn;    // E
    for (int e = threadIdx.x; e < (int)nn; e += blockDim.x) { A1[e] = G[e]; A3[e] = EW[e]; }
    __syncthreads();
    cta_symmetrize(A1, n, n);
    cta_symmetrize(A3, n, n);
    cta_jacobi_eig(A1, n, n, V, n, true, ds);
    if (threadIdx.x == 0) {
        double smax = 0.0;
        for (int j = 0; j < n; ++j) smax = fmax(smax, A1[j + (size_t)j * n]);
        int r = 0;
        for (int j = 0; j < n; ++j)
            if (smax > 0.0 && A1[j + (size_t)j * n] > 1e-14 * smax) sel[r++] = j;
        s_rank = r;
    }
    __syncthreads();
    int r = s_rank;
    // T = V[:, sel] diag(S_sel^{-1/2}), compacted to the left in place (sel[q] >= q): column by column
    for (int qc = 0; qc < r; ++qc) {
        const int j = sel[qc];
        const double sc = rsqrt(A1[j + (size_t)j * n]);
        __syncthreads();
        for (int i = threadIdx.x; i < n; i += blockDim.x) V[i + (size_t)qc * n] = V[i + (size_t)j * n] * sc;
    }
    __syncthreads();
    bool fallback = false;
    double cond = 0.0;
    if (r > 0) {
        cta_matmul(n, r, n, A3, 1, n, V, 1, n, A4, n);       // A4 = EW T         (n x r)
        cta_matmul(r, r, n, V, n, 1, A4, 1, n, E, n);        // E  = T^T EW T     (r x r)
        cta_symmetrize(E, n, r);
        for (int e = threadIdx.x; e < r * r; e += blockDim.x) A1[(e % r) + (size_t)(e / r) * n] = E[(e % r) + (size_t)(e / r) * n];
        cta_jacobi_eig(A1, n, r, nullptr, 0, false, ds);
        if (threadIdx.x == 0) {
            double lmin = A1[0], lmax = A1[0];
            for (int j = 1; j < r; ++j) { lmin = fmin(lmin, A1[j + (size_t)j * n]); lmax = fmax(lmax, A1[j + (size_t)j * n]); }
            s_lmin = lmin; s_lmax = lmax;
        }
        __syncthreads();
        cond = (s_lmin > 0.0) ? s_lmax / s_lmin : INFINITY;
        for (int e = threadIdx.x; e < r * r; e += blockDim.x) A4[(e % r) + (size_t)(e / r) * n] = E[(e % r) + (size_t)(e / r) * n];
        bool ok = cta_cholesky(A4, n, r, ds);
        if (!(cond <= 1e10) || !ok) { fallback = true; }
    }
    if (fallback || r == 0) {
        for (int e = threadIdx.x; e < (int)nn; e += blockDim.x) C[e] = 0.0;
        if (threadIdx.x == 0) { info->rank = 0; info->fallback = fallback ? 1 : 0; info->cond_E = cond; }
        return;
    }
    cta_tri_inverse_lower(A4, n, r, A1, n);                  // A1 = L^{-1}
    cta_matmul(r, r, r, A1, n, 1, A1, 1, n, A3, n);          // A3 = L^{-T} L^{-1} = E^{-1}   (sum over k >= max(i,j); zeros above)
    cta_matmul(n, r, r, V, 1, n, A3, 1, n, A4, n);           // A4 = T E^{-1}     (n x r)
    cta_matmul(n, n, r, A4, 1, n, V, n, 1, C, n);            // C  = T E^{-1} T^T (n x n)
    cta_symmetrize(C, n, n);
    if (threadIdx.x == 0) { info->rank = r; info->fallback = 0; info->cond_E = cond; }
}

// ---------------------------------------------------------------- eq. (24): energy fraction of the coarse correction
// parts[blockIdx.x * (kp + 1) + j] = sum over this block's rows of Wm[i, j] * b[i]  (j < kp: c = W_I^T b) and, at
// j = kp, of x[i] * Hx[i]  (||x_*||_B^2; x and Hx are zero on J).  Wm column-major with leading dimension ldw:
// each column is a contiguous stream, rows split evenly over the blocks, fixed summation order.
__global__ void __launch_bounds__(256) k_energy_parts(int64_t N, int64_t ldw, int kp, const double* Wm, const double* b,
                                                      const double* x, const double* Hx, double* parts)
{
    __shared__ double scratch[32];
    const int64_t chunk = (N + gridDim.x - 1) / gridDim.x;
    const int64_t i0 = (int64_t)blockIdx.x * chunk, i1 = (i0 + chunk < N) ? i0 + chunk : N;
    for (int j = 0; j <= kp; ++j) {
        const double* u = (j < kp) ? Wm + (size_t)j * ldw : x;
        const double* v = (j < kp) ? b : Hx;
        double a = 0.0;
        for (int64_t i = i0 + threadIdx.x; i < i1; i += blockDim.x) a = fma(ldg_f64(u + i), ldg_f64(v + i), a);
        a = block_sum(a, scratch);
        if (threadIdx.x == 0) parts[(size_t)blockIdx.x * (kp + 1) + j] = a;
    }
}

// One CTA: out[0] = c^T C c = ||Qb||_B^2 (Q = W_I C W_I^T, C E_W C = C), out[1] = ||x_*||_B^2, out[2] = chi = out[0] / out[1].
// v = the reduced vector of k_energy_parts (kp + 1 entries); use_coarse = 0 for rank zero (Q = 0).
__global__ void __launch_bounds__(64) k_energy_fraction(int kp, int use_coarse, const double* C, const double* v, double* out)
{
    __shared__ double scratch[32];
    double a = 0.0;
    if (use_coarse && (int)threadIdx.x < kp) {
        double s = 0.0;
        for (int l = 0; l < kp; ++l) s = fma(C[(size_t)l * kp + threadIdx.x], v[l], s);
        a = v[threadIdx.x] * s;
    }
    a = block_sum(a, scratch);
    if (threadIdx.x == 0) {
        out[0] = a;
        out[1] = v[kp];
        out[2] = v[kp] > 0.0 ? a / v[kp] : 0.0;
    }
}

}  // namespace rd
