// coarse.cuh -- S1 (restriction of the reference) and S2 (coarse setup) of every PDAS step.
//
//   S1  Wm = chi_I W               direct restriction, eq. (12); for the zero-extension
//                                  comparator rows whose DOF was active at an earlier restriction of the
//                                  sequence are zero as well, eq. (13) PAPER.md:158-162.
//   S2  G = Wm^T Wm                Gram matrix of the restricted candidate basis on the FP64 tensor cores (mma.sync DMMA)
//       T from G = V S V^T        rank-revealing transform T = V_r S_r^{-1/2} (keep S_j > 1e-14 S_max)
//       Zm = Wm T                 the basis Z of eq. (18), formed EXPLICITLY (orthonormal up to the rounding of G),
//                                 column-major and tile-major (k_alg1_v3's ring)
//       HZm = chi_I H Zm          r masked operator applies as a blocked SpMM (the cached "BZ")
//       E = Zm^T HZm              second DMMA contraction; cond(E) guard, Cholesky, C = E^{-1}
// E is formed from the Z that the iteration really uses, so Q = Z E^{-1} Z^T is the Galerkin projector of span(Z) to
// working accuracy however ill-conditioned W_I is (forming E = T^T (W_I^T H W_I) T instead amplifies the rounding of
// the k x k products by 1/S_min and breaks down on small or clustered inactive sets).
#pragma once
#include "dense.cuh"
#include "operator.cuh"

namespace rd {

// ---------------------------------------------------------------- S1
__global__ void k_restrict(int64_t N, int64_t ldw, int k, int kp, const double* W, const uint8_t* act,
                           const uint8_t* hist, int zeroext, double* Wm)
{
    for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < N; i += (int64_t)gridDim.x * blockDim.x) {
        const bool keep = !act[i] && !(zeroext && hist[i]);
        for (int j = 0; j < kp; ++j)
            Wm[i + (size_t)j * ldw] = (keep && j < k) ? ldg_f64(W + i + (size_t)j * ldw) : 0.0;
    }
}

// Zm = Wm T (N x kp by kp x kp; columns of T beyond the retained rank are zero), written column-major and, if Zt != NULL,
// tile-major for k_alg1_v3's ring: element (i, j) at (i / 32) * 32 kp + 32 j + i % 32 (one 32-row x kp tile = one
// contiguous 256 kp bytes).  One thread per row and 8 output columns (blockIdx.y = column chunk); T sits in shared
// memory and is read as broadcasts.
__global__ void __launch_bounds__(256) k_basis_transform(int64_t N, int64_t ldw, int kp, const double* Wm, const double* T,
                                                         double* Zm, double* Zt)
{
    extern __shared__ double sT[];  // kp x 8: the 8 columns of T of this chunk
    const int j0 = blockIdx.y * 8;
    for (int e = threadIdx.x; e < kp * 8; e += blockDim.x) sT[e] = T[(e % kp) + (size_t)(j0 + e / kp) * kp];
    __syncthreads();
    for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < N; i += (int64_t)gridDim.x * blockDim.x) {
        double acc[8];
#pragma unroll
        for (int q = 0; q < 8; ++q) acc[q] = 0.0;
        for (int l = 0; l < kp; ++l) {
            const double w = ldg_f64(Wm + i + (size_t)l * ldw);
#pragma unroll
            for (int q = 0; q < 8; ++q) acc[q] = fma(w, sT[l + q * kp], acc[q]);
        }
        double* zt = Zt ? Zt + (size_t)(i >> 5) * 32 * kp + (size_t)j0 * 32 + (i & 31) : nullptr;
#pragma unroll
        for (int q = 0; q < 8; ++q) {
            Zm[i + (size_t)(j0 + q) * ldw] = acc[q];
            if (zt) zt[q * 32] = acc[q];
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

// upper_only: the product is symmetric (A^T B with B = A or B = H A) and only the 64 x 64 tiles on or above the diagonal
// are formed; the caller mirrors them (k_mirror_upper_tiles).
__global__ void __launch_bounds__(256) k_gram_dmma(int64_t N, int p, int q, const double* A, int64_t lda,
                                                   const double* B, int64_t ldb, double* Cpart, int upper_only = 0)
{
    __shared__ double sA[64 * RD_GRAM_LD];
    __shared__ double sB[64 * RD_GRAM_LD];
    if (upper_only && blockIdx.z < blockIdx.y) return;
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

// Measurement helper (no arithmetic of the method): back-to-back m8n8k4 FP64 tensor-core operations on registers, eight
// independent accumulator tiles per warp -- the peak the Gram kernels' tensor-pipe utilisation is quoted against.
__global__ void __launch_bounds__(256) k_dmma_peak_probe(int iters, double seed, double* sink)
{
    double acc[8][2];
#pragma unroll
    for (int t = 0; t < 8; ++t) acc[t][0] = acc[t][1] = 0.0;
    double a = seed + 1e-3 * (threadIdx.x & 31), b = seed - 1e-3 * (threadIdx.x & 7);
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int t = 0; t < 8; ++t) dmma_m8n8k4(acc[t][0], acc[t][1], a, b);
        a = -a;  // keeps the accumulators bounded
    }
    double s = 0.0;
#pragma unroll
    for (int t = 0; t < 8; ++t) s += acc[t][0] + acc[t][1];
    if (s == 123.456) sink[0] = s;  // never true: keeps the loop alive
}

// G (p x p): the 64 x 64 tiles below the diagonal <- the transposes of the tiles above it
__global__ void k_mirror_upper_tiles(int p, double* G)
{
    for (int e = blockIdx.x * blockDim.x + threadIdx.x; e < p * p; e += gridDim.x * blockDim.x) {
        const int i = e % p, j = e / p;
        if ((i >> 6) > (j >> 6)) G[e] = G[j + (size_t)i * p];
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

// Step 1 of the k x k part.  In: G = Wm^T Wm (kp x kp).  Work: 2 kp x kp scratch.  Out: T (kp x kp, column-major):
// G = V S V^T (Jacobi), keep S_j > 1e-14 S_max (singular values of W_I above 1e-7 relative; reading A6 of DESIGN.md:
// the paper's QR + SVD threshold is 1e-12), T[:, q] = V[:, sel_q] S_sel_q^{-1/2} for q < rank, zero
// columns beyond; info->rank.
__global__ void __launch_bounds__(1024) k_coarse_T(int kp, const double* G, double* work, double* T, CoarseInfo* info)
{
    __shared__ DenseShared ds;
    __shared__ int sel[RD_MAX_K];
    __shared__ int s_rank;
    const int n = kp;
    const size_t nn = (size_t)n * n;
    double* A1 = work;       // G -> eigenvalues on the diagonal
    double* V = work + nn;   // eigenvectors
    for (int e = threadIdx.x; e < (int)nn; e += blockDim.x) A1[e] = G[e];
    __syncthreads();
    cta_symmetrize(A1, n, n);
    cta_jacobi_eig(A1, n, n, V, n, true, ds);
    if (threadIdx.x == 0) {
        double smax = 0.0;
        for (int j = 0; j < n; ++j) smax = fmax(smax, A1[j + (size_t)j * n]);
        int r = 0;
        for (int j = 0; j < n; ++j)
            if (smax > 0.0 && A1[j + (size_t)j * n] > 1e-14 * smax) sel[r++] = j;
        s_rank = r;
        info->rank = r;
        info->fallback = 0;
        info->cond_E = 0.0;
    }
    __syncthreads();
    const int r = s_rank;
    for (int e = threadIdx.x; e < (int)nn; e += blockDim.x) {
        const int i = e % n, q = e / n;
        double v = 0.0;
        if (q < r) { const int j = sel[q]; v = V[i + (size_t)j * n] * rsqrt(A1[j + (size_t)j * n]); }
        T[e] = v;
    }
}

// Step 2 of the k x k part.  In: E_raw = Zm^T HZm (kp x kp; rows / columns >= rank are zero), T, rank.  Work: 4 kp x kp.
// Out: E (kp x kp, symmetrised, zero outside the leading rank x rank block), C = E^{-1} (same padding): the coarse solve
// of eq. (18) in Z coordinates, CW = T E^{-1} T^T: the same solve in W_I coordinates (diagnostics: rd_coarse_setup,
// rd_energy_fraction), cond_2(E) from a Jacobi eigensolve, rank-zero fallback above 1e10 or if E is not SPD.
__global__ void __launch_bounds__(1024) k_coarse_E(int kp, const double* Eraw, const double* T, double* work, double* E,
                                                   double* C, double* CW, CoarseInfo* info)
{
    __shared__ DenseShared ds;
    __shared__ double s_lmin, s_lmax;
    const int n = kp;
    const size_t nn = (size_t)n * n;
    const int r = info->rank;
    double* A1 = work;            // copy of E for the eigenvalues; later L^{-1}
    double* A4 = work + nn;       // L (Cholesky of E); later T E^{-1}
    double* A3 = work + 2 * nn;   // E^{-1} (r x r)
    for (int e = threadIdx.x; e < (int)nn; e += blockDim.x) {
        const int i = e % n, j = e / n;
        E[e] = (i < r && j < r) ? 0.5 * (Eraw[i + (size_t)j * n] + Eraw[j + (size_t)i * n]) : 0.0;
        C[e] = 0.0;
        CW[e] = 0.0;
    }
    __syncthreads();
    if (r == 0) return;
    for (int e = threadIdx.x; e < (int)nn; e += blockDim.x) { A1[e] = E[e]; A4[e] = E[e]; }
    __syncthreads();
    cta_jacobi_eig(A1, n, r, nullptr, 0, false, ds);
    if (threadIdx.x == 0) {
        double lmin = A1[0], lmax = A1[0];
        for (int j = 1; j < r; ++j) { lmin = fmin(lmin, A1[j + (size_t)j * n]); lmax = fmax(lmax, A1[j + (size_t)j * n]); }
        s_lmin = lmin; s_lmax = lmax;
    }
    __syncthreads();
    const double cond = (s_lmin > 0.0) ? s_lmax / s_lmin : INFINITY;
    const bool ok = cta_cholesky(A4, n, r, ds);
    if (!(cond <= 1e10) || !ok) {
        if (threadIdx.x == 0) { info->rank = 0; info->fallback = 1; info->cond_E = cond; }
        return;
    }
    cta_tri_inverse_lower(A4, n, r, A1, n);                  // A1 = L^{-1}
    cta_matmul(r, r, r, A1, n, 1, A1, 1, n, A3, n);          // A3 = L^{-T} L^{-1} = E^{-1}
    for (int e = threadIdx.x; e < r * r; e += blockDim.x) {
        const int i = e % r, j = e / r;
        C[i + (size_t)j * n] = 0.5 * (A3[i + (size_t)j * n] + A3[j + (size_t)i * n]);
    }
    __syncthreads();
    cta_matmul(n, r, r, T, 1, n, C, 1, n, A4, n);            // A4 = T E^{-1}     (n x r)
    cta_matmul(n, n, r, A4, 1, n, T, n, 1, CW, n);           // CW = T E^{-1} T^T (n x n)
    cta_symmetrize(CW, n, n);
    if (threadIdx.x == 0) { info->fallback = 0; info->cond_E = cond; }
}

// ---------------------------------------------------------------- eq. (23): spectrum the deflated, Jacobi-preconditioned CG sees
// The step lengths a_j and direction coefficients beta_j of a CG run define the Lanczos tridiagonal matrix of the
// operator CG iterates with -- for Algorithm 1 that is D^{-1/2} B P D^{-1/2} = B^ - D^{-1/2} B Z E^{-1} Z^T B D^{-1/2}, the
// matrix of eq. (23), on the complement of its null space:
//     T_jj = 1/a_j + beta_j / a_{j-1},    T_{j,j-1} = sqrt(beta_j) / a_{j-1}        (beta = 0 where the direction restarts)
// Its eigenvalues (Ritz values) lie inside the nonzero spectrum and the extreme ones converge to its ends.  One CTA:
// the last restart-free segment of the m recorded pairs, extreme eigenvalues by multisection on Sturm counts.
// out[0] = smallest, out[1] = largest Ritz value, out[2] = segment length.
__global__ void __launch_bounds__(1024) k_ritz_extremes(int m, const double2* coef, double* out)
{
    __shared__ int s_start;
    __shared__ double s_lo[2], s_hi[2];
    __shared__ int s_pick[2];
    if (threadIdx.x == 0) {
        int st = 0;
        for (int j = m - 1; j > 0; --j)
            if (coef[j].y == 0.0) { st = j; break; }
        // a trailing restart (the replacement branch that ends a solve) leaves a segment of length one: take the one before
        if (m - st < 3) {
            const int end = st;
            st = 0;
            for (int j = end - 1; j > 0; --j)
                if (coef[j].y == 0.0) { st = j; break; }
            m = end;
        }
        s_start = st;
        s_pick[0] = m;  // reuse: segment end
    }
    __syncthreads();
    const int j0 = s_start, j1 = s_pick[0], len = j1 - j0;
    __syncthreads();
    if (len < 1) {
        if (threadIdx.x == 0) { out[0] = 0.0; out[1] = 0.0; out[2] = 0.0; }
        return;
    }
    auto diag = [&](int j) { return 1.0 / coef[j].x + (j > j0 ? coef[j].y / coef[j - 1].x : 0.0); };
    auto off2 = [&](int j) { return coef[j].y / (coef[j - 1].x * coef[j - 1].x); };  // T_{j,j-1}^2, j > j0
    if (threadIdx.x == 0) {  // Gershgorin bounds
        double lo = 1e300, hi = -1e300;
        for (int j = j0; j < j1; ++j) {
            const double d = diag(j);
            const double r = (j > j0 ? sqrt(off2(j)) : 0.0) + (j + 1 < j1 ? sqrt(off2(j + 1)) : 0.0);
            lo = fmin(lo, d - r);
            hi = fmax(hi, d + r);
        }
        lo = fmax(lo, 0.0);  // the operator is positive semidefinite
        s_lo[0] = s_lo[1] = lo;
        s_hi[0] = s_hi[1] = hi * (1.0 + 1e-12) + 1e-300;
    }
    __syncthreads();
    // number of eigenvalues of T below x (Sturm sequence of the LDL^T pivots)
    auto count_below = [&](double x) {
        int cnt = 0;
        double q = 1.0;
        for (int j = j0; j < j1; ++j) {
            q = diag(j) - x - (j > j0 ? off2(j) / q : 0.0);
            if (q == 0.0) q = -1e-300;
            cnt += q < 0.0;
        }
        return cnt;
    };
    for (int which = 0; which < 2; ++which) {  // 0: smallest (first x with count >= 1), 1: largest (first x with count >= len)
        const int want = which == 0 ? 1 : len;
        for (int round = 0; round < 7; ++round) {
            const double lo = s_lo[which], hi = s_hi[which];
            const double x = lo + (hi - lo) * (double)(threadIdx.x + 1) / (double)(blockDim.x + 1);
            const bool ok = count_below(x) >= want;
            if (threadIdx.x == 0) s_pick[1] = blockDim.x;
            __syncthreads();
            if (ok) atomicMin(&s_pick[1], (int)threadIdx.x);
            __syncthreads();
            const int t = s_pick[1];
            __syncthreads();
            if (threadIdx.x == 0) {
                const double w = (hi - lo) / (double)(blockDim.x + 1);
                s_lo[which] = lo + w * t;          // count(lo + w t) < want (or t = 0: lo itself)
                s_hi[which] = lo + w * (t + 1);    // count >= want (or t = blockDim: hi itself)
            }
            __syncthreads();
        }
    }
    if (threadIdx.x == 0) {
        out[0] = 0.5 * (s_lo[0] + s_hi[0]);
        out[1] = 0.5 * (s_lo[1] + s_hi[1]);
        out[2] = (double)len;
    }
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
