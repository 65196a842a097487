// eigs.cuh -- S0: reference construction.  The k lowest eigenpairs of the full H = M + sigma K^T M^{-1} K
// (BASELINE.json north_star; nearest paper text: Alg. 2 step 2 "lowest ... eigenvectors", built
// once before the sequence) by a block Krylov method written for the GPU: Chebyshev-filtered
// subspace iteration with Rayleigh-Ritz on a block of b = k + guard vectors.
//
//   filter   Y_{j+1} = c1 (H Y_j - c Y_j) + c2 Y_{j-1}   two blocked SpMMs per degree, nothing else: no
//                                                        reductions, no host round trip inside a sweep
//   orth     G = X^T X on the FP64 tensor cores, Jacobi-scaled, b x b eigensolve in one CTA, X <- X T
//   RR       A = X^T (H X), eigensolve, X <- X V, residuals ||H x_j - theta_j x_j||
//
// Every degree of the filter applies H to all b columns at once, 8 columns per pass over K and K^T, so the
// matrices stream once per 8 vectors and the work is bandwidth-bound instead of latency-bound.  A Krylov method
// with one vector (Lanczos) needs fewer operator applies in total but runs them one after another.
#pragma once
#include "coarse.cuh"

namespace rd {

#define RD_EIG_CB 8      // columns per SpMM pass
#define RD_EIG_MAXB 128  // block size limit (k <= 64 plus guard)

// (Round 2 tried kernels specialised on the uniform row width with all indices / values loaded before the gathers and the
// row's own Y / Yprev entries prefetched: slower on B200 -- config 2 build 10.05 s against 9.02 s, config 3 7.9 s against
// 6.9 s, 78 registers in the K^T kernel -- so the rolled loops below stay.)
// (Also tried in round 2, commit d22bb87: 4 and 16 columns per pass.  Build times 8 / 4 / 16 columns: config 2 9.05 / 10.08 /
// 9.95 s, config 3 6.69 / 6.31 / 5.91 s, config 5 123.4 / 127.0 / 128.0 s: 8 stays.  ncu: the two kernels run at 35-43 % of
// the DRAM peak with 54 % warp occupancy -- bound by the latency of the gathers, not by bytes; profiles/r2_summary.md.)
// T[:, chunk] = M^{-1} K Y[:, chunk]; chunk = blockIdx.y selects RD_EIG_CB columns
#define CB RD_EIG_CB
__global__ void k_blk_K(Ell K, int64_t N, int64_t ld, const double* minv, const double* Y, double* T)
{
    const int lane = threadIdx.x & 31;
    const int64_t gw = ((int64_t)blockIdx.x * blockDim.x + threadIdx.x) >> 5;
    const int64_t nwt = ((int64_t)gridDim.x * blockDim.x) >> 5;
    const size_t cofs = (size_t)blockIdx.y * CB * ld;
    const double* V = Y + cofs;
    double* O = T + cofs;
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
            for (int q = 0; q < CB; ++q) acc[q] = fma(a, V[c + (size_t)q * ld], acc[q]);
        }
        if (row < N) {
            const double mi = minv[row];
#pragma unroll
            for (int q = 0; q < CB; ++q) O[row + (size_t)q * ld] = acc[q] * mi;
        }
    }
}

// Ynext[:, chunk] = c1 ( (m .* Y + sigma K^T T) - cshift Y ) + c2 Yprev     (Yprev may be NULL when c2 == 0)
// c1 = 1, cshift = 0, c2 = 0 gives the plain block apply H Y.
__global__ void k_blk_KT(Ell KT, int64_t N, int64_t ld, const double* m, double sigma, double c1, double cshift,
                         double c2, const double* Y, const double* T, const double* Yprev, double* Ynext)
{
    const int lane = threadIdx.x & 31;
    const int64_t gw = ((int64_t)blockIdx.x * blockDim.x + threadIdx.x) >> 5;
    const int64_t nwt = ((int64_t)gridDim.x * blockDim.x) >> 5;
    const size_t cofs = (size_t)blockIdx.y * CB * ld;
    const double* Tc = T + cofs;
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
            for (int q = 0; q < CB; ++q) acc[q] = fma(a, Tc[c + (size_t)q * ld], acc[q]);
        }
        if (row < N) {
            const double mi = m[row] - cshift;
#pragma unroll
            for (int q = 0; q < CB; ++q) {
                const size_t idx = cofs + row + (size_t)q * ld;
                double h = fma(sigma, acc[q], mi * Y[idx]);
                h *= c1;
                if (Yprev) h = fma(c2, Yprev[idx], h);
                Ynext[idx] = h;
            }
        }
    }
}

#undef CB

// Upper bound of the spectrum (Gershgorin on |H| <= M + sigma |K|^T M^{-1} |K|):
//   s_r = (1/m_r) sum_c |K_rc|,   bound = max_i ( m_i + sigma sum_r |K_ri| s_r )
__global__ void k_abs_rowsum(Ell K, int64_t N, const double* minv, double* s)
{
    const int lane = threadIdx.x & 31;
    const int64_t gw = ((int64_t)blockIdx.x * blockDim.x + threadIdx.x) >> 5;
    const int64_t nwt = ((int64_t)gridDim.x * blockDim.x) >> 5;
    for (int64_t sl = gw; sl < K.nslices; sl += nwt) {
        const int64_t row = sl * RD_SLICE + lane;
        const int64_t o = K.off[sl];
        const int wd = (int)((K.off[sl + 1] - o) >> 5);
        double acc = 0.0;
        for (int e = 0; e < wd; ++e) acc += fabs(K.val[o + e * 32 + lane]);
        if (row < N) s[row] = acc * minv[row];
    }
}
__global__ void k_gershgorin(Ell KT, int64_t N, const double* m, double sigma, const double* s,
                             unsigned long long* bound_bits)
{
    const int lane = threadIdx.x & 31;
    const int64_t gw = ((int64_t)blockIdx.x * blockDim.x + threadIdx.x) >> 5;
    const int64_t nwt = ((int64_t)gridDim.x * blockDim.x) >> 5;
    double mx = 0.0;
    for (int64_t sl = gw; sl < KT.nslices; sl += nwt) {
        const int64_t row = sl * RD_SLICE + lane;
        const int64_t o = KT.off[sl];
        const int wd = (int)((KT.off[sl + 1] - o) >> 5);
        double acc = 0.0;
        for (int e = 0; e < wd; ++e) acc = fma(fabs(KT.val[o + e * 32 + lane]), s[KT.col[o + e * 32 + lane]], acc);
        if (row < N) mx = fmax(mx, fma(sigma, acc, m[row]));
    }
    mx = warp_max(mx);
    if (lane == 0) atomicMax(bound_bits, (unsigned long long)__double_as_longlong(mx));  // non-negative doubles
}

// Start block: counter-based uniform numbers in (-1, 1) (splitmix64 of seed, row, column); rows >= N stay 0.
__global__ void k_rand_block(int64_t N, int64_t ld, int b, unsigned long long seed, double* X)
{
    const int64_t total = (int64_t)b * N;
    for (int64_t e = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; e < total; e += (int64_t)gridDim.x * blockDim.x) {
        const int64_t j = e / N, i = e - j * N;
        unsigned long long z = seed + 0x9E3779B97F4A7C15ULL * (unsigned long long)(e + 1);
        z = (z ^ (z >> 30)) * 0xBF58476D1CE4E5B9ULL;
        z = (z ^ (z >> 27)) * 0x94D049BB133111EBULL;
        z = z ^ (z >> 31);
        X[i + (size_t)j * ld] = ((double)(z >> 11) + 0.5) * (2.0 / 9007199254740992.0) - 1.0;
    }
}

// Out = X Tm  (X: N x b column-major ld; Tm: b x bo column-major, ld b).  One row per thread, 8 output columns
// per pass (the row of X is re-read from L1/L2 for every pass); Tm lives in shared memory.
__global__ void __launch_bounds__(256) k_right_mult(int64_t N, int64_t ld, int b, int bo, const double* X,
                                                    const double* Tm, double* Out)
{
    extern __shared__ double sT[];  // b * bo
    for (int e = threadIdx.x; e < b * bo; e += blockDim.x) sT[e] = Tm[e];
    __syncthreads();
    for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < N; i += (int64_t)gridDim.x * blockDim.x) {
        for (int j0 = 0; j0 < bo; j0 += 8) {
            double acc[8];
#pragma unroll
            for (int q = 0; q < 8; ++q) acc[q] = 0.0;
            for (int l = 0; l < b; ++l) {
                const double x = X[i + (size_t)l * ld];
#pragma unroll
                for (int q = 0; q < 8; ++q) acc[q] = fma(x, sT[l + (size_t)(j0 + q) * b], acc[q]);  // bo is a multiple of 8
            }
#pragma unroll
            for (int q = 0; q < 8; ++q) Out[i + (size_t)(j0 + q) * ld] = acc[q];
        }
    }
}

// part[blockIdx.x][j] = sum over this CTA's rows of (HX_ij - theta_j X_ij)^2     (deterministic two-phase norm)
__global__ void __launch_bounds__(256) k_resid_parts(int64_t N, int64_t ld, int b, const double* X, const double* HX,
                                                     const double* theta, double* part)
{
    __shared__ double red[32];
    const int64_t per = (N + gridDim.x - 1) / gridDim.x;
    const int64_t r0 = min((int64_t)blockIdx.x * per, N), r1 = min(r0 + per, N);
    for (int j = 0; j < b; ++j) {
        const double th = theta[j];
        double a = 0.0;
        for (int64_t i = r0 + threadIdx.x; i < r1; i += blockDim.x) {
            const double r = fma(-th, X[i + (size_t)j * ld], HX[i + (size_t)j * ld]);
            a = fma(r, r, a);
        }
        a = block_sum(a, red);
        if (threadIdx.x == 0) part[(size_t)blockIdx.x * b + j] = a;
    }
}

// b x b, one CTA: Jacobi-scaled Gram -> Tm with (X Tm)^T (X Tm) = I.
//   G' = D^{-1/2} G D^{-1/2}, G' = V S V^T, Tm = D^{-1/2} V S^{-1/2}   (S clamped at 1e-13 S_max)
// work: 2 b*b doubles.
__global__ void __launch_bounds__(1024) k_orth_small(int b, const double* G, double* work, double* Tm)
{
    __shared__ DenseShared ds;
    __shared__ double dsc[RD_EIG_MAXB];
    __shared__ double s_max;
    double* A = work;
    double* V = work + (size_t)b * b;
    for (int j = threadIdx.x; j < b; j += blockDim.x) {
        const double g = G[j + (size_t)j * b];
        dsc[j] = (g > 0.0) ? rsqrt(g) : 0.0;
    }
    __syncthreads();
    for (int e = threadIdx.x; e < b * b; e += blockDim.x) {
        const int i = e % b, j = e / b;
        A[e] = 0.5 * (G[i + (size_t)j * b] + G[j + (size_t)i * b]) * dsc[i] * dsc[j];
    }
    __syncthreads();
    cta_jacobi_eig(A, b, b, V, b, true, ds);
    if (threadIdx.x == 0) {
        double mx = 0.0;
        for (int j = 0; j < b; ++j) mx = fmax(mx, A[j + (size_t)j * b]);
        s_max = mx;
    }
    __syncthreads();
    for (int e = threadIdx.x; e < b * b; e += blockDim.x) {
        const int i = e % b, j = e / b;
        const double s = fmax(A[j + (size_t)j * b], 1e-13 * s_max);
        Tm[e] = (s > 0.0) ? dsc[i] * V[e] * rsqrt(s) : 0.0;
    }
}

// b x b, one CTA: Rayleigh-Ritz.  A = X^T H X (symmetrised), A = V Theta V^T with Theta ascending.
// work: b*b doubles.  Vout: b x b, theta: b.
__global__ void __launch_bounds__(1024) k_rr_small(int b, const double* Ain, double* work, double* Vout, double* theta)
{
    __shared__ DenseShared ds;
    __shared__ int perm[RD_EIG_MAXB];
    double* A = work;
    for (int e = threadIdx.x; e < b * b; e += blockDim.x) {
        const int i = e % b, j = e / b;
        A[e] = 0.5 * (Ain[i + (size_t)j * b] + Ain[j + (size_t)i * b]);
    }
    __syncthreads();
    double* V = work + (size_t)b * b;
    cta_jacobi_eig(A, b, b, V, b, true, ds);
    if (threadIdx.x == 0) {  // insertion sort of the b eigenvalues
        for (int j = 0; j < b; ++j) perm[j] = j;
        for (int j = 1; j < b; ++j) {
            const int pj = perm[j];
            const double v = A[pj + (size_t)pj * b];
            int q = j - 1;
            while (q >= 0 && A[perm[q] + (size_t)perm[q] * b] > v) { perm[q + 1] = perm[q]; --q; }
            perm[q + 1] = pj;
        }
    }
    __syncthreads();
    for (int e = threadIdx.x; e < b * b; e += blockDim.x) {
        const int i = e % b, j = e / b;
        Vout[e] = V[i + (size_t)perm[j] * b];
    }
    for (int j = threadIdx.x; j < b; j += blockDim.x) theta[j] = A[perm[j] + (size_t)perm[j] * b];
}

// ---- NEXT-3: Jacobi-scaled reference.  S H S with S = diag(H)^{-1/2} has the structure of H itself:
// S H S = (S M S) + sigma (K S)^T M^{-1} (K S), so the eigensolver above runs unchanged on column-scaled copies of the
// values of K (K S), row-scaled copies of the values of K^T (S K^T) and the diagonal m / d.
__global__ void k_scale_ell(Ell A, int64_t N, const double* d, int by_row, double* val_out)
{
    const int lane = threadIdx.x & 31;
    const int64_t gw = ((int64_t)blockIdx.x * blockDim.x + threadIdx.x) >> 5;
    const int64_t nwt = ((int64_t)gridDim.x * blockDim.x) >> 5;
    for (int64_t s = gw; s < A.nslices; s += nwt) {
        const int64_t row = s * RD_SLICE + lane;
        const int64_t o = A.off[s];
        const int wd = (int)((A.off[s + 1] - o) >> 5);
        for (int e = 0; e < wd; ++e) {
            const int64_t pos = o + e * 32 + lane;
            const double a = A.val[pos];
            double sc = 0.0;
            if (row < N && a != 0.0) sc = rsqrt(by_row ? d[row] : d[A.col[pos]]);
            val_out[pos] = a * sc;
        }
    }
}
__global__ void k_div(int64_t N, const double* a, const double* b, double* out)
{
    for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < N; i += (int64_t)gridDim.x * blockDim.x) out[i] = a[i] / b[i];
}
// W[:, j] <- (d^{-1/2} . W[:, j]) / || d^{-1/2} . W[:, j] ||_2, one CTA per column (fixed-order reduction)
__global__ void __launch_bounds__(1024) k_unscale_normalize(int64_t N, int64_t ld, const double* d, double* W)
{
    __shared__ double red[32];
    double* col = W + (size_t)blockIdx.x * ld;
    double acc = 0.0;
    for (int64_t i = threadIdx.x; i < N; i += blockDim.x) {
        const double v = col[i] * rsqrt(d[i]);
        col[i] = v;
        acc = fma(v, v, acc);
    }
    acc = block_sum(acc, red);
    const double inv = acc > 0.0 ? rsqrt(acc) : 0.0;
    for (int64_t i = threadIdx.x; i < N; i += blockDim.x) col[i] *= inv;
}

}  // namespace rd
