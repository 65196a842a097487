// dense.cuh -- small dense linear algebra executed by ONE CTA (all threads of the block cooperate):
// cyclic Jacobi eigensolver, Cholesky, triangular inverse, small products.  Matrices are column-major,
// addressed through generic pointers (shared memory or an L1/L2-resident global scratch area owned by the
// context), sizes up to a few hundred.  Used by the coarse setup of every PDAS step (k <= 64; E = Z^T B Z,
// its Cholesky factor and condition number) and by the Rayleigh-Ritz step of the
// reference eigensolver.  Every routine begins and ends with __syncthreads().
#pragma once
#include "common.cuh"

namespace rd {

#define RD_DENSE_MAXN 256

struct DenseShared {
    double cs[RD_DENSE_MAXN / 2], sn[RD_DENSE_MAXN / 2];
    int pp[RD_DENSE_MAXN / 2], qq[RD_DENSE_MAXN / 2];
    double red[32];
    int flag;
};

// C (M x Nn) = sum_k A(i,k) B(k,j) with explicit strides: A(i,k) = A[i*sai + k*sak], B(k,j) = B[k*sbk + j*sbj].
__device__ inline void cta_matmul(int M, int Nn, int Kk, const double* A, int sai, int sak, const double* B,
                                  int sbk, int sbj, double* C, int ldc)
{
    __syncthreads();
    for (int e = threadIdx.x; e < M * Nn; e += blockDim.x) {
        const int i = e % M, j = e / M;
        double a = 0.0;
        for (int k = 0; k < Kk; ++k) a = fma(A[(size_t)i * sai + (size_t)k * sak], B[(size_t)k * sbk + (size_t)j * sbj], a);
        C[i + (size_t)j * ldc] = a;
    }
    __syncthreads();
}

// A <- (A + A^T)/2
__device__ inline void cta_symmetrize(double* A, int lda, int n)
{
    __syncthreads();
    for (int e = threadIdx.x; e < n * n; e += blockDim.x) {
        const int i = e % n, j = e / n;
        if (i < j) {
            const double v = 0.5 * (A[i + (size_t)j * lda] + A[j + (size_t)i * lda]);
            A[i + (size_t)j * lda] = v;
            A[j + (size_t)i * lda] = v;
        }
    }
    __syncthreads();
}

// Parallel cyclic two-sided Jacobi: A (symmetric n x n, destroyed; eigenvalues end on its diagonal),
// V (n x n, receives the eigenvectors as columns when want_v).  Round-robin ordering: n/2 disjoint
// rotations per round are applied together as one orthogonal similarity A <- R^T A R.
__device__ inline void cta_jacobi_eig(double* A, int lda, int n, double* V, int ldv, bool want_v, DenseShared& ds)
{
    __syncthreads();
    if (want_v)
        for (int e = threadIdx.x; e < n * n; e += blockDim.x) V[(e % n) + (size_t)(e / n) * ldv] = ((e % n) == (e / n)) ? 1.0 : 0.0;
    __syncthreads();
    if (n < 2) return;
    const int np = (n + 1) & ~1;  // players incl. a bye when n is odd
    const int half = np / 2;
    for (int sweep = 0; sweep < 40; ++sweep) {
        double off = 0.0, dg = 0.0;
        for (int e = threadIdx.x; e < n * n; e += blockDim.x) {
            const int i = e % n, j = e / n;
            const double v = A[i + (size_t)j * lda];
            if (i == j) dg = fma(v, v, dg); else off = fma(v, v, off);
        }
        off = block_sum(off, ds.red);
        dg = block_sum(dg, ds.red);
        if (off <= 1e-30 * dg || off == 0.0) break;
        for (int round = 0; round < np - 1; ++round) {
            if (threadIdx.x < half) {
                const int i = threadIdx.x;
                int p = (round + i) % (np - 1);
                int q = (i == 0) ? np - 1 : (round - i + (np - 1)) % (np - 1);
                if (p > q) { const int tmp = p; p = q; q = tmp; }
                double c = 1.0, s = 0.0;
                if (q < n) {
                    const double apq = A[p + (size_t)q * lda];
                    const double app = A[p + (size_t)p * lda], aqq = A[q + (size_t)q * lda];
                    if (apq != 0.0 && fabs(apq) > 1e-300) {
                        const double zeta = (aqq - app) / (2.0 * apq);
                        const double t = ((zeta >= 0.0) ? 1.0 : -1.0) / (fabs(zeta) + sqrt(1.0 + zeta * zeta));
                        c = 1.0 / sqrt(1.0 + t * t);
                        s = c * t;
                    }
                } else {
                    q = -1;  // bye
                }
                ds.cs[i] = c; ds.sn[i] = s; ds.pp[i] = p; ds.qq[i] = q;
            }
            __syncthreads();
            // columns p,q of A and V
            for (int e = threadIdx.x; e < half * n; e += blockDim.x) {
                const int i = e / n, r = e % n;
                const int p = ds.pp[i], q = ds.qq[i];
                if (q < 0) continue;
                const double c = ds.cs[i], s = ds.sn[i];
                if (s == 0.0) continue;
                const double x = A[r + (size_t)p * lda], y = A[r + (size_t)q * lda];
                A[r + (size_t)p * lda] = c * x - s * y;
                A[r + (size_t)q * lda] = s * x + c * y;
                if (want_v) {
                    const double vx = V[r + (size_t)p * ldv], vy = V[r + (size_t)q * ldv];
                    V[r + (size_t)p * ldv] = c * vx - s * vy;
                    V[r + (size_t)q * ldv] = s * vx + c * vy;
                }
            }
            __syncthreads();
            // rows p,q of A
            for (int e = threadIdx.x; e < half * n; e += blockDim.x) {
                const int i = e / n, cc = e % n;
                const int p = ds.pp[i], q = ds.qq[i];
                if (q < 0) continue;
                const double c = ds.cs[i], s = ds.sn[i];
                if (s == 0.0) continue;
                const double x = A[p + (size_t)cc * lda], y = A[q + (size_t)cc * lda];
                A[p + (size_t)cc * lda] = c * x - s * y;
                A[q + (size_t)cc * lda] = s * x + c * y;
            }
            __syncthreads();
        }
    }
    __syncthreads();
}

// In-place lower Cholesky A = L L^T (upper part left untouched).  Returns false if a pivot is <= 0 or NaN.
__device__ inline bool cta_cholesky(double* A, int lda, int n, DenseShared& ds)
{
    __syncthreads();
    if (threadIdx.x == 0) ds.flag = 1;
    __syncthreads();
    for (int j = 0; j < n; ++j) {
        if (threadIdx.x == 0) {
            const double s = A[j + (size_t)j * lda];
            if (!(s > 0.0)) ds.flag = 0; else A[j + (size_t)j * lda] = sqrt(s);
        }
        __syncthreads();
        if (!ds.flag) break;
        const double ljj = A[j + (size_t)j * lda];
        for (int i = j + 1 + threadIdx.x; i < n; i += blockDim.x) A[i + (size_t)j * lda] /= ljj;
        __syncthreads();
        const int rem = n - j - 1;
        for (int e = threadIdx.x; e < rem * rem; e += blockDim.x) {
            const int i = j + 1 + e % rem, c = j + 1 + e / rem;
            if (i >= c) A[i + (size_t)c * lda] = fma(-A[i + (size_t)j * lda], A[c + (size_t)j * lda], A[i + (size_t)c * lda]);
        }
        __syncthreads();
    }
    const bool ok = ds.flag != 0;
    __syncthreads();
    return ok;
}

// X = L^{-1} (lower triangular inverse), one column per thread by forward substitution.
__device__ inline void cta_tri_inverse_lower(const double* L, int ldl, int n, double* X, int ldx)
{
    __syncthreads();
    for (int c = threadIdx.x; c < n; c += blockDim.x) {
        for (int i = 0; i < c; ++i) X[i + (size_t)c * ldx] = 0.0;
        for (int i = c; i < n; ++i) {
            double s = (i == c) ? 1.0 : 0.0;
            for (int q = c; q < i; ++q) s = fma(-L[i + (size_t)q * ldl], X[q + (size_t)c * ldx], s);
            X[i + (size_t)c * ldx] = s / L[i + (size_t)i * ldl];
        }
    }
    __syncthreads();
}

}  // namespace rd
