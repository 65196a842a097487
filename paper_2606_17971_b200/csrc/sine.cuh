// sine.cuh -- NEXT-1 of SURVEY.md 8(f): the analytical Cartesian spatial reference of PAPER.md:186-192 (section
// 2.2.3, eq. (15)) in its cell-centred form: the r lowest products of 1-D sine factors of the constant-coefficient
// Dirichlet Laplacian,
//     v_q(j) = sqrt(2/n) sin(pi q (j + 1/2)/n)   (sqrt(1/n) for q = n),   j = 0..n-1, q = 1..n,
// x fastest.  "Evaluating the selected products costs O(N_s r) work and storage": two kernels, one for
// the 1-D tables (d * qmax * n entries), one streaming write of W.  HBM-bound: 8 N k bytes written.
#pragma once
#include "common.cuh"
#include "dense.cuh"

namespace rd {

// tab[(a * qmax + (q - 1)) * nmax + j] = v_q(j) of axis a
__global__ void k_sine_tables(int d, int qmax, int nmax, int n0, int n1, int n2, double* tab)
{
    const int total = d * qmax * nmax;
    for (int e = blockIdx.x * blockDim.x + threadIdx.x; e < total; e += gridDim.x * blockDim.x) {
        const int j = e % nmax, q = (e / nmax) % qmax + 1, a = e / (nmax * qmax);
        const int n = a == 0 ? n0 : (a == 1 ? n1 : n2);
        double v = 0.0;
        if (j < n && q <= n) v = sqrt((q == n ? 1.0 : 2.0) / (double)n) * sinpi((double)q * ((double)j + 0.5) / (double)n);
        tab[e] = v;
    }
}

// W[i, c] = prod_a v_{modes[c][a]}(i_a), i = i_0 + n0 (i_1 + n1 i_2); columns c >= k (up to kp) are zero
__global__ void k_sine_product(int64_t N, int64_t ld, int d, int qmax, int nmax, int n0, int n1, int k, int kp,
                               const int32_t* modes /* k x 3 */, const double* tab, double* W)
{
    for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < N; i += (int64_t)gridDim.x * blockDim.x) {
        const int i0 = (int)(i % n0);
        const int64_t r = i / n0;
        const int i1 = d > 1 ? (int)(r % n1) : 0;
        const int i2 = d > 2 ? (int)(r / n1) : 0;
        for (int c = 0; c < kp; ++c) {
            double v = 0.0;
            if (c < k) {
                v = tab[(size_t)(0 * qmax + modes[c * 3 + 0] - 1) * nmax + i0];
                if (d > 1) v = tab[(size_t)(1 * qmax + modes[c * 3 + 1] - 1) * nmax + i1] * v;
                if (d > 2) v = tab[(size_t)(2 * qmax + modes[c * 3 + 2] - 1) * nmax + i2] * v;
            }
            W[i + (size_t)c * ld] = v;
        }
    }
}

// ---- NEXT-2: mode-dependent temporal reference, eq. (16)-(17).  For spatial mode i (Laplacian
// eigenvalue mu_i) the temporal matrix S_i = (mu_i I + L)^T (mu_i I + L), L lower bidiagonal (1/dt, -1/dt), shares its
// eigenvectors with H_i = W_t + alpha (mu_i I + L)^T W_t (mu_i I + L) (W_t = I) and nu = h^d (1 + alpha s) grows with s.
// One CTA per spatial mode: cyclic Jacobi in global scratch, eigenvalues sorted ascending, each eigenvector with its
// largest-magnitude component (lowest index on ties) positive.
//   A, V : scratch, gridDim.x x nt x nt.   s_out[i * nt + j], Q_out[(i * nt + j) * nt + t]
__global__ void __launch_bounds__(256) k_temporal_eigs(int nt, double inv_dt, const double* mu, double* A, double* V,
                                                        double* s_out, double* Q_out)
{
    __shared__ DenseShared ds;
    __shared__ int order[RD_DENSE_MAXN];
    const int i = blockIdx.x;
    double* Ai = A + (size_t)i * nt * nt;
    double* Vi = V + (size_t)i * nt * nt;
    const double dg = mu[i] + inv_dt;  // diagonal of B = mu I + L; sub-diagonal -1/dt
    for (int e = threadIdx.x; e < nt * nt; e += blockDim.x) {
        const int a = e % nt, b = e / nt;
        double v = 0.0;
        if (a == b) v = dg * dg + (a + 1 < nt ? inv_dt * inv_dt : 0.0);
        else if (a == b + 1 || b == a + 1) v = -inv_dt * dg;
        Ai[e] = v;
    }
    __syncthreads();
    cta_jacobi_eig(Ai, nt, nt, Vi, nt, true, ds);
    __syncthreads();
    if (threadIdx.x == 0) {  // ascending order of the eigenvalues (insertion sort, nt <= 256)
        for (int j = 0; j < nt; ++j) order[j] = j;
        for (int j = 1; j < nt; ++j) {
            const int o = order[j];
            const double v = Ai[o + (size_t)o * nt];
            int p = j - 1;
            while (p >= 0 && Ai[order[p] + (size_t)order[p] * nt] > v) { order[p + 1] = order[p]; --p; }
            order[p + 1] = o;
        }
    }
    __syncthreads();
    for (int j = threadIdx.x; j < nt; j += blockDim.x) {
        const int o = order[j];
        s_out[(size_t)i * nt + j] = Ai[o + (size_t)o * nt];
        const double* q = Vi + (size_t)o * nt;
        int big = 0;
        for (int t = 1; t < nt; ++t) if (fabs(q[t]) > fabs(q[big])) big = t;
        const double sign = q[big] > 0.0 ? 1.0 : -1.0;
        for (int t = 0; t < nt; ++t) Q_out[((size_t)i * nt + j) * nt + t] = sign * q[t];
    }
}

// W[sidx + Ns t, c] = Q[sel_i[c]][sel_j[c]][t] * prod_a v_{modes[sel_i[c]][a]}(sidx_a); columns c >= k are zero
__global__ void k_kron_product(int64_t Ns, int nt, int64_t ld, int d, int qmax, int nmax, int n0, int n1, int k, int kp,
                               const int32_t* modes /* rs x 3 */, const int32_t* sel /* k x 2: (i, j) */,
                               const double* tab, const double* Q, double* W)
{
    const int64_t N = Ns * nt;
    for (int64_t r = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; r < N; r += (int64_t)gridDim.x * blockDim.x) {
        const int64_t sidx = r % Ns;
        const int t = (int)(r / Ns);
        const int i0 = (int)(sidx % n0);
        const int64_t rr = sidx / n0;
        const int i1 = d > 1 ? (int)(rr % n1) : 0;
        const int i2 = d > 2 ? (int)(rr / n1) : 0;
        for (int c = 0; c < kp; ++c) {
            double v = 0.0;
            if (c < k) {
                const int mi = sel[2 * c], mj = sel[2 * c + 1];
                double phi = tab[(size_t)(0 * qmax + modes[mi * 3 + 0] - 1) * nmax + i0];
                if (d > 1) phi = tab[(size_t)(1 * qmax + modes[mi * 3 + 1] - 1) * nmax + i1] * phi;
                if (d > 2) phi = tab[(size_t)(2 * qmax + modes[mi * 3 + 2] - 1) * nmax + i2] * phi;
                v = Q[((size_t)mi * nt + mj) * nt + t] * phi;
            }
            W[r + (size_t)c * ld] = v;
        }
    }
}

}  // namespace rd
