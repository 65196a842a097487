// sine.cuh -- NEXT-1 of SURVEY.md 8(f): the analytical Cartesian spatial reference of PAPER.md:186-192 (section
// 2.2.3, eq. (15)) in its cell-centred form: the r lowest products of 1-D sine factors of the constant-coefficient
// Dirichlet Laplacian,
//     v_q(j) = sqrt(2/n) sin(pi q (j + 1/2)/n)   (sqrt(1/n) for q = n),   j = 0..n-1, q = 1..n,
// x fastest.  "Evaluating the selected products costs O(N_s r) work and storage": two kernels, one for
// the 1-D tables (d * qmax * n entries), one streaming write of W.  HBM-bound: 8 N k bytes written.
#pragma once
#include "common.cuh"

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

}  // namespace rd
