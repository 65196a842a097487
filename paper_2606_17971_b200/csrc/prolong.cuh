// prolong.cuh -- coarse-mesh reference: P1 prolongation to the fine grid and Euclidean column normalisation
// ("P1 prolongation maps these vectors to the full fine mesh, where each column is normalized in the Euclidean
// norm", section 2.2.2), for the cell-centred Cartesian grids of the configs (reading A20):
// the d-linear interpolant of the coarse cell-centre values, 0 on the boundary of the unit box, at the fine centres.
// HBM-bound data movement: one read of the coarse block (gathers hit L2: 2^d coarse neighbours are shared by
// (n_f/n_c)^d fine cells), one write + one read + one read-modify-write of the fine N x k block.
#pragma once
#include "common.cuh"

namespace rd {

// Interval and weight of fine cell i (0-based) among the nodes 0 | coarse centres | 1 of one axis, in exact integer
// arithmetic in units of 1/(2 nf nc): x = (2i+1) nc, node j (1..nc) at (2j-1) nf, node 0 at 0, node nc+1 at 2 nf nc.
// Returns j = the last node not to the right of x (0..nc); the neighbours are j and j+1, weights 1-t and t.
__device__ __forceinline__ int p1_interval(int i, int nc, int nf, double* t)
{
    const long long x = (long long)(2 * i + 1) * nc;
    long long j = (x + nf) / (2LL * nf);
    if (j > nc) j = nc;
    const long long xj = j == 0 ? 0LL : (2 * j - 1) * (long long)nf;
    const long long len = (j == 0 || j == nc) ? (long long)nf : 2LL * nf;
    *t = (double)(x - xj) / (double)len;
    return (int)j;
}

// W[r, c] = sum over the 2^d corners of the product of the axis weights times Wc[corner, c]; columns k..kp-1 zero.
__global__ void k_prolong_p1(int64_t N, int64_t ld, int d, int c0, int c1, int c2, int f0, int f1, int f2, int k, int kp,
                             const double* __restrict__ Wc, int64_t ldc, double* __restrict__ W)
{
    for (int64_t r = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; r < N; r += (int64_t)gridDim.x * blockDim.x) {
        const int i0 = (int)(r % f0);
        const int64_t rr = r / f0;
        const int i1 = d > 1 ? (int)(rr % f1) : 0;
        const int i2 = d > 2 ? (int)(rr / f1) : 0;
        double t0, t1 = 0.0, t2 = 0.0;
        const int j0 = p1_interval(i0, c0, f0, &t0);
        const int j1 = d > 1 ? p1_interval(i1, c1, f1, &t1) : 1;
        const int j2 = d > 2 ? p1_interval(i2, c2, f2, &t2) : 1;
        // corner weights and coarse row numbers (-1: a boundary node, value 0); corner bit a = upper node of axis a
        double wgt[8];
        int64_t cid[8];
        const int ncorner = 1 << d;
#pragma unroll
        for (int q = 0; q < 8; ++q) {
            if (q >= ncorner) { wgt[q] = 0.0; cid[q] = -1; continue; }
            const int b0 = q & 1, b1 = (q >> 1) & 1, b2 = (q >> 2) & 1;
            const int n0 = j0 + b0, n1 = j1 + b1, n2 = j2 + b2;
            double w = b0 ? t0 : 1.0 - t0;
            bool in = n0 >= 1 && n0 <= c0;
            if (d > 1) { w *= b1 ? t1 : 1.0 - t1; in = in && n1 >= 1 && n1 <= c1; }
            if (d > 2) { w *= b2 ? t2 : 1.0 - t2; in = in && n2 >= 1 && n2 <= c2; }
            wgt[q] = w;
            cid[q] = in ? (int64_t)(n0 - 1) + (int64_t)c0 * ((d > 1 ? n1 - 1 : 0) + (int64_t)c1 * (d > 2 ? n2 - 1 : 0)) : -1;
        }
        for (int c = 0; c < kp; ++c) {
            double v = 0.0;
            if (c < k) {
                const double* col = Wc + (size_t)c * ldc;
#pragma unroll
                for (int q = 0; q < 8; ++q)
                    if (cid[q] >= 0) v += wgt[q] * ldg_f64(col + cid[q]);
            }
            W[r + (size_t)c * ld] = v;
        }
    }
}

// parts[c * gridDim.x + blockIdx.x] = sum of squares of this block's contiguous share of column c (blockIdx.y = c)
__global__ void k_col_sumsq_parts(int64_t N, int64_t ld, const double* __restrict__ W, double* __restrict__ parts)
{
    __shared__ double scratch[32];
    const int c = blockIdx.y;
    const int64_t per = (N + gridDim.x - 1) / gridDim.x;
    const int64_t lo = per * blockIdx.x, hi = lo + per < N ? lo + per : N;
    const double* col = W + (size_t)c * ld;
    double s = 0.0;
    for (int64_t r = lo + threadIdx.x; r < hi; r += blockDim.x) {
        const double v = col[r];
        s += v * v;
    }
    s = block_sum(s, scratch);
    if (threadIdx.x == 0) parts[(size_t)c * gridDim.x + blockIdx.x] = s;
}

// W[:, c] /= sqrt(sum of the column's parts, fixed order); norms[c] = that root; a zero column is left alone
__global__ void k_col_normalise(int64_t N, int64_t ld, int nparts, const double* __restrict__ parts, double* __restrict__ W,
                                double* __restrict__ norms)
{
    const int c = blockIdx.y;
    double s = 0.0;
    for (int p = 0; p < nparts; ++p) s += parts[(size_t)c * nparts + p];
    const double nrm = sqrt(s);
    if (blockIdx.x == 0 && threadIdx.x == 0) norms[c] = nrm;
    if (!(nrm > 0.0)) return;
    double* col = W + (size_t)c * ld;
    for (int64_t r = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; r < N; r += (int64_t)gridDim.x * blockDim.x) col[r] /= nrm;
}

}  // namespace rd
