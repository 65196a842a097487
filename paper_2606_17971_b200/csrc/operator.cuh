// operator.cuh -- S3: the matrix-free reduced Hessian H = M + sigma K^T M^{-1} K (eq. (5))
// and its masked principal submatrix B = H_II (eq. (7)) as two sliced-ELL SpMVs.
//
// Storage: sliced ELL, slice height 32 (one warp, one row per lane).  Slice s holds rows 32s..32s+31,
// padded to the longest row of the slice; entry e of lane l sits at off[s] + 32 e + l, so a warp reads
// 32 consecutive values (256 B) and 32 consecutive indices (128 B) per entry.  Padding entries carry
// value 0 and the row's own column.  K and K^T are both stored (values 8 B + index 4 B per nonzero each).
#pragma once
#include "common.cuh"

namespace rd {

struct Ell {
    const int32_t* col;
    const double* val;
    const int64_t* off;  // nslices + 1, in entries
    int64_t nslices;
    int32_t uwd;  // entries per row if every slice has the same width (off[s] = 32 uwd s, no lookup needed), else -1
};

// One row of a sliced-ELL product with an on-the-fly combined input  v0[c] + beta v1[c]  (v1 may be
// NULL: plain v0).  Returns sum_e A[row,e] * vin[col_e].  All lanes of the warp must call it (same slice).
template <bool COMBINE>
__device__ __forceinline__ double ell_row_dot(const Ell& A, int64_t s, int lane, const double* v0,
                                              const double* v1, double beta)
{
    const int64_t o = A.off[s];
    const int wd = (int)((A.off[s + 1] - o) >> 5);
    const int32_t* cp = A.col + o + lane;
    const double* vp = A.val + o + lane;
    double acc = 0.0;
    int e = 0;
    // groups of 4 entries: indices and values first, then the gathers (keeps 8-12 loads in flight per lane)
    for (; e + 4 <= wd; e += 4) {
        int c0 = ldg_i32(cp + (e + 0) * 32), c1 = ldg_i32(cp + (e + 1) * 32);
        int c2 = ldg_i32(cp + (e + 2) * 32), c3 = ldg_i32(cp + (e + 3) * 32);
        double a0 = ldg_f64(vp + (e + 0) * 32), a1 = ldg_f64(vp + (e + 1) * 32);
        double a2 = ldg_f64(vp + (e + 2) * 32), a3 = ldg_f64(vp + (e + 3) * 32);
        double x0 = v0[c0], x1 = v0[c1], x2 = v0[c2], x3 = v0[c3];
        if (COMBINE) {
            x0 = fma(beta, v1[c0], x0);
            x1 = fma(beta, v1[c1], x1);
            x2 = fma(beta, v1[c2], x2);
            x3 = fma(beta, v1[c3], x3);
        }
        acc = fma(a0, x0, acc);
        acc = fma(a1, x1, acc);
        acc = fma(a2, x2, acc);
        acc = fma(a3, x3, acc);
    }
    for (; e < wd; ++e) {
        int c0 = ldg_i32(cp + e * 32);
        double a0 = ldg_f64(vp + e * 32);
        double x0 = v0[c0];
        if (COMBINE) x0 = fma(beta, v1[c0], x0);
        acc = fma(a0, x0, acc);
    }
    return acc;
}

// Stage "K" over slices [s0, s1) handled by the warps of this CTA:
//   t_r = (1/m_r) sum_c K_rc vin_c,  vin = v0 + beta v1;  if pnew != NULL also pnew_r = vin_r
// (the CG direction update p <- z + beta p of Alg. 1 line 23 is fused here).
template <bool COMBINE>
__device__ __forceinline__ void stage_K(const Ell& K, int64_t N, int64_t s0, int64_t s1, const double* minv,
                                        const double* v0, const double* v1, double beta, double* pnew, double* t)
{
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5, nw = blockDim.x >> 5;
    for (int64_t s = s0 + warp; s < s1; s += nw) {
        const int64_t row = s * RD_SLICE + lane;
        double acc = ell_row_dot<COMBINE>(K, s, lane, v0, v1, beta);
        if (row < N) {
            t[row] = acc * ldg_f64(minv + row);
            if (pnew) {
                double x = v0[row];
                if (COMBINE) x = fma(beta, v1[row], x);
                pnew[row] = x;
            }
        }
    }
}

// Stage "K^T" over slices [s0, s1):
//   w_i = m_i v_i + sigma sum_r K_ri t_r   (i inactive, or act == NULL),  w_i = 0 (i active)
// returns this thread's partial of  v^T w  (Alg. 1 line 9).
__device__ __forceinline__ double stage_KT(const Ell& KT, int64_t N, int64_t s0, int64_t s1, const double* m,
                                           double sigma, const uint8_t* act, const double* v, const double* t,
                                           double* w)
{
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5, nw = blockDim.x >> 5;
    double dot = 0.0;
    for (int64_t s = s0 + warp; s < s1; s += nw) {
        const int64_t row = s * RD_SLICE + lane;
        double acc = ell_row_dot<false>(KT, s, lane, t, nullptr, 0.0);
        if (row < N) {
            const double vi = v[row];
            double wi = fma(sigma, acc, ldg_f64(m + row) * vi);
            if (act && act[row]) wi = 0.0;
            w[row] = wi;
            dot = fma(vi, wi, dot);
        }
    }
    return dot;
}

// ---- stand-alone launches (setup, PDAS update, tests): any grid, warps stride over all slices ---------
__global__ void k_apply_K(Ell K, int64_t N, const double* scale /*NULL or 1/m*/, const double* v, double* out)
{
    const int lane = threadIdx.x & 31;
    const int64_t gw = ((int64_t)blockIdx.x * blockDim.x + threadIdx.x) >> 5;
    const int64_t nwt = ((int64_t)gridDim.x * blockDim.x) >> 5;
    for (int64_t s = gw; s < K.nslices; s += nwt) {
        const int64_t row = s * RD_SLICE + lane;
        double acc = ell_row_dot<false>(K, s, lane, v, nullptr, 0.0);
        if (row < N) out[row] = scale ? acc * scale[row] : acc;
    }
}

__global__ void k_apply_KT_H(Ell KT, int64_t N, const double* m, double sigma, const uint8_t* act,
                             const double* v, const double* t, double* out)
{
    const int lane = threadIdx.x & 31;
    const int64_t gw = ((int64_t)blockIdx.x * blockDim.x + threadIdx.x) >> 5;
    const int64_t nwt = ((int64_t)gridDim.x * blockDim.x) >> 5;
    for (int64_t s = gw; s < KT.nslices; s += nwt) {
        const int64_t row = s * RD_SLICE + lane;
        double acc = ell_row_dot<false>(KT, s, lane, t, nullptr, 0.0);
        if (row < N) {
            double wi = fma(sigma, acc, m[row] * v[row]);
            if (act && act[row]) wi = 0.0;
            out[row] = wi;
        }
    }
}

// out = act ? 0 : v   (chi_I v: the zero extension R_I^T R_I v of eq. (7))
__global__ void k_mask_copy(int64_t N, const uint8_t* act, const double* v, double* out)
{
    for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < N; i += (int64_t)gridDim.x * blockDim.x)
        out[i] = (act && act[i]) ? 0.0 : v[i];
}

// d_i = m_i + sigma sum_r K_ri^2 / m_r = m_i + sigma sum_e KT[i,e]^2 * minv[col_e]   (diagonal of eq. (5))
__global__ void k_diag_H(Ell KT, int64_t N, const double* m, const double* minv, double sigma, int jacobi,
                         double* d, double* dinv)
{
    const int lane = threadIdx.x & 31;
    const int64_t gw = ((int64_t)blockIdx.x * blockDim.x + threadIdx.x) >> 5;
    const int64_t nwt = ((int64_t)gridDim.x * blockDim.x) >> 5;
    for (int64_t s = gw; s < KT.nslices; s += nwt) {
        const int64_t row = s * RD_SLICE + lane;
        const int64_t o = KT.off[s];
        const int wd = (int)((KT.off[s + 1] - o) >> 5);
        double acc = 0.0;
        for (int e = 0; e < wd; ++e) {
            const int c = KT.col[o + e * 32 + lane];
            const double a = KT.val[o + e * 32 + lane];
            acc = fma(a * a, minv[c], acc);
        }
        if (row < N) {
            const double di = fma(sigma, acc, m[row]);
            d[row] = di;
            dinv[row] = jacobi ? 1.0 / di : 1.0;
        }
    }
}

}  // namespace rd
