// pdas.cuh -- S6 (PDAS update, eq. (7)-(8) PAPER.md:102-117) and S7 (control recovery eq. (9) PAPER.md:119-123,
// KKT measures eq. (25)).  The active set lives on the device as one byte per DOF
// (1 = active); a packed LSB-first bitset is produced per step for the report / hash.
#pragma once
#include <math_constants.h>
#include "operator.cuh"

namespace rd {

struct PdasCounters {
    unsigned long long margin_bits;  // min |lambda_i + c_i (y_i - psi_i)| as the bit pattern of a non-negative double
    unsigned long long kkt_bits[6];  // five maxima of eq. (25) (unnormalised) and max |l_i|
    int changed;                     // |J_new xor J|
    int n_active_new;
};

#define RD_GRID_STRIDE(i, N) \
    for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < (N); i += (int64_t)gridDim.x * blockDim.x)

// l = M y_d   (eq. (5) with f = 0)
__global__ void k_ell(int64_t N, const double* m, const double* yd, double* ell)
{
    RD_GRID_STRIDE(i, N) ell[i] = m[i] * yd[i];
}

// Initial active set (reading A5): mode 1 all active, 2 all inactive, 3 given, -1 keep; psi = +inf never active.
__global__ void k_init_active(int64_t N, int mode, const uint8_t* J0, const double* psi, uint8_t* act)
{
    RD_GRID_STRIDE(i, N)
    {
        uint8_t a = (mode == 1) ? 1 : (mode == 2) ? 0 : (mode == 3) ? (J0[i] ? 1 : 0) : act[i];
        if (isinf(psi[i])) a = 0;
        act[i] = a;
    }
}

// Start of a step: y <- y_state with y_J <- psi_J; tmp <- chi_J psi (for b = l_I - H_IJ psi_J); x0 <- chi_I y_state.
__global__ void k_step_begin(int64_t N, const uint8_t* act, const double* psi, const double* ystate, double* y,
                             double* tmp, double* x0)
{
    RD_GRID_STRIDE(i, N)
    {
        const bool a = act[i] != 0;
        const double ys = ystate[i];
        y[i] = a ? psi[i] : ys;
        tmp[i] = a ? psi[i] : 0.0;
        x0[i] = a ? 0.0 : ys;
    }
}

// b = chi_I (l - H chi_J psi)   (eq. (7))
__global__ void k_rhs(int64_t N, const uint8_t* act, const double* ell, const double* Hpsi, double* b)
{
    RD_GRID_STRIDE(i, N) b[i] = act[i] ? 0.0 : ell[i] - Hpsi[i];
}

// y_I <- x
__global__ void k_scatter_solution(int64_t N, const uint8_t* act, const double* x, double* y)
{
    RD_GRID_STRIDE(i, N) if (!act[i]) y[i] = x[i];
}

// eq. (8): lambda = l - H y on J, exactly 0 on I (reading A4); J_new = { psi_i finite, lambda_i + c_i (y_i - psi_i) > 0 }.
__global__ void k_pdas_update(int64_t N, const uint8_t* act, const double* ell, const double* Hy, const double* y,
                              const double* psi, const double* d, int c_is_diag, double* lambda, uint8_t* act_new,
                              double* ystate, PdasCounters* cnt)
{
    __shared__ double red[32];
    __shared__ int ired[2];
    if (threadIdx.x < 2) ired[threadIdx.x] = 0;
    __syncthreads();
    double margin = CUDART_INF;
    int changed = 0, nact = 0;
    RD_GRID_STRIDE(i, N)
    {
        const bool a = act[i] != 0;
        const double lam = a ? ell[i] - Hy[i] : 0.0;
        lambda[i] = lam;
        ystate[i] = y[i];
        uint8_t an = 0;
        if (!isinf(psi[i])) {
            const double ci = c_is_diag ? d[i] : 1.0;
            const double g = lam + ci * (y[i] - psi[i]);
            an = (g > 0.0) ? 1 : 0;
            margin = fmin(margin, fabs(g));
        }
        act_new[i] = an;
        changed += (an != (uint8_t)a);
        nact += an;
    }
    margin = warp_min(margin);
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    if (lane == 0) red[warp] = margin;
    for (int o = 16; o > 0; o >>= 1) {
        changed += __shfl_xor_sync(0xffffffffu, changed, o);
        nact += __shfl_xor_sync(0xffffffffu, nact, o);
    }
    if (lane == 0) { atomicAdd(&ired[0], changed); atomicAdd(&ired[1], nact); }
    __syncthreads();
    if (threadIdx.x == 0) {
        double mm = CUDART_INF;
        for (int w = 0; w < (int)(blockDim.x >> 5); ++w) mm = fmin(mm, red[w]);
        atomicMin(&cnt->margin_bits, (unsigned long long)__double_as_longlong(mm));
        atomicAdd(&cnt->changed, ired[0]);
        atomicAdd(&cnt->n_active_new, ired[1]);
    }
}

// bits[byte] = sum_b act[8 byte + b] << b   (LSB first); also counts the active DOFs
__global__ void k_pack_bits(int64_t N, const uint8_t* act, uint8_t* bits, int* n_active)
{
    const int64_t nbytes = (N + 7) / 8;
    int cnt = 0;
    RD_GRID_STRIDE(bidx, nbytes)
    {
        unsigned v = 0;
        for (int b = 0; b < 8; ++b) {
            const int64_t i = bidx * 8 + b;
            if (i < N && act[i]) { v |= 1u << b; cnt++; }
        }
        bits[bidx] = (uint8_t)v;
    }
    for (int o = 16; o > 0; o >>= 1) cnt += __shfl_xor_sync(0xffffffffu, cnt, o);
    if ((threadIdx.x & 31) == 0 && cnt) atomicAdd(n_active, cnt);
}

// ---- S6 compaction, at the granularity of the 32-row slices / tiles every stage of Algorithm 1 works on -----------
// ("restrict the reference on the GPU", Alg. 2 step 12; "rebuild bitset / index list
// by a prefix scan").  Vectors stay full-domain and zero on J, so a slice whose 32 rows are all active holds no row of
// the inactive system: nothing of it has to be read or written by an iteration.  Two compact, ascending lists:
//   listB  slices with at least one inactive row                      -> K^T product, vector updates, HW_I / W_I tiles
//   listA  slices where t = M^{-1} K p~ can be nonzero (p~ = 0 on J): some stored K entry of a row of the slice sits
//          in an inactive column, or the slice is in listB; entry = 2 s + [s in listB]
// flags[s]: bit 0 = in listA, bit 1 = in listB.
__global__ void k_slice_flags(Ell K, int64_t N, const uint8_t* act, uint8_t* flags)
{
    const int lane = threadIdx.x & 31;
    const int64_t gw = ((int64_t)blockIdx.x * blockDim.x + threadIdx.x) >> 5;
    const int64_t nwt = ((int64_t)gridDim.x * blockDim.x) >> 5;
    for (int64_t s = gw; s < K.nslices; s += nwt) {
        const int64_t row = s * RD_SLICE + lane;
        const bool inactive = row < N && !act[row];
        const int64_t o = K.off[s];
        const int wd = (int)((K.off[s + 1] - o) >> 5);
        bool hit = false;
        for (int e = 0; e < wd; ++e) {
            const int c = ldg_i32(K.col + o + e * 32 + lane);
            const double a = ldg_f64(K.val + o + e * 32 + lane);
            hit = hit || (a != 0.0 && !act[c]);
        }
        const unsigned anyB = __ballot_sync(0xffffffffu, inactive);
        const unsigned anyA = __ballot_sync(0xffffffffu, hit);
        if (lane == 0) flags[s] = (uint8_t)(((anyA | anyB) ? 1 : 0) | (anyB ? 2 : 0));
    }
}

// One CTA: exclusive scan of the two flag bits over all slices, compact lists, counts[0] = |listA|, counts[1] = |listB|.
__global__ void __launch_bounds__(1024) k_slice_lists(int64_t nslices, const uint8_t* flags, int32_t* listA, int32_t* listB,
                                                      int32_t* counts)
{
    __shared__ int sa[1024], sb[1024];
    const int tid = threadIdx.x;
    const int64_t per = (nslices + blockDim.x - 1) / blockDim.x;
    const int64_t s0 = min((int64_t)tid * per, nslices), s1 = min(s0 + per, nslices);
    int ca = 0, cb = 0;
    for (int64_t s = s0; s < s1; ++s) { const int f = flags[s]; ca += f & 1; cb += (f >> 1) & 1; }
    sa[tid] = ca;
    sb[tid] = cb;
    __syncthreads();
    for (int o = 1; o < (int)blockDim.x; o <<= 1) {  // Hillis-Steele inclusive scan
        const int va = (tid >= o) ? sa[tid - o] : 0, vb = (tid >= o) ? sb[tid - o] : 0;
        __syncthreads();
        sa[tid] += va;
        sb[tid] += vb;
        __syncthreads();
    }
    int pa = sa[tid] - ca, pb = sb[tid] - cb;
    for (int64_t s = s0; s < s1; ++s) {
        const int f = flags[s];
        if (f & 1) listA[pa++] = (int32_t)(2 * s + ((f >> 1) & 1));
        if (f & 2) listB[pb++] = (int32_t)s;
    }
    if (tid == (int)blockDim.x - 1) { counts[0] = sa[tid]; counts[1] = sb[tid]; }
}

// one launch instead of seven memsets: the work vectors of a solve start at zero (rows of slices outside the lists
// are never written by the kernel and must read as zero)
__global__ void k_zero_vectors(int64_t n, double* a, double* b, double* c, double* d, double* e, double* f)
{
    RD_GRID_STRIDE(i, n) { a[i] = 0.0; b[i] = 0.0; c[i] = 0.0; d[i] = 0.0; e[i] = 0.0; f[i] = 0.0; }
}

__device__ __forceinline__ void atomic_max_nonneg(unsigned long long* p, double v)
{
    atomicMax(p, (unsigned long long)__double_as_longlong(v));  // order of non-negative doubles = order of their bits
}

// eq. (25) with g = H y - l: max |g + lambda|, max [y - psi]_+, max [-lambda]_+, max |lambda (psi - y)|,
// max |y - min(psi, y - g)|, and max |l| for s = max(1, ||l||_inf).  psi = +inf contributes 0 to the 2nd,
// 4th; min(inf, y - g) = y - g in the 5th.
__global__ void k_kkt(int64_t N, const double* ell, const double* Hy, const double* y, const double* psi,
                      const double* lambda, PdasCounters* cnt)
{
    double k0 = 0, k1 = 0, k2 = 0, k3 = 0, k4 = 0, k5 = 0;
    RD_GRID_STRIDE(i, N)
    {
        const double g = Hy[i] - ell[i];
        const double lam = lambda[i];
        k0 = fmax(k0, fabs(g + lam));
        k2 = fmax(k2, lam < 0.0 ? -lam : 0.0);
        if (isinf(psi[i])) {
            k4 = fmax(k4, fabs(g));
        } else {
            k1 = fmax(k1, y[i] > psi[i] ? y[i] - psi[i] : 0.0);
            k3 = fmax(k3, fabs(lam * (psi[i] - y[i])));
            const double mn = (psi[i] < y[i] - g) ? psi[i] : (y[i] - g);
            k4 = fmax(k4, fabs(y[i] - mn));
        }
        k5 = fmax(k5, fabs(ell[i]));
    }
    k0 = warp_max(k0); k1 = warp_max(k1); k2 = warp_max(k2); k3 = warp_max(k3); k4 = warp_max(k4); k5 = warp_max(k5);
    if ((threadIdx.x & 31) == 0) {
        atomic_max_nonneg(&cnt->kkt_bits[0], k0);
        atomic_max_nonneg(&cnt->kkt_bits[1], k1);
        atomic_max_nonneg(&cnt->kkt_bits[2], k2);
        atomic_max_nonneg(&cnt->kkt_bits[3], k3);
        atomic_max_nonneg(&cnt->kkt_bits[4], k4);
        atomic_max_nonneg(&cnt->kkt_bits[5], k5);
    }
}

}  // namespace rd
