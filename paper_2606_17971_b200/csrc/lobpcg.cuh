// lobpcg.cuh -- S0, second eigensolver: locally optimal block preconditioned CG for the k lowest eigenpairs of
// H = M + sigma K^T M^{-1} K on a Cartesian grid, preconditioned by the exact inverse of the HOMOGENEOUS operator of the
// same grid, which the paper's analytical reference diagonalises (eq. (15): products of 1-D sine
// vectors v_q with Laplacian eigenvalues mu_q; sine.cuh builds them as a reference, here they are a preconditioner):
//
//     T = S^T diag( 1 / (mbar (1 + sigma kappa_ref^2 mu^2)) ) S,      S = S_x (x) S_y (x) S_z,  S_a[q, j] = v_q(j)
//
// applied axis by axis as dense n_a x n_a products on the FP64 tensor cores (k_dgemm_dmma).  The Chebyshev filter of
// eigs.cuh needs a polynomial degree ~ sqrt(theta_max / gap) per sweep (22,500 in total on the 160^3 mesh); with T the
// spectrum LOBPCG sees is bounded independently of the mesh (coefficient contrast and Peclet number only), and every
// iteration costs one block apply of H, one of T, two Gram products and four tall-skinny products, all blocked.
//
// One iteration, basis S = [X, W, P] (N x 3b, one contiguous block; HS = [HX, HW, HP] beside it):
//   R = HX - X diag(theta);  W = T R;  HW = H W
//   Gs = S^T S, Gh = S^T HS                          (k_gram_dmma)
//   k_lobpcg_rr: Jacobi-scaled Gs = V s V^T, Tm = D^{-1/2} V s^{-1/2} (directions with s below 1e-12 s_max dropped),
//                A' = Tm^T Gh Tm = U theta U^T, C = Tm U[:, lowest b]                                   (one CTA)
//   P' = [W, P] C[b:, :],  X' = X C[:b, :] + P'      and the same combinations of HW, HP, HX        (k_dgemm_dmma)
// No reorthogonalisation pass over the N x 3b block is needed: the Gram-based Rayleigh-Ritz works in the metric Gs.
#pragma once
#include "eigs.cuh"

namespace rd {

// ---------------------------------------------------------------------------------------------------------------------
// D[m, n] = sum_k A[m, k] B[k, n] (+ E[m, n]) with explicit strides, on m8n8k4 FP64 tensor-core tiles.
//   A[m sam + k sak], B[k sbk + n sbn], D and E [m sdm + n sdn]; blockIdx.z = batch: z1 = z / nb2, z2 = z % nb2 select
//   the offsets z1 * bs1 + z2 * bs2 of each operand (0 strides: shared operand).
// CTA = 8 warps, tile 64 (m) x 8 TN (n); warp w owns rows [8w, 8w + 8) and TN accumulator tiles; the contraction runs in
// chunks of 32 staged in shared memory.  AM: A is contiguous along m (sam == 1), else along k (sak == 1); BN: B is
// contiguous along n (sbn == 1), else along k (sbk == 1).  The shared layouts put the contiguous index last, padded so
// that both the staging stores and the fragment loads are bank-conflict free (leading dimension = 4 mod 16 doubles).
struct GemmOp {
    const double* p;
    int64_t s0, s1;    // strides of the two matrix indices
    int64_t bs1, bs2;  // batch strides
};

template <bool AM, bool BN, int TN>
__global__ void __launch_bounds__(256, 2) k_dgemm_dmma(int M, int Nn, int Kk, int nb2, GemmOp A, GemmOp B, GemmOp E, GemmOp D)
{
    constexpr int TNC = 8 * TN;                  // n columns per CTA
    constexpr int LDA_M = 64 + 4, LDA_K = 32 + 4;
    constexpr int LDB_N = (TNC % 16 == 4 % 16) ? TNC : TNC + ((4 - TNC % 16) + 16) % 16, LDB_K = 32 + 4;
    __shared__ double sA[AM ? 32 * LDA_M : 64 * LDA_K];
    __shared__ double sB[BN ? 32 * LDB_N : TNC * LDB_K];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int am = lane >> 2, ak = lane & 3;
    const int m0 = blockIdx.x * 64, n0 = blockIdx.y * TNC;
    const int64_t z1 = blockIdx.z / nb2, z2 = blockIdx.z % nb2;
    const double* Ap = A.p + z1 * A.bs1 + z2 * A.bs2;
    const double* Bp = B.p + z1 * B.bs1 + z2 * B.bs2;
    double acc[TN][2];
#pragma unroll
    for (int t = 0; t < TN; ++t) acc[t][0] = acc[t][1] = 0.0;
    const bool live = (m0 + warp * 8) < M;
    // Register-staged pipeline: the global loads of chunk c + 1 are issued before the tensor-core work on chunk c and land in
    // shared memory after it, so their latency overlaps the DMMAs of this CTA as well as those of the other resident CTAs.
    constexpr int NA = (64 * 32) / 256, NB = (TNC * 32) / 256;
    double ra[NA], rb[NB];
    auto fetch = [&](int k0) {
#pragma unroll
        for (int u = 0; u < NA; ++u) {
            const int e = threadIdx.x + u * 256;
            const int mm = AM ? (e & 63) : (e >> 5), kk = AM ? (e >> 6) : (e & 31);
            const int gm = m0 + mm, gk = k0 + kk;
            ra[u] = (gm < M && gk < Kk) ? ldg_f64(Ap + (int64_t)gm * A.s0 + (int64_t)gk * A.s1) : 0.0;
        }
#pragma unroll
        for (int u = 0; u < NB; ++u) {
            const int e = threadIdx.x + u * 256;
            const int kk = BN ? (e / TNC) : (e & 31), nn = BN ? (e - (e / TNC) * TNC) : (e >> 5);
            const int gn = n0 + nn, gk = k0 + kk;
            rb[u] = (gn < Nn && gk < Kk) ? ldg_f64(Bp + (int64_t)gk * B.s0 + (int64_t)gn * B.s1) : 0.0;
        }
    };
    auto stage = [&]() {
#pragma unroll
        for (int u = 0; u < NA; ++u) {
            const int e = threadIdx.x + u * 256;
            if (AM) sA[(e >> 6) * LDA_M + (e & 63)] = ra[u];   // sA[k][m], lanes along m
            else sA[(e >> 5) * LDA_K + (e & 31)] = ra[u];      // sA[m][k], lanes along k
        }
#pragma unroll
        for (int u = 0; u < NB; ++u) {
            const int e = threadIdx.x + u * 256;
            if (BN) sB[(e / TNC) * LDB_N + (e - (e / TNC) * TNC)] = rb[u];  // sB[k][n], lanes along n
            else sB[(e >> 5) * LDB_K + (e & 31)] = rb[u];                   // sB[n][k], lanes along k
        }
    };
    fetch(0);
    for (int k0 = 0; k0 < Kk; k0 += 32) {
        __syncthreads();  // every warp is done with the previous chunk
        stage();
        __syncthreads();
        if (k0 + 32 < Kk) fetch(k0 + 32);
        if (live) {
#pragma unroll
            for (int kk = 0; kk < 32; kk += 4) {
                const double a = AM ? sA[(kk + ak) * LDA_M + warp * 8 + am] : sA[(warp * 8 + am) * LDA_K + kk + ak];
#pragma unroll
                for (int t = 0; t < TN; ++t) {
                    const double b = BN ? sB[(kk + ak) * LDB_N + t * 8 + am] : sB[(t * 8 + am) * LDB_K + kk + ak];
                    dmma_m8n8k4(acc[t][0], acc[t][1], a, b);
                }
            }
        }
    }
    if (!live) return;
    const int gm = m0 + warp * 8 + am;
    if (gm >= M) return;
    double* Dp = const_cast<double*>(D.p) + z1 * D.bs1 + z2 * D.bs2 + (int64_t)gm * D.s0;
    const double* Ep = E.p ? E.p + z1 * E.bs1 + z2 * E.bs2 + (int64_t)gm * E.s0 : nullptr;
#pragma unroll
    for (int t = 0; t < TN; ++t) {
        const int gn = n0 + t * 8 + 2 * ak;
#pragma unroll
        for (int e = 0; e < 2; ++e) {
            if (gn + e < Nn) {
                double v = acc[t][e];
                if (Ep) v += Ep[(int64_t)(gn + e) * E.s1];
                Dp[(int64_t)(gn + e) * D.s1] = v;
            }
        }
    }
}

// ---------------------------------------------------------------------------------------------------------------------
// 1-D sine vectors of one axis (cell-centred form of sine.cuh): S[q][j] = v_{q+1}(j+1), row-major n x n,
// its transpose, and the Laplacian eigenvalues mu_{q+1} = 4 n^2 sin^2(pi (q+1) / (2n)).
__global__ void k_sine_axis_tables(int n, double* S, double* St, double* mu)
{
    for (int e = blockIdx.x * blockDim.x + threadIdx.x; e < n * n; e += gridDim.x * blockDim.x) {
        const int q = e / n + 1, j = e % n + 1;
        // sin(pi q (2j - 1) / (2n)) with the argument reduced in integers: period 4n in q (2j - 1)
        const long long r = ((long long)q * (2 * j - 1)) % (4LL * n);
        const double v = sqrt((q == n ? 1.0 : 2.0) / (double)n) * sinpi((double)r / (2.0 * n));
        S[(size_t)(q - 1) * n + (j - 1)] = v;
        St[(size_t)(j - 1) * n + (q - 1)] = v;
        if (j == 1) {
            const double s = sinpi((double)q / (2.0 * n));
            mu[q - 1] = 4.0 * (double)n * (double)n * s * s;
        }
    }
}

// Y[i, c] *= 1 / (mbar (1 + sigma kap^2 (mu_x[qx] + mu_y[qy] + mu_z[qz])^2)),  i = qx + nx (qy + ny qz): the inverse of
// the homogeneous operator in the sine basis (eq. (5) with K = kap mbar L, M = mbar I).
__global__ void k_sine_scale(int64_t N, int64_t ld, int ncols, int nx, int ny, const double* mux, const double* muy,
                             const double* muz, double mbar, double sk2, double* Y)
{
    for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < N; i += (int64_t)gridDim.x * blockDim.x) {
        const int qx = (int)(i % nx);
        const int64_t r = i / nx;
        const int qy = (int)(r % ny), qz = (int)(r / ny);
        double mu = mux[qx];
        if (muy) mu += muy[qy];
        if (muz) mu += muz[qz];
        const double w = 1.0 / (mbar * fma(sk2, mu * mu, 1.0));
        for (int c = 0; c < ncols; ++c) Y[i + (size_t)c * ld] *= w;
    }
}

// R[:, j] = HX[:, j] - theta_j X[:, j] and part[blockIdx.x][j] = this CTA's share of ||R[:, j]||^2 (fixed order)
__global__ void __launch_bounds__(256) k_resid_write_parts(int64_t N, int64_t ld, int b, const double* X, const double* HX,
                                                           const double* theta, double* R, double* part)
{
    __shared__ double red[32];
    const int64_t per = (N + gridDim.x - 1) / gridDim.x;
    const int64_t r0 = min((int64_t)blockIdx.x * per, N), r1 = min(r0 + per, N);
    for (int j = 0; j < b; ++j) {
        const double th = theta[j];
        double a = 0.0;
        for (int64_t i = r0 + threadIdx.x; i < r1; i += blockDim.x) {
            const double r = fma(-th, X[i + (size_t)j * ld], HX[i + (size_t)j * ld]);
            R[i + (size_t)j * ld] = r;
            a = fma(r, r, a);
        }
        a = block_sum(a, red);
        if (threadIdx.x == 0) part[(size_t)blockIdx.x * b + j] = a;
    }
}

// ---------------------------------------------------------------------------------------------------------------------
// The ns x ns part of one LOBPCG iteration (ns = b + 2 na <= RD_DENSE_MAXN):
//   Gs = S^T S, Gh = S^T H S  ->  C (ns x b, column-major, ld ns) and theta (b) with
//   (S C)^T (S C) = I, (S C)^T H (S C) = diag(theta), theta the b lowest Ritz values of span(S).
// Two symmetric eigenproblems of size <= ns.  One CTA running cta_jacobi_eig on matrices of this size in global memory is
// bound by the L2 bandwidth and latency of a single SM (600 ms at ns = 240); k_jacobi_grid spreads the n/2 disjoint
// rotations of a round over n/2 CTAs with one grid barrier per round, and the products around it are plain grid kernels.
//
// k_jacobi_grid: parallel cyclic two-sided Jacobi, round-robin ordering as in cta_jacobi_eig.  n even (callers pad), grid =
// at least n/2 CTAs of 256 threads, cooperative launch.  CTA i owns the pair (p_i, q_i) of the round: it forms ALL rotations
// of the round from the current matrix (3 n/2 loads, redundantly in every CTA), then writes columns p_i, q_i of
// A' = R^T A R into the other buffer (reads only its own two columns of the current one) and rotates columns p_i, q_i of V
// in place.  Result: eigenvalues on the diagonal of A0, eigenvectors in V.  n_ptr (may be NULL): the size, read on the device.
__global__ void __launch_bounds__(256) k_jacobi_grid(int n_in, const int* n_ptr, double* A0, double* A1, double* V, GridBarrier* bar,
                                                     double* partials, const int* skip)
{
    if (skip && *skip) return;  // uniform over the grid
    __shared__ double cs[RD_DENSE_MAXN / 2], sn[RD_DENSE_MAXN / 2];
    __shared__ int pp[RD_DENSE_MAXN / 2], qq[RD_DENSE_MAXN / 2];
    __shared__ double red[32];
    const int n = n_ptr ? *n_ptr : n_in;
    const int lda = n, ldv = n;
    const int half = n / 2;
    const int i = blockIdx.x;
    const unsigned int G = gridDim.x;
    if (n < 2) return;  // uniform over the grid
    if (i < half)
        for (int e = threadIdx.x; e < 2 * n; e += blockDim.x) {
            const int c = 2 * i + e / n, r = e % n;
            V[r + (size_t)c * ldv] = (r == c) ? 1.0 : 0.0;
        }
    double* cur = A0;
    double* nxt = A1;
    for (int sweep = 0; sweep < 40; ++sweep) {
        // off-diagonal and diagonal weight, partial sums over columns 2i, 2i + 1 in a fixed order
        double off = 0.0, dg = 0.0;
        if (i < half)
            for (int e = threadIdx.x; e < 2 * n; e += blockDim.x) {
                const int c = 2 * i + e / n, r = e % n;
                const double v = cur[r + (size_t)c * lda];
                if (r == c) dg = fma(v, v, dg); else off = fma(v, v, off);
            }
        off = block_sum(off, red);
        dg = block_sum(dg, red);
        if (threadIdx.x == 0 && i < half) { partials[i] = off; partials[half + i] = dg; }
        grid_barrier(bar, G);
        double toff = 0.0, tdg = 0.0;
        for (int e = 0; e < half; ++e) { toff += partials[e]; tdg += partials[half + e]; }
        grid_barrier(bar, G);  // partials are rewritten in the next sweep
        if (toff <= 1e-30 * tdg || toff == 0.0) break;
        for (int round = 0; round < n - 1; ++round) {
            if (threadIdx.x < half) {
                const int t = threadIdx.x;
                int p = (round + t) % (n - 1);
                int q = (t == 0) ? n - 1 : (round - t + (n - 1)) % (n - 1);
                if (p > q) { const int tmp = p; p = q; q = tmp; }
                double c = 1.0, s = 0.0;
                const double apq = cur[p + (size_t)q * lda];
                if (apq != 0.0 && fabs(apq) > 1e-300) {
                    const double app = cur[p + (size_t)p * lda], aqq = cur[q + (size_t)q * lda];
                    const double zeta = (aqq - app) / (2.0 * apq);
                    const double tt = ((zeta >= 0.0) ? 1.0 : -1.0) / (fabs(zeta) + sqrt(1.0 + zeta * zeta));
                    c = 1.0 / sqrt(1.0 + tt * tt);
                    s = c * tt;
                }
                cs[t] = c; sn[t] = s; pp[t] = p; qq[t] = q;
            }
            __syncthreads();
            if (i < half) {
                const int p = pp[i], q = qq[i];
                const double c = cs[i], s = sn[i];
                const double* cp = cur + (size_t)p * lda;
                const double* cq = cur + (size_t)q * lda;
                double* np_ = nxt + (size_t)p * lda;
                double* nq_ = nxt + (size_t)q * lda;
                for (int t = threadIdx.x; t < half; t += blockDim.x) {
                    const int rp = pp[t], rq = qq[t];
                    const double ct = cs[t], st = sn[t];
                    // columns p, q rotated by (c, s), then rows rp, rq by (ct, st)
                    const double a_pp = cp[rp], a_pq = cq[rp], a_qp = cp[rq], a_qq = cq[rq];  // (row, column): rp/rq x p/q
                    const double u_p = c * a_pp - s * a_pq, u_q = s * a_pp + c * a_pq;          // row rp
                    const double w_p = c * a_qp - s * a_qq, w_q = s * a_qp + c * a_qq;          // row rq
                    np_[rp] = ct * u_p - st * w_p;
                    np_[rq] = st * u_p + ct * w_p;
                    nq_[rp] = ct * u_q - st * w_q;
                    nq_[rq] = st * u_q + ct * w_q;
                }
                double* vp = V + (size_t)p * ldv;
                double* vq = V + (size_t)q * ldv;
                for (int r = threadIdx.x; r < n; r += blockDim.x) {
                    const double x = vp[r], y = vq[r];
                    vp[r] = c * x - s * y;
                    vq[r] = s * x + c * y;
                }
            }
            double* tmp = cur; cur = nxt; nxt = tmp;
            grid_barrier(bar, G);
        }
    }
    if (cur != A0 && i < half)  // the diagonal (all the callers read) back into A0; every CTA copies its two columns
        for (int e = threadIdx.x; e < 2 * n; e += blockDim.x) {
            const int c = 2 * i + e / n, r = e % n;
            A0[r + (size_t)c * lda] = cur[r + (size_t)c * lda];
        }
}

// Step 1: dsc = diag(Gs)^{-1/2}, A0 = D^{-1/2} sym(Gs) D^{-1/2}, GhS = sym(Gh)
__global__ void k_rr_scale(int ns, const double* Gs, const double* Gh, double* dsc, double* A0, double* GhS)
{
    for (int e = blockIdx.x * blockDim.x + threadIdx.x; e < ns * ns; e += gridDim.x * blockDim.x) {
        const int i = e % ns, j = e / ns;
        const double gi = Gs[i + (size_t)i * ns], gj = Gs[j + (size_t)j * ns];
        const double di = (gi > 0.0 && isfinite(gi)) ? rsqrt(gi) : 0.0, dj = (gj > 0.0 && isfinite(gj)) ? rsqrt(gj) : 0.0;
        A0[e] = 0.5 * (Gs[i + (size_t)j * ns] + Gs[j + (size_t)i * ns]) * di * dj;
        GhS[e] = 0.5 * (Gh[i + (size_t)j * ns] + Gh[j + (size_t)i * ns]);
        if (j == 0) dsc[i] = di;
    }
}
// Step 2 (one CTA): keep the directions with Gram eigenvalue above 1e-12 of the largest; Tm = D^{-1/2} V_kept s^{-1/2}.
// info[0] = r (kept), info[1] = r rounded up to even (the size of the second eigenproblem).
__global__ void __launch_bounds__(1024) k_rr_select(int ns, const double* A0, const double* V, const double* dsc, double* Tm, int* info)
{
    __shared__ int sel[RD_DENSE_MAXN];
    __shared__ int s_r;
    if (info[2]) return;  // the Cholesky path already produced Tm
    if (threadIdx.x == 0) {
        double mx = 0.0;
        for (int j = 0; j < ns; ++j) mx = fmax(mx, A0[j + (size_t)j * ns]);
        int r = 0;
        for (int j = 0; j < ns; ++j)
            if (A0[j + (size_t)j * ns] > 1e-12 * mx) sel[r++] = j;
        s_r = r;
        info[0] = r;
        info[1] = (r + 1) & ~1;
    }
    __syncthreads();
    const int r = s_r;
    for (int e = threadIdx.x; e < ns * r; e += blockDim.x) {
        const int i = e % ns, q = e / ns;
        const int j = sel[q];
        Tm[i + (size_t)q * ns] = dsc[i] * V[i + (size_t)j * ns] * rsqrt(A0[j + (size_t)j * ns]);
    }
}
// Step 2, fast path (one CTA): Cholesky of the scaled Gram, A0 = L L^T; Tm = D^{-1/2} L^{-T}, all ns directions kept.
// info[2] = 1 on success; a pivot below 1e-10 (a basis that is dependent to working accuracy) leaves info[2] = 0 and the
// eigenvalue path (k_jacobi_grid + k_rr_select) runs instead.  Linv: ns x ns scratch.
__global__ void __launch_bounds__(1024) k_rr_chol(int ns, double* A0, const double* dsc, double* Linv, double* Tm, int* info, int force_fallback)
{
    __shared__ DenseShared ds;
    __shared__ int s_ok;
    const bool ok = !force_fallback && cta_cholesky(A0, ns, ns, ds);
    if (threadIdx.x == 0) {
        int good = ok ? 1 : 0;
        for (int j = 0; j < ns && good; ++j)
            if (!(A0[j + (size_t)j * ns] > 1e-5)) good = 0;  // L_jj^2 = pivot check: L_jj^2 is the pivot of the unit-diagonal Gram, 1e-10 = a direction dependent to 1e-5
        s_ok = good;
        info[2] = good;
        if (good) { info[0] = ns; info[1] = (ns + 1) & ~1; }
    }
    __syncthreads();
    if (!s_ok) return;
    cta_tri_inverse_lower(A0, ns, ns, Linv, ns);
    for (int e = threadIdx.x; e < ns * ns; e += blockDim.x) {
        const int i = e % ns, q = e / ns;
        Tm[e] = (i <= q) ? dsc[i] * Linv[q + (size_t)i * ns] : 0.0;  // (L^{-T})[i, q] = Linv[q, i]
    }
}

// Step 3: Q = GhS Tm (ns x r)
__global__ void k_rr_q(int ns, const int* info, const double* GhS, const double* Tm, double* Q)
{
    const int r = info[0];
    for (int e = blockIdx.x * blockDim.x + threadIdx.x; e < ns * r; e += gridDim.x * blockDim.x) {
        const int i = e % ns, q = e / ns;
        double a = 0.0;
        for (int l = 0; l < ns; ++l) a = fma(GhS[i + (size_t)l * ns], Tm[l + (size_t)q * ns], a);  // GhS symmetric: row i = column i
        Q[e] = a;
    }
}
// Step 4: A' = sym(Tm^T Q), r x r inside an re x re matrix (re = r rounded up to even; the pad index is decoupled and sorts last)
__global__ void k_rr_a(int ns, const int* info, const double* Tm, const double* Q, double* A0)
{
    const int r = info[0], re = info[1];
    for (int e = blockIdx.x * blockDim.x + threadIdx.x; e < re * re; e += gridDim.x * blockDim.x) {
        const int p = e % re, q = e / re;
        double a = 0.0;
        if (p < r && q < r) {
            double a1 = 0.0, a2 = 0.0;
            for (int i = 0; i < ns; ++i) {
                a1 = fma(Tm[i + (size_t)p * ns], Q[i + (size_t)q * ns], a1);
                a2 = fma(Tm[i + (size_t)q * ns], Q[i + (size_t)p * ns], a2);
            }
            a = 0.5 * (a1 + a2);
        } else if (p == q) {
            a = 1e300;
        }
        A0[e] = a;
    }
}
// Step 5 (one CTA): ascending order of the Ritz values, C = Tm U[:, lowest b], theta
__global__ void __launch_bounds__(1024) k_rr_finish(int ns, int b, const int* info, const double* A0, const double* U, const double* Tm,
                                                    double* C, double* theta)
{
    __shared__ int sel[RD_DENSE_MAXN];
    const int r = info[0], re = info[1];
    if (threadIdx.x == 0) {
        for (int j = 0; j < re; ++j) sel[j] = j;
        for (int j = 1; j < re; ++j) {
            const int pj = sel[j];
            const double v = A0[pj + (size_t)pj * re];
            int q = j - 1;
            while (q >= 0 && A0[sel[q] + (size_t)sel[q] * re] > v) { sel[q + 1] = sel[q]; --q; }
            sel[q + 1] = pj;
        }
    }
    __syncthreads();
    const int bo = min(b, r);
    for (int e = threadIdx.x; e < ns * b; e += blockDim.x) {
        const int i = e % ns, j = e / ns;
        double a = 0.0;
        if (j < bo) {
            const double* u = U + (size_t)sel[j] * re;
            for (int q = 0; q < r; ++q) a = fma(Tm[i + (size_t)q * ns], u[q], a);
        }
        C[i + (size_t)j * ns] = a;
    }
    for (int j = threadIdx.x; j < b; j += blockDim.x) theta[j] = (j < bo) ? A0[sel[j] + (size_t)sel[j] * re] : 0.0;
}

}  // namespace rd
