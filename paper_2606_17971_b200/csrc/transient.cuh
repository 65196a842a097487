// Transient variant of the coarse-mesh reference, eq. (14) (section 2.2.2; reading A21):
// every spatial vector phi_i defines  H_i = (I (x) phi_i)^T H (I (x) phi_i),  D_i = (I (x) phi_i)^T diag(H) (I (x) phi_i)
// and the small generalized problem  H_i q = nu D_i q.   Layout of the all-at-once DOFs: id = space + N_s * t.
#pragma once
#include "common.cuh"
#include "dense.cuh"

namespace rd {

// v = e_t (x) phi: the slab t of v holds phi, every other slab is zero
__global__ void k_slab_vector(int64_t Ns, int nt, int t, const double* phi, double* v)
{
    const int64_t N = Ns * nt;
    for (int64_t r = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; r < N; r += (int64_t)gridDim.x * blockDim.x)
        v[r] = (r / Ns == t) ? phi[r % Ns] : 0.0;
}

// out[s] = sum_x a[s N_s + x] phi[x] (phi[x] once more if sq): one CTA per slab s, fixed summation order.
// Column t of H_i is (e_s (x) phi)^T (H (e_t (x) phi)) over s; D_i is the same sum with a = diag(H) and sq = 1.
__global__ void __launch_bounds__(256) k_slab_dots(int64_t Ns, const double* a, const double* phi, int sq, double* out)
{
    __shared__ double scratch[32];
    const double* as = a + (size_t)blockIdx.x * Ns;
    double acc = 0.0;
    for (int64_t x = threadIdx.x; x < Ns; x += blockDim.x) {
        const double p = phi[x];
        acc = fma(as[x], sq ? p * p : p, acc);
    }
    acc = block_sum(acc, scratch);
    if (threadIdx.x == 0) out[blockIdx.x] = acc;
}

// One CTA per spatial vector i: H_i q = nu D_i q through the symmetric scaling D_i^{-1/2} H_i D_i^{-1/2} p = nu p,
// q = D_i^{-1/2} p (so q^T D_i q = 1); cyclic Jacobi in global scratch, nu ascending, each q with its largest-magnitude
// component (lowest index on ties) positive.
//   Hs: gridDim.x x nt x nt (column-major, symmetrised here), Ds: gridDim.x x nt;  A, V: scratch of the size of Hs.
//   nu_out[i * nt + j], Q_out[(i * nt + j) * nt + t]
__global__ void __launch_bounds__(256) k_transient_eigs(int nt, const double* Hs, const double* Ds, double* A, double* V,
                                                         double* nu_out, double* Q_out)
{
    __shared__ DenseShared ds;
    __shared__ int order[RD_DENSE_MAXN];
    const int i = blockIdx.x;
    const double* Hi = Hs + (size_t)i * nt * nt;
    const double* Di = Ds + (size_t)i * nt;
    double* Ai = A + (size_t)i * nt * nt;
    double* Vi = V + (size_t)i * nt * nt;
    for (int e = threadIdx.x; e < nt * nt; e += blockDim.x) {
        const int a = e % nt, b = e / nt;
        Ai[e] = 0.5 * (Hi[a + (size_t)b * nt] + Hi[b + (size_t)a * nt]) / (sqrt(Di[a]) * sqrt(Di[b]));
    }
    __syncthreads();
    cta_jacobi_eig(Ai, nt, nt, Vi, nt, true, ds);
    __syncthreads();
    if (threadIdx.x == 0) {
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
        nu_out[(size_t)i * nt + j] = Ai[o + (size_t)o * nt];
        const double* p = Vi + (size_t)o * nt;
        double* q = Q_out + ((size_t)i * nt + j) * nt;
        int big = 0;
        for (int t = 0; t < nt; ++t) {
            q[t] = p[t] / sqrt(Di[t]);
            if (fabs(q[t]) > fabs(q[big])) big = t;
        }
        if (!(q[big] > 0.0))
            for (int t = 0; t < nt; ++t) q[t] = -q[t];
    }
}

// ---- compact (Kronecker-factored) reference: "the reference stores N_s r_s + N_t r floating-point values and
// r spatial-column indices.  Restriction evaluates a selected product at its inactive space-time entries."
//   W[x + N_s t, c] = Qc[t + nt c] * Phi[x + N_s sp[c]]       Phi: N_s x r_s,  Qc: nt x k,  sp: k spatial-column indices
// k_restrict_kron is S1 (eq. (12) / eq. (13)) straight from the factors: Wm = chi_I W without a stored dense W.
__global__ void k_restrict_kron(int64_t Ns, int nt, int64_t ldw, int k, int kp, const double* Phi, const double* Qc,
                                const int32_t* sp, const uint8_t* act, const uint8_t* hist, int zeroext, double* Wm)
{
    const int64_t N = Ns * nt;
    for (int64_t r = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; r < N; r += (int64_t)gridDim.x * blockDim.x) {
        const int64_t x = r % Ns;
        const int t = (int)(r / Ns);
        const bool keep = !act[r] && !(zeroext && hist[r]);
        for (int c = 0; c < kp; ++c)
            Wm[r + (size_t)c * ldw] = (keep && c < k) ? Qc[t + (size_t)nt * c] * ldg_f64(Phi + x + (size_t)Ns * sp[c]) : 0.0;
    }
}
// the dense N x k block of a compact reference (rd_get_reference), leading dimension ld
__global__ void k_kron_dense(int64_t Ns, int nt, int64_t ld, int k, const double* Phi, const double* Qc, const int32_t* sp, double* W)
{
    const int64_t N = Ns * nt;
    for (int64_t r = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; r < N; r += (int64_t)gridDim.x * blockDim.x) {
        const int64_t x = r % Ns;
        const int t = (int)(r / Ns);
        for (int c = 0; c < k; ++c) W[r + (size_t)c * ld] = Qc[t + (size_t)nt * c] * ldg_f64(Phi + x + (size_t)Ns * sp[c]);
    }
}
// Qc[:, c] = Q[sel_i[c]][sel_j[c]][:] * scale_c, sp[c] = position of sel_i[c] among the distinct spatial columns used
// (cols[]: their indices, rs_used entries).  scale_c = 1 (normalise = 0) or 1 / (||q||_2 ||phi_i||_2) (unit Euclidean
// columns of q (x) phi; phin2[i] = ||phi_i||_2^2).  One thread per reference column.
__global__ void k_kron_pack(int nt, int k, int rs_used, const int32_t* cols, const int32_t* sel, const double* Q,
                            int normalise, const double* phin2, double* Qc, int32_t* sp)
{
    const int c = blockIdx.x * blockDim.x + threadIdx.x;
    if (c >= k) return;
    const int mi = sel[2 * c], mj = sel[2 * c + 1];
    int pos = 0;
    for (int q = 0; q < rs_used; ++q)
        if (cols[q] == mi) pos = q;
    sp[c] = pos;
    const double* q = Q + ((size_t)mi * nt + mj) * nt;
    double scale = 1.0;
    if (normalise) {
        double s2 = 0.0;
        for (int t = 0; t < nt; ++t) s2 = fma(q[t], q[t], s2);
        scale = 1.0 / sqrt(s2 * phin2[mi]);
    }
    for (int t = 0; t < nt; ++t) Qc[t + (size_t)nt * c] = q[t] * scale;
}
// out[i] = sum_x Phi[x, i]^2 (one CTA per column, fixed order)
__global__ void __launch_bounds__(256) k_col_norm2(int64_t Ns, const double* Phi, double* out)
{
    __shared__ double scratch[32];
    const double* col = Phi + (size_t)blockIdx.x * Ns;
    double a = 0.0;
    for (int64_t x = threadIdx.x; x < Ns; x += blockDim.x) a = fma(col[x], col[x], a);
    a = block_sum(a, scratch);
    if (threadIdx.x == 0) out[blockIdx.x] = a;
}

// W[x + N_s t, c] = Q[sel_i[c]][sel_j[c]][t] * Phi[x, sel_i[c]]; columns c >= k are zero
__global__ void k_kron_vectors(int64_t Ns, int nt, int64_t ld, int k, int kp, const int32_t* sel, const double* Phi, const double* Q,
                               double* W)
{
    const int64_t N = Ns * nt;
    for (int64_t r = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; r < N; r += (int64_t)gridDim.x * blockDim.x) {
        const int64_t x = r % Ns;
        const int t = (int)(r / Ns);
        for (int c = 0; c < kp; ++c) {
            double v = 0.0;
            if (c < k) {
                const int mi = sel[2 * c], mj = sel[2 * c + 1];
                v = Q[((size_t)mi * nt + mj) * nt + t] * Phi[x + (size_t)mi * Ns];
            }
            W[r + (size_t)c * ld] = v;
        }
    }
}

}  // namespace rd
