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
