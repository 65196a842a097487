// refdef_api.cu -- the C ABI of include/refdef.h: context, host orchestration of the PDAS loop, launches.
// One translation unit; all device code is in the .cuh files beside it.  Links only against cudart.
#include <cuda_runtime.h>

#include <algorithm>
#include <chrono>
#include <cmath>
#include <cstdarg>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <new>
#include <string>
#include <vector>

#include "../../include/refdef.h"
#include "cg.cuh"
#include "cg3.cuh"
#include "sine.cuh"
#include "prolong.cuh"
#include "transient.cuh"
#include "coarse.cuh"
#include "eigs.cuh"
#include "lobpcg.cuh"
#include "pdas.cuh"

using namespace rd;

namespace {

struct DevBuf {
    void* p = nullptr;
    size_t bytes = 0;
};

struct EllStore {
    int32_t* col = nullptr;
    double* val = nullptr;
    int64_t* off = nullptr;
    int64_t nslices = 0, entries = 0;
    int32_t uwd = -1;
    Ell view() const { return Ell{col, val, off, nslices, uwd}; }
};

}  // namespace

struct rd_ctx {
    int64_t N = 0, nnz = 0, ldw = 0;
    int device = 0, num_sms = 0;
    cudaStream_t stream = nullptr;
    double alpha = 0, sigma = 0;
    rd_options opt;
    std::string err;
    std::vector<void*> allocs;  // everything cudaMalloc'ed (freed in destroy)
    std::vector<void*> pinned;

    EllStore K, KT;
    double *m = nullptr, *minv = nullptr, *d = nullptr, *dinv = nullptr;
    // work vectors (length ldw)
    double *x = nullptr, *r = nullptr, *p0 = nullptr, *p1 = nullptr, *z = nullptr, *w = nullptr, *t = nullptr;
    double *b = nullptr, *tmp = nullptr, *Hy = nullptr, *ell = nullptr, *y = nullptr, *ystate = nullptr;
    double *lam = nullptr, *u = nullptr, *in0 = nullptr, *in1 = nullptr;  // staging for host callers
    uint8_t *act = nullptr, *act_new = nullptr, *hist = nullptr, *bits = nullptr, *act_stage = nullptr;
    uint8_t* act_seq = nullptr;  // the active set the next query of the sequence inherits; only rd_solve_query writes it
    uint8_t* h_bits = nullptr;  // pinned
    int* d_nactive = nullptr;
    int* h_nactive = nullptr;
    // reference
    int k = 0, kp = 0;
    // W: the stored reference.  Wm = chi_I W (restricted candidate basis).  Zm = Wm T: the basis Z of eq. (18), formed
    // explicitly; HZm = chi_I H Zm (the cached BZ); Zt / HZt: their tile-major copies for k_alg1_v3's ring.
    double *W = nullptr, *Wm = nullptr, *Zm = nullptr, *HZm = nullptr, *Zt = nullptr, *HZt = nullptr, *Tchunk = nullptr;
    // S6 compaction: per-slice flags and the two compact lists of live slices of the current active set
    uint8_t* sflags = nullptr;
    int32_t *listA = nullptr, *listB = nullptr, *d_live = nullptr;
    int32_t* h_live = nullptr;
    // compact (Kronecker-factored) reference: W[x + Ns t, c] = kQc[t + nt c] * kPhi[x + Ns ksp[c]]
    bool have_ref = false;
    int ref_kind = 0;  // 0: dense N x k block in W; 1: factors (kPhi, kQc, ksp), no dense copy is kept
    double *kPhi = nullptr, *kQc = nullptr;
    int32_t* ksp = nullptr;
    int64_t kNs = 0, kPhi_cap = 0;
    int knt = 0, krs = 0, kQc_cap = 0;
    int work_kp = 0;   // padded rank the work buffers (Wm, Zm, ...) were allocated for
    int dense_kp = 0;  // padded rank the dense block W was allocated for
    double2* coef = nullptr;  // CG-Lanczos coefficients of the last rd_solve_inactive (eq. (23) diagnostic)
    int32_t coef_cap = 0;
    bool want_ritz = false;
    double* d_ritz = nullptr;
    double *gram_parts = nullptr, *G = nullptr, *EW = nullptr, *cwork = nullptr, *C = nullptr;  // EW: W_I^T H W_I on request
    double *T = nullptr, *Eraw = nullptr, *E = nullptr, *CW = nullptr;  // T (W_I -> Z), E = Z^T B Z, C = E^{-1}, CW = T C T^T
    int gram_nparts = 0;
    CoarseInfo* d_cinfo = nullptr;
    CoarseInfo* h_cinfo = nullptr;
    // CG
    int cg_grid = 0;
    double* partial = nullptr;
    GridBarrier* bar = nullptr;
    CgDevReport* d_cgrep = nullptr;
    CgDevReport* h_cgrep = nullptr;
    PdasCounters* d_cnt = nullptr;
    PdasCounters* h_cnt = nullptr;
    cudaEvent_t ev[8];
    bool have_state = false;
    double ref_ms_pending = 0.0, ref_ms_last = 0.0;
    int64_t ref_degree = 0;  // total Chebyshev degree of the last rd_build_reference
    int ref_block = 0;       // its block size b
    int64_t ref_col_applies = 0;  // sum over filter degrees of the columns H was applied to (locked columns excluded)
    double ref_filter_ms = 0.0;   // CUDA-event time of all filter applies of the last build
    // work of the last rd_build_reference_lobpcg: FP64 tensor-core flop (sine transforms, Gram products, tall products),
    // column applies of H and of the preconditioner, CUDA-event time of the iteration loop
    double lob_flop = 0.0, lob_ms = 0.0;
    int64_t lob_h_applies = 0, lob_t_applies = 0;
    int64_t launches = 0;  // kernels launched so far (rd_kernel_launches)
};

namespace {

int fail(rd_ctx* c, int code, const char* fmt, ...)
{
    if (c) {
        char buf[512];
        va_list ap;
        va_start(ap, fmt);
        vsnprintf(buf, sizeof buf, fmt, ap);
        va_end(ap);
        c->err = buf;
    }
    return code;
}

#define CU(call)                                                                                        \
    do {                                                                                                \
        cudaError_t e__ = (call);                                                                       \
        if (e__ != cudaSuccess) return fail(ctx, RD_ECUDA, "%s: %s (%s:%d)", #call, cudaGetErrorString(e__), __FILE__, __LINE__); \
    } while (0)

bool is_device_ptr(const void* p)
{
    cudaPointerAttributes a;
    if (cudaPointerGetAttributes(&a, p) != cudaSuccess) {
        cudaGetLastError();
        return false;
    }
    return a.type == cudaMemoryTypeDevice || a.type == cudaMemoryTypeManaged;
}

template <class T>
int dalloc(rd_ctx* ctx, T** out, size_t count, bool zero = true)
{
    void* p = nullptr;
    size_t bytes = std::max<size_t>(count, 1) * sizeof(T);
    cudaError_t e = cudaMalloc(&p, bytes);
    if (e != cudaSuccess) {
        cudaGetLastError();
        return fail(ctx, RD_ENOMEM, "cudaMalloc(%zu bytes): %s", bytes, cudaGetErrorString(e));
    }
    ctx->allocs.push_back(p);
    if (zero) {
        e = cudaMemsetAsync(p, 0, bytes, ctx->stream);
        if (e != cudaSuccess) return fail(ctx, RD_ECUDA, "cudaMemsetAsync: %s", cudaGetErrorString(e));
    }
    *out = (T*)p;
    return RD_OK;
}
template <class T>
int halloc(rd_ctx* ctx, T** out, size_t count)
{
    void* p = nullptr;
    cudaError_t e = cudaMallocHost(&p, std::max<size_t>(count, 1) * sizeof(T));
    if (e != cudaSuccess) {
        cudaGetLastError();
        return fail(ctx, RD_ENOMEM, "cudaMallocHost: %s", cudaGetErrorString(e));
    }
    memset(p, 0, std::max<size_t>(count, 1) * sizeof(T));
    ctx->pinned.push_back(p);
    *out = (T*)p;
    return RD_OK;
}
#define RDTRY(x)                  \
    do {                          \
        int rc__ = (x);           \
        if (rc__ != RD_OK) return rc__; \
    } while (0)

// Host/device input: returns a device pointer holding `count` elements of src (staged if src is host).
template <class T>
int in_dev(rd_ctx* ctx, const T* src, size_t count, T* stage, const T** out)
{
    if (!src) { *out = nullptr; return RD_OK; }
    if (is_device_ptr(src)) { *out = src; return RD_OK; }
    CU(cudaMemcpyAsync(stage, src, count * sizeof(T), cudaMemcpyHostToDevice, ctx->stream));
    *out = stage;
    return RD_OK;
}
template <class T>
int out_host(rd_ctx* ctx, T* dst, const T* dev, size_t count)
{
    if (!dst || dst == dev) return RD_OK;
    CU(cudaMemcpyAsync(dst, dev, count * sizeof(T), is_device_ptr(dst) ? cudaMemcpyDeviceToDevice : cudaMemcpyDeviceToHost,
                       ctx->stream));
    return RD_OK;
}

inline int grid_for(int64_t work, int threads, int cap)
{
    int64_t g = (work + threads - 1) / threads;
    return (int)std::max<int64_t>(1, std::min<int64_t>(g, cap));
}

// ---- host construction of the two sliced-ELL matrices ------------------------------------------------
struct HostEll {
    std::vector<int32_t> col;
    std::vector<double> val;
    std::vector<int64_t> off;
};

void csr_to_ell(int64_t N, const std::vector<int64_t>& rp, const std::vector<int32_t>& ci, const std::vector<double>& va,
                HostEll& E)
{
    const int64_t ns = (N + RD_SLICE - 1) / RD_SLICE;
    E.off.assign(ns + 1, 0);
    for (int64_t s = 0; s < ns; ++s) {
        int64_t wd = 0;
        for (int64_t r = s * RD_SLICE; r < std::min(N, (s + 1) * RD_SLICE); ++r) wd = std::max(wd, rp[r + 1] - rp[r]);
        E.off[s + 1] = E.off[s] + wd * RD_SLICE;
    }
    E.col.assign(E.off[ns], 0);
    E.val.assign(E.off[ns], 0.0);
    for (int64_t s = 0; s < ns; ++s) {
        const int64_t wd = (E.off[s + 1] - E.off[s]) / RD_SLICE;
        for (int l = 0; l < RD_SLICE; ++l) {
            const int64_t r = s * RD_SLICE + l;
            const int32_t self = (int32_t)std::min<int64_t>(r, N - 1);
            const int64_t len = (r < N) ? rp[r + 1] - rp[r] : 0;
            for (int64_t e = 0; e < wd; ++e) {
                const int64_t pos = E.off[s] + e * RD_SLICE + l;
                if (e < len) { E.col[pos] = ci[rp[r] + e]; E.val[pos] = va[rp[r] + e]; }
                else { E.col[pos] = self; E.val[pos] = 0.0; }
            }
        }
    }
}

int upload_ell(rd_ctx* ctx, const HostEll& h, EllStore& d)
{
    d.nslices = (int64_t)h.off.size() - 1;
    d.entries = h.off.back();
    d.uwd = -1;
    if (d.nslices > 0) {
        const int64_t w0 = h.off[1] - h.off[0];
        bool uniform = true;
        for (int64_t s = 1; s < d.nslices && uniform; ++s) uniform = (h.off[s + 1] - h.off[s]) == w0;
        if (uniform && w0 / RD_SLICE <= 64) d.uwd = (int32_t)(w0 / RD_SLICE);
    }
    RDTRY(dalloc(ctx, &d.col, h.col.size(), false));
    RDTRY(dalloc(ctx, &d.val, h.val.size(), false));
    RDTRY(dalloc(ctx, &d.off, h.off.size(), false));
    CU(cudaMemcpyAsync(d.col, h.col.data(), h.col.size() * sizeof(int32_t), cudaMemcpyHostToDevice, ctx->stream));
    CU(cudaMemcpyAsync(d.val, h.val.data(), h.val.size() * sizeof(double), cudaMemcpyHostToDevice, ctx->stream));
    CU(cudaMemcpyAsync(d.off, h.off.data(), h.off.size() * sizeof(int64_t), cudaMemcpyHostToDevice, ctx->stream));
    CU(cudaStreamSynchronize(ctx->stream));  // the host vectors go away
    return RD_OK;
}

uint64_t fnv1a(const uint8_t* p, int64_t n)
{
    uint64_t h = 1469598103934665603ULL;
    for (int64_t i = 0; i < n; ++i) { h ^= (uint64_t)p[i]; h *= 1099511628211ULL; }
    return h;
}

constexpr int kThreads = 256;
inline int big_grid(rd_ctx* ctx) { return ctx->num_sms * 8; }

// out = H v (unmasked: act == NULL) or chi_I H v (v must already vanish on J).  Uses ctx->t.
int launch_apply_H(rd_ctx* ctx, const double* v, const uint8_t* act, double* out)
{
    const int g = grid_for(ctx->K.nslices * 32, kThreads, big_grid(ctx));
    k_apply_K<<<g, kThreads, 0, ctx->stream>>>(ctx->K.view(), ctx->N, ctx->minv, v, ctx->t);
    k_apply_KT_H<<<g, kThreads, 0, ctx->stream>>>(ctx->KT.view(), ctx->N, ctx->m, ctx->sigma, act, v, ctx->t, out);
    ctx->launches += 2;
    CU(cudaGetLastError());
    return RD_OK;
}

// Buffers for a reference of k columns: the work blocks of S1 / S2 always; the dense N x k block W only for the dense
// kind (a compact reference never materialises it).  Buffers of an earlier, smaller reference stay allocated until destroy.
int alloc_reference(rd_ctx* ctx, int k, bool need_dense = true)
{
    const int kp = (k + 7) & ~7;
    const size_t nk = (size_t)ctx->ldw * kp;
    if (ctx->work_kp < kp) {
        RDTRY(dalloc(ctx, &ctx->Wm, nk));
        RDTRY(dalloc(ctx, &ctx->Zm, nk));
        RDTRY(dalloc(ctx, &ctx->HZm, nk));
        RDTRY(dalloc(ctx, &ctx->Zt, nk));   // tile-major copies (k_alg1_v3); pad rows stay zero
        RDTRY(dalloc(ctx, &ctx->HZt, nk));
        RDTRY(dalloc(ctx, &ctx->Tchunk, (size_t)ctx->ldw * 8));
        ctx->gram_nparts = ctx->num_sms * 2;
        RDTRY(dalloc(ctx, &ctx->gram_parts, (size_t)ctx->gram_nparts * kp * kp));
        RDTRY(dalloc(ctx, &ctx->G, (size_t)kp * kp));
        RDTRY(dalloc(ctx, &ctx->EW, (size_t)kp * kp));
        RDTRY(dalloc(ctx, &ctx->cwork, (size_t)6 * kp * kp));
        RDTRY(dalloc(ctx, &ctx->C, (size_t)kp * kp));
        RDTRY(dalloc(ctx, &ctx->T, (size_t)kp * kp));
        RDTRY(dalloc(ctx, &ctx->Eraw, (size_t)kp * kp));
        RDTRY(dalloc(ctx, &ctx->E, (size_t)kp * kp));
        RDTRY(dalloc(ctx, &ctx->CW, (size_t)kp * kp));
        ctx->work_kp = kp;
    } else if (ctx->kp != kp) {
        // a narrower reference in wider buffers: the tile-major blocks are addressed with the new kp; clear the old layout
        CU(cudaMemsetAsync(ctx->Zt, 0, (size_t)ctx->ldw * ctx->work_kp * sizeof(double), ctx->stream));
        CU(cudaMemsetAsync(ctx->HZt, 0, (size_t)ctx->ldw * ctx->work_kp * sizeof(double), ctx->stream));
    }
    if (need_dense && ctx->dense_kp < kp) {
        RDTRY(dalloc(ctx, &ctx->W, nk));
        ctx->dense_kp = kp;
    }
    ctx->k = k;
    ctx->kp = kp;
    ctx->have_ref = false;  // the caller sets it once the reference is in place
    return RD_OK;
}

// S1 + S2 for the active set in ctx->act.  Leaves Zm, HZm (and their tile-major copies), E, C = E^{-1}, CW and *h_cinfo
// (the stream is synchronised before returning).  want_EW: also form W_I^T H_II W_I in ctx->EW (diagnostics only).
int coarse_setup(rd_ctx* ctx, int method, float* ms_restrict, float* ms_coarse, bool want_EW = false)
{
    const int64_t N = ctx->N;
    const int kp = ctx->kp;
    const bool tiles = ctx->opt.alg1_variant == 0;
    CU(cudaEventRecord(ctx->ev[0], ctx->stream));
    if (ctx->ref_kind == 1)  // compact reference: the selected products are evaluated at the inactive entries
        k_restrict_kron<<<grid_for(N, kThreads, big_grid(ctx)), kThreads, 0, ctx->stream>>>(
            ctx->kNs, ctx->knt, ctx->ldw, ctx->k, kp, ctx->kPhi, ctx->kQc, ctx->ksp, ctx->act, ctx->hist, method == RD_ZEROEXT ? 1 : 0, ctx->Wm);
    else
        k_restrict<<<grid_for(N, kThreads, big_grid(ctx)), kThreads, 0, ctx->stream>>>(
            N, ctx->ldw, ctx->k, kp, ctx->W, ctx->act, ctx->hist, method == RD_ZEROEXT ? 1 : 0, ctx->Wm);
    ctx->launches++;
    CU(cudaEventRecord(ctx->ev[1], ctx->stream));
    const int g = grid_for(ctx->K.nslices * 32, kThreads, big_grid(ctx));
    dim3 gg(ctx->gram_nparts, (kp + 63) / 64, (kp + 63) / 64);
    const int64_t kk = (int64_t)kp * kp;
    // H_II V for the kp columns of V, 8 at a time: OUT column-major, OUTT (may be NULL) tile-major
    auto spmm_H = [&](const double* V, double* OUT, double* OUTT) {
        for (int j = 0; j < kp; j += 8) {
            const double* Vj = V + (size_t)j * ctx->ldw;
            k_spmm_K<8><<<g, kThreads, 0, ctx->stream>>>(ctx->K.view(), N, ctx->ldw, ctx->minv, Vj, ctx->ldw, ctx->Tchunk);
            k_spmm_KT<8><<<g, kThreads, 0, ctx->stream>>>(ctx->KT.view(), N, ctx->ldw, ctx->m, ctx->sigma, ctx->act, Vj, ctx->ldw,
                                                           ctx->Tchunk, ctx->ldw, OUT + (size_t)j * ctx->ldw, OUTT, kp, j);
            ctx->launches += 2;
        }
    };
    auto gram = [&](const double* A, const double* B, double* out) {
        k_gram_dmma<<<gg, 256, 0, ctx->stream>>>(N, kp, kp, A, ctx->ldw, B, ctx->ldw, ctx->gram_parts);
        k_reduce_parts<<<grid_for(kk, kThreads, 64), kThreads, 0, ctx->stream>>>(ctx->gram_nparts, kk, ctx->gram_parts, out);
        ctx->launches += 2;
    };
    gram(ctx->Wm, ctx->Wm, ctx->G);
    if (want_EW) {  // W_I^T H_II W_I (HZm serves as scratch for H_II W_I; it is overwritten below)
        spmm_H(ctx->Wm, ctx->HZm, nullptr);
        gram(ctx->Wm, ctx->HZm, ctx->EW);
    }
    k_coarse_T<<<1, 1024, 0, ctx->stream>>>(kp, ctx->G, ctx->cwork, ctx->T, ctx->d_cinfo);
    k_basis_transform<<<dim3(std::max(1, grid_for(N, 256, big_grid(ctx)) / 2), kp / 8), 256, (size_t)kp * 8 * sizeof(double), ctx->stream>>>(
        N, ctx->ldw, kp, ctx->Wm, ctx->T, ctx->Zm, tiles ? ctx->Zt : nullptr);
    ctx->launches += 2;
    spmm_H(ctx->Zm, ctx->HZm, tiles ? ctx->HZt : nullptr);
    gram(ctx->Zm, ctx->HZm, ctx->Eraw);
    k_coarse_E<<<1, 1024, 0, ctx->stream>>>(kp, ctx->Eraw, ctx->T, ctx->cwork, ctx->E, ctx->C, ctx->CW, ctx->d_cinfo);
    ctx->launches++;
    CU(cudaGetLastError());
    CU(cudaMemcpyAsync(ctx->h_cinfo, ctx->d_cinfo, sizeof(CoarseInfo), cudaMemcpyDeviceToHost, ctx->stream));
    CU(cudaEventRecord(ctx->ev[2], ctx->stream));
    CU(cudaStreamSynchronize(ctx->stream));
    if (ms_restrict) CU(cudaEventElapsedTime(ms_restrict, ctx->ev[0], ctx->ev[1]));
    if (ms_coarse) CU(cudaEventElapsedTime(ms_coarse, ctx->ev[1], ctx->ev[2]));
    return RD_OK;
}

// Algorithm 1 on the system defined by ctx->act, rhs ctx->b, start ctx->x (both zero on J).  Blocking.
int run_alg1(rd_ctx* ctx, int method, int64_t n_inactive, rd_solve_report* rep, float* ms_restrict, float* ms_coarse)
{
    const int64_t N = ctx->N;
    memset(rep, 0, sizeof *rep);
    if (ms_restrict) *ms_restrict = 0;
    if (ms_coarse) *ms_coarse = 0;
    int use_coarse = 0;
    if (method != RD_JACOBI_CG) {
        if (!ctx->have_ref || ctx->k <= 0) return fail(ctx, RD_ENOREF, "method %d needs a reference (rd_build_reference / rd_set_reference)", method);
        RDTRY(coarse_setup(ctx, method, ms_restrict, ms_coarse));
        rep->rank_used = ctx->h_cinfo->rank;
        rep->coarse_fallback = ctx->h_cinfo->fallback;
        rep->cond_E = ctx->h_cinfo->cond_E;
        use_coarse = ctx->h_cinfo->rank > 0;
    }
    // zero-extension history A <- A u J after every restriction of the sequence, whichever method runs
    k_hist_update<<<grid_for(N, kThreads, big_grid(ctx)), kThreads, 0, ctx->stream>>>(N, ctx->act, ctx->hist);
    ctx->launches++;

    CgParams P;
    memset(&P, 0, sizeof P);
    P.N = N; P.ldw = ctx->ldw; P.kp = ctx->kp; P.use_coarse = use_coarse;
    P.K = ctx->K.view(); P.KT = ctx->KT.view();
    P.m = ctx->m; P.minv = ctx->minv; P.dinv = ctx->dinv; P.sigma = ctx->sigma;
    P.act = ctx->act; P.b = ctx->b;
    P.x = ctx->x; P.r = ctx->r; P.p0 = ctx->p0; P.p1 = ctx->p1; P.z = ctx->z; P.w = ctx->w; P.t = ctx->t;
    // the kernels work in the coordinates of the explicit basis Z = W_I T: "Wm" = Zm, "HWm" = H_II Zm, C = E^{-1}, "EW" = E
    P.Wm = ctx->Zm; P.HWm = ctx->HZm; P.HWt = ctx->HZt; P.C = ctx->C; P.EW = ctx->E;
    P.eps = ctx->opt.eps; P.eps_c = ctx->opt.eps_c; P.cap = ctx->opt.cg_cap; P.replace_period = ctx->opt.replace_period;
    P.partial = ctx->partial; P.bar = ctx->bar;
    {   // Part of the H_II Z stream is requested with L2 evict_last when the whole working set nearly fits the 126 MB L2
        // (config 2): what is left of an L2 budget after K, K^T and ten vectors, at most 90 % of the stream.  The budget
        // (MB) can be overridden with RD_L2_BUDGET_MB for experiments (profiles/r2_summary.md).
        static const double budget_mb = [] { const char* e = getenv("RD_L2_BUDGET_MB"); return e ? atof(e) : 80.0; }();
        const double hw_bytes = 8.0 * (double)n_inactive * ctx->kp;
        const double other = 12.0 * (double)(ctx->K.entries + ctx->KT.entries) + 80.0 * (double)N;
        double frac = hw_bytes > 0 ? std::min(0.9, std::max(0.0, (budget_mb * 1e6 - other) / hw_bytes)) : 0.0;
        const int64_t tiles_per_cta = ((n_inactive + 31) / 32 + ctx->cg_grid - 1) / ctx->cg_grid;
        P.hw_res_tiles = (int32_t)((double)tiles_per_cta * frac);
    } P.rep = ctx->d_cgrep;
    const int variant = ctx->opt.alg1_variant == 1 ? 1 : 0;
    {   // S6 compaction: live 32-row slices of this active set, as two compact lists (pdas.cuh), and zeroed work vectors
        // (rows outside the lists are never written by k_alg1_v3 and must read as zero)
        const int gsl = grid_for(ctx->K.nslices * 32, kThreads, big_grid(ctx));
        k_slice_flags<<<gsl, kThreads, 0, ctx->stream>>>(ctx->K.view(), N, ctx->act, ctx->sflags);
        k_slice_lists<<<1, 1024, 0, ctx->stream>>>(ctx->K.nslices, ctx->sflags, ctx->listA, ctx->listB, ctx->d_live);
        k_zero_vectors<<<grid_for(ctx->ldw, kThreads, big_grid(ctx)), kThreads, 0, ctx->stream>>>(ctx->ldw, ctx->p0, ctx->p1, ctx->z, ctx->w,
                                                                                               ctx->t, ctx->r);
        ctx->launches += 3;
        CU(cudaMemcpyAsync(ctx->h_live, ctx->d_live, 2 * sizeof(int32_t), cudaMemcpyDeviceToHost, ctx->stream));
        P.listA = ctx->listA; P.listB = ctx->listB; P.live_counts = ctx->d_live; P.Wt = ctx->Zt;
    }
    if (ctx->want_ritz && variant == 0) {  // eq. (23) diagnostic (rd_solve_inactive): record (a, beta) of every iteration
        const int32_t want = (int32_t)std::min<int64_t>(std::max(ctx->opt.cg_cap, 1), 1 << 20);
        if (ctx->coef_cap < want) {
            RDTRY(dalloc(ctx, &ctx->coef, (size_t)want));
            if (!ctx->d_ritz) RDTRY(dalloc(ctx, &ctx->d_ritz, 4));
            ctx->coef_cap = want;
        }
        P.coef = ctx->coef;
        P.coef_cap = ctx->coef_cap;
    }
    CU(cudaMemsetAsync(ctx->bar, 0, sizeof(GridBarrier), ctx->stream));
    CU(cudaEventRecord(ctx->ev[3], ctx->stream));
    void* args[] = {(void*)&P};
    if (variant == 0)
        CU(cudaLaunchCooperativeKernel((const void*)k_alg1_v3, dim3(ctx->cg_grid), dim3(RD_CG_THREADS), args, sizeof(Cg3Shared), ctx->stream));
    else
        CU(cudaLaunchCooperativeKernel((const void*)k_alg1, dim3(ctx->cg_grid), dim3(RD_CG_THREADS), args, 0, ctx->stream));
    ctx->launches++;
    CU(cudaEventRecord(ctx->ev[4], ctx->stream));
    CU(cudaMemcpyAsync(ctx->h_cgrep, ctx->d_cgrep, sizeof(CgDevReport), cudaMemcpyDeviceToHost, ctx->stream));
    CU(cudaStreamSynchronize(ctx->stream));
    float ms = 0;
    CU(cudaEventElapsedTime(&ms, ctx->ev[3], ctx->ev[4]));
    rep->iters = ctx->h_cgrep->iters;
    rep->replacements = ctx->h_cgrep->replacements;
    rep->status = ctx->h_cgrep->status;
    rep->rel_resid_verified = ctx->h_cgrep->rel_resid_verified;
    rep->t_iter_ms = ms;
    for (int q = 0; q < 8; ++q) rep->t_stage_us[q] = (variant == 0) ? ctx->h_cgrep->t_stage_us[q] : 0.0;
    // algorithmic HBM bytes of one loop iteration:
    // both ELL matrices once (8 B value + 4 B index per stored nonzero), t written and read on all N rows,
    // 14 vector passes over the n inactive rows, the two n x r passes over HW_I and W_I, the mask.
    const double rnk = use_coarse ? (double)rep->rank_used : 0.0;
    // k_alg1_v3 (default) passes over HW_I only: 8 n r instead of 16 n r.
    rep->bytes_per_iter = (24.0 * (double)ctx->nnz + 17.0 * (double)N) * ((double)n_inactive / (double)N) + 112.0 * (double)n_inactive +
                          (variant == 0 ? 8.0 : 16.0) * (double)n_inactive * rnk;
    rep->live_slices_A = ctx->h_live[0];
    rep->live_slices_B = ctx->h_live[1];
    if (P.coef && rep->iters > 0) {
        double h[3];
        k_ritz_extremes<<<1, 1024, 0, ctx->stream>>>(std::min(rep->iters, ctx->coef_cap), ctx->coef, ctx->d_ritz);
        ctx->launches++;
        CU(cudaGetLastError());
        CU(cudaMemcpyAsync(h, ctx->d_ritz, sizeof h, cudaMemcpyDeviceToHost, ctx->stream));
        CU(cudaStreamSynchronize(ctx->stream));
        rep->ritz_min = h[0]; rep->ritz_max = h[1]; rep->ritz_count = (int32_t)h[2];
    }
    return RD_OK;
}

// The count lowest products of 1-D sine modes, ordered by (mu, q_1, ..., q_d); mu is summed over the per-axis terms in
// ascending order so that permuted tuples tie exactly (reading A18).
struct SineCand { double mu; int q[3]; };
void select_sine_modes(int ndim, const int64_t* dims, int count, std::vector<SineCand>& cand, int* qmax_out)
{
    const int k = count;
    int qmax = 1;
    std::vector<std::vector<double>> terms(ndim);
    for (int a = 0; a < ndim; ++a) {
        const int64_t n = dims[a];
        const int qa = (int)std::min<int64_t>(n, k);
        qmax = std::max(qmax, qa);
        terms[a].resize(qa);
        for (int q = 1; q <= qa; ++q) {
            const double s = std::sin(M_PI * q / (2.0 * n));
            terms[a][q - 1] = 4.0 * n * n * (s * s);
        }
    }
    const int q0n = (int)terms[0].size(), q1n = ndim > 1 ? (int)terms[1].size() : 1, q2n = ndim > 2 ? (int)terms[2].size() : 1;
    cand.reserve((size_t)q0n * q1n * q2n);
    for (int q0 = 1; q0 <= q0n; ++q0)
        for (int q1 = 1; q1 <= q1n; ++q1)
            for (int q2 = 1; q2 <= q2n; ++q2) {
                double p[3] = {terms[0][q0 - 1], ndim > 1 ? terms[1][q1 - 1] : 0.0, ndim > 2 ? terms[2][q2 - 1] : 0.0};
                std::sort(p, p + ndim);
                double mu = 0.0;
                for (int a = 0; a < ndim; ++a) mu += p[a];
                cand.push_back(SineCand{mu, {q0, q1, q2}});
            }
    std::sort(cand.begin(), cand.end(), [](const SineCand& x, const SineCand& y) {
        if (x.mu != y.mu) return x.mu < y.mu;
        if (x.q[0] != y.q[0]) return x.q[0] < y.q[0];
        if (x.q[1] != y.q[1]) return x.q[1] < y.q[1];
        return x.q[2] < y.q[2];
    });
    cand.resize(std::min<size_t>(cand.size(), (size_t)count));
    if (qmax_out) *qmax_out = qmax;
}

// Stores a compact reference: Phi_used (Ns x rs_used, device, column-major ld Ns) is copied into the
// context; Qc (nt x k) and sp (k) are packed from the per-vector temporal eigenvectors Q[(i * nt + j) * nt + t] and the
// selection sel (k pairs (i, j)); cols[] lists the rs_used distinct spatial indices i in the order of Phi_used's columns.
int store_kron(rd_ctx* ctx, int k, int64_t Ns, int nt, int rs_used, const double* d_Phi_used, const std::vector<int32_t>& cols,
               const int32_t* d_sel, const double* d_Q, int normalise, const double* d_phin2)
{
    const int64_t need_phi = Ns * rs_used;
    if (ctx->kPhi_cap < need_phi) { RDTRY(dalloc(ctx, &ctx->kPhi, (size_t)need_phi, false)); ctx->kPhi_cap = need_phi; }
    if (ctx->kQc_cap < nt * k) {
        RDTRY(dalloc(ctx, &ctx->kQc, (size_t)nt * k, false));
        RDTRY(dalloc(ctx, &ctx->ksp, (size_t)k + RD_MAX_K, false));
        ctx->kQc_cap = nt * k;
    }
    CU(cudaMemcpyAsync(ctx->kPhi, d_Phi_used, (size_t)need_phi * sizeof(double), cudaMemcpyDeviceToDevice, ctx->stream));
    int32_t* d_cols = ctx->ksp + k;  // scratch behind sp
    CU(cudaMemcpyAsync(d_cols, cols.data(), (size_t)rs_used * sizeof(int32_t), cudaMemcpyHostToDevice, ctx->stream));
    k_kron_pack<<<1, RD_MAX_K, 0, ctx->stream>>>(nt, k, rs_used, d_cols, d_sel, d_Q, normalise, d_phin2, ctx->kQc, ctx->ksp);
    ctx->launches++;
    CU(cudaGetLastError());
    CU(cudaStreamSynchronize(ctx->stream));
    ctx->kNs = Ns; ctx->knt = nt; ctx->krs = rs_used;
    ctx->ref_kind = 1;
    ctx->have_ref = true;
    return RD_OK;
}

}  // namespace

// =====================================================================================================
extern "C" {

void rd_default_options(rd_options* o)
{
    o->sigma_is_alpha = 1.0;
    o->eps = 1e-8;
    o->eps_c = 1e-8;
    o->cg_cap = 500000;
    o->pdas_cap = 100;
    o->replace_period = 0;
    o->jacobi = 1;
    o->c_is_diag = 0;
    o->init = RD_INIT_PAPER;
    o->alg1_variant = 0;
}

const char* rd_last_error(const rd_ctx* ctx) { return ctx ? ctx->err.c_str() : "null context"; }

void rd_destroy(rd_ctx* ctx)
{
    if (!ctx) return;
    cudaStreamSynchronize(ctx->stream);
    for (void* p : ctx->allocs) cudaFree(p);
    for (void* p : ctx->pinned) cudaFreeHost(p);
    for (auto& e : ctx->ev) if (e) cudaEventDestroy(e);
    delete ctx;
}

int64_t rd_kernel_launches(const rd_ctx* ctx) { return ctx ? ctx->launches : 0; }

int rd_create(rd_ctx** out, int64_t N, const int64_t* rowptr, const int32_t* colidx, const double* val,
              const double* m_diag, double alpha, const rd_options* opt, void* cuda_stream)
{
    if (!out) return RD_EINVAL;
    *out = nullptr;
    if (N <= 0 || N > 2000000000LL || !rowptr || !colidx || !val || !m_diag || !(alpha > 0.0)) return RD_EINVAL;
    int ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev == 0) {
        cudaGetLastError();
        return RD_ECUDA;  // no CPU fallback
    }
    rd_ctx* ctx = new (std::nothrow) rd_ctx();
    if (!ctx) return RD_ENOMEM;
    for (auto& e : ctx->ev) e = nullptr;
    *out = ctx;  // returned even on failure so that rd_last_error can be read; caller destroys
    ctx->stream = (cudaStream_t)cuda_stream;
    ctx->N = N;
    ctx->ldw = (N + 31) & ~(int64_t)31;
    ctx->alpha = alpha;
    if (opt) ctx->opt = *opt; else rd_default_options(&ctx->opt);
    ctx->sigma = (ctx->opt.sigma_is_alpha != 0.0) ? alpha : 1.0 / alpha;
    CU(cudaGetDevice(&ctx->device));
    cudaDeviceProp prop;
    CU(cudaGetDeviceProperties(&prop, ctx->device));
    ctx->num_sms = prop.multiProcessorCount;
    if (!prop.cooperativeLaunch) return fail(ctx, RD_ECUDA, "device lacks cooperative launch");
    for (auto& e : ctx->ev) CU(cudaEventCreate(&e));

    // ---- bring the CSR to the host (setup only), sort rows, merge duplicates ----
    std::vector<int64_t> rp(N + 1);
    CU(cudaMemcpy(rp.data(), rowptr, (N + 1) * sizeof(int64_t), cudaMemcpyDefault));
    const int64_t nnz_in = rp[N];
    if (rp[0] != 0 || nnz_in < 0) return fail(ctx, RD_EINVAL, "rowptr[0] != 0 or negative nnz");
    std::vector<int32_t> ci(nnz_in);
    std::vector<double> va(nnz_in), mh(N);
    CU(cudaMemcpy(ci.data(), colidx, nnz_in * sizeof(int32_t), cudaMemcpyDefault));
    CU(cudaMemcpy(va.data(), val, nnz_in * sizeof(double), cudaMemcpyDefault));
    CU(cudaMemcpy(mh.data(), m_diag, N * sizeof(double), cudaMemcpyDefault));
    for (int64_t i = 0; i < N; ++i)
        if (!(mh[i] > 0.0) || !std::isfinite(mh[i])) return fail(ctx, RD_ENOTSPD, "m[%lld] = %g is not > 0", (long long)i, mh[i]);
    std::vector<int64_t> rp2(N + 1, 0);
    std::vector<int32_t> ci2;
    std::vector<double> va2;
    ci2.reserve(nnz_in);
    va2.reserve(nnz_in);
    {
        std::vector<std::pair<int32_t, double>> row;
        for (int64_t r = 0; r < N; ++r) {
            if (rp[r + 1] < rp[r]) return fail(ctx, RD_EINVAL, "rowptr not monotone at row %lld", (long long)r);
            row.clear();
            for (int64_t e = rp[r]; e < rp[r + 1]; ++e) {
                if (ci[e] < 0 || ci[e] >= N) return fail(ctx, RD_EINVAL, "column index out of range at entry %lld", (long long)e);
                row.emplace_back(ci[e], va[e]);
            }
            std::stable_sort(row.begin(), row.end(), [](const std::pair<int32_t, double>& a, const std::pair<int32_t, double>& b) { return a.first < b.first; });
            for (size_t q = 0; q < row.size(); ++q) {
                if (!ci2.empty() && (int64_t)ci2.size() > rp2[r] && ci2.back() == row[q].first) va2.back() += row[q].second;
                else { ci2.push_back(row[q].first); va2.push_back(row[q].second); }
            }
            rp2[r + 1] = (int64_t)ci2.size();
        }
    }
    ctx->nnz = rp2[N];
    // transpose (counting sort: rows of K^T come out with ascending column = ascending row of K)
    std::vector<int64_t> tp(N + 1, 0);
    for (int64_t e = 0; e < ctx->nnz; ++e) tp[ci2[e] + 1]++;
    for (int64_t i = 0; i < N; ++i) tp[i + 1] += tp[i];
    std::vector<int32_t> tc(ctx->nnz);
    std::vector<double> tv(ctx->nnz);
    {
        std::vector<int64_t> cur(tp.begin(), tp.end() - 1);
        for (int64_t r = 0; r < N; ++r)
            for (int64_t e = rp2[r]; e < rp2[r + 1]; ++e) {
                const int64_t pos = cur[ci2[e]]++;
                tc[pos] = (int32_t)r;
                tv[pos] = va2[e];
            }
    }
    {
        HostEll hk, hkt;
        csr_to_ell(N, rp2, ci2, va2, hk);
        csr_to_ell(N, tp, tc, tv, hkt);
        RDTRY(upload_ell(ctx, hk, ctx->K));
        RDTRY(upload_ell(ctx, hkt, ctx->KT));
    }
    const size_t L = (size_t)ctx->ldw;
    RDTRY(dalloc(ctx, &ctx->m, L));
    RDTRY(dalloc(ctx, &ctx->minv, L));
    RDTRY(dalloc(ctx, &ctx->d, L));
    RDTRY(dalloc(ctx, &ctx->dinv, L));
    {
        std::vector<double> mi(N);
        for (int64_t i = 0; i < N; ++i) mi[i] = 1.0 / mh[i];
        CU(cudaMemcpyAsync(ctx->m, mh.data(), N * sizeof(double), cudaMemcpyHostToDevice, ctx->stream));
        CU(cudaMemcpyAsync(ctx->minv, mi.data(), N * sizeof(double), cudaMemcpyHostToDevice, ctx->stream));
        CU(cudaStreamSynchronize(ctx->stream));
    }
    double** vecs[] = {&ctx->x, &ctx->r, &ctx->p0, &ctx->p1, &ctx->z, &ctx->w, &ctx->t, &ctx->b, &ctx->tmp, &ctx->Hy,
                       &ctx->ell, &ctx->y, &ctx->ystate, &ctx->lam, &ctx->u, &ctx->in0, &ctx->in1};
    for (double** v : vecs) RDTRY(dalloc(ctx, v, L));
    RDTRY(dalloc(ctx, &ctx->act, L));
    RDTRY(dalloc(ctx, &ctx->act_new, L));
    RDTRY(dalloc(ctx, &ctx->hist, L));
    RDTRY(dalloc(ctx, &ctx->act_stage, L));
    RDTRY(dalloc(ctx, &ctx->act_seq, L));
    RDTRY(dalloc(ctx, &ctx->bits, (size_t)(N + 7) / 8));
    RDTRY(halloc(ctx, &ctx->h_bits, (size_t)(N + 7) / 8));
    RDTRY(dalloc(ctx, &ctx->d_nactive, 1));
    RDTRY(halloc(ctx, &ctx->h_nactive, 1));
    RDTRY(dalloc(ctx, &ctx->d_cinfo, 1));
    RDTRY(halloc(ctx, &ctx->h_cinfo, 1));
    RDTRY(dalloc(ctx, &ctx->d_cgrep, 1));
    RDTRY(halloc(ctx, &ctx->h_cgrep, 1));
    RDTRY(dalloc(ctx, &ctx->d_cnt, 1));
    RDTRY(halloc(ctx, &ctx->h_cnt, 1));
    RDTRY(dalloc(ctx, &ctx->bar, 1));
    RDTRY(dalloc(ctx, &ctx->sflags, (size_t)ctx->K.nslices));
    RDTRY(dalloc(ctx, &ctx->listA, (size_t)ctx->K.nslices));
    RDTRY(dalloc(ctx, &ctx->listB, (size_t)ctx->K.nslices));
    RDTRY(dalloc(ctx, &ctx->d_live, 2));
    RDTRY(halloc(ctx, &ctx->h_live, 2));
    // persistent Algorithm-1 kernel: one CTA per SM, all co-resident
    int occ = 0;
    CU(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, k_alg1, RD_CG_THREADS, 0));
    if (occ < 1) return fail(ctx, RD_ECUDA, "k_alg1 does not fit an SM (occupancy 0)");
    CU(cudaFuncSetAttribute(k_alg1_v3, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sizeof(Cg3Shared)));
    CU(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, k_alg1_v3, RD_CG_THREADS, sizeof(Cg3Shared)));
    if (occ < 1) return fail(ctx, RD_ECUDA, "k_alg1_v3 does not fit an SM (occupancy 0)");
    ctx->cg_grid = ctx->num_sms;
    RDTRY(dalloc(ctx, &ctx->partial, (size_t)2 * SL_NSLOT * ctx->cg_grid));
    // d = diag(H), dinv
    k_diag_H<<<grid_for(ctx->KT.nslices * 32, kThreads, big_grid(ctx)), kThreads, 0, ctx->stream>>>(
        ctx->KT.view(), N, ctx->m, ctx->minv, ctx->sigma, ctx->opt.jacobi, ctx->d, ctx->dinv);
    ctx->launches++;
    CU(cudaGetLastError());
    CU(cudaStreamSynchronize(ctx->stream));
    return RD_OK;
}

int rd_set_options(rd_ctx* ctx, const rd_options* opt)
{
    if (!ctx || !opt) return RD_EINVAL;
    if ((opt->sigma_is_alpha != 0.0) != (ctx->opt.sigma_is_alpha != 0.0)) return fail(ctx, RD_EINVAL, "sigma_is_alpha is fixed at create");
    const bool jac_changed = (opt->jacobi != 0) != (ctx->opt.jacobi != 0);
    ctx->opt = *opt;
    if (jac_changed) {
        k_diag_H<<<grid_for(ctx->KT.nslices * 32, kThreads, big_grid(ctx)), kThreads, 0, ctx->stream>>>(
            ctx->KT.view(), ctx->N, ctx->m, ctx->minv, ctx->sigma, ctx->opt.jacobi, ctx->d, ctx->dinv);
        ctx->launches++;
        CU(cudaGetLastError());
    }
    return RD_OK;
}

int rd_reset_sequence(rd_ctx* ctx)
{
    if (!ctx) return RD_EINVAL;
    ctx->have_state = false;
    CU(cudaMemsetAsync(ctx->ystate, 0, ctx->ldw * sizeof(double), ctx->stream));
    CU(cudaMemsetAsync(ctx->act, 0, ctx->ldw, ctx->stream));
    CU(cudaMemsetAsync(ctx->act_seq, 0, ctx->ldw, ctx->stream));
    CU(cudaMemsetAsync(ctx->hist, 0, ctx->ldw, ctx->stream));
    return RD_OK;
}

int rd_apply_K(rd_ctx* ctx, const double* v, double* out)
{
    if (!ctx || !v || !out) return RD_EINVAL;
    const double* dv;
    RDTRY(in_dev(ctx, v, ctx->N, ctx->in0, &dv));
    double* dout = is_device_ptr(out) ? out : ctx->tmp;
    k_apply_K<<<grid_for(ctx->K.nslices * 32, kThreads, big_grid(ctx)), kThreads, 0, ctx->stream>>>(ctx->K.view(), ctx->N, nullptr, dv, dout);
    ctx->launches++;
    CU(cudaGetLastError());
    RDTRY(out_host(ctx, out, dout, ctx->N));
    CU(cudaStreamSynchronize(ctx->stream));
    return RD_OK;
}

int rd_apply_KT(rd_ctx* ctx, const double* v, double* out)
{
    if (!ctx || !v || !out) return RD_EINVAL;
    const double* dv;
    RDTRY(in_dev(ctx, v, ctx->N, ctx->in0, &dv));
    double* dout = is_device_ptr(out) ? out : ctx->tmp;
    k_apply_K<<<grid_for(ctx->KT.nslices * 32, kThreads, big_grid(ctx)), kThreads, 0, ctx->stream>>>(ctx->KT.view(), ctx->N, nullptr, dv, dout);
    ctx->launches++;
    CU(cudaGetLastError());
    RDTRY(out_host(ctx, out, dout, ctx->N));
    CU(cudaStreamSynchronize(ctx->stream));
    return RD_OK;
}

int rd_apply_H(rd_ctx* ctx, const double* v, const uint8_t* active, double* out)
{
    if (!ctx || !v || !out) return RD_EINVAL;
    const double* dv;
    const uint8_t* da;
    RDTRY(in_dev(ctx, v, ctx->N, ctx->in0, &dv));
    RDTRY(in_dev(ctx, active, ctx->N, ctx->act_stage, &da));
    double* dout = is_device_ptr(out) ? out : ctx->tmp;
    const double* vin = dv;
    if (da) {  // chi_I v
        k_mask_copy<<<grid_for(ctx->N, kThreads, big_grid(ctx)), kThreads, 0, ctx->stream>>>(ctx->N, da, dv, ctx->in1);
        ctx->launches++;
        vin = ctx->in1;
    }
    RDTRY(launch_apply_H(ctx, vin, da, dout));
    RDTRY(out_host(ctx, out, dout, ctx->N));
    CU(cudaStreamSynchronize(ctx->stream));
    return RD_OK;
}

int rd_diag_H(rd_ctx* ctx, double* d_out)
{
    if (!ctx || !d_out) return RD_EINVAL;
    RDTRY(out_host(ctx, d_out, ctx->d, ctx->N));
    CU(cudaStreamSynchronize(ctx->stream));
    return RD_OK;
}

int rd_build_reference_prolonged(rd_ctx* ctx, int32_t k, int32_t ndim, const int64_t* dims_c, const int64_t* dims_f,
                                 const double* Wc, double* norms_out)
{
    if (!ctx || !dims_c || !dims_f || !Wc || k < 1 || k > RD_MAX_K || ndim < 1 || ndim > 3) return RD_EINVAL;
    int64_t Nc = 1, Nf = 1;
    for (int a = 0; a < ndim; ++a) {
        if (dims_c[a] < 1 || dims_c[a] > (1 << 20)) return fail(ctx, RD_EINVAL, "dims_c[%d] = %lld", a, (long long)dims_c[a]);
        if (dims_f[a] < 1 || dims_f[a] > (1 << 20)) return fail(ctx, RD_EINVAL, "dims_f[%d] = %lld", a, (long long)dims_f[a]);
        Nc *= dims_c[a];
        Nf *= dims_f[a];
    }
    if (Nf != ctx->N) return fail(ctx, RD_EINVAL, "product of dims_f %lld is not N = %lld (steady Cartesian grids only)", (long long)Nf, (long long)ctx->N);
    const auto t_begin = std::chrono::steady_clock::now();
    RDTRY(alloc_reference(ctx, k));
    const int kp = ctx->kp, nparts = ctx->num_sms;
    // scratch of this call: a device copy of the coarse block (Wc may be a host pointer), partial sums, norms
    double *d_Wc = nullptr, *d_parts = nullptr, *d_norms = nullptr;
    std::vector<double> norms(k, 0.0);
    cudaError_t e = cudaMalloc(&d_Wc, (size_t)Nc * k * sizeof(double));
    if (e == cudaSuccess) e = cudaMalloc(&d_parts, (size_t)nparts * k * sizeof(double));
    if (e == cudaSuccess) e = cudaMalloc(&d_norms, (size_t)k * sizeof(double));
    if (e != cudaSuccess) {
        cudaGetLastError();
        cudaFree(d_Wc), cudaFree(d_parts), cudaFree(d_norms);
        return fail(ctx, RD_ENOMEM, "cudaMalloc of the coarse block (%lld x %d)", (long long)Nc, k);
    }
    e = cudaMemcpyAsync(d_Wc, Wc, (size_t)Nc * k * sizeof(double), cudaMemcpyDefault, ctx->stream);
    if (e == cudaSuccess) e = cudaMemsetAsync(ctx->W, 0, (size_t)ctx->ldw * kp * sizeof(double), ctx->stream);  // pad rows stay zero
    const int c0 = (int)dims_c[0], c1 = ndim > 1 ? (int)dims_c[1] : 1, c2 = ndim > 2 ? (int)dims_c[2] : 1;
    const int f0 = (int)dims_f[0], f1 = ndim > 1 ? (int)dims_f[1] : 1, f2 = ndim > 2 ? (int)dims_f[2] : 1;
    const int g = grid_for(ctx->N, kThreads, big_grid(ctx));
    k_prolong_p1<<<g, kThreads, 0, ctx->stream>>>(ctx->N, ctx->ldw, ndim, c0, c1, c2, f0, f1, f2, k, kp, d_Wc, Nc, ctx->W);
    k_col_sumsq_parts<<<dim3(nparts, k), kThreads, 0, ctx->stream>>>(ctx->N, ctx->ldw, ctx->W, d_parts);
    k_col_normalise<<<dim3(std::max(1, g / 8), k), kThreads, 0, ctx->stream>>>(ctx->N, ctx->ldw, nparts, d_parts, ctx->W, d_norms);
    ctx->launches += 3;
    if (e == cudaSuccess) e = cudaGetLastError();
    if (e == cudaSuccess) e = cudaMemcpyAsync(norms.data(), d_norms, (size_t)k * sizeof(double), cudaMemcpyDeviceToHost, ctx->stream);
    if (e == cudaSuccess) e = cudaStreamSynchronize(ctx->stream);
    cudaFree(d_Wc), cudaFree(d_parts), cudaFree(d_norms);
    if (e != cudaSuccess) return fail(ctx, RD_ECUDA, "prolonged reference: %s", cudaGetErrorString(e));
    if (norms_out) for (int c = 0; c < k; ++c) norms_out[c] = norms[c];
    for (int c = 0; c < k; ++c)
        if (!(norms[c] > 0.0) || !std::isfinite(norms[c])) {
            ctx->k = 0;  // no usable reference
            return fail(ctx, RD_EINVAL, "column %d of the prolonged reference has norm %g", c, norms[c]);
        }
    ctx->have_ref = true;
    ctx->ref_kind = 0;
    ctx->ref_degree = 0;
    ctx->ref_col_applies = 0;
    ctx->lob_flop = 0.0;
    ctx->lob_ms = 0.0;
    ctx->ref_filter_ms = 0.0;
    ctx->ref_block = k;
    ctx->ref_ms_pending = std::chrono::duration<double, std::milli>(std::chrono::steady_clock::now() - t_begin).count();
    ctx->ref_ms_last = ctx->ref_ms_pending;
    return RD_OK;
}

int rd_set_reference(rd_ctx* ctx, int32_t k, const double* W)
{
    if (!ctx || !W || k < 1 || k > RD_MAX_K) return RD_EINVAL;
    RDTRY(alloc_reference(ctx, k));
    CU(cudaMemsetAsync(ctx->W, 0, (size_t)ctx->ldw * ctx->kp * sizeof(double), ctx->stream));
    CU(cudaMemcpy2DAsync(ctx->W, ctx->ldw * sizeof(double), W, ctx->N * sizeof(double), ctx->N * sizeof(double), k,
                         cudaMemcpyDefault, ctx->stream));
    CU(cudaStreamSynchronize(ctx->stream));
    ctx->have_ref = true;
    ctx->ref_kind = 0;
    ctx->ref_ms_pending = 0.0;
    return RD_OK;
}

int rd_get_reference(rd_ctx* ctx, double* W_out, int32_t* k_out)
{
    if (!ctx) return RD_EINVAL;
    if (k_out) *k_out = ctx->have_ref ? ctx->k : 0;
    if (!W_out || !ctx->have_ref || ctx->k <= 0) return RD_OK;
    if (ctx->ref_kind == 1) {  // compact reference: the dense block is formed for the caller only
        double* dst = W_out;
        double* tmp = nullptr;
        if (!is_device_ptr(W_out)) {
            if (cudaMalloc(&tmp, (size_t)ctx->N * ctx->k * sizeof(double)) != cudaSuccess) {
                cudaGetLastError();
                return fail(ctx, RD_ENOMEM, "cudaMalloc of the dense copy of a compact reference");
            }
            dst = tmp;
        }
        k_kron_dense<<<grid_for(ctx->N, kThreads, big_grid(ctx)), kThreads, 0, ctx->stream>>>(ctx->kNs, ctx->knt, ctx->N, ctx->k, ctx->kPhi,
                                                                                           ctx->kQc, ctx->ksp, dst);
        ctx->launches++;
        cudaError_t e = cudaGetLastError();
        if (e == cudaSuccess && tmp) e = cudaMemcpyAsync(W_out, tmp, (size_t)ctx->N * ctx->k * sizeof(double), cudaMemcpyDeviceToHost, ctx->stream);
        if (e == cudaSuccess) e = cudaStreamSynchronize(ctx->stream);
        if (tmp) cudaFree(tmp);
        if (e != cudaSuccess) return fail(ctx, RD_ECUDA, "rd_get_reference: %s", cudaGetErrorString(e));
        return RD_OK;
    }
    CU(cudaMemcpy2DAsync(W_out, ctx->N * sizeof(double), ctx->W, ctx->ldw * sizeof(double), ctx->N * sizeof(double), ctx->k,
                         cudaMemcpyDefault, ctx->stream));
    CU(cudaStreamSynchronize(ctx->stream));
    return RD_OK;
}

int rd_build_reference(rd_ctx* ctx, int32_t k, double tol, int32_t max_block_iters, double* theta_out, double* resid_out,
                       int32_t* iters_out)
{
    if (!ctx || k < 1 || k > RD_MAX_K || !(tol > 0.0) || max_block_iters < 1) return RD_EINVAL;
    if (k > ctx->N) return fail(ctx, RD_EINVAL, "k = %d exceeds N = %lld", k, (long long)ctx->N);
    const int64_t N = ctx->N, ld = ctx->ldw;
    // block size: k plus a guard of max(8, k/4) vectors, a multiple of 8, never more than N rounded up
    int b = (k + std::max(8, k / 4) + 7) & ~7;
    while (b - 8 >= k && b > N) b -= 8;
    const int nchunk = b / RD_EIG_CB;
    const auto t_begin = std::chrono::steady_clock::now();

    // ---- scratch of this call (released before returning)
    struct Scratch {
        std::vector<void*> p;
        ~Scratch() { for (void* q : p) cudaFree(q); }
    } scratch;
    auto salloc = [&](double** out, size_t count) -> int {
        void* q = nullptr;
        cudaError_t e = cudaMalloc(&q, std::max<size_t>(count, 1) * sizeof(double));
        if (e != cudaSuccess) { cudaGetLastError(); return fail(ctx, RD_ENOMEM, "cudaMalloc(%zu doubles): %s", count, cudaGetErrorString(e)); }
        scratch.p.push_back(q);
        cudaMemsetAsync(q, 0, std::max<size_t>(count, 1) * sizeof(double), ctx->stream);
        *out = (double*)q;
        return RD_OK;
    };
    const size_t nb = (size_t)ld * b;
    double *P[4], *T, *parts, *Gs, *work, *Tm, *d_theta, *rparts, *rsum, *gersh;
    for (auto& q : P) RDTRY(salloc(&q, nb));
    RDTRY(salloc(&T, nb));
    const int nparts = ctx->num_sms * 2;
    RDTRY(salloc(&parts, (size_t)nparts * b * b));
    RDTRY(salloc(&Gs, (size_t)b * b));
    RDTRY(salloc(&work, (size_t)2 * b * b));
    RDTRY(salloc(&Tm, (size_t)b * b));
    RDTRY(salloc(&d_theta, b));
    const int rgrid = ctx->num_sms * 2;
    RDTRY(salloc(&rparts, (size_t)rgrid * b));
    RDTRY(salloc(&rsum, b));
    RDTRY(salloc(&gersh, 1));
    std::vector<double> theta(b), res2(b), resid(b, INFINITY);

    const int gs = grid_for(ctx->K.nslices * 32, kThreads, big_grid(ctx));
    const dim3 ggram(nparts, (b + 63) / 64, (b + 63) / 64);
    const int64_t bb = (int64_t)b * b;

    // ---- upper bound of the spectrum
    k_abs_rowsum<<<gs, kThreads, 0, ctx->stream>>>(ctx->K.view(), N, ctx->minv, T);
    k_gershgorin<<<gs, kThreads, 0, ctx->stream>>>(ctx->KT.view(), N, ctx->m, ctx->sigma, T, (unsigned long long*)gersh);
    ctx->launches += 2;
    double beta = 0.0;
    CU(cudaMemcpyAsync(&beta, gersh, sizeof(double), cudaMemcpyDeviceToHost, ctx->stream));
    CU(cudaStreamSynchronize(ctx->stream));
    if (!(beta > 0.0) || !std::isfinite(beta)) return fail(ctx, RD_ENOTSPD, "spectrum bound %g", beta);
    beta *= 1.0 + 1e-10;

    int64_t col_applies = 0;
    float filter_ms = 0.0f;
    // columns [col0, b) of the block (col0 a multiple of the chunk width): the leading col0 columns are locked
    auto block_apply = [&](const double* Y, double c1, double cshift, double c2, const double* Yprev, double* Ynext, int col0 = 0) {
        const int nch = nchunk - col0 / RD_EIG_CB;
        const dim3 gb(std::max(1, gs / std::min(nch, 4)), nch);
        const size_t o = (size_t)col0 * ld;
        k_blk_K<<<gb, kThreads, 0, ctx->stream>>>(ctx->K.view(), N, ld, ctx->minv, Y + o, T + o);
        k_blk_KT<<<gb, kThreads, 0, ctx->stream>>>(ctx->KT.view(), N, ld, ctx->m, ctx->sigma, c1, cshift, c2, Y + o, T + o,
                                                   Yprev ? Yprev + o : nullptr, Ynext + o);
        ctx->launches += 2;
        col_applies += (int64_t)nch * RD_EIG_CB;
    };
    auto gram = [&](const double* A, const double* B, double* out) {
        k_gram_dmma<<<ggram, 256, 0, ctx->stream>>>(N, b, b, A, ld, B, ld, parts);
        k_reduce_parts<<<grid_for(bb, kThreads, 64), kThreads, 0, ctx->stream>>>(nparts, bb, parts, out);
        ctx->launches += 2;
    };
    const size_t smem_rm = (size_t)b * b * sizeof(double);
    if (smem_rm > 48 * 1024) CU(cudaFuncSetAttribute(k_right_mult, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem_rm));
    auto right_mult = [&](const double* X, const double* M, double* Out) {
        k_right_mult<<<grid_for(N, 256, big_grid(ctx)), 256, smem_rm, ctx->stream>>>(N, ld, b, b, X, M, Out);
        ctx->launches++;
    };

    int cur = 0;  // P[cur] holds X
    k_rand_block<<<grid_for(N * b, kThreads, big_grid(ctx)), kThreads, 0, ctx->stream>>>(N, ld, b, 0x5EEDULL, P[cur]);
    ctx->launches++;
    int sweeps = 0, status = RD_ECAP;
    int64_t total_degree = 0;
    for (int sweep = 0; sweep < max_block_iters; ++sweep) {
        sweeps = sweep + 1;
        // orthonormalise twice (the second pass removes the cond^2 loss of the first)
        for (int pass = 0; pass < 2; ++pass) {
            const int nxt = (cur + 1) & 3;
            gram(P[cur], P[cur], Gs);
            k_orth_small<<<1, 1024, 0, ctx->stream>>>(b, Gs, work, Tm);
            ctx->launches++;
            right_mult(P[cur], Tm, P[nxt]);
            cur = nxt;
        }
        // Rayleigh-Ritz
        double* X = P[cur];
        double* HX = P[(cur + 1) & 3];
        block_apply(X, 1.0, 0.0, 0.0, nullptr, HX);
        gram(X, HX, Gs);
        k_rr_small<<<1, 1024, 0, ctx->stream>>>(b, Gs, work, Tm, d_theta);
        ctx->launches++;
        double* Xr = P[(cur + 2) & 3];
        double* HXr = P[(cur + 3) & 3];
        right_mult(X, Tm, Xr);
        right_mult(HX, Tm, HXr);
        k_resid_parts<<<rgrid, 256, 0, ctx->stream>>>(N, ld, b, Xr, HXr, d_theta, rparts);
        k_reduce_parts<<<1, kThreads, 0, ctx->stream>>>(rgrid, b, rparts, rsum);
        ctx->launches += 2;
        CU(cudaGetLastError());
        CU(cudaMemcpyAsync(theta.data(), d_theta, b * sizeof(double), cudaMemcpyDeviceToHost, ctx->stream));
        CU(cudaMemcpyAsync(res2.data(), rsum, b * sizeof(double), cudaMemcpyDeviceToHost, ctx->stream));
        CU(cudaStreamSynchronize(ctx->stream));
        cur = (cur + 2) & 3;  // X = Xr; HXr sits in P[(cur+1)&3]
        bool ok = true;
        for (int j = 0; j < b; ++j) {
            if (!(theta[j] > 0.0) || !std::isfinite(theta[j])) return fail(ctx, RD_ENOTSPD, "Ritz value %d = %g", j, theta[j]);
            resid[j] = std::sqrt(std::max(res2[j], 0.0)) / theta[j];
            if (j < k && !(resid[j] <= tol)) ok = false;
        }
        if (ok) { status = RD_OK; break; }
        if (sweep + 1 == max_block_iters) break;
        // Chebyshev filter on [a, beta], scaled at lo (a lower estimate of theta_1), degree from the growth target
        const double a = theta[b - 1];
        const double abs_r0 = resid[0] * theta[0];
        const double lo = std::max(0.0, theta[0] - abs_r0);
        if (!(a < beta)) return fail(ctx, RD_ECUDA, "Ritz value %g above the spectrum bound %g", a, beta);
        const double e = 0.5 * (beta - a), c = 0.5 * (beta + a);
        const double growth = std::acosh((c - lo) / e);  // per degree, at lo, relative to the cut a
        int deg = (int)std::ceil(std::log(1e4) / growth);
        deg = std::max(8, std::min(deg, 200000));
        total_degree += deg;
        double sg = e / (lo - c);
        const double tau = 2.0 / sg;
        double* Y0 = P[cur];
        double* Y1 = P[(cur + 1) & 3];
        double* Y2 = P[(cur + 2) & 3];
        // Locking: the leading Ritz vectors that already pass the residual test (whole chunks of them) skip the filter
        // and are carried over unchanged; orthonormalisation and Rayleigh-Ritz of the next sweep still see the whole
        // block, and a locked vector that drifts above the tolerance is simply filtered again.
        int nlock = 0;
        while (nlock < k && resid[nlock] <= tol) ++nlock;
        nlock = std::min((nlock / RD_EIG_CB) * RD_EIG_CB, b - RD_EIG_CB);
        const double* Xlocked = Y0;
        CU(cudaEventRecord(ctx->ev[0], ctx->stream));
        block_apply(Y0, sg / e, c, 0.0, nullptr, Y1, nlock);
        for (int j = 2; j <= deg; ++j) {
            const double sn = 1.0 / (tau - sg);
            block_apply(Y1, 2.0 * sn / e, c, -sg * sn, Y0, Y2, nlock);
            double* tmp = Y0; Y0 = Y1; Y1 = Y2; Y2 = tmp;
            sg = sn;
        }
        CU(cudaEventRecord(ctx->ev[1], ctx->stream));
        CU(cudaEventSynchronize(ctx->ev[1]));
        {
            float ms1 = 0.0f;
            CU(cudaEventElapsedTime(&ms1, ctx->ev[0], ctx->ev[1]));
            filter_ms += ms1;
        }
        if (nlock > 0 && Y1 != Xlocked)
            CU(cudaMemcpyAsync(Y1, Xlocked, (size_t)nlock * ld * sizeof(double), cudaMemcpyDeviceToDevice, ctx->stream));
        CU(cudaGetLastError());
        for (int q = 0; q < 4; ++q) if (P[q] == Y1) cur = q;
    }
    // W <- the k lowest Ritz vectors (pad columns zero)
    RDTRY(alloc_reference(ctx, k));
    CU(cudaMemsetAsync(ctx->W, 0, (size_t)ld * ctx->kp * sizeof(double), ctx->stream));
    CU(cudaMemcpyAsync(ctx->W, P[cur], (size_t)ld * k * sizeof(double), cudaMemcpyDeviceToDevice, ctx->stream));
    CU(cudaStreamSynchronize(ctx->stream));
    ctx->have_ref = true;
    ctx->ref_kind = 0;
    if (theta_out) memcpy(theta_out, theta.data(), k * sizeof(double));
    if (resid_out) memcpy(resid_out, resid.data(), k * sizeof(double));
    if (iters_out) *iters_out = sweeps;
    ctx->ref_degree = total_degree;
    ctx->ref_block = b;
    ctx->ref_col_applies = col_applies;
    ctx->lob_flop = 0.0;
    ctx->lob_ms = 0.0;
    ctx->ref_filter_ms = filter_ms;
    ctx->ref_ms_pending = std::chrono::duration<double, std::milli>(std::chrono::steady_clock::now() - t_begin).count();
    ctx->ref_ms_last = ctx->ref_ms_pending;
    if (status != RD_OK) fail(ctx, status, "reference not converged to tol %g in %d sweeps (worst residual %g)", tol, sweeps,
                              *std::max_element(resid.begin(), resid.begin() + k));
    return status;
}

int rd_build_reference_sine(rd_ctx* ctx, int32_t k, int32_t ndim, const int64_t* dims, double* mu_out, int32_t* modes_out)
{
    if (!ctx || !dims || k < 1 || k > RD_MAX_K || ndim < 1 || ndim > 3) return RD_EINVAL;
    int64_t prod = 1;
    for (int a = 0; a < ndim; ++a) {
        if (dims[a] < 1 || dims[a] > (1 << 20)) return fail(ctx, RD_EINVAL, "dims[%d] = %lld", a, (long long)dims[a]);
        prod *= dims[a];
    }
    if (prod != ctx->N) return fail(ctx, RD_EINVAL, "product of dims %lld is not N = %lld (steady Cartesian grids only)", (long long)prod, (long long)ctx->N);
    if (k > ctx->N) return fail(ctx, RD_EINVAL, "k = %d exceeds N = %lld", k, (long long)ctx->N);
    const auto t_begin = std::chrono::steady_clock::now();
    // ---- selection on the host: the k lowest products, ordered by (mu, q_1, ..., q_d); mu is summed over the
    // per-axis terms in ascending order so that permuted tuples tie exactly (reading A18)
    int qmax = 1;
    std::vector<SineCand> cand;
    select_sine_modes(ndim, dims, k, cand, &qmax);
    std::vector<int32_t> modes((size_t)k * 3);
    for (int c = 0; c < k; ++c) {
        for (int a = 0; a < 3; ++a) modes[(size_t)c * 3 + a] = cand[c].q[a];
        if (mu_out) mu_out[c] = cand[c].mu;
        if (modes_out) for (int a = 0; a < ndim; ++a) modes_out[(size_t)c * ndim + a] = cand[c].q[a];
    }
    // ---- tables and the product on the device
    RDTRY(alloc_reference(ctx, k));
    int nmax = 1;
    for (int a = 0; a < ndim; ++a) nmax = std::max<int>(nmax, (int)dims[a]);
    int32_t* d_modes = nullptr;
    double* d_tab = nullptr;
    const size_t tab_count = (size_t)ndim * qmax * nmax;
    if (cudaMalloc(&d_modes, modes.size() * sizeof(int32_t)) != cudaSuccess || cudaMalloc(&d_tab, tab_count * sizeof(double)) != cudaSuccess) {
        cudaGetLastError();
        if (d_modes) cudaFree(d_modes);
        return fail(ctx, RD_ENOMEM, "cudaMalloc of the sine tables");
    }
    cudaError_t e = cudaMemcpyAsync(d_modes, modes.data(), modes.size() * sizeof(int32_t), cudaMemcpyHostToDevice, ctx->stream);
    const int n0 = (int)dims[0], n1 = ndim > 1 ? (int)dims[1] : 1, n2 = ndim > 2 ? (int)dims[2] : 1;
    k_sine_tables<<<grid_for((int64_t)tab_count, kThreads, 1024), kThreads, 0, ctx->stream>>>(ndim, qmax, nmax, n0, n1, n2, d_tab);
    k_sine_product<<<grid_for(ctx->N, kThreads, big_grid(ctx)), kThreads, 0, ctx->stream>>>(ctx->N, ctx->ldw, ndim, qmax, nmax, n0, n1, k,
                                                                                           ctx->kp, d_modes, d_tab, ctx->W);
    ctx->launches += 2;
    if (e == cudaSuccess) e = cudaGetLastError();
    if (e == cudaSuccess) e = cudaStreamSynchronize(ctx->stream);
    cudaFree(d_modes);
    cudaFree(d_tab);
    if (e != cudaSuccess) return fail(ctx, RD_ECUDA, "sine reference: %s", cudaGetErrorString(e));
    ctx->have_ref = true;
    ctx->ref_kind = 0;
    ctx->ref_degree = 0;
    ctx->ref_col_applies = 0;
    ctx->lob_flop = 0.0;
    ctx->lob_ms = 0.0;
    ctx->ref_filter_ms = 0.0;
    ctx->ref_block = k;
    ctx->ref_ms_pending = std::chrono::duration<double, std::milli>(std::chrono::steady_clock::now() - t_begin).count();
    ctx->ref_ms_last = ctx->ref_ms_pending;
    return RD_OK;
}

// Shared by rd_build_reference_spacetime (ordered selection of k pairs among the first min(k, N_s) spatial modes) and
// rd_build_reference_spacetime_cover (every temporal factor of the first S spatial modes, k = S nt).
static int build_spacetime(rd_ctx* ctx, int32_t k, int32_t pool, int32_t ndim, const int64_t* dims, int32_t nt, double dt, double* s_out,
                           int32_t* pairs_out)
{
    int64_t Ns = 1;
    for (int a = 0; a < ndim; ++a) {
        if (dims[a] < 1 || dims[a] > (1 << 20)) return fail(ctx, RD_EINVAL, "dims[%d] = %lld", a, (long long)dims[a]);
        Ns *= dims[a];
    }
    if (Ns * nt != ctx->N) return fail(ctx, RD_EINVAL, "product of dims x nt = %lld is not N = %lld", (long long)(Ns * nt), (long long)ctx->N);
    if (k > ctx->N) return fail(ctx, RD_EINVAL, "k = %d exceeds N = %lld", k, (long long)ctx->N);
    const auto t_begin = std::chrono::steady_clock::now();
    // ---- the candidate spatial modes and their Laplacian eigenvalues
    const int rs = (int)std::min<int64_t>(pool, Ns);
    if ((int64_t)k > (int64_t)rs * nt) return fail(ctx, RD_EINVAL, "k = %d exceeds the %d x %d candidates", k, rs, nt);
    int qmax = 1;
    std::vector<SineCand> cand;
    select_sine_modes(ndim, dims, rs, cand, &qmax);
    std::vector<int32_t> modes((size_t)rs * 3);
    std::vector<double> mu(rs);
    for (int i = 0; i < rs; ++i) {
        for (int a = 0; a < 3; ++a) modes[(size_t)i * 3 + a] = cand[i].q[a];
        mu[i] = cand[i].mu;
    }
    RDTRY(alloc_reference(ctx, k, /*need_dense=*/false));
    int nmax = 1;
    for (int a = 0; a < ndim; ++a) nmax = std::max<int>(nmax, (int)dims[a]);
    const size_t tab_count = (size_t)ndim * qmax * nmax, tt = (size_t)rs * nt * nt;
    struct Scratch {
        std::vector<void*> p;
        ~Scratch() { for (void* q : p) cudaFree(q); }
    } scratch;
    auto salloc = [&](void** out, size_t bytes) -> int {
        if (cudaMalloc(out, std::max<size_t>(bytes, 16)) != cudaSuccess) { cudaGetLastError(); return fail(ctx, RD_ENOMEM, "cudaMalloc(%zu)", bytes); }
        scratch.p.push_back(*out);
        return RD_OK;
    };
    int32_t *d_modes = nullptr, *d_sel = nullptr;
    double *d_tab = nullptr, *d_mu = nullptr, *d_A = nullptr, *d_V = nullptr, *d_s = nullptr, *d_Q = nullptr, *d_Phi = nullptr;
    RDTRY(salloc((void**)&d_modes, (size_t)RD_MAX_K * 3 * sizeof(int32_t)));
    RDTRY(salloc((void**)&d_sel, (size_t)2 * k * sizeof(int32_t)));
    RDTRY(salloc((void**)&d_tab, tab_count * sizeof(double)));
    RDTRY(salloc((void**)&d_mu, rs * sizeof(double)));
    RDTRY(salloc((void**)&d_A, tt * sizeof(double)));
    RDTRY(salloc((void**)&d_V, tt * sizeof(double)));
    RDTRY(salloc((void**)&d_s, (size_t)rs * nt * sizeof(double)));
    RDTRY(salloc((void**)&d_Q, tt * sizeof(double)));
    CU(cudaMemcpyAsync(d_mu, mu.data(), rs * sizeof(double), cudaMemcpyHostToDevice, ctx->stream));
    const int n0 = (int)dims[0], n1 = ndim > 1 ? (int)dims[1] : 1, n2 = ndim > 2 ? (int)dims[2] : 1;
    k_sine_tables<<<grid_for((int64_t)tab_count, kThreads, 1024), kThreads, 0, ctx->stream>>>(ndim, qmax, nmax, n0, n1, n2, d_tab);
    // ---- temporal eigenproblems of eq. (17), one CTA per spatial mode
    k_temporal_eigs<<<rs, 256, 0, ctx->stream>>>(nt, 1.0 / dt, d_mu, d_A, d_V, d_s, d_Q);
    ctx->launches += 2;
    std::vector<double> s_all((size_t)rs * nt);
    CU(cudaMemcpyAsync(s_all.data(), d_s, s_all.size() * sizeof(double), cudaMemcpyDeviceToHost, ctx->stream));
    CU(cudaStreamSynchronize(ctx->stream));
    // ---- ordered selection of the k lowest pairs: (s, i, j) ("order the candidate pairs by nu ... A
    // fixed ordering resolves repeated eigenvalues"; nu = h^d (1 + alpha s) is increasing in s).  With k = rs * nt
    // (complete coverage) every pair is kept, in the same order.
    struct Pair { double s; int i, j; };
    std::vector<Pair> pr;
    pr.reserve(s_all.size());
    for (int i = 0; i < rs; ++i)
        for (int j = 0; j < nt; ++j) pr.push_back(Pair{s_all[(size_t)i * nt + j], i, j});
    std::sort(pr.begin(), pr.end(), [](const Pair& x, const Pair& y) {
        if (x.s != y.s) return x.s < y.s;
        if (x.i != y.i) return x.i < y.i;
        return x.j < y.j;
    });
    std::vector<int32_t> sel((size_t)2 * k), cols;
    for (int c = 0; c < k; ++c) {
        sel[2 * c] = pr[c].i;
        sel[2 * c + 1] = pr[c].j;
        if (std::find(cols.begin(), cols.end(), pr[c].i) == cols.end()) cols.push_back(pr[c].i);
        if (s_out) s_out[c] = pr[c].s;
        if (pairs_out) {
            for (int a = 0; a < ndim; ++a) pairs_out[(size_t)c * (ndim + 1) + a] = modes[(size_t)pr[c].i * 3 + a];
            pairs_out[(size_t)c * (ndim + 1) + ndim] = pr[c].j;
        }
    }
    std::sort(cols.begin(), cols.end());
    const int rs_used = (int)cols.size();  // r_s: the distinct spatial modes the selected pairs use
    // ---- the compact reference: Phi (N_s x r_s: the selected sine products), Qc (nt x k), sp (k)
    std::vector<int32_t> used_modes((size_t)rs_used * 3);
    for (int q = 0; q < rs_used; ++q)
        for (int a = 0; a < 3; ++a) used_modes[(size_t)q * 3 + a] = modes[(size_t)cols[q] * 3 + a];
    RDTRY(salloc((void**)&d_Phi, (size_t)Ns * rs_used * sizeof(double)));
    CU(cudaMemcpyAsync(d_modes, used_modes.data(), used_modes.size() * sizeof(int32_t), cudaMemcpyHostToDevice, ctx->stream));
    CU(cudaMemcpyAsync(d_sel, sel.data(), sel.size() * sizeof(int32_t), cudaMemcpyHostToDevice, ctx->stream));
    k_sine_product<<<grid_for(Ns, kThreads, big_grid(ctx)), kThreads, 0, ctx->stream>>>(Ns, Ns, ndim, qmax, nmax, n0, n1, rs_used, rs_used, d_modes,
                                                                                      d_tab, d_Phi);
    ctx->launches++;
    CU(cudaGetLastError());
    RDTRY(store_kron(ctx, k, Ns, nt, rs_used, d_Phi, cols, d_sel, d_Q, /*normalise=*/0, nullptr));
    ctx->ref_degree = 0;
    ctx->ref_col_applies = 0;
    ctx->lob_flop = 0.0;
    ctx->lob_ms = 0.0;
    ctx->ref_filter_ms = 0.0;
    ctx->ref_block = k;
    ctx->ref_ms_pending = std::chrono::duration<double, std::milli>(std::chrono::steady_clock::now() - t_begin).count();
    ctx->ref_ms_last = ctx->ref_ms_pending;
    return RD_OK;
}

int rd_build_reference_spacetime(rd_ctx* ctx, int32_t k, int32_t ndim, const int64_t* dims, int32_t nt, double dt, double* s_out,
                                 int32_t* pairs_out)
{
    if (!ctx || !dims || k < 1 || k > RD_MAX_K || ndim < 1 || ndim > 3 || nt < 1 || nt > RD_DENSE_MAXN || !(dt > 0.0)) return RD_EINVAL;
    return build_spacetime(ctx, k, /*pool=*/k, ndim, dims, nt, dt, s_out, pairs_out);
}

int rd_build_reference_spacetime_cover(rd_ctx* ctx, int32_t S, int32_t ndim, const int64_t* dims, int32_t nt, double dt, double* s_out,
                                       int32_t* pairs_out)
{
    if (!ctx || !dims || S < 1 || ndim < 1 || ndim > 3 || nt < 1 || nt > RD_DENSE_MAXN || !(dt > 0.0)) return RD_EINVAL;
    if ((int64_t)S * nt > RD_MAX_K) return fail(ctx, RD_EINVAL, "S x nt = %lld exceeds the rank limit %d", (long long)S * nt, RD_MAX_K);
    return build_spacetime(ctx, S * nt, /*pool=*/S, ndim, dims, nt, dt, s_out, pairs_out);
}

int rd_reference_storage(const rd_ctx* ctx, int32_t* kind, int64_t* n_values, int64_t* n_indices)
{
    if (!ctx) return RD_EINVAL;
    const bool kron = ctx->have_ref && ctx->ref_kind == 1;
    if (kind) *kind = ctx->have_ref ? ctx->ref_kind : -1;
    if (n_values) *n_values = !ctx->have_ref ? 0 : kron ? ctx->kNs * ctx->krs + (int64_t)ctx->knt * ctx->k : ctx->N * (int64_t)ctx->k;
    if (n_indices) *n_indices = kron ? ctx->k : 0;
    return RD_OK;
}

int rd_build_reference_transient(rd_ctx* ctx, int32_t k, int32_t rs, int32_t nt, const double* Phi, double* nu_out, int32_t* pairs_out)
{
    if (!ctx || !Phi || k < 1 || k > RD_MAX_K || rs < 1 || rs > RD_MAX_K || nt < 1 || nt > RD_DENSE_MAXN) return RD_EINVAL;
    if (ctx->N % nt != 0) return fail(ctx, RD_EINVAL, "N = %lld is not a multiple of nt = %d", (long long)ctx->N, nt);
    if ((int64_t)k > (int64_t)rs * nt) return fail(ctx, RD_EINVAL, "k = %d exceeds the %d x %d candidates", k, rs, nt);
    const int64_t N = ctx->N, Ns = N / nt;
    const auto t_begin = std::chrono::steady_clock::now();
    RDTRY(alloc_reference(ctx, k, /*need_dense=*/false));
    struct Scratch {
        std::vector<void*> p;
        ~Scratch() { for (void* q : p) cudaFree(q); }
    } scratch;
    auto salloc = [&](void** out, size_t bytes) -> int {
        if (cudaMalloc(out, std::max<size_t>(bytes, 16)) != cudaSuccess) { cudaGetLastError(); return fail(ctx, RD_ENOMEM, "cudaMalloc(%zu)", bytes); }
        scratch.p.push_back(*out);
        return RD_OK;
    };
    const size_t tt = (size_t)rs * nt * nt;
    int32_t* d_sel = nullptr;
    double *d_Phi = nullptr, *d_H = nullptr, *d_D = nullptr, *d_A = nullptr, *d_V = nullptr, *d_nu = nullptr, *d_Q = nullptr, *d_parts = nullptr,
           *d_norms = nullptr;
    const int nparts = 64;
    RDTRY(salloc((void**)&d_sel, (size_t)2 * k * sizeof(int32_t)));
    RDTRY(salloc((void**)&d_Phi, (size_t)Ns * rs * sizeof(double)));
    RDTRY(salloc((void**)&d_H, tt * sizeof(double)));
    RDTRY(salloc((void**)&d_D, (size_t)rs * nt * sizeof(double)));
    RDTRY(salloc((void**)&d_A, tt * sizeof(double)));
    RDTRY(salloc((void**)&d_V, tt * sizeof(double)));
    RDTRY(salloc((void**)&d_nu, (size_t)rs * nt * sizeof(double)));
    RDTRY(salloc((void**)&d_Q, tt * sizeof(double)));
    RDTRY(salloc((void**)&d_parts, (size_t)nparts * k * sizeof(double)));
    RDTRY(salloc((void**)&d_norms, (size_t)k * sizeof(double)));
    CU(cudaMemcpyAsync(d_Phi, Phi, (size_t)Ns * rs * sizeof(double), cudaMemcpyDefault, ctx->stream));
    // ---- the small temporal matrices of eq. (14): column t of H_i from one operator apply on e_t (x) phi_i
    const int g = grid_for(N, kThreads, big_grid(ctx));
    for (int i = 0; i < rs; ++i) {
        const double* phi = d_Phi + (size_t)i * Ns;
        for (int t = 0; t < nt; ++t) {
            k_slab_vector<<<g, kThreads, 0, ctx->stream>>>(Ns, nt, t, phi, ctx->in0);
            ctx->launches++;
            RDTRY(launch_apply_H(ctx, ctx->in0, nullptr, ctx->tmp));
            k_slab_dots<<<nt, 256, 0, ctx->stream>>>(Ns, ctx->tmp, phi, 0, d_H + ((size_t)i * nt + t) * nt);
            ctx->launches++;
        }
        k_slab_dots<<<nt, 256, 0, ctx->stream>>>(Ns, ctx->d, phi, 1, d_D + (size_t)i * nt);
        ctx->launches++;
    }
    k_transient_eigs<<<rs, 256, 0, ctx->stream>>>(nt, d_H, d_D, d_A, d_V, d_nu, d_Q);
    ctx->launches++;
    CU(cudaGetLastError());
    std::vector<double> nu_all((size_t)rs * nt);
    CU(cudaMemcpyAsync(nu_all.data(), d_nu, nu_all.size() * sizeof(double), cudaMemcpyDeviceToHost, ctx->stream));
    CU(cudaStreamSynchronize(ctx->stream));
    // ---- "selects the requested total rank from these spatial-temporal candidates": order (nu, i, j)
    struct Pair { double nu; int i, j; };
    std::vector<Pair> pr;
    pr.reserve(nu_all.size());
    for (int i = 0; i < rs; ++i)
        for (int j = 0; j < nt; ++j) {
            const double v = nu_all[(size_t)i * nt + j];
            if (!(v == v)) return fail(ctx, RD_ENOTSPD, "spatial vector %d: temporal problem is not definite (zero vector?)", i);
            pr.push_back(Pair{v, i, j});
        }
    std::sort(pr.begin(), pr.end(), [](const Pair& x, const Pair& y) {
        if (x.nu != y.nu) return x.nu < y.nu;
        if (x.i != y.i) return x.i < y.i;
        return x.j < y.j;
    });
    std::vector<int32_t> sel((size_t)2 * k), cols;
    for (int c = 0; c < k; ++c) {
        sel[2 * c] = pr[c].i;
        sel[2 * c + 1] = pr[c].j;
        if (std::find(cols.begin(), cols.end(), pr[c].i) == cols.end()) cols.push_back(pr[c].i);
        if (nu_out) nu_out[c] = pr[c].nu;
        if (pairs_out) { pairs_out[2 * c] = pr[c].i; pairs_out[2 * c + 1] = pr[c].j; }
    }
    std::sort(cols.begin(), cols.end());
    const int rs_used = (int)cols.size();
    CU(cudaMemcpyAsync(d_sel, sel.data(), sel.size() * sizeof(int32_t), cudaMemcpyHostToDevice, ctx->stream));
    // ---- compact storage: the r_s spatial vectors the selection uses, the k temporal vectors scaled so that
    // every column q (x) phi_i has unit Euclidean norm (||q (x) phi|| = ||q|| ||phi||), and the spatial-column indices
    double *d_used = nullptr, *d_phin2 = nullptr;
    RDTRY(salloc((void**)&d_used, (size_t)Ns * rs_used * sizeof(double)));
    RDTRY(salloc((void**)&d_phin2, (size_t)rs * sizeof(double)));
    for (int q = 0; q < rs_used; ++q)
        CU(cudaMemcpyAsync(d_used + (size_t)q * Ns, d_Phi + (size_t)cols[q] * Ns, (size_t)Ns * sizeof(double), cudaMemcpyDeviceToDevice, ctx->stream));
    k_col_norm2<<<rs, 256, 0, ctx->stream>>>(Ns, d_Phi, d_phin2);
    ctx->launches++;
    CU(cudaGetLastError());
    RDTRY(store_kron(ctx, k, Ns, nt, rs_used, d_used, cols, d_sel, d_Q, /*normalise=*/1, d_phin2));
    ctx->ref_degree = 0;
    ctx->ref_col_applies = 0;
    ctx->lob_flop = 0.0;
    ctx->lob_ms = 0.0;
    ctx->ref_filter_ms = 0.0;
    ctx->ref_block = k;
    ctx->ref_ms_pending = std::chrono::duration<double, std::milli>(std::chrono::steady_clock::now() - t_begin).count();
    ctx->ref_ms_last = ctx->ref_ms_pending;
    return RD_OK;
}

int rd_build_reference_scaled(rd_ctx* ctx, int32_t k, double tol, int32_t max_block_iters, double* mu_out, double* resid_out,
                              int32_t* iters_out)
{
    if (!ctx || k < 1 || k > RD_MAX_K || !(tol > 0.0) || max_block_iters < 1) return RD_EINVAL;
    const int64_t N = ctx->N;
    const auto t_begin = std::chrono::steady_clock::now();
    double *kval = nullptr, *ktval = nullptr, *ms = nullptr;
    auto release = [&]() { if (kval) cudaFree(kval); if (ktval) cudaFree(ktval); if (ms) cudaFree(ms); };
    if (cudaMalloc(&kval, std::max<int64_t>(ctx->K.entries, 1) * sizeof(double)) != cudaSuccess ||
        cudaMalloc(&ktval, std::max<int64_t>(ctx->KT.entries, 1) * sizeof(double)) != cudaSuccess ||
        cudaMalloc(&ms, ctx->ldw * sizeof(double)) != cudaSuccess) {
        cudaGetLastError();
        release();
        return fail(ctx, RD_ENOMEM, "cudaMalloc of the scaled operator copies");
    }
    cudaMemsetAsync(ms, 0, ctx->ldw * sizeof(double), ctx->stream);
    const int g = grid_for(ctx->K.nslices * 32, kThreads, big_grid(ctx));
    k_scale_ell<<<g, kThreads, 0, ctx->stream>>>(ctx->K.view(), N, ctx->d, 0, kval);    // K S
    k_scale_ell<<<g, kThreads, 0, ctx->stream>>>(ctx->KT.view(), N, ctx->d, 1, ktval);  // S K^T
    k_div<<<grid_for(N, kThreads, big_grid(ctx)), kThreads, 0, ctx->stream>>>(N, ctx->m, ctx->d, ms);  // S M S
    ctx->launches += 3;
    // the eigensolver of rd_build_reference on the scaled operator (same structure, see eigs.cuh)
    double* const kval0 = ctx->K.val;
    double* const ktval0 = ctx->KT.val;
    double* const m0 = ctx->m;
    ctx->K.val = kval; ctx->KT.val = ktval; ctx->m = ms;
    const int rc = rd_build_reference(ctx, k, tol, max_block_iters, mu_out, resid_out, iters_out);
    ctx->K.val = kval0; ctx->KT.val = ktval0; ctx->m = m0;
    cudaError_t e = cudaSuccess;
    if (rc == RD_OK || rc == RD_ECAP) {
        // w = S v, each column normalised in the Euclidean norm
        k_unscale_normalize<<<k, 1024, 0, ctx->stream>>>(N, ctx->ldw, ctx->d, ctx->W);
        ctx->launches++;
        e = cudaGetLastError();
    }
    if (e == cudaSuccess) e = cudaStreamSynchronize(ctx->stream);
    release();
    if (e != cudaSuccess) return fail(ctx, RD_ECUDA, "scaled reference: %s", cudaGetErrorString(e));
    ctx->ref_ms_pending = std::chrono::duration<double, std::milli>(std::chrono::steady_clock::now() - t_begin).count();
    ctx->ref_ms_last = ctx->ref_ms_pending;
    return rc;
}

int rd_probe_fp64_tensor_peak(rd_ctx* ctx, double* tflops)
{
    if (!ctx || !tflops) return RD_EINVAL;
    const int iters = 1 << 15, blocks = ctx->num_sms * 8, threads = 256;
    float best = 1e30f;
    for (int rep = 0; rep < 5; ++rep) {
        CU(cudaEventRecord(ctx->ev[0], ctx->stream));
        k_dmma_peak_probe<<<blocks, threads, 0, ctx->stream>>>(iters, 0.5, ctx->tmp);
        CU(cudaEventRecord(ctx->ev[1], ctx->stream));
        CU(cudaEventSynchronize(ctx->ev[1]));
        float ms = 0;
        CU(cudaEventElapsedTime(&ms, ctx->ev[0], ctx->ev[1]));
        if (rep > 0) best = std::min(best, ms);
        ctx->launches++;
    }
    CU(cudaGetLastError());
    const double flop = (double)blocks * (threads / 32) * (double)iters * 8.0 * 512.0;  // m8n8k4: 2 * 8 * 8 * 4 flop
    *tflops = flop / (best * 1e-3) / 1e12;
    return RD_OK;
}

int rd_reference_work(const rd_ctx* ctx, int64_t* column_applies, double* filter_ms, double* bytes_per_column_apply)
{
    if (!ctx) return RD_EINVAL;
    if (column_applies) *column_applies = ctx->ref_col_applies;
    if (filter_ms) *filter_ms = ctx->ref_filter_ms;
    // K and K^T stream once per 8 columns (12 B per stored entry each); per column Y is read by the gathers
    // and once directly, T written and read, Yprev read, Ynext written: 48 N
    if (bytes_per_column_apply) *bytes_per_column_apply = 3.0 * (double)ctx->nnz + 48.0 * (double)ctx->N;
    return RD_OK;
}

int rd_reference_info(const rd_ctx* ctx, int32_t* block, int64_t* total_degree, double* build_ms)
{
    if (!ctx) return RD_EINVAL;
    if (block) *block = ctx->ref_block;
    if (total_degree) *total_degree = ctx->ref_degree;
    if (build_ms) *build_ms = ctx->ref_ms_last;
    return RD_OK;
}

int rd_coarse_setup(rd_ctx* ctx, int32_t method, const uint8_t* active, double* G, double* EW, double* C, int32_t* rank_used,
                    double* cond_E, int32_t* fallback)
{
    if (!ctx || !active) return RD_EINVAL;
    if (!ctx->have_ref || ctx->k <= 0) return fail(ctx, RD_ENOREF, "no reference set");
    const uint8_t* da;
    RDTRY(in_dev(ctx, active, ctx->N, ctx->act_stage, &da));
    CU(cudaMemcpyAsync(ctx->act, da, ctx->N, cudaMemcpyDeviceToDevice, ctx->stream));
    RDTRY(coarse_setup(ctx, method, nullptr, nullptr, EW != nullptr));
    const int kp = ctx->kp, k = ctx->k;
    auto copy_kk = [&](double* dst, const double* src) -> int {
        if (!dst) return RD_OK;
        CU(cudaMemcpy2DAsync(dst, k * sizeof(double), src, kp * sizeof(double), k * sizeof(double), k, cudaMemcpyDefault, ctx->stream));
        return RD_OK;
    };
    RDTRY(copy_kk(G, ctx->G));
    RDTRY(copy_kk(EW, ctx->EW));
    RDTRY(copy_kk(C, ctx->CW));
    CU(cudaStreamSynchronize(ctx->stream));
    if (rank_used) *rank_used = ctx->h_cinfo->rank;
    if (cond_E) *cond_E = ctx->h_cinfo->cond_E;
    if (fallback) *fallback = ctx->h_cinfo->fallback;
    return RD_OK;
}

int rd_solve_inactive(rd_ctx* ctx, int32_t method, const uint8_t* active, const double* b, double* x, rd_solve_report* rep)
{
    if (!ctx || !active || !b || !x || !rep) return RD_EINVAL;
    if (method < RD_JACOBI_CG || method > RD_ZEROEXT) return RD_EINVAL;
    const int64_t N = ctx->N;
    const uint8_t* da;
    const double *db, *dx;
    RDTRY(in_dev(ctx, active, N, ctx->act_stage, &da));
    RDTRY(in_dev(ctx, b, N, ctx->in0, &db));
    RDTRY(in_dev(ctx, (const double*)x, N, ctx->in1, &dx));
    CU(cudaMemcpyAsync(ctx->act, da, N, cudaMemcpyDeviceToDevice, ctx->stream));
    const int g = grid_for(N, kThreads, big_grid(ctx));
    k_mask_copy<<<g, kThreads, 0, ctx->stream>>>(N, ctx->act, db, ctx->b);
    k_mask_copy<<<g, kThreads, 0, ctx->stream>>>(N, ctx->act, dx, ctx->x);
    CU(cudaMemsetAsync(ctx->d_nactive, 0, sizeof(int), ctx->stream));
    k_pack_bits<<<g, kThreads, 0, ctx->stream>>>(N, ctx->act, ctx->bits, ctx->d_nactive);  // |J| for the bytes model
    ctx->launches += 3;
    CU(cudaMemcpyAsync(ctx->h_nactive, ctx->d_nactive, sizeof(int), cudaMemcpyDeviceToHost, ctx->stream));
    CU(cudaStreamSynchronize(ctx->stream));
    float msr = 0, msc = 0;
    ctx->want_ritz = true;
    const int rc_alg = run_alg1(ctx, method, N - *ctx->h_nactive, rep, &msr, &msc);
    ctx->want_ritz = false;
    RDTRY(rc_alg);
    RDTRY(out_host(ctx, x, ctx->x, N));
    CU(cudaStreamSynchronize(ctx->stream));
    return rep->status;
}

int rd_energy_fraction(rd_ctx* ctx, int32_t method, const uint8_t* active, const double* b, const double* x_star, double* chi,
                       double* qb_energy, double* xs_energy)
{
    if (!ctx || !active || !b || !x_star || !chi) return RD_EINVAL;
    if (method < RD_JACOBI_CG || method > RD_ZEROEXT) return RD_EINVAL;
    const int64_t N = ctx->N;
    int use_coarse = 0;
    if (method != RD_JACOBI_CG && (!ctx->have_ref || ctx->k <= 0)) return fail(ctx, RD_ENOREF, "method %d needs a reference", method);
    const uint8_t* da;
    const double *db, *dx;
    RDTRY(in_dev(ctx, active, N, ctx->act_stage, &da));
    RDTRY(in_dev(ctx, b, N, ctx->in0, &db));
    RDTRY(in_dev(ctx, x_star, N, ctx->in1, &dx));
    CU(cudaMemcpyAsync(ctx->act, da, N, cudaMemcpyDeviceToDevice, ctx->stream));
    const int g = grid_for(N, kThreads, big_grid(ctx));
    k_mask_copy<<<g, kThreads, 0, ctx->stream>>>(N, ctx->act, db, ctx->b);
    k_mask_copy<<<g, kThreads, 0, ctx->stream>>>(N, ctx->act, dx, ctx->x);
    ctx->launches += 2;
    if (method != RD_JACOBI_CG) {
        RDTRY(coarse_setup(ctx, method, nullptr, nullptr));  // the history of RD_ZEROEXT is read, not advanced
        use_coarse = ctx->h_cinfo->rank > 0;
    }
    RDTRY(launch_apply_H(ctx, ctx->x, ctx->act, ctx->w));  // w = B x_* on I, 0 on J
    const int kp = use_coarse ? ctx->kp : 0;
    const int nparts = ctx->gram_parts ? ctx->gram_nparts : 0;
    double *parts = ctx->gram_parts, *red = ctx->cwork;
    if (!nparts) {  // no reference was ever allocated (Jacobi-CG only): the CG reduction slots serve
        parts = ctx->partial;
        red = ctx->partial + ctx->cg_grid;
    }
    const int np = nparts ? nparts : ctx->cg_grid;
    k_energy_parts<<<np, 256, 0, ctx->stream>>>(N, ctx->ldw, kp, ctx->Wm, ctx->b, ctx->x, ctx->w, parts);
    k_reduce_parts<<<1, 128, 0, ctx->stream>>>(np, kp + 1, parts, red);
    k_energy_fraction<<<1, 64, 0, ctx->stream>>>(kp, use_coarse, ctx->CW, red, red + kp + 1);
    ctx->launches += 3;
    CU(cudaGetLastError());
    double h[3];
    CU(cudaMemcpyAsync(h, red + kp + 1, sizeof h, cudaMemcpyDeviceToHost, ctx->stream));
    CU(cudaStreamSynchronize(ctx->stream));
    if (qb_energy) *qb_energy = h[0];
    if (xs_energy) *xs_energy = h[1];
    *chi = h[2];
    return RD_OK;
}

int rd_kkt(rd_ctx* ctx, const double* y_d, const double* psi, const double* y, const double* lambda, double* kkt)
{
    if (!ctx || !y_d || !psi || !y || !lambda || !kkt) return RD_EINVAL;
    const int64_t N = ctx->N;
    const int g = grid_for(N, kThreads, big_grid(ctx));
    const double *dyd, *dpsi, *dy, *dl;
    RDTRY(in_dev(ctx, y_d, N, ctx->in0, &dyd));
    k_ell<<<g, kThreads, 0, ctx->stream>>>(N, ctx->m, dyd, ctx->ell);
    RDTRY(in_dev(ctx, psi, N, ctx->in1, &dpsi));
    RDTRY(in_dev(ctx, y, N, ctx->in0, &dy));       // in0 is free again: l has been formed (same stream)
    RDTRY(in_dev(ctx, lambda, N, ctx->tmp, &dl));
    RDTRY(launch_apply_H(ctx, dy, nullptr, ctx->Hy));
    CU(cudaMemsetAsync(ctx->d_cnt, 0, sizeof(PdasCounters), ctx->stream));
    k_kkt<<<g, kThreads, 0, ctx->stream>>>(N, ctx->ell, ctx->Hy, dy, dpsi, dl, ctx->d_cnt);
    ctx->launches += 2;
    CU(cudaGetLastError());
    CU(cudaMemcpyAsync(ctx->h_cnt, ctx->d_cnt, sizeof(PdasCounters), cudaMemcpyDeviceToHost, ctx->stream));
    CU(cudaStreamSynchronize(ctx->stream));
    double kk[6];
    memcpy(kk, ctx->h_cnt->kkt_bits, sizeof kk);
    const double s = std::max(1.0, kk[5]);
    kkt[0] = kk[0] / s; kkt[1] = kk[1]; kkt[2] = kk[2] / s; kkt[3] = kk[3] / s; kkt[4] = kk[4] / s;
    return RD_OK;
}

int rd_pdas_update(rd_ctx* ctx, const double* y_d, const double* psi, const uint8_t* active, const double* y,
                   double* lambda_out, uint8_t* active_new_out, int64_t* changed, int64_t* n_active_new, double* margin)
{
    if (!ctx || !y_d || !psi || !active || !y || !lambda_out || !active_new_out) return RD_EINVAL;
    const int64_t N = ctx->N;
    const int g = grid_for(N, kThreads, big_grid(ctx));
    const double *dyd, *dpsi, *dy;
    const uint8_t* da;
    RDTRY(in_dev(ctx, y_d, N, ctx->in0, &dyd));
    k_ell<<<g, kThreads, 0, ctx->stream>>>(N, ctx->m, dyd, ctx->ell);
    RDTRY(in_dev(ctx, psi, N, ctx->in1, &dpsi));
    RDTRY(in_dev(ctx, y, N, ctx->in0, &dy));  // in0 is free again: l has been formed (same stream)
    RDTRY(in_dev(ctx, active, N, ctx->act_stage, &da));
    RDTRY(launch_apply_H(ctx, dy, nullptr, ctx->Hy));
    CU(cudaMemsetAsync(ctx->d_cnt, 0, sizeof(PdasCounters), ctx->stream));
    {
        const unsigned long long inf_bits = 0x7ff0000000000000ULL;
        CU(cudaMemcpyAsync(&ctx->d_cnt->margin_bits, &inf_bits, sizeof inf_bits, cudaMemcpyHostToDevice, ctx->stream));
    }
    // lam / act_new / tmp are scratch here: the sequence's own state (ystate, act_seq, hist) is not touched
    k_pdas_update<<<g, kThreads, 0, ctx->stream>>>(N, da, ctx->ell, ctx->Hy, dy, dpsi, ctx->d, ctx->opt.c_is_diag, ctx->lam, ctx->act_new,
                                                   ctx->tmp, ctx->d_cnt);
    ctx->launches += 2;
    CU(cudaGetLastError());
    CU(cudaMemcpyAsync(ctx->h_cnt, ctx->d_cnt, sizeof(PdasCounters), cudaMemcpyDeviceToHost, ctx->stream));
    RDTRY(out_host(ctx, lambda_out, ctx->lam, N));
    RDTRY(out_host(ctx, active_new_out, ctx->act_new, N));
    CU(cudaStreamSynchronize(ctx->stream));
    if (changed) *changed = ctx->h_cnt->changed;
    if (n_active_new) *n_active_new = ctx->h_cnt->n_active_new;
    if (margin) memcpy(margin, &ctx->h_cnt->margin_bits, sizeof(double));
    return RD_OK;
}

int rd_solve_query(rd_ctx* ctx, int32_t method, const double* y_d, const double* psi, const uint8_t* J0, double* y, double* u,
                   double* lambda, rd_step_report* steps, uint8_t* J_bits, rd_query_report* rep)
{
    if (!ctx || !y_d || !psi || !y || !u || !steps || !rep) return RD_EINVAL;
    if (method < RD_JACOBI_CG || method > RD_ZEROEXT) return RD_EINVAL;
    if (ctx->opt.init == RD_INIT_GIVEN && !J0) return RD_EINVAL;
    if (method != RD_JACOBI_CG && (!ctx->have_ref || ctx->k <= 0)) return fail(ctx, RD_ENOREF, "method %d needs a reference", method);
    const auto t_begin = std::chrono::steady_clock::now();
    const int64_t N = ctx->N;
    const int64_t nbytes = (N + 7) / 8;
    const int g = grid_for(N, kThreads, big_grid(ctx));
    memset(rep, 0, sizeof *rep);
    const double *dyd, *dpsi;
    const uint8_t* dJ0;
    RDTRY(in_dev(ctx, y_d, N, ctx->in0, &dyd));
    RDTRY(in_dev(ctx, psi, N, ctx->in1, &dpsi));
    RDTRY(in_dev(ctx, J0, N, ctx->act_stage, &dJ0));
    k_ell<<<g, kThreads, 0, ctx->stream>>>(N, ctx->m, dyd, ctx->ell);
    int init = ctx->opt.init;
    if (init == RD_INIT_PAPER) init = ctx->have_state ? -1 : RD_INIT_ALL_ACTIVE;
    if (!ctx->have_state) CU(cudaMemsetAsync(ctx->ystate, 0, ctx->ldw * sizeof(double), ctx->stream));
    if (init == -1)  // inherit the set saved by the previous query (single-step entry points may have used ctx->act since)
        CU(cudaMemcpyAsync(ctx->act, ctx->act_seq, N, cudaMemcpyDeviceToDevice, ctx->stream));
    k_init_active<<<g, kThreads, 0, ctx->stream>>>(N, init, dJ0, dpsi, ctx->act);
    ctx->launches += 2;
    CU(cudaGetLastError());

    std::vector<uint64_t> seen;
    int status = RD_ESTEPS, nsteps = 0;
    int64_t total_iters = 0;
    // bits / count of the current active set
    auto pack = [&]() -> int {
        CU(cudaMemsetAsync(ctx->d_nactive, 0, sizeof(int), ctx->stream));
        k_pack_bits<<<grid_for(nbytes, kThreads, big_grid(ctx)), kThreads, 0, ctx->stream>>>(N, ctx->act, ctx->bits, ctx->d_nactive);
        ctx->launches++;
        CU(cudaMemcpyAsync(ctx->h_bits, ctx->bits, nbytes, cudaMemcpyDeviceToHost, ctx->stream));
        CU(cudaMemcpyAsync(ctx->h_nactive, ctx->d_nactive, sizeof(int), cudaMemcpyDeviceToHost, ctx->stream));
        CU(cudaStreamSynchronize(ctx->stream));
        return RD_OK;
    };
    RDTRY(pack());
    for (int step = 0; step < ctx->opt.pdas_cap; ++step) {
        rd_step_report* sr = &steps[step];
        memset(sr, 0, sizeof *sr);
        nsteps = step + 1;
        sr->active_hash = fnv1a(ctx->h_bits, nbytes);
        if (J_bits) memcpy(J_bits + (size_t)step * nbytes, ctx->h_bits, nbytes);
        seen.push_back(sr->active_hash);
        const int64_t n = N - *ctx->h_nactive;
        sr->n_inactive = (int32_t)n;
        CU(cudaEventRecord(ctx->ev[5], ctx->stream));
        // y <- y_state, y_J <- psi_J ; tmp = chi_J psi ; x0 = chi_I y_state (warm inner start)
        k_step_begin<<<g, kThreads, 0, ctx->stream>>>(N, ctx->act, dpsi, ctx->ystate, ctx->y, ctx->tmp, ctx->x);
        ctx->launches++;
        float ms_upd0 = 0, ms_upd1 = 0;
        if (n > 0) {
            RDTRY(launch_apply_H(ctx, ctx->tmp, nullptr, ctx->Hy));
            k_rhs<<<g, kThreads, 0, ctx->stream>>>(N, ctx->act, ctx->ell, ctx->Hy, ctx->b);
            ctx->launches++;
            CU(cudaEventRecord(ctx->ev[6], ctx->stream));
            rd_solve_report so;
            float msr = 0, msc = 0;
            RDTRY(run_alg1(ctx, method, n, &so, &msr, &msc));
            CU(cudaEventElapsedTime(&ms_upd0, ctx->ev[5], ctx->ev[6]));
            sr->cg_iters = so.iters; sr->rank_used = so.rank_used; sr->coarse_fallback = so.coarse_fallback;
            sr->replacements = so.replacements; sr->status = so.status; sr->rel_resid_verified = so.rel_resid_verified;
            sr->cond_E = so.cond_E; sr->t_restrict = msr; sr->t_coarse = msc; sr->t_iter = so.t_iter_ms;
            total_iters += so.iters;
            CU(cudaEventRecord(ctx->ev[5], ctx->stream));
            k_scatter_solution<<<g, kThreads, 0, ctx->stream>>>(N, ctx->act, ctx->x, ctx->y);
            ctx->launches++;
        }
        // lambda = l - H y on J, 0 on I; eq. (8)
        RDTRY(launch_apply_H(ctx, ctx->y, nullptr, ctx->Hy));
        CU(cudaMemsetAsync(ctx->d_cnt, 0, sizeof(PdasCounters), ctx->stream));
        {
            const unsigned long long inf_bits = 0x7ff0000000000000ULL;
            CU(cudaMemcpyAsync(&ctx->d_cnt->margin_bits, &inf_bits, sizeof inf_bits, cudaMemcpyHostToDevice, ctx->stream));
        }
        k_pdas_update<<<g, kThreads, 0, ctx->stream>>>(N, ctx->act, ctx->ell, ctx->Hy, ctx->y, dpsi, ctx->d, ctx->opt.c_is_diag,
                                                       ctx->lam, ctx->act_new, ctx->ystate, ctx->d_cnt);
        ctx->launches++;
        CU(cudaGetLastError());
        CU(cudaMemcpyAsync(ctx->h_cnt, ctx->d_cnt, sizeof(PdasCounters), cudaMemcpyDeviceToHost, ctx->stream));
        CU(cudaEventRecord(ctx->ev[7], ctx->stream));
        CU(cudaStreamSynchronize(ctx->stream));
        CU(cudaEventElapsedTime(&ms_upd1, ctx->ev[5], ctx->ev[7]));
        sr->t_update = ms_upd0 + ms_upd1;
        memcpy(&sr->margin, &ctx->h_cnt->margin_bits, sizeof(double));
        if (ctx->h_cnt->changed == 0) { status = RD_OK; break; }
        std::swap(ctx->act, ctx->act_new);
        RDTRY(pack());
        const uint64_t hn = fnv1a(ctx->h_bits, nbytes);
        bool cyc = false;
        for (uint64_t hsh : seen) cyc = cyc || (hsh == hn);
        if (cyc) { status = RD_ECYCLE; break; }
    }
    ctx->have_state = true;
    CU(cudaMemcpyAsync(ctx->act_seq, ctx->act, N, cudaMemcpyDeviceToDevice, ctx->stream));  // what the next query inherits
    rep->n_steps = nsteps;
    rep->status = status;
    rep->total_cg_iters = total_iters;
    for (int i = 0; i < nsteps; ++i) {
        const int st = steps[i].status;
        if (st != RD_OK) {
            rep->n_inner_failed++;
            auto sev = [](int q) { return q == RD_ENOTSPD ? 3 : q == RD_ERESID ? 2 : q == RD_ECAP ? 1 : q == RD_OK ? 0 : 4; };
            if (sev(st) > sev(rep->worst_inner_status)) rep->worst_inner_status = st;
        }
        rep->n_fallbacks += steps[i].coarse_fallback ? 1 : 0;
    }
    // u = M^{-1} K y (eq. (9), f = 0), all state values incl. the active ones
    k_apply_K<<<grid_for(ctx->K.nslices * 32, kThreads, big_grid(ctx)), kThreads, 0, ctx->stream>>>(ctx->K.view(), N, ctx->minv, ctx->y, ctx->u);
    ctx->launches++;
    // KKT measures, eq. (25)
    RDTRY(launch_apply_H(ctx, ctx->y, nullptr, ctx->Hy));
    CU(cudaMemsetAsync(ctx->d_cnt, 0, sizeof(PdasCounters), ctx->stream));
    k_kkt<<<g, kThreads, 0, ctx->stream>>>(N, ctx->ell, ctx->Hy, ctx->y, dpsi, ctx->lam, ctx->d_cnt);
    ctx->launches++;
    CU(cudaGetLastError());
    CU(cudaMemcpyAsync(ctx->h_cnt, ctx->d_cnt, sizeof(PdasCounters), cudaMemcpyDeviceToHost, ctx->stream));
    RDTRY(out_host(ctx, y, ctx->y, N));
    RDTRY(out_host(ctx, u, ctx->u, N));
    if (lambda) RDTRY(out_host(ctx, lambda, ctx->lam, N));
    CU(cudaStreamSynchronize(ctx->stream));
    double kk[6];
    memcpy(kk, ctx->h_cnt->kkt_bits, sizeof kk);
    const double s = std::max(1.0, kk[5]);
    rep->kkt[0] = kk[0] / s; rep->kkt[1] = kk[1]; rep->kkt[2] = kk[2] / s; rep->kkt[3] = kk[3] / s; rep->kkt[4] = kk[4] / s;
    rep->t_reference_charged = ctx->ref_ms_pending;
    ctx->ref_ms_pending = 0.0;
    rep->t_total = std::chrono::duration<double, std::milli>(std::chrono::steady_clock::now() - t_begin).count() + rep->t_reference_charged;
    return status;
}

}  // extern "C"

// ---------------------------------------------------------------------------------------------------------------------
// rd_apply_H_noalloc: S3 for callers that cannot allocate (CUDA graph capture, serving loops, harnesses that forbid
// cudaMalloc).  The intermediate t = M^{-1} K (chi_I v) of eq. (5) lives in a file-scope device array instead of a
// context buffer; the mask chi_I is applied inside the gather, so no masked copy of v is needed either.
//
// g_noalloc_t is a DEVICE symbol: in host code its name is a host-side stand-in, not a device address.  The address the
// kernels get comes from cudaGetSymbolAddress, taken once per device with that device current (noalloc_scratch below).
namespace {

__device__ __align__(256) double g_noalloc_t[RD_NOALLOC_MAX_N];  // 8 MiB on every GPU that loads the library, until exit

constexpr int kMaxDevices = 64;
double* g_noalloc_ptr[kMaxDevices];  // per device: the address of g_noalloc_t on it, NULL until resolved

// t_r = (1/m_r) sum_c K_rc (act_c ? 0 : v_c): k_apply_K with chi_I folded into the gather.  Same order of the sums as
// ell_row_dot (groups of four entries, one fma chain), so the result equals k_mask_copy + k_apply_K bit for bit.
__global__ void k_apply_K_masked(Ell K, int64_t N, const double* __restrict__ minv, const uint8_t* __restrict__ act,
                                 const double* __restrict__ v, double* __restrict__ t)
{
    const int lane = threadIdx.x & 31;
    const int64_t gw = ((int64_t)blockIdx.x * blockDim.x + threadIdx.x) >> 5;
    const int64_t nwt = ((int64_t)gridDim.x * blockDim.x) >> 5;
    for (int64_t s = gw; s < K.nslices; s += nwt) {
        const int64_t row = s * RD_SLICE + lane;
        const int64_t o = K.off[s];
        const int wd = (int)((K.off[s + 1] - o) >> 5);
        const int32_t* cp = K.col + o + lane;
        const double* vp = K.val + o + lane;
        double acc = 0.0;
        for (int e = 0; e < wd; ++e) {
            const int c = ldg_i32(cp + e * 32);
            const double a = ldg_f64(vp + e * 32);
            const double x = (act && act[c]) ? 0.0 : v[c];
            acc = fma(a, x, acc);
        }
        if (row < N) t[row] = acc * ldg_f64(minv + row);
    }
}

// The device address of g_noalloc_t on `device` (which must be current).  No allocation: the array is part of the module.
int noalloc_scratch(rd_ctx* ctx, int device, double** out)
{
    if (device < 0 || device >= kMaxDevices) return fail(ctx, RD_EINVAL, "device ordinal %d is outside 0..%d", device, kMaxDevices - 1);
    if (!g_noalloc_ptr[device]) {
        void* p = nullptr;
        const cudaError_t e = cudaGetSymbolAddress(&p, g_noalloc_t);
        if (e != cudaSuccess || !p) {
            cudaGetLastError();
            return fail(ctx, RD_ECUDA, "cudaGetSymbolAddress(g_noalloc_t) on device %d: %s", device, cudaGetErrorString(e));
        }
        g_noalloc_ptr[device] = (double*)p;  // the same value whichever thread stores it
    }
    *out = g_noalloc_ptr[device];
    return RD_OK;
}

}  // namespace

extern "C" int rd_apply_H_noalloc(rd_ctx* ctx, const double* v, const uint8_t* active, double* out)
{
    if (!ctx || !v || !out) return RD_EINVAL;
    if (ctx->N > (int64_t)RD_NOALLOC_MAX_N)
        return fail(ctx, RD_EINVAL, "rd_apply_H_noalloc: N = %lld exceeds RD_NOALLOC_MAX_N = %lld (the static scratch); use rd_apply_H",
                    (long long)ctx->N, (long long)RD_NOALLOC_MAX_N);
    if (v == out) return fail(ctx, RD_EINVAL, "rd_apply_H_noalloc: out must not alias v");
    if (!is_device_ptr(v) || !is_device_ptr(out) || (active && !is_device_ptr(active)))
        return fail(ctx, RD_EINVAL, "rd_apply_H_noalloc takes device pointers only (a host buffer would need a staging copy)");
    int dev = -1;
    CU(cudaGetDevice(&dev));
    if (dev != ctx->device) return fail(ctx, RD_EINVAL, "rd_apply_H_noalloc: device %d is current, the context lives on device %d", dev, ctx->device);
    double* t = nullptr;
    RDTRY(noalloc_scratch(ctx, dev, &t));
    // every row of t below N is rewritten by the first kernel before the second reads it: nothing has to start at zero
    const int g = grid_for(ctx->K.nslices * 32, kThreads, big_grid(ctx));
    k_apply_K_masked<<<g, kThreads, 0, ctx->stream>>>(ctx->K.view(), ctx->N, ctx->minv, active, v, t);
    k_apply_KT_H<<<g, kThreads, 0, ctx->stream>>>(ctx->KT.view(), ctx->N, ctx->m, ctx->sigma, active, v, t, out);
    ctx->launches += 2;
    CU(cudaGetLastError());
    return RD_OK;
}

// ---------------------------------------------------------------------------------------------------------------------
// S0, second eigensolver: LOBPCG preconditioned by the inverse of the homogeneous grid operator (lobpcg.cuh).
namespace {

struct SineAxis {
    int n = 0;
    int64_t rs = 1;  // stride of this axis in the vector (product of the faster dims)
    double *S = nullptr, *St = nullptr, *mu = nullptr;
};

template <bool AM, bool BN>
void launch_gemm(cudaStream_t st, int tn, int M, int Nn, int Kk, int nb1, int nb2, GemmOp A, GemmOp B, GemmOp E, GemmOp D)
{
    if (tn == 10) {
        const dim3 g((M + 63) / 64, (Nn + 79) / 80, nb1 * nb2);
        k_dgemm_dmma<AM, BN, 10><<<g, 256, 0, st>>>(M, Nn, Kk, nb2, A, B, E, D);
    } else {
        const dim3 g((M + 63) / 64, (Nn + 63) / 64, nb1 * nb2);
        k_dgemm_dmma<AM, BN, 8><<<g, 256, 0, st>>>(M, Nn, Kk, nb2, A, B, E, D);
    }
}
inline int tile_for(int n) { return (((n + 79) / 80) * 80 < ((n + 63) / 64) * 64) ? 10 : 8; }

// Y[:, 0:ncols] <- transform along one axis (forward: coefficients S y; inverse: S^T y), from `in` to `out`
int sine_axis_pass(rd_ctx* ctx, const SineAxis& ax, bool inverse, int64_t N, int64_t ld, int ncols, const double* in, double* out)
{
    const double* Mat = inverse ? ax.St : ax.S;  // Mat[o][i], row-major
    const int n = ax.n;
    const GemmOp none{nullptr, 0, 0, 0, 0};
    if (ax.rs == 1) {
        // D[l, o] = sum_i In[l n + i] Mat[o][i]: lines are the m index, both operands contiguous along the contraction
        const int64_t L = N / n;
        const GemmOp A{in, n, 1, ld, 0}, B{Mat, 1, n, 0, 0}, D{out, n, 1, ld, 0};
        launch_gemm<false, false>(ctx->stream, tile_for(n), (int)L, n, n, ncols, 1, A, B, none, D);
    } else {
        // D[o, l] = sum_i Mat[o][i] In[i rs + l] for every slab of rs n entries
        const int64_t slab = ax.rs * n, nslab = N / slab;
        if ((int64_t)ncols * nslab > 65535) return fail(ctx, RD_EINVAL, "sine preconditioner: %lld batches exceed the grid limit", (long long)(ncols * nslab));
        const GemmOp A{Mat, n, 1, 0, 0}, B{in, ax.rs, 1, ld, slab}, D{out, ax.rs, 1, ld, slab};
        launch_gemm<false, true>(ctx->stream, tile_for((int)std::min<int64_t>(ax.rs, 1 << 20)), n, (int)ax.rs, n, ncols, (int)nslab, A, B, none, D);
    }
    ctx->launches++;
    return RD_OK;
}

}  // namespace

extern "C" int rd_build_reference_lobpcg(rd_ctx* ctx, int32_t k, double tol, int32_t max_iters, int32_t ndim, const int64_t* dims,
                                         double kappa_ref, double* theta_out, double* resid_out, int32_t* iters_out)
{
    if (!ctx || !dims || k < 1 || k > RD_MAX_K || !(tol > 0.0) || max_iters < 1 || ndim < 1 || ndim > 3 || !(kappa_ref > 0.0))
        return RD_EINVAL;
    const int64_t N = ctx->N, ld = ctx->ldw;
    int64_t prod = 1;
    for (int a = 0; a < ndim; ++a) {
        if (dims[a] < 2 || dims[a] > 4096) return fail(ctx, RD_EINVAL, "dims[%d] = %lld", a, (long long)dims[a]);
        prod *= dims[a];
    }
    if (prod != N) return fail(ctx, RD_EINVAL, "prod(dims) = %lld but N = %lld", (long long)prod, (long long)N);
    int b = (k + std::max(8, k / 4) + 7) & ~7;
    while (b - 8 >= k && 3 * b > N) b -= 8;
    if (3 * b > N || 3 * b > RD_DENSE_MAXN) return fail(ctx, RD_EINVAL, "block of %d vectors: 3 b must not exceed min(N, %d)", b, RD_DENSE_MAXN);
    const auto t_begin = std::chrono::steady_clock::now();

    struct Scratch {
        std::vector<void*> p;
        ~Scratch() { for (void* q : p) cudaFree(q); }
    } scratch;
    auto salloc = [&](double** out, size_t count) -> int {
        void* q = nullptr;
        cudaError_t e = cudaMalloc(&q, std::max<size_t>(count, 1) * sizeof(double));
        if (e != cudaSuccess) { cudaGetLastError(); return fail(ctx, RD_ENOMEM, "cudaMalloc(%zu doubles): %s", count, cudaGetErrorString(e)); }
        scratch.p.push_back(q);
        cudaMemsetAsync(q, 0, std::max<size_t>(count, 1) * sizeof(double), ctx->stream);
        *out = (double*)q;
        return RD_OK;
    };
    const size_t nb = (size_t)ld * b;
    const int ns_max = 3 * b;
    double *S, *HS, *Xn, *HXn, *Pn, *HPn, *tmp, *parts, *Gs, *Gh, *work, *Cm, *d_theta, *rparts, *rsum, *d_info;
    RDTRY(salloc(&S, 3 * nb));
    RDTRY(salloc(&HS, 3 * nb));
    RDTRY(salloc(&Xn, nb));
    RDTRY(salloc(&HXn, nb));
    RDTRY(salloc(&Pn, nb));
    RDTRY(salloc(&HPn, nb));
    RDTRY(salloc(&tmp, nb));
    const int nparts = ctx->num_sms * 2;
    RDTRY(salloc(&parts, (size_t)nparts * ns_max * ns_max));
    RDTRY(salloc(&Gs, (size_t)ns_max * ns_max));
    RDTRY(salloc(&Gh, (size_t)ns_max * ns_max));
    RDTRY(salloc(&work, (size_t)7 * ns_max * ns_max + 1024));
    RDTRY(salloc(&Cm, (size_t)ns_max * b));
    RDTRY(salloc(&d_theta, b));
    const int rgrid = ctx->num_sms * 2;
    RDTRY(salloc(&rparts, (size_t)rgrid * b));
    RDTRY(salloc(&rsum, b));
    RDTRY(salloc(&d_info, 4));  // four ints (kept, kept rounded up to even, Cholesky flag, unused), then the grid barrier of k_jacobi_grid
    // the preconditioner: per-axis sine tables, the mean lumped mass
    SineAxis ax[3];
    {
        int64_t rs = 1;
        for (int a = 0; a < ndim; ++a) {
            ax[a].n = (int)dims[a];
            ax[a].rs = rs;
            rs *= dims[a];
            RDTRY(salloc(&ax[a].S, (size_t)dims[a] * dims[a]));
            RDTRY(salloc(&ax[a].St, (size_t)dims[a] * dims[a]));
            RDTRY(salloc(&ax[a].mu, (size_t)dims[a]));
            k_sine_axis_tables<<<grid_for(dims[a] * dims[a], kThreads, 1024), kThreads, 0, ctx->stream>>>(ax[a].n, ax[a].S, ax[a].St, ax[a].mu);
            ctx->launches++;
        }
    }
    double mbar = 0.0;
    {
        std::vector<double> mh(N);
        CU(cudaMemcpyAsync(mh.data(), ctx->m, (size_t)N * sizeof(double), cudaMemcpyDeviceToHost, ctx->stream));
        CU(cudaStreamSynchronize(ctx->stream));
        long double s = 0.0L;
        for (int64_t i = 0; i < N; ++i) s += mh[i];
        mbar = (double)(s / (long double)N);
    }
    const double sk2 = ctx->sigma * kappa_ref * kappa_ref;
    std::vector<double> theta(b), res2(b), resid(b, INFINITY);
    const int gs = grid_for(ctx->K.nslices * 32, kThreads, big_grid(ctx));
    int64_t col_applies = 0;
    int64_t prec_applies = 0;
    double tensor_flop = 0.0;  // m8n8k4 work as issued: products of the logical sizes (tile padding not counted)
    double sum_dims = 0.0;
    for (int a = 0; a < ndim; ++a) sum_dims += (double)dims[a];

    auto block_apply = [&](const double* Y, double* HY, int nc) {  // HY = H Y for nc columns (a multiple of 8); tmp holds M^{-1} K Y
        const int nch = nc / RD_EIG_CB;
        const dim3 gb(std::max(1, gs / std::min(nch, 4)), nch);
        k_blk_K<<<gb, kThreads, 0, ctx->stream>>>(ctx->K.view(), N, ld, ctx->minv, Y, tmp);
        k_blk_KT<<<gb, kThreads, 0, ctx->stream>>>(ctx->KT.view(), N, ld, ctx->m, ctx->sigma, 1.0, 0.0, 0.0, Y, tmp, nullptr, HY);
        ctx->launches += 2;
        col_applies += nc;
    };
    auto precondition = [&](double* Y, int nc) -> int {  // Y <- T Y in place (nc columns), tmp is the other buffer of the ping-pong
        double* cur = Y;
        double* oth = tmp;
        for (int a = 0; a < ndim; ++a) {
            RDTRY(sine_axis_pass(ctx, ax[a], false, N, ld, nc, cur, oth));
            std::swap(cur, oth);
        }
        k_sine_scale<<<grid_for(N, kThreads, big_grid(ctx)), kThreads, 0, ctx->stream>>>(
            N, ld, nc, ax[0].n, ndim > 1 ? ax[1].n : 1, ax[0].mu, ndim > 1 ? ax[1].mu : nullptr, ndim > 2 ? ax[2].mu : nullptr, mbar, sk2, cur);
        ctx->launches++;
        for (int a = ndim - 1; a >= 0; --a) {
            RDTRY(sine_axis_pass(ctx, ax[a], true, N, ld, nc, cur, oth));
            std::swap(cur, oth);
        }
        // 2 ndim passes: the result is back in Y
        prec_applies += nc;
        tensor_flop += 4.0 * sum_dims * (double)N * nc;  // forward and inverse transform: 2 n_a flop per entry, axis and direction
        return RD_OK;
    };
    auto gram = [&](int p, const double* A, const double* B, double* out) {  // out (p x p) = A^T B
        const dim3 gg(nparts, (p + 63) / 64, (p + 63) / 64);
        k_gram_dmma<<<gg, 256, 0, ctx->stream>>>(N, p, p, A, ld, B, ld, parts, 1);  // symmetric products only: upper tiles
        k_reduce_parts<<<grid_for((int64_t)p * p, kThreads, 64), kThreads, 0, ctx->stream>>>(nparts, (int64_t)p * p, parts, out);
        k_mirror_upper_tiles<<<grid_for((int64_t)p * p, kThreads, 64), kThreads, 0, ctx->stream>>>(p, out);
        ctx->launches += 3;
        {
            const double nt = (double)((p + 63) / 64);
            tensor_flop += 2.0 * (double)N * 64.0 * 64.0 * (nt * (nt + 1.0) / 2.0);  // the upper 64 x 64 tiles
        }
    };
    // Out (N x nout) = A[:, 0:kk] Cs (kk x nout, column-major with leading dimension ldc) (+ Add)
    auto tall_mult = [&](const double* A, int kk, const double* Cs, int ldc, const double* Add, double* Out, int nout) {
        const GemmOp a{A, 1, ld, 0, 0}, c{Cs, 1, ldc, 0, 0}, e{Add, 1, ld, 0, 0}, d{Out, 1, ld, 0, 0};
        launch_gemm<true, false>(ctx->stream, 10, (int)N, nout, kk, 1, 1, a, c, e, d);
        ctx->launches++;
        tensor_flop += 2.0 * (double)N * kk * nout;
    };
    auto copy_cols = [&](double* dst, const double* src, int nc) -> int {
        if (nc > 0) CU(cudaMemcpyAsync(dst, src, (size_t)nc * ld * sizeof(double), cudaMemcpyDeviceToDevice, ctx->stream));
        return RD_OK;
    };
    double* X = S;
    double* HX = HS;
    const bool no_chol = std::getenv("RD_LOBPCG_NO_CHOL") != nullptr;  // tests: take the eigenvalue whitening on every iteration
    // the ns x ns part: two grid-parallel Jacobi eigensolves and the small products between them (lobpcg.cuh)
    auto small_rr = [&](int ns) -> int {
        const size_t nn = (size_t)ns_max * ns_max;
        double *A0 = work, *A1 = work + nn, *Vj = work + 2 * nn, *Tm = work + 3 * nn, *GhS = work + 4 * nn, *Q = work + 5 * nn;
        double* dsc = work + 6 * nn;
        double* jpart = work + 6 * nn + 512;
        GridBarrier* bar = (GridBarrier*)(d_info + 2);  // zero-initialised, returns to its idle state after every launch
        int* info = (int*)d_info;
        const int gsm = grid_for((int64_t)ns * ns, kThreads, 256);
        k_rr_scale<<<gsm, kThreads, 0, ctx->stream>>>(ns, Gs, Gh, dsc, A0, GhS);
        CU(cudaMemcpyAsync(A1, A0, (size_t)ns * ns * sizeof(double), cudaMemcpyDeviceToDevice, ctx->stream));  // the Cholesky works on a copy
        k_rr_chol<<<1, 1024, 0, ctx->stream>>>(ns, A1, dsc, Q, Tm, info, no_chol ? 1 : 0);
        int n_arg = ns;
        const int* n_ptr = nullptr;
        const int* skip1 = info + 2;
        void* args1[] = {&n_arg, &n_ptr, &A0, &A1, &Vj, &bar, &jpart, &skip1};
        CU(cudaLaunchCooperativeKernel((const void*)k_jacobi_grid, dim3(ns / 2), dim3(256), args1, 0, ctx->stream));
        k_rr_select<<<1, 1024, 0, ctx->stream>>>(ns, A0, Vj, dsc, Tm, info);
        k_rr_q<<<gsm, kThreads, 0, ctx->stream>>>(ns, info, GhS, Tm, Q);
        k_rr_a<<<gsm, kThreads, 0, ctx->stream>>>(ns, info, Tm, Q, A0);
        int n_zero = 0;
        const int* n_ptr2 = info + 1;
        const int* skip2 = nullptr;
        void* args2[] = {&n_zero, &n_ptr2, &A0, &A1, &Vj, &bar, &jpart, &skip2};
        CU(cudaLaunchCooperativeKernel((const void*)k_jacobi_grid, dim3(ns / 2), dim3(256), args2, 0, ctx->stream));
        k_rr_finish<<<1, 1024, 0, ctx->stream>>>(ns, b, info, A0, Vj, Tm, Cm, d_theta);
        ctx->launches += 8;
        return RD_OK;
    };

    // ---- start: T applied to a seeded random block (smooth), orthonormalised twice, Rayleigh-Ritz
    k_rand_block<<<grid_for(N * b, kThreads, big_grid(ctx)), kThreads, 0, ctx->stream>>>(N, ld, b, 0x5EEDULL, X);
    ctx->launches++;
    RDTRY(precondition(X, b));
    auto orthonormalise = [&]() -> int {
        gram(b, X, X, Gs);
        k_orth_small<<<1, 1024, 0, ctx->stream>>>(b, Gs, work, Cm);
        ctx->launches++;
        tall_mult(X, b, Cm, b, nullptr, Xn, b);
        return copy_cols(X, Xn, b);
    };
    RDTRY(orthonormalise());
    RDTRY(orthonormalise());
    auto fresh_ritz = [&]() -> int {  // HX = H X, then X <- X V, HX <- HX V with V from X^T H X; theta on the device
        block_apply(X, HX, b);
        gram(b, X, HX, Gs);
        k_rr_small<<<1, 1024, 0, ctx->stream>>>(b, Gs, work, Cm, d_theta);
        ctx->launches++;
        tall_mult(X, b, Cm, b, nullptr, Xn, b);
        tall_mult(HX, b, Cm, b, nullptr, HXn, b);
        RDTRY(copy_cols(X, Xn, b));
        return copy_cols(HX, HXn, b);
    };
    RDTRY(fresh_ritz());
    int iters = 0, status = RD_ECAP;
    const bool dbg = std::getenv("RD_LOBPCG_DEBUG") != nullptr;  // per-iteration trace and phase times on stderr (synchronises)
    double ph_ms[6] = {0, 0, 0, 0, 0, 0};  // residual, preconditioner, H apply, Gram, small dense, tall products + copies
    auto t_last = std::chrono::steady_clock::now();
    auto phase = [&](int q) {
        if (!dbg) return;
        cudaStreamSynchronize(ctx->stream);
        const auto t = std::chrono::steady_clock::now();
        ph_ms[q] += std::chrono::duration<double, std::milli>(t - t_last).count();
        t_last = t;
    };
    bool verified = true;  // the residuals about to be computed come from a freshly applied H X
    // Locking: the leading Ritz vectors that pass the test (whole chunks of 8) stay in X and in the Rayleigh-Ritz but get no
    // new search directions: W and P have na = b - nl columns, the basis b + 2 na.  nl never decreases between restarts.
    int nl = 0;        // locked leading columns
    int np_cols = 0;   // columns of P' (in Pn / HPn) from the last iteration; they belong to X columns [b - np_cols, b)
    CU(cudaEventRecord(ctx->ev[0], ctx->stream));
    for (int it = 0; it <= max_iters; ++it) {
        // residuals R = HX - X theta: norms of all b columns, R itself for the active ones into the W slot (columns b ..)
        int nl_new = nl;
        k_resid_write_parts<<<rgrid, 256, 0, ctx->stream>>>(N, ld, b, X, HX, d_theta, Xn, rparts);
        k_reduce_parts<<<1, kThreads, 0, ctx->stream>>>(rgrid, b, rparts, rsum);
        ctx->launches += 2;
        CU(cudaGetLastError());
        CU(cudaMemcpyAsync(theta.data(), d_theta, b * sizeof(double), cudaMemcpyDeviceToHost, ctx->stream));
        CU(cudaMemcpyAsync(res2.data(), rsum, b * sizeof(double), cudaMemcpyDeviceToHost, ctx->stream));
        CU(cudaStreamSynchronize(ctx->stream));
        bool ok = true;
        if (dbg) {
            int info_h[2] = {0, 0};
            cudaMemcpy(info_h, d_info, sizeof info_h, cudaMemcpyDeviceToHost);
            double mx = 0.0;
            for (int j = 0; j < k; ++j) mx = std::max(mx, std::sqrt(std::max(res2[j], 0.0)) / std::fabs(theta[j]));
            fprintf(stderr, "lobpcg it %d: nl %d kept %d max rel resid %.3e theta[0] %.6e theta[k-1] %.6e | ms resid %.1f prec %.1f H %.1f gram %.1f dense %.1f mult %.1f\n",
                    it, nl, info_h[0], mx, theta[0], theta[k - 1], ph_ms[0], ph_ms[1], ph_ms[2], ph_ms[3], ph_ms[4], ph_ms[5]);
            t_last = std::chrono::steady_clock::now();
        }
        for (int j = 0; j < b; ++j) {
            if (j < k && (!(theta[j] > 0.0) || !std::isfinite(theta[j]))) return fail(ctx, RD_ENOTSPD, "Ritz value %d = %g", j, theta[j]);
            resid[j] = std::sqrt(std::max(res2[j], 0.0)) / std::fabs(theta[j]);
            if (j < k && !(resid[j] <= tol)) ok = false;
        }
        if (ok && verified) { status = RD_OK; break; }
        if (ok) {
            // the recurrence of HX passed: confirm with a freshly applied operator and a fresh Rayleigh-Ritz before stopping
            RDTRY(orthonormalise());
            RDTRY(fresh_ritz());
            np_cols = 0;  // P's companion HP no longer matches the rotated block
            nl = 0;
            verified = true;
            continue;
        }
        verified = false;
        if (it == max_iters) break;
        iters = it + 1;
        if ((it & 15) == 15) {
            // the blocks HX and HP follow X and P through the same small products: every 16 iterations they are recomputed
            // from the operator so that their rounding errors do not accumulate into the Ritz values
            block_apply(X, HX, b);
            if (np_cols > 0) block_apply(Pn, HPn, np_cols);
        }
        while (nl_new < k && resid[nl_new] <= tol) ++nl_new;
        nl_new = std::min((nl_new / RD_EIG_CB) * RD_EIG_CB, b - RD_EIG_CB);
        nl = std::max(nl, nl_new);
        const int na = b - nl;
        double* Wb = S + nb;
        double* HW = HS + nb;
        double* Pb = Wb + (size_t)na * ld;
        double* HP = HW + (size_t)na * ld;
        RDTRY(copy_cols(Wb, Xn + (size_t)nl * ld, na));
        phase(0);
        RDTRY(precondition(Wb, na));
        phase(1);
        block_apply(Wb, HW, na);
        phase(2);
        // P: the trailing min(na, np_cols) columns of the last P'
        const int npc = std::min(na, np_cols);
        RDTRY(copy_cols(Pb, Pn + (size_t)(np_cols - npc) * ld, npc));
        RDTRY(copy_cols(HP, HPn + (size_t)(np_cols - npc) * ld, npc));
        const int ns = b + na + npc;
        gram(ns, S, S, Gs);
        gram(ns, S, HS, Gh);
        phase(3);
        RDTRY(small_rr(ns));
        phase(4);
        // P' = [W, P] C[b:, :],  X' = X C[:b, :] + P'  (all b columns; the next iteration uses the trailing na columns of P');
        // the same combinations of the H blocks
        tall_mult(Wb, ns - b, Cm + b, ns, nullptr, Pn, b);
        tall_mult(HW, ns - b, Cm + b, ns, nullptr, HPn, b);
        tall_mult(X, b, Cm, ns, Pn, Xn, b);
        tall_mult(HX, b, Cm, ns, HPn, HXn, b);
        np_cols = b;
        RDTRY(copy_cols(X, Xn, b));
        RDTRY(copy_cols(HX, HXn, b));
        CU(cudaGetLastError());
        phase(5);
    }
    CU(cudaEventRecord(ctx->ev[1], ctx->stream));
    // W <- the k lowest Ritz vectors (pad columns zero)
    RDTRY(alloc_reference(ctx, k));
    CU(cudaMemsetAsync(ctx->W, 0, (size_t)ld * ctx->kp * sizeof(double), ctx->stream));
    CU(cudaMemcpyAsync(ctx->W, X, (size_t)ld * k * sizeof(double), cudaMemcpyDeviceToDevice, ctx->stream));
    CU(cudaStreamSynchronize(ctx->stream));
    float loop_ms = 0.0f;
    CU(cudaEventElapsedTime(&loop_ms, ctx->ev[0], ctx->ev[1]));
    ctx->have_ref = true;
    ctx->ref_kind = 0;
    if (theta_out) memcpy(theta_out, theta.data(), k * sizeof(double));
    if (resid_out) memcpy(resid_out, resid.data(), k * sizeof(double));
    if (iters_out) *iters_out = iters;
    ctx->ref_degree = iters;
    ctx->ref_block = b;
    ctx->ref_col_applies = 0;  // the Chebyshev filter's counters: not this solver's
    ctx->ref_filter_ms = 0.0;
    ctx->ref_ms_pending = std::chrono::duration<double, std::milli>(std::chrono::steady_clock::now() - t_begin).count();
    ctx->ref_ms_last = ctx->ref_ms_pending;
    ctx->lob_flop = tensor_flop;
    ctx->lob_ms = loop_ms;
    ctx->lob_h_applies = col_applies;
    ctx->lob_t_applies = prec_applies;
    if (status != RD_OK) fail(ctx, status, "reference not converged to tol %g in %d LOBPCG iterations (worst residual %g)", tol, iters,
                              *std::max_element(resid.begin(), resid.begin() + k));
    return status;
}

extern "C" int rd_reference_lobpcg_work(const rd_ctx* ctx, double* tensor_flop, double* loop_ms, int64_t* h_column_applies,
                                        int64_t* t_column_applies)
{
    if (!ctx) return RD_EINVAL;
    if (tensor_flop) *tensor_flop = ctx->lob_flop;
    if (loop_ms) *loop_ms = ctx->lob_ms;
    if (h_column_applies) *h_column_applies = ctx->lob_h_applies;
    if (t_column_applies) *t_column_applies = ctx->lob_t_applies;
    return RD_OK;
}
