/*
 * refdef.h -- C ABI of the B200-native hot path of arxiv/paper_2606_17971
 * ("Reference-Space Reuse for Steady and Transient State-Constrained Conjugate Heat Transfer").
 *
 * Citations are PAPER.md:line (the text of the paper) plus section / equation / algorithm.
 * Names follow BASELINE.json: K state operator (N x N sparse, integrated form), m the lumped mass
 * diagonal (> 0), sigma the penalty scalar, H = M + sigma K^T M^{-1} K the SPD reduced Hessian
 * (the paper's "M", eq. (5) PAPER.md:91-95 with A = M_l^{-1}K, W = M_l/m-bar of PAPER.md:133;
 * the common factor 1/m-bar is dropped), W the full-domain reference (the paper's Phi, N x k),
 * J the active set, I its complement, B = H_II the inactive system matrix (eq. (7)).
 *
 * POINTER CONVENTION.  Unless an argument says "host", every array argument may be a HOST pointer or a
 * DEVICE pointer: the library asks the CUDA runtime (cudaPointerGetAttributes) and stages host data
 * through its own device buffers with cudaMemcpyAsync on the context's stream.  Device pointers are used
 * in place.  The library never frees or keeps caller memory: K, m and W are copied at create /
 * set_reference.  All arithmetic of the path runs in CUDA kernels on the device the context was created
 * on; there is no CPU fallback: without a usable CUDA device every entry point returns RD_ECUDA.
 *
 * ERRORS.  Every int-returning function returns an rd_status.  Hard errors (RD_EINVAL, RD_ENOMEM,
 * RD_ECUDA, RD_ENOREF) leave outputs unspecified.  The soft statuses of a solve (RD_ENOTSPD, RD_ECAP,
 * RD_ESTEPS, RD_ECYCLE, RD_ERESID) still return the last iterate and a complete report: the paper records
 * such failures separately and keeps going.  No C++ exception crosses this boundary and
 * there is no global state: one context = one operator = one reference.
 *
 * THREADS/STREAMS.  A context is not thread safe.  All work is enqueued on the stream given at create
 * (NULL = the legacy default stream); calls that return host results synchronise that stream.
 */
#ifndef REFDEF_H
#define REFDEF_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct rd_ctx rd_ctx; /* opaque; owns device copies of K, K^T, m, d, W and all work buffers */

typedef enum {
    RD_OK = 0,
    RD_EINVAL = -1,
    RD_ENOMEM = -2,
    RD_ECUDA = -3,
    RD_ENOREF = -4,  /* a deflated method was asked for but no reference is set */
    RD_ENOTSPD = -5, /* m_i <= 0, or non-positive curvature / rho inside CG (Alg. 1 line 9) */
    RD_ECAP = -6,    /* CG iteration cap reached */
    RD_ESTEPS = -7,  /* PDAS step cap reached */
    RD_ECYCLE = -8,  /* an active set repeated within one query */
    RD_ERESID = -9   /* Verify failed: recurrence converged but the recomputed residual is above eps */
} rd_status;

/* Inner solver variants (PAPER.md:331-335 lists the paper's comparison set; BASELINE.json keeps three). */
typedef enum {
    RD_JACOBI_CG = 0, /* rank-zero execution of Algorithm 1 = Jacobi-preconditioned CG */
    RD_REFDEF = 1,    /* direct restriction Z~ = R_I W, eq. (12) */
    RD_ZEROEXT = 2    /* zero-extension transfer, eq. (13) PAPER.md:158-162 (cumulative over a sequence) */
} rd_method;

/* Initial active set of a query (the first query starts with every DOF active, later
 * queries inherit state and active set; the cold-start variant resets to all active). */
typedef enum {
    RD_INIT_PAPER = 0,        /* first query of a sequence all active, later queries warm */
    RD_INIT_ALL_ACTIVE = 1,
    RD_INIT_ALL_INACTIVE = 2,
    RD_INIT_GIVEN = 3         /* J0 flags supplied by the caller */
} rd_init;

typedef struct {
    double sigma_is_alpha; /* 1: sigma = alpha (paper, eq. (5)); 0: sigma = 1/alpha (BASELINE.json's literal text) */
    double eps;            /* Verify tolerance on ||b - Bx||/||b||; BASELINE.json: 1e-8 */
    double eps_c;          /* recurrence trigger tau = eps_c ||b|| (Alg. 1 line 1) */
    int32_t cg_cap;        /* CG iteration cap */
    int32_t pdas_cap;      /* PDAS step cap */
    int32_t replace_period;/* scheduled residual replacement period, 0 = only at candidate convergence */
    int32_t jacobi;        /* 1: J = diag(B)^{-1}; 0: identity */
    int32_t c_is_diag;     /* eq. (8): c_i = H_ii (1) or c = 1 (0, BASELINE.json configs) */
    int32_t init;          /* rd_init */
    int32_t alg1_variant;  /* 0: projection carried in coefficient form, one pass over H_II W_I per iteration, operands
                              staged through shared memory by TMA bulk copies, work restricted to the 32-row slices that
                              hold inactive rows (default);
                              1: the literal recurrence of Alg. 1 (passes over H_II W_I and W_I), register-staged, all
                              rows visited and masked.  Same method, same results up to rounding */
} rd_options;

/* One PDAS step (one inactive system).  Times are milliseconds measured with CUDA events on the stream. */
typedef struct {
    int32_t n_inactive;     /* |I| at the start of the step */
    int32_t cg_iters;       /* executions of Alg. 1 line 9 (operator applies inside the loop) */
    int32_t rank_used;      /* retained rank r_I of the restricted basis */
    int32_t coarse_fallback;/* 1: cond(E) > 1e10 or E not SPD -> rank-zero execution */
    int32_t replacements;   /* times the replacement branch (Alg. 1 lines 11-20) was entered */
    int32_t status;         /* rd_status of the inner solve */
    double rel_resid_verified; /* Verify: ||b - Bx||_2/||b||_2 from a fresh apply */
    double cond_E;          /* 2-norm condition number of E = Z^T B Z (eq. (18)) */
    double margin;          /* min_i |lambda_i + c_i (y_i - psi_i)| over finite psi_i: distance of eq. (8) to a tie */
    uint64_t active_hash;   /* FNV-1a (64 bit) of the packed active set at the start of the step */
    double t_restrict, t_coarse, t_iter, t_update; /* ms: S1, S2, Algorithm 1, rhs + multiplier/active-set update */
} rd_step_report;

typedef struct {
    int32_t n_steps, status; /* status: outcome of the PDAS loop (RD_OK: the active set repeated; RD_ESTEPS; RD_ECYCLE) */
    double kkt[5];    /* eq. (25): stationarity, primal, dual, complementarity, projected gradient */
    double t_total;   /* ms, whole call */
    double t_reference_charged; /* ms of rd_build_reference charged to this query (first query after a build) */
    int64_t total_cg_iters;
    /* Inner solves are recorded separately from the outer loop ("Caps, cycles, ... and residual failures
     * are recorded separately"): a query is a time-to-solution only if status == RD_OK, worst_inner_status == RD_OK
     * and every kkt[i] <= 1e-8. */
    int32_t worst_inner_status; /* the most severe steps[i].status of this query: RD_OK unless some Algorithm-1 solve ended
                                   RD_ENOTSPD (-5, most severe), RD_ERESID (-9) or RD_ECAP (-6) */
    int32_t n_inner_failed;     /* number of steps whose inner solve did not return RD_OK */
    int32_t n_fallbacks;        /* number of steps that took the rank-zero fallback of PAPER.md:265 (cond(E) > 1e10) */
    int32_t reserved;
} rd_query_report;

/* Report of one Algorithm-1 solve through rd_solve_inactive. */
typedef struct {
    int32_t iters, rank_used, coarse_fallback, replacements, status;
    double rel_resid_verified, cond_E, t_iter_ms;
    double bytes_per_iter; /* algorithmic HBM bytes one loop iteration moves for this (N, n, nnz, rank) */
    double t_stage_us[8];  /* alg1_variant 0: microseconds CTA 0 spent in  [0] stage A (K product)  [1] grid barrier
                              [2] stage B (K^T product)  [3] grid barrier + reduction  [4] k x k coefficient updates
                              [5] stage C (updates + H_II W_I pass)  [6] grid barrier + reduction  [7] outside the loop;
                              zeros for the other variants */
    /* eq. (23), alg1_variant 0 through rd_solve_inactive only: extreme Ritz values of the operator the
     * deflated, Jacobi-preconditioned CG iterates with, D^{-1/2} B P D^{-1/2} = B^ - D^{-1/2} B Z E^{-1} Z^T B D^{-1/2}, from the
     * Lanczos tridiagonal matrix of the last restart-free run of ritz_count iterations.  They lie inside the nonzero
     * spectrum of that matrix and converge to its ends: ritz_max / ritz_min estimates the effective condition number.
     * Zero when nothing was recorded. */
    double ritz_min, ritz_max;
    int32_t ritz_count;
    int32_t live_slices_A, live_slices_B; /* S6 compaction: 32-row slices the K product / the K^T product, vector updates
                              and tall-skinny pass of this solve touch (of ceil(N/32)); all others are skipped */
    int32_t reserved;
} rd_solve_report;

void rd_default_options(rd_options* opt);

/* Step 1 of Algorithm 2: take the assembled operator.  K in CSR (rowptr: N+1 int64,
 * colidx: nnz int32, val: nnz double; any order inside a row; duplicates are summed) and the lumped mass
 * diagonal m (N doubles, all > 0 else RD_ENOTSPD).  alpha > 0.  Builds sliced-ELL copies of K and K^T, 1/m
 * and d = diag(H), d_i = m_i + sigma sum_r K_ri^2/m_r (eq. (5)).  opt may be NULL (defaults).
 * cuda_stream: a cudaStream_t or NULL. */
int rd_create(rd_ctx** out, int64_t N, const int64_t* rowptr, const int32_t* colidx, const double* val,
              const double* m_diag, double alpha, const rd_options* opt, void* cuda_stream);
void rd_destroy(rd_ctx* ctx);
const char* rd_last_error(const rd_ctx* ctx); /* host string owned by the context; "" if none */
int64_t rd_kernel_launches(const rd_ctx* ctx); /* CUDA kernels this context has launched so far */
int rd_set_options(rd_ctx* ctx, const rd_options* opt); /* sigma_is_alpha cannot change after create (RD_EINVAL) */

/* Steps 2-4 of Algorithm 2, BASELINE.json variant: the k lowest eigenpairs of the full
 * H (the paper builds its reference once, before the sequence, and charges it to the first
 * query).  Block Krylov method: Chebyshev-filtered subspace iteration on a block of
 * b = k + max(8, k/4) vectors (rounded up to a multiple of 8) with Rayleigh-Ritz after every filter sweep,
 * started from a fixed counter-based random block, run until every
 * ||H w_j - theta_j w_j||_2 <= tol * theta_j (||w_j|| = 1, j < k) or max_block_iters sweeps (then RD_ECAP is
 * returned and the best block so far is kept as the reference).  W is stored on the device (N x k,
 * orthonormal columns).  theta_out: k doubles (ascending), may be NULL.  resid_out: k doubles (relative
 * residuals reached), may be NULL.  iters_out: sweeps used, may be NULL.  All three are host pointers.
 * 1 <= k <= 64, k <= N.  The wall time is remembered and charged to the next query.  W is unique only up to
 * sign and rotation inside clusters: compare by eigenvalues and principal angles, never by columns. */
int rd_build_reference(rd_ctx* ctx, int32_t k, double tol, int32_t max_block_iters, double* theta_out,
                       double* resid_out, int32_t* iters_out);
/* Facts about the last rd_build_reference: block size b, total Chebyshev degree (each degree = one application
 * of H to all b columns), wall milliseconds.  Any pointer may be NULL. */
int rd_reference_info(const rd_ctx* ctx, int32_t* block, int64_t* total_degree, double* build_ms);
/* Work of the Chebyshev filter of the last rd_build_reference / rd_build_reference_scaled (zeros for the other
 * constructions): column_applies = the number of (column, degree) pairs H was applied to (locked columns excluded),
 * filter_ms = CUDA-event time of those applies, bytes_per_column_apply = the algorithmic HBM bytes of one of them,
 * 3 nnz + 48 N (K and K^T stream once per 8 columns; six vector passes per column).  The filter's GB/s is
 * column_applies * bytes_per_column_apply / filter_ms.  Any pointer may be NULL. */
int rd_reference_work(const rd_ctx* ctx, int64_t* column_applies, double* filter_ms, double* bytes_per_column_apply);
/* Measurement helper: the FP64 tensor-core throughput of this device in TFLOP/s (back-to-back mma.sync m8n8k4 f64 on
 * registers, best of four timed launches): the denominator for the tensor-pipe share of the S2 Gram kernels. */
int rd_probe_fp64_tensor_peak(rd_ctx* ctx, double* tflops);
/* The Jacobi-scaled variant of rd_build_reference (the paper's "generalized eigenproblem M_c phi = mu D_c phi supplies
 * low modes in Jacobi-scaled coordinates ... each column is normalized in the Euclidean norm", here on the
 * fine operator): the k lowest pairs of H w = mu D w, D = diag(H), by the same block method applied to
 * D^{-1/2} H D^{-1/2}; the stored reference has unit columns (D-orthogonal up to that scaling, not orthogonal: the
 * coarse setup orthogonalises the restricted basis anyway).  Arguments and statuses as rd_build_reference; mu_out
 * receives the generalized eigenvalues, the residual test is ||H w - mu D w|| in the scaled coordinates. */
int rd_build_reference_scaled(rd_ctx* ctx, int32_t k, double tol, int32_t max_block_iters, double* mu_out,
                              double* resid_out, int32_t* iters_out);
/* rd_build_reference for operators on a Cartesian grid of the unit box (dims as in rd_build_reference_sine): the same
 * k lowest eigenpairs of H (same tolerance test, same outputs, same stored reference) by a locally optimal block
 * preconditioned CG (LOBPCG) whose preconditioner is the exact inverse of the HOMOGENEOUS operator of that grid,
 * T = S^T diag(1 / (mbar (1 + sigma kappa_ref^2 mu^2))) S, with S the products of the 1-D sine vectors of eq. (15)
 * and mu their Laplacian eigenvalues, mbar the mean of m; S is applied axis by axis as dense
 * products on the FP64 tensor cores.  kappa_ref > 0: the conductivity of the homogeneous comparison medium (the
 * background conductivity of the problem; it changes the number of iterations, never the result).  max_iters: cap on
 * LOBPCG iterations (RD_ECAP as a soft status, the best block so far stays as the reference); iters_out: iterations
 * used.  The result is checked with a freshly applied H before RD_OK is returned.  3 (k + guard) <= 256 and <= N. */
int rd_build_reference_lobpcg(rd_ctx* ctx, int32_t k, double tol, int32_t max_iters, int32_t ndim, const int64_t* dims,
                              double kappa_ref, double* theta_out, double* resid_out, int32_t* iters_out);
/* Work of the last rd_build_reference_lobpcg (zeros otherwise): tensor_flop = FP64 flop issued to the tensor cores
 * (sine transforms 4 sum(dims) N per column apply of T, the upper tiles of the two Gram products, the tall products),
 * loop_ms = CUDA-event time of the iteration loop, and the numbers of column applies of H and of T.  tensor_flop /
 * loop_ms against rd_probe_fp64_tensor_peak is the solver's share of the FP64 tensor peak.  Any pointer may be NULL. */
int rd_reference_lobpcg_work(const rd_ctx* ctx, double* tensor_flop, double* loop_ms, int64_t* h_column_applies,
                             int64_t* t_column_applies);
/* The analytical Cartesian spatial reference of the paper (section 2.2.3, eq. (15)) for steady
 * problems on a Cartesian grid of dims[0] x ... x dims[ndim-1] cells (ndim <= 3, x = dims[0] fastest, product = N,
 * else RD_EINVAL): the k lowest products of the 1-D sine modes of the constant-coefficient Dirichlet Laplacian,
 * v_q(j) = sqrt(2/n) sin(pi q (j + 1/2)/n) for the cell-centred grids used here (the paper's grid is node-centred),
 * ordered by (mu, q_1, ..., q_d), mu = sum_a 4 n_a^2 sin^2(pi q_a/(2 n_a)) ("Lexicographic ordering fixes the choice
 * within repeated eigenvalues").  The reference is homogeneous; the operator keeps its interfaces and transport.
 * O(N k) work: replaces rd_build_reference when the grid is Cartesian.  mu_out: host, k doubles, may be NULL.
 * modes_out: host, k x ndim int32 (row c = q_1..q_d of column c), may be NULL.  The build time is charged to the next
 * query like rd_build_reference's. */
int rd_build_reference_sine(rd_ctx* ctx, int32_t k, int32_t ndim, const int64_t* dims, double* mu_out, int32_t* modes_out);
/* The mode-dependent temporal reference of the paper (section 2.2.4, eq. (16)-(17)) for the
 * backward-Euler all-at-once operator K_st = I (x) K_s + L (x) M_s on a Cartesian grid of dims cells (ndim <= 3) and nt
 * uniform slabs of length dt (product of dims x nt = N, ordering space + N_s * time, else RD_EINVAL; nt <= 256).
 * For each of the first min(k, N_s) spatial sine modes phi_i (Laplacian eigenvalue mu_i, rd_build_reference_sine's
 * order) the temporal matrix S_i = (mu_i I + L)^T (mu_i I + L) is diagonalised (it shares its eigenvectors with H_i of
 * eq. (17); capacity c_0 = 1, W_t = I); the candidate pairs are ordered by (s, i, j) and the k lowest retained;
 * column c of the reference is q_{i,j} (x) phi_i, each q with its largest-magnitude component positive.
 * s_out: host, k doubles (reference eigenvalue nu = h^d (1 + sigma s)), may be NULL.  pairs_out: host, k x (ndim + 1)
 * int32 (q_1..q_d of the spatial mode, then j), may be NULL.  Build time charged to the next query.
 * Stored compactly (rd_reference_storage): the r_s distinct sine products used and the k temporal vectors. */
int rd_build_reference_spacetime(rd_ctx* ctx, int32_t k, int32_t ndim, const int64_t* dims, int32_t nt, double dt,
                                 double* s_out, int32_t* pairs_out);
/* Complete temporal coverage ("The timed Cartesian trajectories keep all temporal factors of S spatial
 * modes ... which pairs each retained mode with every time level"; :210): the reference of rd_build_reference_spacetime
 * restricted to the first S spatial sine modes, ALL nt temporal eigenvectors of each: rank k = S * nt (<= 64, else
 * RD_EINVAL), columns in the order (s, i, j) as above.  s_out: k doubles, pairs_out: k x (ndim + 1) int32, may be NULL. */
int rd_build_reference_spacetime_cover(rd_ctx* ctx, int32_t S, int32_t ndim, const int64_t* dims, int32_t nt, double dt,
                                       double* s_out, int32_t* pairs_out);
/* How the reference is held ("If the selected pairs use r_s distinct spatial modes, the reference stores
 * N_s r_s + N_t r floating-point values and r spatial-column indices.  Restriction evaluates a selected product at its
 * inactive space-time entries.").  kind: -1 none, 0 dense N x k block, 1 compact space-time factors (the two
 * rd_build_reference_spacetime* calls and rd_build_reference_transient): no dense copy exists on the device, S1 forms
 * the restricted candidate W_I from the factors and rd_get_reference forms the dense block for the caller only.
 * n_values: doubles stored (N k, or N_s r_s + N_t k); n_indices: int32 stored (0 or k).  Any pointer may be NULL. */
int rd_reference_storage(const rd_ctx* ctx, int32_t* kind, int64_t* n_values, int64_t* n_indices);
/* The paper's coarse-mesh reference (section 2.2.2): "P1 prolongation maps these vectors to the full
 * fine mesh, where each column is normalized in the Euclidean norm."  Wc: N_c x k column-major (ld N_c), host or
 * device: vectors on a coarser Cartesian grid of dims_c cells of the same unit box, typically the Jacobi-scaled low
 * modes of the coarse operator (rd_build_reference_scaled on a context created from the coarse K, then
 * rd_get_reference).  dims_f: the fine grid (ndim <= 3, x = dims[0] fastest on both grids, product of dims_f = N else
 * RD_EINVAL; any ratio dims_f[a]/dims_c[a], also non-integer).  P1 on the cell-centred grids used here = the d-linear
 * interpolant of the coarse cell-centre values, extended by the Dirichlet value 0 on the boundary, evaluated at the
 * fine cell centres (reading A20).  norms_out: host, k doubles, the Euclidean norms of the prolonged columns
 * before the normalisation, may be NULL; a zero or non-finite column is RD_EINVAL and leaves no reference.
 * The time of this call is charged to the next query (the coarse eigensolve ran elsewhere: the caller adds it). */
int rd_build_reference_prolonged(rd_ctx* ctx, int32_t k, int32_t ndim, const int64_t* dims_c, const int64_t* dims_f,
                                 const double* Wc, double* norms_out);
/* Inject a reference (e.g. the oracle's): W is N x k column-major with leading dimension N. */
int rd_set_reference(rd_ctx* ctx, int32_t k, const double* W);
/* Copy the stored reference out: W_out N x k column-major (ld N); returns k via k_out (0 if none). */
int rd_get_reference(rd_ctx* ctx, double* W_out, int32_t* k_out);

/* Steps 9-15 of Algorithm 2 for one query: PDAS, eq. (7)-(8) PAPER.md:102-117, with
 * Algorithm 1 on every inactive system; then u = M^{-1} K y (eq. (9), f = 0)
 * and the KKT measures of eq. (25).  y_d, psi: N doubles (psi_i = +inf allowed: never active).
 * J0: N bytes (non-zero = active), used only with RD_INIT_GIVEN, else may be NULL.
 * y, u, lambda: N doubles out (lambda may be NULL).  steps: host array of opt.pdas_cap entries.
 * J_bits: NULL or host array of pdas_cap * ceil(N/8) bytes: the active set at the start of each step,
 * packed LSB first.  rep: host. */
int rd_solve_query(rd_ctx* ctx, int32_t method, const double* y_d, const double* psi, const uint8_t* J0,
                   double* y, double* u, double* lambda, rd_step_report* steps, uint8_t* J_bits,
                   rd_query_report* rep);
/* Forget the warm-start state and the zero-extension history (start of a new sequence). */
int rd_reset_sequence(rd_ctx* ctx);

/* ---- single steps of the path, exported so that each can be checked against the oracle ---- */

/* out = K v, out = K^T v (N doubles each). */
int rd_apply_K(rd_ctx* ctx, const double* v, double* out);
int rd_apply_KT(rd_ctx* ctx, const double* v, double* out);
/* S3: out = H v (eq. (5)).  active: NULL (full operator) or N bytes (non-zero = active): then the masked
 * operator of eq. (7), out_i = (H (chi_I v))_i on I and 0 on J. */
int rd_apply_H(rd_ctx* ctx, const double* v, const uint8_t* active, double* out);
int rd_diag_H(rd_ctx* ctx, double* d_out);
/* S3 without any allocation (callers under CUDA graph capture, serving loops, harnesses that forbid cudaMalloc):
 * out = H v, or with active != NULL the masked operator of eq. (7) exactly as rd_apply_H computes it (same kernels'
 * order of sums: bit-identical results).  The intermediate t = M^-1 K (chi_I v) lives in a file-scope
 * `static __device__` array of RD_NOALLOC_MAX_N doubles (8 MiB, held by every GPU that loads the library until the
 * process exits) instead of a context buffer.
 *   v, out : N doubles, DEVICE pointers, out must not alias v; active: NULL or N bytes, DEVICE pointer.  The caller owns
 *            all three; host pointers are RD_EINVAL (they would need a staging copy).
 *   N > RD_NOALLOC_MAX_N is RD_EINVAL with a message in rd_last_error; rd_apply_H has no such limit.
 * The call enqueues two kernels on the context's stream and returns WITHOUT synchronising; it calls no cudaMalloc,
 * cudaFree or allocating library routine (the first call on a device resolves the array's address with
 * cudaGetSymbolAddress: make that call outside a capture).  Every call on a device shares the one array, which keeps
 * the previous call's contents: each call rewrites all N entries it reads, so nothing needs clearing, but two calls
 * that overlap on the GPU (different streams, or two contexts) race on it.  The device of the context must be current. */
#define RD_NOALLOC_MAX_N (1 << 20)
int rd_apply_H_noalloc(rd_ctx* ctx, const double* v, const uint8_t* active, double* out);
/* Algorithm 1 on one inactive system (S1-S5): active = N bytes; b, x: N doubles in full-domain indexing
 * (entries on J are ignored on input and 0 on output); x holds x0 on entry.  Deflated methods use the
 * stored reference and, for RD_ZEROEXT, update the zero-extension history. */
int rd_solve_inactive(rd_ctx* ctx, int32_t method, const uint8_t* active, const double* b, double* x,
                      rd_solve_report* rep);
/* S1+S2 for one active set: restricted basis, Gram G = W_I^T W_I and E_W = W_I^T H_II W_I (both k x k
 * column-major, may be NULL), and C = T E^{-1} T^T (k x k, the coarse solve in W_I coordinates, may be NULL);
 * rank / cond / fallback as in rd_step_report.
 * SEQUENCE STATE.  The single-step entry points (rd_coarse_setup, rd_solve_inactive, rd_energy_fraction) work on
 * their own copy of the active flags: the active set and state a later rd_solve_query inherits under
 * RD_INIT_PAPER are kept apart and are not touched by them.  The zero-extension history (eq. (13),
 * DESIGN.md reading A9) is advanced by rd_solve_inactive (every restriction of the sequence counts, whichever
 * method runs) and only read by rd_coarse_setup and rd_energy_fraction. */
int rd_coarse_setup(rd_ctx* ctx, int32_t method, const uint8_t* active, double* G, double* EW, double* C,
                    int32_t* rank_used, double* cond_E, int32_t* fallback);

/* S7, the acceptance measures of eq. (25) for ANY pair (y, lambda), as rd_solve_query computes them for
 * its result: with g = H y - l, l = M y_d, s = max(1, ||l||_inf),
 *   kkt[0] = ||g + lambda||_inf / s,  kkt[1] = ||[y - psi]_+||_inf (absolute),  kkt[2] = ||[-lambda]_+||_inf / s,
 *   kkt[3] = ||lambda .* (psi - y)||_inf / s,  kkt[4] = ||y - min(psi, y - g)||_inf / s.
 * y_d, psi, y, lambda: N doubles, host or device (psi_i = +inf allowed).  kkt: 5 host doubles. */
int rd_kkt(rd_ctx* ctx, const double* y_d, const double* psi, const double* y, const double* lambda, double* kkt);

/* S6, one multiplier / active-set update of PDAS (eq. (7)-(8)) for ANY state y and active set, as
 * rd_solve_query performs it after every inner solve: lambda = l - H y on the active set and exactly 0 on the inactive
 * set (reading A4), active_new_i = [psi_i finite and lambda_i + c_i (y_i - psi_i) > 0] with c_i = 1 or H_ii
 * (rd_options.c_is_diag), margin = min_i |lambda_i + c_i (y_i - psi_i)| over finite psi_i.
 * y_d, psi, y: N doubles; active: N bytes (non-zero = active); lambda_out: N doubles; active_new_out: N bytes; all host or
 * device.  changed (number of DOFs whose membership changes), n_active_new, margin: host scalars, may be NULL.
 * Touches neither the sequence state nor the zero-extension history. */
int rd_pdas_update(rd_ctx* ctx, const double* y_d, const double* psi, const uint8_t* active, const double* y,
                   double* lambda_out, uint8_t* active_new_out, int64_t* changed, int64_t* n_active_new, double* margin);

/* Transient variant of the coarse-mesh reference, eq. (14) (section 2.2.2; reading A21).
 * The context holds the all-at-once operator of N = N_s * nt DOFs in the layout id = space + N_s * t.  Phi: N_s x rs
 * spatial vectors, column-major, host or device (e.g. prolonged coarse vectors, or the reference of a steady
 * context read with rd_get_reference), none zero.  For every column phi_i the nt x nt matrices
 *     H_i = (I (x) phi_i)^T H (I (x) phi_i),   D_i = (I (x) phi_i)^T diag(H) (I (x) phi_i),   H_i q = nu D_i q
 * are formed (nt operator applies per vector) and solved on the device; the k lowest of the rs * nt candidates in
 * the order (nu, i, j) become the reference: column = q (x) phi_i, the component of q of largest magnitude
 * positive, unit Euclidean norm.  nu_out: k host doubles or NULL; pairs_out: 2k host int32 (i, j) or NULL.
 * RD_EINVAL: k > rs * nt, k or rs > 64, nt > the dense limit, N not a multiple of nt; RD_ENOTSPD: a zero vector. */
int rd_build_reference_transient(rd_ctx* ctx, int32_t k, int32_t rs, int32_t nt, const double* Phi, double* nu_out,
                                 int32_t* pairs_out);

/* Energy fraction removed by the coarse correction, eq. (24): for an independent solution
 * x_* of B x = b (B = H_II on the inactive set of `active`) and a zero initial guess,
 *     chi = ||Q b||_B^2 / ||x_*||_B^2,   ||v||_B^2 = v^T B v,   Q = Z E^{-1} Z^T (Algorithm 1 line 2)
 * with the basis of `method` on this active set (S1 + S2 are run; rank zero and RD_JACOBI_CG give chi = 0;
 * the zero-extension history is read, not advanced).  Computed as c^T C c with c = W_I^T b and C of
 * rd_coarse_setup (Q = W_I C W_I^T and C E_W C = C), and x_*^T (B x_*) from one masked operator apply.
 * active: N bytes; b, x_star: N doubles in full-domain indexing (entries on J ignored), host or device.
 * chi, qb_energy (= ||Qb||_B^2), xs_energy (= ||x_*||_B^2): host doubles out; the last two may be NULL.
 * The complementary fraction ||x_* - Qb||_B^2 / ||x_*||_B^2 equals 1 - chi when x_* solves the system. */
int rd_energy_fraction(rd_ctx* ctx, int32_t method, const uint8_t* active, const double* b, const double* x_star,
                       double* chi, double* qb_energy, double* xs_energy);

#ifdef __cplusplus
}
#endif
#endif /* REFDEF_H */
