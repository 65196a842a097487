/*
 * refdef_oracle.c -- TEST INFRASTRUCTURE, NOT PRODUCT CODE.
 *
 * Plain, slow, single-threaded fp64 CPU oracle for the hot path of
 * "Reference-Space Reuse for Steady and Transient State-Constrained Conjugate Heat
 * Transfer" (arxiv/paper_2606_17971; citations are PAPER.md:line).  Only tests/,
 * __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may
 * build, load or call this file.  It shares no code, header, table or helper with
 * the CUDA path under paper_2606_17971_b200/ and neither imports the other.
 *
 * Names follow BASELINE.json: K state operator (CSR), m lumped mass diagonal,
 * sigma penalty scalar, H = M + sigma K^T M^{-1} K reduced Hessian (the paper's "M",
 * eq. (5) PAPER.md:93 with A = M_l^{-1}K, W = M_l/m-bar of PAPER.md:133; the common
 * factor 1/m-bar is dropped, reading A2), W the full-domain reference
 * (the paper's Phi), J active set, I inactive set, B = H_II.
 *
 * What is written out here, in the paper's order and notation:
 *   O1  operator       eq. (5)  PAPER.md:91-95        orc_apply_H, orc_diag_H
 *   O3  Algorithm 1    PAPER.md:214-259, :261-275     orc_alg1 (+ orc_coarse_*)
 *   O2  PDAS           eq. (7)-(8) PAPER.md:102-117   orc_solve_query
 *   O4  KKT measures   eq. (25) PAPER.md:343-346      inside orc_solve_query
 *       recovery       eq. (9)  PAPER.md:119-123      u = M^{-1} K y - f (f = 0)
 *
 * Pins (tests/test_oracle_*.py, -m "not gpu"): dense Cholesky / brute-force active sets
 * on tiny grids, symmetry + definiteness, KKT complementarity, unconstrained limit,
 * projector identities, restriction-residual identity eq. (20)-(21),
 * closed-form spectrum, rank-zero == Jacobi-CG, Fig. 2 transfer pattern, energy fraction
 * eq. (24); and (tests/test_oracle_pins_kkt_init.py) the five KKT measures of eq. (25) on a perturbed pair with
 * ||l||_inf > 1, the cond(E) > 1e10 fallback on both sides of its threshold, the query starts (given J0, all
 * inactive, inherited state and set), c = H_ii and the margin -- each shown to fail under listed mutations.
 * Unpinned: CG iteration counts at full size ("parity unpinned").
 *
 * Threads.  The parity tests use the plain build (gcc -O2, single thread, the loops exactly as written).
 * The TIMING legs of bench.py (cpu_baseline, --impl reference) may build the same file with -fopenmp: the
 * ORC_PAR_FOR / ORC_PAR_SUM marks below then split the row loops over the host cores in static chunks
 * (sums change their order, nothing else changes; K^T t becomes a row loop over a transposed copy whose
 * entries are in the order of the scatter, so that product is bit-identical).  Without -fopenmp the marks
 * are empty.  tests/test_oracle_pins.py checks the threaded build against the plain one.
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#define ORC_PRAGMA(x) _Pragma(#x)
#define ORC_PAR_FOR ORC_PRAGMA(omp parallel for schedule(static))
#define ORC_PAR_SUM(v) ORC_PRAGMA(omp parallel for schedule(static) reduction(+ : v))
#else
#define ORC_PAR_FOR
#define ORC_PAR_SUM(v)
#endif

#define ORC_OK 0
#define ORC_EINVAL (-1)
#define ORC_ENOMEM (-2)
#define ORC_ENOTSPD (-5)
#define ORC_ECAP (-6)
#define ORC_ESTEPS (-7)
#define ORC_ECYCLE (-8)
#define ORC_ERESID (-9)

#define ORC_JACOBI_CG 0
#define ORC_REFDEF 1
#define ORC_ZEROEXT 2

#define ORC_INIT_PAPER 0
#define ORC_INIT_ALL_ACTIVE 1
#define ORC_INIT_ALL_INACTIVE 2
#define ORC_INIT_GIVEN 3

typedef struct {
    int64_t N, nnz;
    int64_t *rowptr;
    int32_t *colidx;
    double *val;
    double *m;     /* lumped mass diagonal */
    double sigma;  /* penalty scalar (reading A1: sigma = alpha) */
    double *d;     /* diag(H) */
    double *t, *full_in, *full_out; /* scratch, length N */
    /* sequence state (PAPER.md:339 warm starts; reading A9 zero-extension history) */
    int have_state;
    double *y_state;
    uint8_t *J_state;   /* 1 = active */
    uint8_t *A_hist;    /* 1 = DOF was active at an earlier restriction of this sequence */
#ifdef _OPENMP
    int64_t *t_rowptr; int32_t *t_row; double *t_val; /* K^T by rows, entries of a row in ascending row of K */
#endif
} orc_ctx;

/* threads the timing build uses (1 for the plain build) */
int orc_threads(void)
{
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

typedef struct {
    int32_t n_inactive, cg_iters, rank_used, coarse_fallback, replacements, status;
    double rel_resid_verified, cond_E, margin;
    uint64_t active_hash;
} orc_step_report;

typedef struct {
    int32_t n_steps, status;
    double kkt[5];
} orc_query_report;

typedef struct {
    double eps, eps_c;
    int32_t cg_cap, pdas_cap, replace_period, jacobi, c_is_diag, init;
} orc_options;

/* ------------------------------------------------------------------ O1: operator */

orc_ctx *orc_create(int64_t N, const int64_t *rowptr, const int32_t *colidx, const double *val,
                    const double *m, double sigma)
{
    if (N <= 0 || !rowptr || !colidx || !val || !m) return NULL;
    for (int64_t i = 0; i < N; i++) if (!(m[i] > 0.0)) return NULL;
    orc_ctx *c = (orc_ctx *)calloc(1, sizeof(orc_ctx));
    if (!c) return NULL;
    c->N = N;
    c->nnz = rowptr[N];
    c->sigma = sigma;
    c->rowptr = (int64_t *)malloc((size_t)(N + 1) * sizeof(int64_t));
    c->colidx = (int32_t *)malloc((size_t)c->nnz * sizeof(int32_t));
    c->val = (double *)malloc((size_t)c->nnz * sizeof(double));
    c->m = (double *)malloc((size_t)N * sizeof(double));
    c->d = (double *)calloc((size_t)N, sizeof(double));
    c->t = (double *)malloc((size_t)N * sizeof(double));
    c->full_in = (double *)malloc((size_t)N * sizeof(double));
    c->full_out = (double *)malloc((size_t)N * sizeof(double));
    c->y_state = (double *)calloc((size_t)N, sizeof(double));
    c->J_state = (uint8_t *)calloc((size_t)N, 1);
    c->A_hist = (uint8_t *)calloc((size_t)N, 1);
    memcpy(c->rowptr, rowptr, (size_t)(N + 1) * sizeof(int64_t));
    memcpy(c->colidx, colidx, (size_t)c->nnz * sizeof(int32_t));
    memcpy(c->val, val, (size_t)c->nnz * sizeof(double));
    memcpy(c->m, m, (size_t)N * sizeof(double));
    /* d_i = m_i + sigma * sum_r K_ri^2 / m_r  (diagonal of eq. (5)) */
    for (int64_t i = 0; i < N; i++) c->d[i] = m[i];
    for (int64_t r = 0; r < N; r++)
        for (int64_t e = rowptr[r]; e < rowptr[r + 1]; e++)
            c->d[colidx[e]] += sigma * val[e] * val[e] / m[r];
#ifdef _OPENMP
    /* transposed copy for the threaded K^T t (counting sort: ascending row of K inside each row of K^T) */
    c->t_rowptr = (int64_t *)calloc((size_t)(N + 1), sizeof(int64_t));
    c->t_row = (int32_t *)malloc((size_t)c->nnz * sizeof(int32_t));
    c->t_val = (double *)malloc((size_t)c->nnz * sizeof(double));
    for (int64_t e = 0; e < c->nnz; e++) c->t_rowptr[colidx[e] + 1]++;
    for (int64_t i = 0; i < N; i++) c->t_rowptr[i + 1] += c->t_rowptr[i];
    {
        int64_t *cur = (int64_t *)malloc((size_t)N * sizeof(int64_t));
        memcpy(cur, c->t_rowptr, (size_t)N * sizeof(int64_t));
        for (int64_t r = 0; r < N; r++)
            for (int64_t e = rowptr[r]; e < rowptr[r + 1]; e++) {
                int64_t pos = cur[colidx[e]]++;
                c->t_row[pos] = (int32_t)r; c->t_val[pos] = val[e];
            }
        free(cur);
    }
#endif
    return c;
}

void orc_destroy(orc_ctx *c)
{
    if (!c) return;
    free(c->rowptr); free(c->colidx); free(c->val); free(c->m); free(c->d);
    free(c->t); free(c->full_in); free(c->full_out);
    free(c->y_state); free(c->J_state); free(c->A_hist);
#ifdef _OPENMP
    free(c->t_rowptr); free(c->t_row); free(c->t_val);
#endif
    free(c);
}

void orc_reset_sequence(orc_ctx *c)
{
    c->have_state = 0;
    memset(c->y_state, 0, (size_t)c->N * sizeof(double));
    memset(c->J_state, 0, (size_t)c->N);
    memset(c->A_hist, 0, (size_t)c->N);
}

/* out = K v */
void orc_apply_K(const orc_ctx *c, const double *v, double *out)
{
    ORC_PAR_FOR
    for (int64_t r = 0; r < c->N; r++) {
        double s = 0.0;
        for (int64_t e = c->rowptr[r]; e < c->rowptr[r + 1]; e++) s += c->val[e] * v[c->colidx[e]];
        out[r] = s;
    }
}

/* out = K^T t */
void orc_apply_KT(const orc_ctx *c, const double *t, double *out)
{
#ifdef _OPENMP
    ORC_PAR_FOR
    for (int64_t i = 0; i < c->N; i++) {
        double s = 0.0;
        for (int64_t e = c->t_rowptr[i]; e < c->t_rowptr[i + 1]; e++) s += c->t_val[e] * t[c->t_row[e]];
        out[i] = s;
    }
#else
    for (int64_t i = 0; i < c->N; i++) out[i] = 0.0;
    for (int64_t r = 0; r < c->N; r++)
        for (int64_t e = c->rowptr[r]; e < c->rowptr[r + 1]; e++) out[c->colidx[e]] += c->val[e] * t[r];
#endif
}

/* out = H v = m.*v + sigma K^T ((K v)./m)   (eq. (5); mass-weighted form :133) */
void orc_apply_H(orc_ctx *c, const double *v, double *out)
{
    orc_apply_K(c, v, c->t);
    ORC_PAR_FOR
    for (int64_t r = 0; r < c->N; r++) c->t[r] /= c->m[r];
    orc_apply_KT(c, c->t, out);
    ORC_PAR_FOR
    for (int64_t i = 0; i < c->N; i++) out[i] = c->m[i] * v[i] + c->sigma * out[i];
}

void orc_diag_H(const orc_ctx *c, double *d_out) { memcpy(d_out, c->d, (size_t)c->N * sizeof(double)); }

/* B x = (H R_I^T x)_I, B = H_II (eq. (7)): extend by zero, apply, restrict */
static void apply_B(orc_ctx *c, const int64_t *idx, int64_t n, const double *x, double *out)
{
    memset(c->full_in, 0, (size_t)c->N * sizeof(double));
    ORC_PAR_FOR
    for (int64_t q = 0; q < n; q++) c->full_in[idx[q]] = x[q];
    orc_apply_H(c, c->full_in, c->full_out);
    ORC_PAR_FOR
    for (int64_t q = 0; q < n; q++) out[q] = c->full_out[idx[q]];
}

void orc_apply_B(orc_ctx *c, const int64_t *idx, int64_t n, const double *x, double *out) { apply_B(c, idx, n, x, out); }

/* ------------------------------------------------------------------ small dense algebra */

static double dot(const double *a, const double *b, int64_t n)
{
    double s = 0.0;
    ORC_PAR_SUM(s)
    for (int64_t i = 0; i < n; i++) s += a[i] * b[i];
    return s;
}
static double nrm2(const double *a, int64_t n) { return sqrt(dot(a, a, n)); }

/* Thin Householder QR of A (n x k, column-major).  p = min(n,k).
 * Out: Q (n x p, column-major, orthonormal columns), R (p x k, column-major, upper trapezoidal). */
static void householder_qr(const double *A, int64_t n, int k, double *Q, double *R)
{
    int p = (n < k) ? (int)n : k;
    double *W = (double *)malloc((size_t)n * k * sizeof(double));
    double *V = (double *)calloc((size_t)n * p, sizeof(double)); /* reflector vectors */
    double *beta = (double *)calloc((size_t)p, sizeof(double));
    memcpy(W, A, (size_t)n * k * sizeof(double));
    for (int j = 0; j < p; j++) {
        double *col = W + (size_t)j * n;
        double normx = nrm2(col + j, n - j);
        double *v = V + (size_t)j * n;
        if (normx == 0.0) { beta[j] = 0.0; continue; }
        double a0 = col[j];
        double s = (a0 >= 0.0) ? -normx : normx; /* resulting diagonal entry */
        for (int64_t i = j; i < n; i++) v[i] = col[i];
        v[j] = a0 - s;
        double vtv = dot(v + j, v + j, n - j);
        beta[j] = (vtv > 0.0) ? 2.0 / vtv : 0.0;
        for (int c2 = j; c2 < k; c2++) {
            double *cc = W + (size_t)c2 * n;
            double f = beta[j] * dot(v + j, cc + j, n - j);
            ORC_PAR_FOR
            for (int64_t i = j; i < n; i++) cc[i] -= f * v[i];
        }
    }
    for (int c2 = 0; c2 < k; c2++)
        for (int i = 0; i < p; i++) R[(size_t)c2 * p + i] = (i <= c2) ? W[(size_t)c2 * n + i] : 0.0;
    /* Q = H_0 ... H_{p-1} [I_p; 0] */
    for (int c2 = 0; c2 < p; c2++) {
        double *q = Q + (size_t)c2 * n;
        for (int64_t i = 0; i < n; i++) q[i] = (i == c2) ? 1.0 : 0.0;
        for (int j = p - 1; j >= 0; j--) {
            const double *v = V + (size_t)j * n;
            if (beta[j] == 0.0) continue;
            double f = beta[j] * dot(v + j, q + j, n - j);
            ORC_PAR_FOR
            for (int64_t i = j; i < n; i++) q[i] -= f * v[i];
        }
    }
    free(W); free(V); free(beta);
}

/* One-sided (Hestenes) Jacobi on the columns of A (rows x cols, column-major): A V = U S.
 * Out: V (cols x cols, column-major), s (cols) = column norms of A V, sorted descending. */
static void jacobi_svd_right(double *A, int rows, int cols, double *V, double *s)
{
    for (int i = 0; i < cols; i++)
        for (int j = 0; j < cols; j++) V[(size_t)j * cols + i] = (i == j) ? 1.0 : 0.0;
    for (int sweep = 0; sweep < 60; sweep++) {
        int rotated = 0;
        for (int p = 0; p < cols - 1; p++)
            for (int q = p + 1; q < cols; q++) {
                double *ap = A + (size_t)p * rows, *aq = A + (size_t)q * rows;
                double app = dot(ap, ap, rows), aqq = dot(aq, aq, rows), apq = dot(ap, aq, rows);
                if (fabs(apq) <= 1e-15 * sqrt(app * aqq) || apq == 0.0) continue;
                rotated = 1;
                double zeta = (aqq - app) / (2.0 * apq);
                double t = ((zeta >= 0.0) ? 1.0 : -1.0) / (fabs(zeta) + sqrt(1.0 + zeta * zeta));
                double cs = 1.0 / sqrt(1.0 + t * t), sn = cs * t;
                for (int i = 0; i < rows; i++) {
                    double x = ap[i], y = aq[i];
                    ap[i] = cs * x - sn * y;
                    aq[i] = sn * x + cs * y;
                }
                double *vp = V + (size_t)p * cols, *vq = V + (size_t)q * cols;
                for (int i = 0; i < cols; i++) {
                    double x = vp[i], y = vq[i];
                    vp[i] = cs * x - sn * y;
                    vq[i] = sn * x + cs * y;
                }
            }
        if (!rotated) break;
    }
    for (int j = 0; j < cols; j++) s[j] = nrm2(A + (size_t)j * rows, rows);
    /* selection sort, descending, permuting V's columns alongside */
    for (int a = 0; a < cols - 1; a++) {
        int best = a;
        for (int b2 = a + 1; b2 < cols; b2++) if (s[b2] > s[best]) best = b2;
        if (best != a) {
            double ts = s[a]; s[a] = s[best]; s[best] = ts;
            for (int i = 0; i < cols; i++) {
                double tv = V[(size_t)a * cols + i];
                V[(size_t)a * cols + i] = V[(size_t)best * cols + i];
                V[(size_t)best * cols + i] = tv;
            }
        }
    }
}

/* Cyclic two-sided Jacobi eigenvalues of a symmetric r x r matrix (destroyed). */
static void jacobi_eigvals(double *E, int r, double *lam)
{
    for (int sweep = 0; sweep < 60; sweep++) {
        double off = 0.0, diag = 0.0;
        for (int i = 0; i < r; i++)
            for (int j = 0; j < r; j++) {
                double v = E[(size_t)j * r + i];
                if (i == j) diag += v * v; else off += v * v;
            }
        if (off <= 1e-30 * diag || off == 0.0) break;
        for (int p = 0; p < r - 1; p++)
            for (int q = p + 1; q < r; q++) {
                double apq = E[(size_t)q * r + p];
                if (apq == 0.0) continue;
                double app = E[(size_t)p * r + p], aqq = E[(size_t)q * r + q];
                double zeta = (aqq - app) / (2.0 * apq);
                double t = ((zeta >= 0.0) ? 1.0 : -1.0) / (fabs(zeta) + sqrt(1.0 + zeta * zeta));
                double cs = 1.0 / sqrt(1.0 + t * t), sn = cs * t;
                for (int i = 0; i < r; i++) { /* columns p,q */
                    double x = E[(size_t)p * r + i], y = E[(size_t)q * r + i];
                    E[(size_t)p * r + i] = cs * x - sn * y;
                    E[(size_t)q * r + i] = sn * x + cs * y;
                }
                for (int i = 0; i < r; i++) { /* rows p,q */
                    double x = E[(size_t)i * r + p], y = E[(size_t)i * r + q];
                    E[(size_t)i * r + p] = cs * x - sn * y;
                    E[(size_t)i * r + q] = sn * x + cs * y;
                }
            }
    }
    for (int i = 0; i < r; i++) lam[i] = E[(size_t)i * r + i];
}

/* In-place lower Cholesky of a symmetric r x r matrix (column-major). Returns 0 on success. */
static int cholesky(double *E, int r)
{
    for (int j = 0; j < r; j++) {
        double s = E[(size_t)j * r + j];
        for (int q = 0; q < j; q++) s -= E[(size_t)q * r + j] * E[(size_t)q * r + j];
        if (!(s > 0.0)) return 1;
        double ljj = sqrt(s);
        E[(size_t)j * r + j] = ljj;
        for (int i = j + 1; i < r; i++) {
            double v = E[(size_t)j * r + i];
            for (int q = 0; q < j; q++) v -= E[(size_t)q * r + i] * E[(size_t)q * r + j];
            E[(size_t)j * r + i] = v / ljj;
        }
    }
    return 0;
}
static void chol_solve(const double *L, int r, double *y)
{
    for (int i = 0; i < r; i++) {
        double s = y[i];
        for (int q = 0; q < i; q++) s -= L[(size_t)q * r + i] * y[q];
        y[i] = s / L[(size_t)i * r + i];
    }
    for (int i = r - 1; i >= 0; i--) {
        double s = y[i];
        for (int q = i + 1; q < r; q++) s -= L[(size_t)i * r + q] * y[q];
        y[i] = s / L[(size_t)i * r + i];
    }
}

/* ------------------------------------------------------------------ coarse space, eq. (18) */

typedef struct {
    orc_ctx *c;
    const int64_t *idx;
    int64_t n;
    int r;            /* retained rank r_I */
    int fallback;     /* 1: cond(E) > 1e10 (or E not SPD) -> rank zero */
    double cond_E;
    double *Z, *BZ;   /* n x r, column-major */
    double *E, *L;    /* r x r: E = Z^T B Z (symmetrised), L its Cholesky factor */
    double *small;    /* r scratch */
} orc_coarse;

void orc_coarse_free(orc_coarse *cs)
{
    if (!cs) return;
    free(cs->Z); free(cs->BZ); free(cs->E); free(cs->L); free(cs->small);
    free(cs);
}

/* Rank-revealing orthogonalisation of Z~ (thin QR, SVD of the triangular factor, keep singular
 * values > 1e-12 * largest), then BZ, E = Z^T B Z, Cholesky, cond(E) guard (:263-265). */
orc_coarse *orc_coarse_build(orc_ctx *c, const int64_t *idx, int64_t n, const double *Zt, int k)
{
    orc_coarse *cs = (orc_coarse *)calloc(1, sizeof(orc_coarse));
    cs->c = c; cs->idx = idx; cs->n = n; cs->r = 0; cs->cond_E = 0.0;
    if (k <= 0 || n <= 0 || !Zt) return cs;
    int p = (n < k) ? (int)n : k;
    double *Q = (double *)malloc((size_t)n * p * sizeof(double));
    double *R = (double *)malloc((size_t)p * k * sizeof(double));
    householder_qr(Zt, n, k, Q, R);
    /* SVD of R (p x k): one-sided Jacobi on the columns of R^T (k x p): R^T V = U' S, so R = V S U'^T
     * and the LEFT singular vectors of R are the columns of V. */
    double *Rt = (double *)malloc((size_t)k * p * sizeof(double));
    for (int i = 0; i < p; i++)
        for (int j = 0; j < k; j++) Rt[(size_t)i * k + j] = R[(size_t)j * p + i];
    double *V = (double *)malloc((size_t)p * p * sizeof(double));
    double *s = (double *)malloc((size_t)p * sizeof(double));
    jacobi_svd_right(Rt, k, p, V, s);
    int r = 0;
    for (int j = 0; j < p; j++) if (s[0] > 0.0 && s[j] > 1e-12 * s[0]) r++;
    if (r > 0) {
        cs->Z = (double *)malloc((size_t)n * r * sizeof(double));
        cs->BZ = (double *)malloc((size_t)n * r * sizeof(double));
        cs->E = (double *)malloc((size_t)r * r * sizeof(double));
        cs->L = (double *)malloc((size_t)r * r * sizeof(double));
        cs->small = (double *)malloc((size_t)r * sizeof(double));
        for (int j = 0; j < r; j++) {
            ORC_PAR_FOR
            for (int64_t i = 0; i < n; i++) {
                double acc = 0.0;
                for (int q = 0; q < p; q++) acc += Q[(size_t)q * n + i] * V[(size_t)j * p + q];
                cs->Z[(size_t)j * n + i] = acc;
            }
        }
        for (int j = 0; j < r; j++) apply_B(c, idx, n, cs->Z + (size_t)j * n, cs->BZ + (size_t)j * n);
        for (int a = 0; a < r; a++)
            for (int b2 = 0; b2 < r; b2++)
                cs->E[(size_t)b2 * r + a] = dot(cs->Z + (size_t)a * n, cs->BZ + (size_t)b2 * n, n);
        for (int a = 0; a < r; a++)
            for (int b2 = a + 1; b2 < r; b2++) {
                double v = 0.5 * (cs->E[(size_t)b2 * r + a] + cs->E[(size_t)a * r + b2]);
                cs->E[(size_t)b2 * r + a] = v; cs->E[(size_t)a * r + b2] = v;
            }
        /* 2-norm condition number from a Jacobi eigensolve (reading A7) */
        double *tmp = (double *)malloc((size_t)r * r * sizeof(double));
        double *lam = (double *)malloc((size_t)r * sizeof(double));
        memcpy(tmp, cs->E, (size_t)r * r * sizeof(double));
        jacobi_eigvals(tmp, r, lam);
        double lmin = lam[0], lmax = lam[0];
        for (int i = 1; i < r; i++) { if (lam[i] < lmin) lmin = lam[i]; if (lam[i] > lmax) lmax = lam[i]; }
        cs->cond_E = (lmin > 0.0) ? lmax / lmin : INFINITY;
        free(tmp); free(lam);
        memcpy(cs->L, cs->E, (size_t)r * r * sizeof(double));
        int bad = !(cs->cond_E <= 1e10) || cholesky(cs->L, r);
        if (bad) { cs->fallback = 1; r = 0; }
    }
    cs->r = r;
    free(Q); free(R); free(Rt); free(V); free(s);
    return cs;
}

/* out = Q v = Z E^{-1} Z^T v  (eq. (18)) */
void orc_coarse_Q(orc_coarse *cs, const double *v, double *out)
{
    int64_t n = cs->n; int r = cs->r;
    for (int64_t i = 0; i < n; i++) out[i] = 0.0;
    if (r == 0) return;
    for (int j = 0; j < r; j++) cs->small[j] = dot(cs->Z + (size_t)j * n, v, n);
    chol_solve(cs->L, r, cs->small);
    for (int j = 0; j < r; j++) {
        ORC_PAR_FOR
        for (int64_t i = 0; i < n; i++) out[i] += cs->Z[(size_t)j * n + i] * cs->small[j];
    }
}

/* out = P v = v - Z E^{-1} (BZ)^T v  (eq. (18); cached BZ) */
void orc_coarse_P(orc_coarse *cs, const double *v, double *out)
{
    int64_t n = cs->n; int r = cs->r;
    for (int64_t i = 0; i < n; i++) out[i] = v[i];
    if (r == 0) return;
    for (int j = 0; j < r; j++) cs->small[j] = dot(cs->BZ + (size_t)j * n, v, n);
    chol_solve(cs->L, r, cs->small);
    for (int j = 0; j < r; j++) {
        ORC_PAR_FOR
        for (int64_t i = 0; i < n; i++) out[i] -= cs->Z[(size_t)j * n + i] * cs->small[j];
    }
}

int orc_coarse_rank(const orc_coarse *cs) { return cs->r; }
int orc_coarse_fallback(const orc_coarse *cs) { return cs->fallback; }
double orc_coarse_cond(const orc_coarse *cs) { return cs->cond_E; }
void orc_coarse_get(const orc_coarse *cs, double *Z, double *BZ, double *E)
{
    size_t nr = (size_t)cs->n * cs->r, rr = (size_t)cs->r * cs->r;
    if (cs->r == 0) return;
    if (Z) memcpy(Z, cs->Z, nr * sizeof(double));
    if (BZ) memcpy(BZ, cs->BZ, nr * sizeof(double));
    if (E) memcpy(E, cs->E, rr * sizeof(double));
}

/* ------------------------------------------------------------------ O3: Algorithm 1 */

typedef struct {
    int32_t iters, rank_used, coarse_fallback, replacements, status;
    double rel_resid_verified, cond_E;
} orc_solve_report;

/* Verify(x, eps): ||b - Bx||_2/||b||_2 from a fresh apply (||b - Bx||_2 when b = 0) */
static double verify(orc_ctx *c, const int64_t *idx, int64_t n, const double *b, const double *x, double *w)
{
    apply_B(c, idx, n, x, w);
    double s = 0.0;
    for (int64_t i = 0; i < n; i++) { double e = b[i] - w[i]; s += e * e; }
    double nb = nrm2(b, n);
    return (nb > 0.0) ? sqrt(s) / nb : sqrt(s);
}

/* Algorithm 1, line numbers as reconstructed in SURVEY.md §8(c) O3, on a coarse space that
 * line 2 has already built (orc_coarse_build; rank zero = Jacobi-CG).
 * idx: the n inactive DOFs (ascending); b, x: length n (x holds x0 on entry). */
int orc_alg1_cs(orc_ctx *c, const int64_t *idx, int64_t n, const double *b, double *x, orc_coarse *cs,
                double eps, double eps_c, int cap, int replace_period, int jacobi, orc_solve_report *rep)
{
    memset(rep, 0, sizeof(*rep));
    double *r = (double *)malloc((size_t)n * sizeof(double));
    double *z = (double *)malloc((size_t)n * sizeof(double));
    double *p = (double *)malloc((size_t)n * sizeof(double));
    double *w = (double *)malloc((size_t)n * sizeof(double));
    double *Jr = (double *)malloc((size_t)n * sizeof(double));
    double *jac = (double *)malloc((size_t)n * sizeof(double));
    /* 1 */
    double nb = nrm2(b, n);
    double tau = (nb > 0.0) ? eps_c * nb : eps_c;
    /* 2 (done by the caller) */
    rep->rank_used = cs->r; rep->coarse_fallback = cs->fallback; rep->cond_E = cs->cond_E;
    for (int64_t i = 0; i < n; i++) jac[i] = jacobi ? 1.0 / c->d[idx[i]] : 1.0;
    int status = ORC_ECAP, done = 0;
    /* 3: x <- x0 + Q(b - B x0); r <- b - B x */
    apply_B(c, idx, n, x, w);
    for (int64_t i = 0; i < n; i++) r[i] = b[i] - w[i];
    orc_coarse_Q(cs, r, z);
    for (int64_t i = 0; i < n; i++) x[i] += z[i];
    apply_B(c, idx, n, x, w);
    for (int64_t i = 0; i < n; i++) r[i] = b[i] - w[i];
    /* 4-6 */
    if (nrm2(r, n) <= tau) { status = ORC_OK; done = 1; }
    double rho = 0.0;
    if (!done) {
        /* 7: z <- P J r; p <- z; rho <- r^T z */
        for (int64_t i = 0; i < n; i++) Jr[i] = jac[i] * r[i];
        orc_coarse_P(cs, Jr, z);
        memcpy(p, z, (size_t)n * sizeof(double));
        rho = dot(r, z, n);
    }
    /* 8 */
    for (int it = 1; !done && it <= cap; it++) {
        /* 9 */
        apply_B(c, idx, n, p, w);
        rep->iters = it;
        double pw = dot(p, w, n);
        if (!(pw > 0.0) || !(rho > 0.0)) { status = ORC_ENOTSPD; break; }
        /* 10 */
        double a = rho / pw;
        ORC_PAR_FOR
        for (int64_t i = 0; i < n; i++) x[i] += a * p[i];
        ORC_PAR_FOR
        for (int64_t i = 0; i < n; i++) r[i] -= a * w[i];
        /* 11 */
        if (nrm2(r, n) <= tau || (replace_period > 0 && it % replace_period == 0)) {
            rep->replacements++;
            /* 12 */
            apply_B(c, idx, n, x, w);
            ORC_PAR_FOR
            for (int64_t i = 0; i < n; i++) r[i] = b[i] - w[i];
            /* 13-15 */
            if (nrm2(r, n) <= tau) { status = ORC_OK; break; }
            /* 16 */
            orc_coarse_Q(cs, r, z);
            ORC_PAR_FOR
            for (int64_t i = 0; i < n; i++) x[i] += z[i];
            apply_B(c, idx, n, x, w);
            ORC_PAR_FOR
            for (int64_t i = 0; i < n; i++) r[i] = b[i] - w[i];
            /* 17-19 */
            if (nrm2(r, n) <= tau) { status = ORC_OK; break; }
            /* 20 */
            ORC_PAR_FOR
            for (int64_t i = 0; i < n; i++) Jr[i] = jac[i] * r[i];
            orc_coarse_P(cs, Jr, z);
            memcpy(p, z, (size_t)n * sizeof(double));
            rho = dot(r, z, n);
        } else {
            /* 22 */
            ORC_PAR_FOR
            for (int64_t i = 0; i < n; i++) Jr[i] = jac[i] * r[i];
            orc_coarse_P(cs, Jr, z);
            double rho_new = dot(r, z, n);
            /* 23 */
            double beta = rho_new / rho;
            ORC_PAR_FOR
            for (int64_t i = 0; i < n; i++) p[i] = z[i] + beta * p[i];
            rho = rho_new;
        }
    }
    /* 26: Verify with the recorded termination status */
    rep->rel_resid_verified = verify(c, idx, n, b, x, w);
    if (status == ORC_OK && !(rep->rel_resid_verified <= eps)) status = ORC_ERESID;
    rep->status = status;
    free(r); free(z); free(p); free(w); free(Jr); free(jac);
    return status;
}

/* Algorithm 1 with its line 2: Zt = restricted candidate basis Z~ (n x k column-major) or NULL / k = 0 for Jacobi-CG. */
int orc_alg1(orc_ctx *c, const int64_t *idx, int64_t n, const double *b, double *x, const double *Zt, int k,
             double eps, double eps_c, int cap, int replace_period, int jacobi, orc_solve_report *rep)
{
    orc_coarse *cs = orc_coarse_build(c, idx, n, Zt, k);
    int status = orc_alg1_cs(c, idx, n, b, x, cs, eps, eps_c, cap, replace_period, jacobi, rep);
    orc_coarse_free(cs);
    return status;
}

/* ------------------------------------------------------------------ O3a: restriction */

/* Restricted candidate basis of one inactive set (idx ascending, n entries), n x k column-major:
 *   RefDef          Z~ = R_I W                      eq. (12), PAPER.md:152 -- W itself is never changed;
 *   zero-extension  Z~ = R_I (chi_{not A} .* W)     eq. (13), cumulative (reading A9):
 *                   A = every DOF that was ACTIVE at an earlier restriction of this sequence, so a row
 *                   released since then carries zeros ("DOFs released after the first restriction carry
 *                   no reference entries").  The first restriction of a sequence is direct.
 * Afterwards the DOFs outside idx (the current active set) are added to the history A. */
void orc_restrict(orc_ctx *c, int method, const double *W, int k, const int64_t *idx, int64_t n, double *Zt)
{
    int64_t N = c->N;
    if (Zt && W)
        for (int j = 0; j < k; j++)
            for (int64_t q = 0; q < n; q++) {
                int64_t i = idx[q];
                double v = W[(size_t)j * N + i];
                if (method == ORC_ZEROEXT && c->A_hist[i]) v = 0.0;
                Zt[(size_t)j * n + q] = v;
            }
    uint8_t *inact = (uint8_t *)calloc((size_t)N, 1);
    for (int64_t q = 0; q < n; q++) inact[idx[q]] = 1;
    for (int64_t i = 0; i < N; i++) if (!inact[i]) c->A_hist[i] = 1;
    free(inact);
}

/* ------------------------------------------------------------------ O2: PDAS query */

static uint64_t fnv1a_bits(const uint8_t *flags, int64_t N, uint8_t *packed /* ceil(N/8) or NULL */)
{
    uint64_t hsh = 1469598103934665603ULL;
    int64_t nb = (N + 7) / 8;
    for (int64_t byte = 0; byte < nb; byte++) {
        uint8_t v = 0;
        for (int bit = 0; bit < 8; bit++) {
            int64_t i = byte * 8 + bit;
            if (i < N && flags[i]) v |= (uint8_t)(1u << bit);
        }
        if (packed) packed[byte] = v;
        hsh ^= (uint64_t)v;
        hsh *= 1099511628211ULL;
    }
    return hsh;
}

/* O4: the five acceptance measures of eq. (25) for any pair (y, lambda):
 *   g = H y - l,  s = max(1, ||l||_inf)
 *   kkt[0] = ||g + lambda||_inf / s              stationarity
 *   kkt[1] = ||[y - psi]_+||_inf                 primal feasibility ("The primal-feasibility quantity is absolute")
 *   kkt[2] = ||[-lambda]_+||_inf / s             dual feasibility
 *   kkt[3] = ||lambda .* (psi - y)||_inf / s     complementarity
 *   kkt[4] = ||y - min(psi, y - g)||_inf / s     projected gradient
 * psi_i = +inf contributes 0 to [1], [3] and y_i - min(inf, y_i - g_i) = g_i to [4].  ell = M y_d, length N. */
void orc_kkt(orc_ctx *c, const double *ell, const double *psi, const double *y, const double *lambda, double *kkt)
{
    int64_t N = c->N;
    double *Hy = (double *)malloc((size_t)N * sizeof(double));
    orc_apply_H(c, y, Hy);
    double s = 1.0, k0 = 0, k1 = 0, k2 = 0, k3 = 0, k4 = 0;
    for (int64_t i = 0; i < N; i++) if (fabs(ell[i]) > s) s = fabs(ell[i]);
    for (int64_t i = 0; i < N; i++) {
        double g = Hy[i] - ell[i];
        double v0 = fabs(g + lambda[i]);
        double v2 = (lambda[i] < 0.0) ? -lambda[i] : 0.0;
        double v1 = 0.0, v3 = 0.0, v4;
        if (isinf(psi[i])) {
            v4 = fabs(g); /* y - min(inf, y - g) = g */
        } else {
            v1 = (y[i] > psi[i]) ? y[i] - psi[i] : 0.0;
            v3 = fabs(lambda[i] * (psi[i] - y[i]));
            double mn = (psi[i] < y[i] - g) ? psi[i] : (y[i] - g);
            v4 = fabs(y[i] - mn);
        }
        if (v0 > k0) k0 = v0;
        if (v1 > k1) k1 = v1;
        if (v2 > k2) k2 = v2;
        if (v3 > k3) k3 = v3;
        if (v4 > k4) k4 = v4;
    }
    kkt[0] = k0 / s; kkt[1] = k1; kkt[2] = k2 / s; kkt[3] = k3 / s; kkt[4] = k4 / s;
    free(Hy);
}

/* One optimisation query: PDAS (eq. (7)-(8); Alg. 2 steps 9-15, :392-398),
 * control recovery (eq. (9), :121) and the KKT measures (eq. (25), :343-346).
 * W: full-domain reference, N x k column-major (may be NULL for Jacobi-CG).
 * J0: N flags, used only with init = ORC_INIT_GIVEN.
 * Outputs y, u, lambda: length N.  steps: pdas_cap entries.  J_bits: NULL or pdas_cap*ceil(N/8) bytes
 * (the active set AT THE START of each step, packed LSB-first). */
int orc_solve_query(orc_ctx *c, int method, const double *y_d, const double *psi, const uint8_t *J0,
                    const double *W, int k, const orc_options *opt,
                    double *y, double *u, double *lambda,
                    orc_step_report *steps, uint8_t *J_bits, orc_query_report *rep)
{
    int64_t N = c->N;
    int64_t nbytes = (N + 7) / 8;
    uint8_t *J = (uint8_t *)malloc((size_t)N), *Jn = (uint8_t *)malloc((size_t)N);
    double *ell = (double *)malloc((size_t)N * sizeof(double));
    double *tmp = (double *)malloc((size_t)N * sizeof(double));
    double *Hy = (double *)malloc((size_t)N * sizeof(double));
    int64_t *idx = (int64_t *)malloc((size_t)N * sizeof(int64_t));
    double *b = (double *)malloc((size_t)N * sizeof(double));
    double *x = (double *)malloc((size_t)N * sizeof(double));
    uint64_t *seen = (uint64_t *)malloc((size_t)(opt->pdas_cap + 1) * sizeof(uint64_t));
    int nseen = 0;
    memset(rep, 0, sizeof(*rep));

    /* l = M y_d (f = 0), eq. (5) */
    for (int64_t i = 0; i < N; i++) ell[i] = c->m[i] * y_d[i];

    /* initial active set and state (reading A5) */
    int init = opt->init;
    if (init == ORC_INIT_PAPER) init = c->have_state ? -1 : ORC_INIT_ALL_ACTIVE;
    if (init == -1) {
        memcpy(J, c->J_state, (size_t)N);
    } else if (init == ORC_INIT_ALL_ACTIVE) {
        memset(J, 1, (size_t)N);
    } else if (init == ORC_INIT_ALL_INACTIVE) {
        memset(J, 0, (size_t)N);
    } else {
        for (int64_t i = 0; i < N; i++) J[i] = J0[i] ? 1 : 0;
    }
    for (int64_t i = 0; i < N; i++) if (isinf(psi[i])) J[i] = 0; /* psi = +inf is never active */
    if (!c->have_state) memset(c->y_state, 0, (size_t)N * sizeof(double));

    int status = ORC_ESTEPS, nsteps = 0;
    for (int step = 0; step < opt->pdas_cap; step++) {
        orc_step_report *sr = &steps[step];
        memset(sr, 0, sizeof(*sr));
        nsteps = step + 1;
        sr->active_hash = fnv1a_bits(J, N, J_bits ? J_bits + (size_t)step * nbytes : NULL);
        seen[nseen++] = sr->active_hash;
        int64_t n = 0;
        for (int64_t i = 0; i < N; i++) if (!J[i]) idx[n++] = i;
        sr->n_inactive = (int32_t)n;
        /* y <- y_state; y_J <- psi_J */
        for (int64_t i = 0; i < N; i++) y[i] = J[i] ? psi[i] : c->y_state[i];
        if (n > 0) {
            /* b = l_I - H_IJ psi_J  (eq. (7)): one full apply to chi_J .* psi */
            for (int64_t i = 0; i < N; i++) tmp[i] = J[i] ? psi[i] : 0.0;
            orc_apply_H(c, tmp, Hy);
            for (int64_t q = 0; q < n; q++) { b[q] = ell[idx[q]] - Hy[idx[q]]; x[q] = c->y_state[idx[q]]; }
            /* restricted basis (O3a): RefDef eq. (12); zero-extension eq. (13) cumulative (A9) */
            double *Zt = NULL;
            int kk = 0;
            if (method != ORC_JACOBI_CG && W && k > 0) {
                kk = k;
                Zt = (double *)malloc((size_t)n * k * sizeof(double));
            }
            orc_restrict(c, method, W, kk, idx, n, Zt);
            orc_solve_report so;
            orc_alg1(c, idx, n, b, x, Zt, kk, opt->eps, opt->eps_c, opt->cg_cap, opt->replace_period,
                     opt->jacobi, &so);
            free(Zt);
            sr->cg_iters = so.iters; sr->rank_used = so.rank_used; sr->coarse_fallback = so.coarse_fallback;
            sr->replacements = so.replacements; sr->status = so.status;
            sr->rel_resid_verified = so.rel_resid_verified; sr->cond_E = so.cond_E;
            for (int64_t q = 0; q < n; q++) y[idx[q]] = x[q];
        }
        /* lambda = l - H y on all DOFs, then lambda_I := 0 exactly (reading A4) */
        orc_apply_H(c, y, Hy);
        for (int64_t i = 0; i < N; i++) lambda[i] = J[i] ? (ell[i] - Hy[i]) : 0.0;
        /* eq. (8): J_new = { i : lambda_i + c_i (y_i - psi_i) > 0 }, strict (A10); c_i = 1 or d_i (A3) */
        double margin = INFINITY;
        int same = 1;
        for (int64_t i = 0; i < N; i++) {
            if (isinf(psi[i])) { Jn[i] = 0; if (J[i]) same = 0; continue; }
            double ci = opt->c_is_diag ? c->d[i] : 1.0;
            double g = lambda[i] + ci * (y[i] - psi[i]);
            Jn[i] = (g > 0.0) ? 1 : 0;
            if (fabs(g) < margin) margin = fabs(g);
            if (Jn[i] != J[i]) same = 0;
        }
        sr->margin = margin;
        memcpy(c->y_state, y, (size_t)N * sizeof(double));
        if (same) { status = ORC_OK; break; }
        uint64_t hn = fnv1a_bits(Jn, N, NULL);
        int cyc = 0;
        for (int q = 0; q < nseen; q++) if (seen[q] == hn) cyc = 1;
        memcpy(J, Jn, (size_t)N);
        if (cyc) { status = ORC_ECYCLE; break; }
    }
    memcpy(c->J_state, J, (size_t)N);
    c->have_state = 1;
    rep->n_steps = nsteps;
    rep->status = status;

    /* u = M^{-1} K y - f, all state values incl. the active ones (eq. (9)) */
    orc_apply_K(c, y, tmp);
    for (int64_t i = 0; i < N; i++) u[i] = tmp[i] / c->m[i];

    orc_kkt(c, ell, psi, y, lambda, rep->kkt);

    free(J); free(Jn); free(ell); free(tmp); free(Hy); free(idx); free(b); free(x); free(seen);
    return status;
}

/* state accessors for the harness (warm-start state between queries) */
void orc_get_state(const orc_ctx *c, double *y_state, uint8_t *J_flags, uint8_t *A_flags)
{
    if (y_state) memcpy(y_state, c->y_state, (size_t)c->N * sizeof(double));
    if (J_flags) memcpy(J_flags, c->J_state, (size_t)c->N);
    if (A_flags) memcpy(A_flags, c->A_hist, (size_t)c->N);
}
