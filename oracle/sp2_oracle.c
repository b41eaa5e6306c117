/*
 * oracle/sp2_oracle.c -- CPU ORACLE.  TEST INFRASTRUCTURE, NOT PRODUCT CODE.
 *
 * A plain, slow, obviously-correct FP64 implementation of the SP2 ("second-order spectral projection")
 * density-matrix recursion of arxiv 2401.13772 (PAPER.md = /root/reference/PAPER.md, cited as P:<line>):
 *
 *   X_0 = (e_max I - H) / (e_max - e_min)                      Eq. 5, Listing 2
 *   X_{m+1} = X_m^2            if tr X_m >  N_occ              Eq. 6
 *   X_{m+1} = 2 X_m - X_m^2    if tr X_m <= N_occ              Eq. 7, "<=" from Listing 2
 *   D = X_n for enough iterations n
 *
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may build, load or
 * call this file.  It shares no code, header, table or helper with the CUDA path (paper_2401_13772_b200/csrc),
 * and the CUDA path never calls it.  There is deliberately no blocking, tiling or algebraic reordering here:
 * products are the textbook triple loop, sparse products are the textbook Gustavson row merge with a dense
 * accumulator.  OpenMP only distributes independent output rows over threads; every sum that crosses rows is
 * done sequentially in row order, so results do not depend on the thread count.
 *
 * Readings of the paper where it is silent/ambiguous are those of SURVEY.md section 8(c) and DESIGN.md
 * ("Readings"): Gershgorin bounds for e_min/e_max; missing `else` in Listing 2 restored
 * from Eq. 6-7; idempotency measure e_m = ||X_m^2 - X_m||_F / ||X_m||_F with stop rules S1/S2/S3; the returned
 * matrix is X_{m*} (the iterate that was tested); threshold keeps |v| >= tau or the diagonal; ELLPACK-R
 * overflow is a failure (status -3).
 *
 * PINS (tests/test_oracle_pins.py): brute-force Jacobi eigenprojector on tiny N, closed forms (diagonal H, 2x2 H,
 * staggered bipartite lattice), projector invariants, scalar recursion on eigenvalues, shift/scale and
 * permutation invariance, hand-built threshold cases, tau=0 sparse == dense.  The stop-rule constants (1e-2 gate,
 * two-back comparison) are DESIGN.md readings: "parity unpinned" by the paper for those constants only.
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

#define ORACLE_LOG_LEN 128

typedef struct {
    int32_t status;       /* 0 converged (S1), 1 noise floor (S2), 2 max_products (S3), <0 failure          */
    int32_t n_products;   /* number of X^2 products evaluated = m_star + 1                                   */
    int32_t m_star;       /* index of the returned iterate; branch[0..m_star-1] are the recorded decisions   */
    int32_t overflow_row; /* ELLPACK: lowest row that needed more than M slots, else -1                      */
    double emin, emax;    /* Gershgorin bounds used for Eq. 5                                                */
    uint8_t branch[ORACLE_LOG_LEN];      /* b_m: 1 => X <- 2X - X^2, 0 => X <- X^2                          */
    double trace[ORACLE_LOG_LEN];        /* tr X_m                                                           */
    double idem[ORACLE_LOG_LEN];         /* e_m                                                              */
    int32_t max_row_nnz[ORACLE_LOG_LEN]; /* ELLPACK: max over rows of stored nnz of P_m (and X_{m+1})        */
} oracle_stats_t;

/* ---- Neumaier compensated summation: traces and norms carry <= 1 ulp error ---- */
typedef struct { double s, c; } nsum_t;
static inline void nsum_add(nsum_t *a, double x)
{
    double t = a->s + x;
    if (fabs(a->s) >= fabs(x)) a->c += (a->s - t) + x; else a->c += (x - t) + a->s;
    a->s = t;
}
static inline double nsum_get(const nsum_t *a) { return a->s + a->c; }

static void stats_init(oracle_stats_t *st)
{
    memset(st, 0, sizeof(*st));
    st->overflow_row = -1;
}

/* stop rules S1/S2/S3, DESIGN.md "Readings" item 5.  Returns -1 to continue, else the status. */
static int stop_rule(int m, const double *e, double tol, int max_products)
{
    if (e[m] < tol) return 0;                                   /* S1 */
    if (m >= 2 && e[m] < 1e-2 && e[m] >= e[m - 2]) return 1;    /* S2: stagnation on the noise floor */
    if (m + 1 == max_products) return 2;                        /* S3 */
    return -1;
}

/* =============================================== DENSE ================================================ */

/* Gershgorin circle bounds: e_min = min_i(H_ii - sum_{j!=i}|H_ij|), e_max = max_i(H_ii + ...). */
int oracle_gershgorin_dense(const double *H, int64_t N, int64_t ld, double *emin, double *emax)
{
    if (!H || N <= 0 || ld < N) return -1;
    double lo = INFINITY, hi = -INFINITY;
    for (int64_t i = 0; i < N; ++i) {
        nsum_t r = {0, 0};
        for (int64_t j = 0; j < N; ++j)
            if (j != i) nsum_add(&r, fabs(H[i * ld + j]));
        double rad = nsum_get(&r), d = H[i * ld + i];
        if (d - rad < lo) lo = d - rad;
        if (d + rad > hi) hi = d + rad;
    }
    *emin = lo; *emax = hi;
    return 0;
}

/* tr A = sum_i A_ii (Listing 2 `bml_trace`). */
double oracle_trace_dense(const double *A, int64_t N, int64_t ld)
{
    nsum_t t = {0, 0};
    for (int64_t i = 0; i < N; ++i) nsum_add(&t, A[i * ld + i]);
    return nsum_get(&t);
}

/* P = X X by the definition P_ij = sum_k X_ik X_kj, k ascending, separate multiply and add. */
void oracle_x2_dense(const double *X, int64_t N, double *P)
{
#pragma omp parallel for schedule(static)
    for (int64_t i = 0; i < N; ++i) {
        double *Pi = P + i * N;
        for (int64_t j = 0; j < N; ++j) Pi[j] = 0.0;
        for (int64_t k = 0; k < N; ++k) {
            const double a = X[i * N + k];
            const double *Xk = X + k * N;
            for (int64_t j = 0; j < N; ++j) Pi[j] += a * Xk[j];
        }
    }
}

/* Selected entries of X X, one dot product each (full-size sampled parity). */
void oracle_x2_dense_sampled(const double *X, int64_t N, int64_t ld, int64_t ns,
                             const int64_t *rows, const int64_t *cols, double *out)
{
#pragma omp parallel for schedule(static)
    for (int64_t s = 0; s < ns; ++s) {
        const int64_t i = rows[s], j = cols[s];
        nsum_t a = {0, 0};
        for (int64_t k = 0; k < N; ++k) nsum_add(&a, X[i * ld + k] * X[k * ld + j]);
        out[s] = nsum_get(&a);
    }
}

/* Eq. 5 with Gershgorin bounds: X_ij = -s H_ij (i != j), X_ii = s (e_max - H_ii), s = 1/(e_max - e_min). */
void oracle_rescale_dense(const double *H, int64_t N, int64_t ld, double emin, double emax, double *X)
{
    const double s = 1.0 / (emax - emin);
    for (int64_t i = 0; i < N; ++i)
        for (int64_t j = 0; j < N; ++j)
            X[i * N + j] = (i == j) ? s * (emax - H[i * ld + i]) : -s * H[i * ld + j];
}

/* ||P - X||_F^2 and ||X||_F^2, row partials then a sequential compensated sum over rows. */
static void dense_norms(const double *P, const double *X, int64_t N, double *e2, double *x2, double *rowbuf)
{
#pragma omp parallel for schedule(static)
    for (int64_t i = 0; i < N; ++i) {
        nsum_t a = {0, 0}, b = {0, 0};
        for (int64_t j = 0; j < N; ++j) {
            const double d = P[i * N + j] - X[i * N + j];
            nsum_add(&a, d * d);
            nsum_add(&b, X[i * N + j] * X[i * N + j]);
        }
        rowbuf[2 * i] = nsum_get(&a);
        rowbuf[2 * i + 1] = nsum_get(&b);
    }
    nsum_t a = {0, 0}, b = {0, 0};
    for (int64_t i = 0; i < N; ++i) { nsum_add(&a, rowbuf[2 * i]); nsum_add(&b, rowbuf[2 * i + 1]); }
    *e2 = nsum_get(&a); *x2 = nsum_get(&b);
}

/*
 * Dense SP2, SURVEY 8(c) algorithm lines 1-13.  H: N x N row-major with leading dimension ld, exactly symmetric.
 * D: N x N, leading dimension N.  Returns the status (also in st->status).
 */
/* bounds == NULL: Gershgorin (reading 1); else { e_min, e_max } supplied by the caller (oracle/bounds.py, the
 * tighter-bounds option of SURVEY 8(f) f-3).  Nothing else differs. */
int oracle_sp2_dense_bounds(const double *H, int64_t N, int64_t ld, int32_t n_occ, double tol, int32_t max_products,
                            const double *bounds, double *D, oracle_stats_t *st);
int oracle_sp2_dense(const double *H, int64_t N, int64_t ld, int32_t n_occ, double tol, int32_t max_products,
                     double *D, oracle_stats_t *st)
{
    return oracle_sp2_dense_bounds(H, N, ld, n_occ, tol, max_products, NULL, D, st);
}
int oracle_sp2_dense_bounds(const double *H, int64_t N, int64_t ld, int32_t n_occ, double tol, int32_t max_products,
                            const double *bounds, double *D, oracle_stats_t *st)
{
    stats_init(st);
    if (!H || !D || N <= 0 || ld < N || n_occ <= 0 || n_occ >= N || !(tol > 0) || max_products < 1 ||
        max_products > ORACLE_LOG_LEN)
        return st->status = -1;
    for (int64_t i = 0; i < N; ++i)                    /* item 12: symmetry is required exactly */
        for (int64_t j = 0; j < i; ++j)
            if (H[i * ld + j] != H[j * ld + i]) return st->status = -5;
    double emin, emax;
    oracle_gershgorin_dense(H, N, ld, &emin, &emax);                                          /* line 1 */
    if (bounds) { emin = bounds[0]; emax = bounds[1]; }
    st->emin = emin; st->emax = emax;
    if (!(emax - emin > 0)) return st->status = -2;
    double *X = (double *)malloc(sizeof(double) * N * N), *P = (double *)malloc(sizeof(double) * N * N);
    double *rowbuf = (double *)malloc(sizeof(double) * 2 * N);
    if (!X || !P || !rowbuf) { free(X); free(P); free(rowbuf); return st->status = -4; }
    oracle_rescale_dense(H, N, ld, emin, emax, X);                                            /* line 2 */
    int status = 2, m;
    for (m = 0;; ++m) {                                                                       /* line 3 */
        const double t = oracle_trace_dense(X, N, N);                                         /* line 4 */
        oracle_x2_dense(X, N, P);                                                             /* line 5 */
        double e2, x2;
        dense_norms(P, X, N, &e2, &x2, rowbuf);
        st->trace[m] = t;                                                                     /* line 7 */
        st->idem[m] = sqrt(e2) / sqrt(x2);                                                    /* line 6 */
        const int s = stop_rule(m, st->idem, tol, max_products);                              /* lines 8-10 */
        if (s >= 0) { status = s; break; }
        const int b = (t - (double)n_occ <= 0.0);                                             /* line 11 */
        st->branch[m] = (uint8_t)b;
        if (b) { for (int64_t q = 0; q < N * N; ++q) X[q] = 2.0 * X[q] - P[q]; }              /* line 12, Eq. 7 */
        else   { memcpy(X, P, sizeof(double) * N * N); }                                      /*          Eq. 6 */
    }
    memcpy(D, X, sizeof(double) * N * N);                                                     /* line 13 */
    st->m_star = m; st->n_products = m + 1;
    free(X); free(P); free(rowbuf);
    return st->status = status;
}

/* =============================================== ELLPACK-R ============================================ */
/* Listing 1: N rows, M slots per row, value[N*M], index[N*M], nnz[N]; entry p of row i at i*M+p. */

static int cmp_i32(const void *a, const void *b)
{
    const int32_t x = *(const int32_t *)a, y = *(const int32_t *)b;
    return (x > y) - (x < y);
}

/* Gershgorin over stored entries; a missing diagonal counts as 0. */
int oracle_gershgorin_ellpack(int64_t N, int32_t M, const double *value, const int32_t *index,
                              const int32_t *nnz, double *emin, double *emax)
{
    if (!value || !index || !nnz || N <= 0 || M < 1) return -1;
    double lo = INFINITY, hi = -INFINITY;
    for (int64_t i = 0; i < N; ++i) {
        nsum_t r = {0, 0};
        double d = 0.0;
        for (int32_t p = 0; p < nnz[i]; ++p) {
            if (index[i * M + p] == i) d = value[i * M + p];
            else nsum_add(&r, fabs(value[i * M + p]));
        }
        const double rad = nsum_get(&r);
        if (d - rad < lo) lo = d - rad;
        if (d + rad > hi) hi = d + rad;
    }
    *emin = lo; *emax = hi;
    return 0;
}

double oracle_trace_ellpack(int64_t N, int32_t M, const double *value, const int32_t *index, const int32_t *nnz)
{
    nsum_t t = {0, 0};
    for (int64_t i = 0; i < N; ++i)
        for (int32_t p = 0; p < nnz[i]; ++p)
            if (index[i * M + p] == i) nsum_add(&t, value[i * M + p]);
    return nsum_get(&t);
}

/*
 * Eq. 5 on ELLPACK-R: pattern unchanged except that a missing diagonal is inserted; the row is then put in
 * ascending column order.  Returns -1 if ok else the lowest overflowing row.
 */
int64_t oracle_rescale_ellpack(int64_t N, int32_t M, const double *hv, const int32_t *hi, const int32_t *hn,
                               double emin, double emax, double *xv, int32_t *xi, int32_t *xn)
{
    const double s = 1.0 / (emax - emin);
    int64_t bad = -1;
    for (int64_t i = 0; i < N; ++i) {
        int32_t n = hn[i], have_diag = 0;
        int32_t cnt = 0;
        for (int32_t p = 0; p < n; ++p) if (hi[i * M + p] == i) have_diag = 1;
        const int32_t total = n + (have_diag ? 0 : 1);
        if (total > M) { if (bad < 0) bad = i; xn[i] = 0; continue; }
        for (int32_t p = 0; p < n; ++p) xi[i * M + cnt++] = hi[i * M + p];
        if (!have_diag) xi[i * M + cnt++] = (int32_t)i;
        qsort(xi + i * M, (size_t)cnt, sizeof(int32_t), cmp_i32);
        for (int32_t q = 0; q < cnt; ++q) {
            const int32_t j = xi[i * M + q];
            double h = 0.0;
            for (int32_t p = 0; p < n; ++p) if (hi[i * M + p] == j) h = hv[i * M + p];
            xv[i * M + q] = (j == i) ? s * (emax - h) : -s * h;
        }
        for (int32_t q = cnt; q < M; ++q) { xi[i * M + q] = 0; xv[i * M + q] = 0.0; }
        xn[i] = cnt;
    }
    return bad;
}

/*
 * Thresholded row-wise product P = thr_tau(X X), Gustavson row merge with a dense accumulator:
 *   for p ascending over row i (k = idx[i][p]):  for q over row k:  acc[j] = fma(x_ik, x_kj, acc[j])
 *   keep (j, acc[j]) iff |acc[j]| >= tau or j == i, ascending j.
 * Rows of X must be in ascending column order.  Returns -1 if ok else the lowest row with more than M kept
 * entries (its stored row is truncated).  max_nnz (optional) receives the largest kept count.
 */
int64_t oracle_x2_ellpack(int64_t N, int32_t M, const double *xv, const int32_t *xi, const int32_t *xn, double tau,
                          double *pv, int32_t *pi, int32_t *pn, int32_t *max_nnz)
{
    int64_t bad = -1;
    int32_t mx = 0;
#pragma omp parallel
    {
        double *acc = (double *)calloc((size_t)N, sizeof(double));
        uint8_t *seen = (uint8_t *)calloc((size_t)N, 1);
        int32_t *touched = (int32_t *)malloc(sizeof(int32_t) * (size_t)N);
#pragma omp for schedule(dynamic, 64) reduction(max : mx)
        for (int64_t i = 0; i < N; ++i) {
            int32_t nt = 0;
            for (int32_t p = 0; p < xn[i]; ++p) {
                const int32_t k = xi[i * M + p];
                const double a = xv[i * M + p];
                for (int32_t q = 0; q < xn[k]; ++q) {
                    const int32_t j = xi[(int64_t)k * M + q];
                    if (!seen[j]) { seen[j] = 1; acc[j] = 0.0; touched[nt++] = j; }
                    acc[j] = fma(a, xv[(int64_t)k * M + q], acc[j]);
                }
            }
            qsort(touched, (size_t)nt, sizeof(int32_t), cmp_i32);
            int32_t cnt = 0;
            for (int32_t u = 0; u < nt; ++u) {
                const int32_t j = touched[u];
                if (fabs(acc[j]) >= tau || j == i) {
                    if (cnt < M) { pi[i * M + cnt] = j; pv[i * M + cnt] = acc[j]; }
                    ++cnt;
                }
                seen[j] = 0;
            }
            if (cnt > mx) mx = cnt;
            if (cnt > M) {
#pragma omp critical
                { if (bad < 0 || i < bad) bad = i; }
                cnt = M;
            }
            for (int32_t q = cnt; q < M; ++q) { pi[i * M + q] = 0; pv[i * M + q] = 0.0; }
            pn[i] = cnt;
        }
        free(acc); free(seen); free(touched);
    }
    if (max_nnz) *max_nnz = mx;
    return bad;
}

/* ||P - X||_F^2 over the union of the two patterns (absent = 0) and ||X||_F^2. */
static void ell_norms(int64_t N, int32_t M, const double *pv, const int32_t *pi, const int32_t *pn,
                      const double *xv, const int32_t *xi, const int32_t *xn, double *e2, double *x2, double *rowbuf)
{
#pragma omp parallel for schedule(static)
    for (int64_t i = 0; i < N; ++i) {
        nsum_t a = {0, 0}, b = {0, 0};
        int32_t p = 0, q = 0;
        while (p < pn[i] || q < xn[i]) {
            const int32_t jp = p < pn[i] ? pi[i * M + p] : INT32_MAX, jx = q < xn[i] ? xi[i * M + q] : INT32_MAX;
            double d;
            if (jp == jx) { d = pv[i * M + p] - xv[i * M + q]; ++p; ++q; }
            else if (jp < jx) { d = pv[i * M + p]; ++p; }
            else { d = -xv[i * M + q]; ++q; }
            nsum_add(&a, d * d);
        }
        for (q = 0; q < xn[i]; ++q) nsum_add(&b, xv[i * M + q] * xv[i * M + q]);
        rowbuf[2 * i] = nsum_get(&a);
        rowbuf[2 * i + 1] = nsum_get(&b);
    }
    nsum_t a = {0, 0}, b = {0, 0};
    for (int64_t i = 0; i < N; ++i) { nsum_add(&a, rowbuf[2 * i]); nsum_add(&b, rowbuf[2 * i + 1]); }
    *e2 = nsum_get(&a); *x2 = nsum_get(&b);
}

/*
 * X' = thr_tau(2X - P) on the union pattern, diagonal always kept.  Written to (ov, oi, on).
 * Returns -1 if ok else the lowest overflowing row.
 */
int64_t oracle_update_ellpack(int64_t N, int32_t M, const double *xv, const int32_t *xi, const int32_t *xn,
                              const double *pv, const int32_t *pi, const int32_t *pn, double tau,
                              double *ov, int32_t *oi, int32_t *on, int32_t *max_nnz)
{
    int64_t bad = -1;
    int32_t mx = 0;
    for (int64_t i = 0; i < N; ++i) {
        int32_t p = 0, q = 0, cnt = 0;
        while (p < pn[i] || q < xn[i]) {
            const int32_t jp = p < pn[i] ? pi[i * M + p] : INT32_MAX, jx = q < xn[i] ? xi[i * M + q] : INT32_MAX;
            int32_t j; double v;
            if (jp == jx) { j = jp; v = 2.0 * xv[i * M + q] - pv[i * M + p]; ++p; ++q; }
            else if (jp < jx) { j = jp; v = -pv[i * M + p]; ++p; }
            else { j = jx; v = 2.0 * xv[i * M + q]; ++q; }
            if (fabs(v) >= tau || j == i) {
                if (cnt < M) { oi[i * M + cnt] = j; ov[i * M + cnt] = v; }
                ++cnt;
            }
        }
        if (cnt > mx) mx = cnt;
        if (cnt > M) { if (bad < 0) bad = i; cnt = M; }
        for (int32_t u = cnt; u < M; ++u) { oi[i * M + u] = 0; ov[i * M + u] = 0.0; }
        on[i] = cnt;
    }
    if (max_nnz) *max_nnz = mx;
    return bad;
}

/*
 * Sparse SP2 (dense loop with lines 5, 6, 12 replaced by 5s, 6s, 12s).  Input rows may be in any
 * column order; D is returned in ascending column order in (dv, di, dn), all of size N*M / N.
 */
int oracle_sp2_ellpack_bounds(int64_t N, int32_t M, const double *hv, const int32_t *hi, const int32_t *hn, int32_t n_occ,
                              double tol, double tau, int32_t max_products, const double *bounds, double *dv, int32_t *di,
                              int32_t *dn, oracle_stats_t *st);
int oracle_sp2_ellpack(int64_t N, int32_t M, const double *hv, const int32_t *hi, const int32_t *hn, int32_t n_occ,
                       double tol, double tau, int32_t max_products, double *dv, int32_t *di, int32_t *dn,
                       oracle_stats_t *st)
{
    return oracle_sp2_ellpack_bounds(N, M, hv, hi, hn, n_occ, tol, tau, max_products, NULL, dv, di, dn, st);
}
/* bounds as in oracle_sp2_dense_bounds */
int oracle_sp2_ellpack_bounds(int64_t N, int32_t M, const double *hv, const int32_t *hi, const int32_t *hn, int32_t n_occ,
                              double tol, double tau, int32_t max_products, const double *bounds, double *dv, int32_t *di,
                              int32_t *dn, oracle_stats_t *st)
{
    stats_init(st);
    if (!hv || !hi || !hn || !dv || !di || !dn || N <= 0 || M < 1 || n_occ <= 0 || n_occ >= N || !(tol > 0) ||
        !(tau >= 0) || max_products < 1 || max_products > ORACLE_LOG_LEN)
        return st->status = -1;
    for (int64_t i = 0; i < N; ++i) if (hn[i] < 0 || hn[i] > M) return st->status = -1;
    double emin, emax;
    oracle_gershgorin_ellpack(N, M, hv, hi, hn, &emin, &emax);
    if (bounds) { emin = bounds[0]; emax = bounds[1]; }
    st->emin = emin; st->emax = emax;
    if (!(emax - emin > 0)) return st->status = -2;
    const size_t nm = (size_t)N * (size_t)M;
    double *xv = (double *)malloc(sizeof(double) * nm), *pv = (double *)malloc(sizeof(double) * nm),
           *yv = (double *)malloc(sizeof(double) * nm), *rowbuf = (double *)malloc(sizeof(double) * 2 * (size_t)N);
    int32_t *xi = (int32_t *)malloc(sizeof(int32_t) * nm), *pi = (int32_t *)malloc(sizeof(int32_t) * nm),
            *yi = (int32_t *)malloc(sizeof(int32_t) * nm);
    int32_t *xn = (int32_t *)malloc(sizeof(int32_t) * (size_t)N), *pn = (int32_t *)malloc(sizeof(int32_t) * (size_t)N),
            *yn = (int32_t *)malloc(sizeof(int32_t) * (size_t)N);
    int status = 2, m = 0;
    int64_t bad = oracle_rescale_ellpack(N, M, hv, hi, hn, emin, emax, xv, xi, xn);
    if (bad >= 0) { st->overflow_row = (int32_t)bad; status = -3; goto done; }
    for (m = 0;; ++m) {
        const double t = oracle_trace_ellpack(N, M, xv, xi, xn);
        int32_t mxp = 0, mxu = 0;
        bad = oracle_x2_ellpack(N, M, xv, xi, xn, tau, pv, pi, pn, &mxp);
        st->max_row_nnz[m] = mxp;
        st->trace[m] = t;
        if (bad >= 0) { st->overflow_row = (int32_t)bad; status = -3; break; }       /* item 9 */
        double e2, x2;
        ell_norms(N, M, pv, pi, pn, xv, xi, xn, &e2, &x2, rowbuf);
        st->idem[m] = sqrt(e2) / sqrt(x2);
        const int s = stop_rule(m, st->idem, tol, max_products);
        if (s >= 0) { status = s; break; }
        const int b = (t - (double)n_occ <= 0.0);
        st->branch[m] = (uint8_t)b;
        if (b) {
            bad = oracle_update_ellpack(N, M, xv, xi, xn, pv, pi, pn, tau, yv, yi, yn, &mxu);
            if (mxu > st->max_row_nnz[m]) st->max_row_nnz[m] = mxu;
            if (bad >= 0) { st->overflow_row = (int32_t)bad; status = -3; break; }
            memcpy(xv, yv, sizeof(double) * nm); memcpy(xi, yi, sizeof(int32_t) * nm);
            memcpy(xn, yn, sizeof(int32_t) * (size_t)N);
        } else {
            memcpy(xv, pv, sizeof(double) * nm); memcpy(xi, pi, sizeof(int32_t) * nm);
            memcpy(xn, pn, sizeof(int32_t) * (size_t)N);
        }
    }
    if (status >= 0) {
        memcpy(dv, xv, sizeof(double) * nm); memcpy(di, xi, sizeof(int32_t) * nm);
        memcpy(dn, xn, sizeof(int32_t) * (size_t)N);
    }
done:
    st->m_star = m; st->n_products = m + 1;
    free(xv); free(pv); free(yv); free(rowbuf); free(xi); free(pi); free(yi); free(xn); free(pn); free(yn);
    return st->status = status;
}

/* =============================================== ELLBLOCK ============================================= */
/*
 * ELLBLOCK ("a generalization of ELLPACK-R where each element is a block"): N = NB * bs rows in NB block rows of
 * bs x bs dense blocks, MB block slots per block row: block p of block row I is value[((I*MB + p)*bs + r)*bs + c],
 * r, c < bs (row-major inside the block), at block column index[I*MB + p]; nnz[I] blocks are stored.
 * Readings (items E1-E4 -- the paper gives the format's one-line definition only):
 *   E1. one uniform block size bs; N is a multiple of bs;
 *   E2. the threshold acts on BLOCKS: a block of thr(A) is kept iff its Frobenius norm sqrt(sum v^2) >= tau or it is a
 *       diagonal block (I == J) -- for bs = 1 this is the scalar rule |v| >= tau or j == i (sqrt(v*v) == |v| exactly);
 *   E3. accumulation order of a block product chain: blocks K of block row I ascending, and inside one block product
 *       acc[r][c] = fma(A[r][k], B[k][c], acc[r][c]) for k = 0 .. bs-1 ascending -- for bs = 1 the scalar oracle's
 *       order, so bs = 1 must reproduce oracle_x2_ellpack / oracle_sp2_ellpack bit for bit (pinned);
 *   E4. everything else (Gershgorin over stored entries, Eq. 5 with a missing diagonal BLOCK inserted, union-pattern
 *       norms, stop rules, D = X_{m*}, overflow of MB = failure -3) is the ELLPACK-R oracle's, applied per element.
 */
static double blk_norm(const double *b, int32_t bs)
{
    double s = 0.0;
    for (int32_t q = 0; q < bs * bs; ++q) s += b[q] * b[q];
    return sqrt(s);
}

int oracle_gershgorin_ellblock(int64_t NB, int32_t MB, int32_t bs, const double *value, const int32_t *index,
                               const int32_t *nnz, double *emin, double *emax)
{
    if (!value || !index || !nnz || NB <= 0 || MB < 1 || bs < 1) return -1;
    const int64_t bb = (int64_t)bs * bs;
    double lo = INFINITY, hi = -INFINITY;
    for (int64_t I = 0; I < NB; ++I)
        for (int32_t r = 0; r < bs; ++r) {
            nsum_t rad = {0, 0};
            double d = 0.0;
            for (int32_t p = 0; p < nnz[I]; ++p) {
                const double *b = value + (I * MB + p) * bb + (int64_t)r * bs;
                for (int32_t c = 0; c < bs; ++c) {
                    if (index[I * MB + p] == I && c == r) d = b[c];
                    else nsum_add(&rad, fabs(b[c]));
                }
            }
            const double g = nsum_get(&rad);
            if (d - g < lo) lo = d - g;
            if (d + g > hi) hi = d + g;
        }
    *emin = lo; *emax = hi;
    return 0;
}

double oracle_trace_ellblock(int64_t NB, int32_t MB, int32_t bs, const double *value, const int32_t *index,
                             const int32_t *nnz)
{
    const int64_t bb = (int64_t)bs * bs;
    nsum_t t = {0, 0};
    for (int64_t I = 0; I < NB; ++I)
        for (int32_t p = 0; p < nnz[I]; ++p)
            if (index[I * MB + p] == I)
                for (int32_t r = 0; r < bs; ++r) nsum_add(&t, value[(I * MB + p) * bb + (int64_t)r * bs + r]);
    return nsum_get(&t);
}

/* Eq. 5 per element; a missing diagonal block is inserted (H_II = 0); blocks in ascending block-column order.
 * Returns -1 if ok else the lowest block row that needs more than MB slots. */
int64_t oracle_rescale_ellblock(int64_t NB, int32_t MB, int32_t bs, const double *hv, const int32_t *hi, const int32_t *hn,
                                double emin, double emax, double *xv, int32_t *xi, int32_t *xn)
{
    const double s = 1.0 / (emax - emin);
    const int64_t bb = (int64_t)bs * bs;
    int64_t bad = -1;
    for (int64_t I = 0; I < NB; ++I) {
        const int32_t n = hn[I];
        int32_t have = 0, cnt = 0;
        for (int32_t p = 0; p < n; ++p) if (hi[I * MB + p] == I) have = 1;
        if (n + (have ? 0 : 1) > MB) { if (bad < 0) bad = I; xn[I] = 0; continue; }
        for (int32_t p = 0; p < n; ++p) xi[I * MB + cnt++] = hi[I * MB + p];
        if (!have) xi[I * MB + cnt++] = (int32_t)I;
        qsort(xi + I * MB, (size_t)cnt, sizeof(int32_t), cmp_i32);
        for (int32_t q = 0; q < cnt; ++q) {
            const int32_t J = xi[I * MB + q];
            const double *src = NULL;
            for (int32_t p = 0; p < n; ++p) if (hi[I * MB + p] == J) src = hv + (I * MB + p) * bb;
            double *dst = xv + (I * MB + q) * bb;
            for (int32_t r = 0; r < bs; ++r)
                for (int32_t c = 0; c < bs; ++c) {
                    const double h = src ? src[(int64_t)r * bs + c] : 0.0;
                    dst[(int64_t)r * bs + c] = (J == I && r == c) ? s * (emax - h) : -s * h;
                }
        }
        for (int32_t q = cnt; q < MB; ++q) { xi[I * MB + q] = 0; memset(xv + (I * MB + q) * bb, 0, sizeof(double) * bb); }
        xn[I] = cnt;
    }
    return bad;
}

/* P = thr_tau(X X) on blocks (readings E2, E3): Gustavson over block rows with a dense array of accumulator blocks. */
int64_t oracle_x2_ellblock(int64_t NB, int32_t MB, int32_t bs, const double *xv, const int32_t *xi, const int32_t *xn,
                           double tau, double *pv, int32_t *pi, int32_t *pn, int32_t *max_nnz)
{
    const int64_t bb = (int64_t)bs * bs;
    int64_t bad = -1;
    int32_t mx = 0;
#pragma omp parallel
    {
        double *acc = (double *)calloc((size_t)NB * (size_t)bb, sizeof(double));
        uint8_t *seen = (uint8_t *)calloc((size_t)NB, 1);
        int32_t *touched = (int32_t *)malloc(sizeof(int32_t) * (size_t)NB);
#pragma omp for schedule(dynamic, 16) reduction(max : mx)
        for (int64_t I = 0; I < NB; ++I) {
            int32_t nt = 0;
            for (int32_t p = 0; p < xn[I]; ++p) {
                const int32_t K = xi[I * MB + p];
                const double *A = xv + (I * MB + p) * bb;
                for (int32_t q = 0; q < xn[K]; ++q) {
                    const int32_t J = xi[(int64_t)K * MB + q];
                    const double *Bk = xv + ((int64_t)K * MB + q) * bb;
                    double *C = acc + (int64_t)J * bb;
                    if (!seen[J]) { seen[J] = 1; memset(C, 0, sizeof(double) * bb); touched[nt++] = J; }
                    for (int32_t r = 0; r < bs; ++r)
                        for (int32_t c = 0; c < bs; ++c) {
                            double v = C[(int64_t)r * bs + c];
                            for (int32_t k = 0; k < bs; ++k) v = fma(A[(int64_t)r * bs + k], Bk[(int64_t)k * bs + c], v);
                            C[(int64_t)r * bs + c] = v;
                        }
                }
            }
            qsort(touched, (size_t)nt, sizeof(int32_t), cmp_i32);
            int32_t cnt = 0;
            for (int32_t u = 0; u < nt; ++u) {
                const int32_t J = touched[u];
                const double *C = acc + (int64_t)J * bb;
                if (blk_norm(C, bs) >= tau || J == I) {
                    if (cnt < MB) { pi[I * MB + cnt] = J; memcpy(pv + (I * MB + cnt) * bb, C, sizeof(double) * bb); }
                    ++cnt;
                }
                seen[J] = 0;
            }
            if (cnt > mx) mx = cnt;
            if (cnt > MB) {
#pragma omp critical
                { if (bad < 0 || I < bad) bad = I; }
                cnt = MB;
            }
            for (int32_t q = cnt; q < MB; ++q) { pi[I * MB + q] = 0; memset(pv + (I * MB + q) * bb, 0, sizeof(double) * bb); }
            pn[I] = cnt;
        }
        free(acc); free(seen); free(touched);
    }
    if (max_nnz) *max_nnz = mx;
    return bad;
}

/* ||P - X||_F^2 over the union of the two block patterns (an absent block = 0) and ||X||_F^2 */
static void ellblock_norms(int64_t NB, int32_t MB, int32_t bs, const double *pv, const int32_t *pi, const int32_t *pn,
                           const double *xv, const int32_t *xi, const int32_t *xn, double *e2, double *x2)
{
    const int64_t bb = (int64_t)bs * bs;
    nsum_t a = {0, 0}, b = {0, 0};
    for (int64_t I = 0; I < NB; ++I) {
        nsum_t ra = {0, 0}, rb = {0, 0};
        int32_t p = 0, q = 0;
        while (p < pn[I] || q < xn[I]) {
            const int32_t jp = p < pn[I] ? pi[I * MB + p] : INT32_MAX, jx = q < xn[I] ? xi[I * MB + q] : INT32_MAX;
            const double *P = (jp <= jx) ? pv + (I * MB + p) * bb : NULL, *X = (jx <= jp) ? xv + (I * MB + q) * bb : NULL;
            for (int64_t t = 0; t < bb; ++t) {
                const double d = (P ? P[t] : 0.0) - (X ? X[t] : 0.0);
                nsum_add(&ra, d * d);
            }
            if (P) ++p;
            if (X) ++q;
        }
        for (q = 0; q < xn[I]; ++q)
            for (int64_t t = 0; t < bb; ++t) nsum_add(&rb, xv[(I * MB + q) * bb + t] * xv[(I * MB + q) * bb + t]);
        nsum_add(&a, nsum_get(&ra));
        nsum_add(&b, nsum_get(&rb));
    }
    *e2 = nsum_get(&a); *x2 = nsum_get(&b);
}

/* X' = thr_tau(2X - P) on the union of the block patterns; diagonal blocks always kept. */
int64_t oracle_update_ellblock(int64_t NB, int32_t MB, int32_t bs, const double *xv, const int32_t *xi, const int32_t *xn,
                               const double *pv, const int32_t *pi, const int32_t *pn, double tau, double *ov, int32_t *oi,
                               int32_t *on, int32_t *max_nnz)
{
    const int64_t bb = (int64_t)bs * bs;
    int64_t bad = -1;
    int32_t mx = 0;
    double *tmp = (double *)malloc(sizeof(double) * (size_t)bb);
    for (int64_t I = 0; I < NB; ++I) {
        int32_t p = 0, q = 0, cnt = 0;
        while (p < pn[I] || q < xn[I]) {
            const int32_t jp = p < pn[I] ? pi[I * MB + p] : INT32_MAX, jx = q < xn[I] ? xi[I * MB + q] : INT32_MAX;
            const double *P = (jp <= jx) ? pv + (I * MB + p) * bb : NULL, *X = (jx <= jp) ? xv + (I * MB + q) * bb : NULL;
            const int32_t J = jp < jx ? jp : jx;
            for (int64_t t = 0; t < bb; ++t) tmp[t] = X ? (P ? 2.0 * X[t] - P[t] : 2.0 * X[t]) : -P[t];
            if (P) ++p;
            if (X) ++q;
            if (blk_norm(tmp, bs) >= tau || J == I) {
                if (cnt < MB) { oi[I * MB + cnt] = J; memcpy(ov + (I * MB + cnt) * bb, tmp, sizeof(double) * bb); }
                ++cnt;
            }
        }
        if (cnt > mx) mx = cnt;
        if (cnt > MB) { if (bad < 0) bad = I; cnt = MB; }
        for (int32_t u = cnt; u < MB; ++u) { oi[I * MB + u] = 0; memset(ov + (I * MB + u) * bb, 0, sizeof(double) * bb); }
        on[I] = cnt;
    }
    free(tmp);
    if (max_nnz) *max_nnz = mx;
    return bad;
}

/* SP2 on ELLBLOCK: the ELLPACK-R loop (oracle_sp2_ellpack_bounds) with the block operations above. */
int oracle_sp2_ellblock(int64_t NB, int32_t MB, int32_t bs, const double *hv, const int32_t *hi, const int32_t *hn,
                        int32_t n_occ, double tol, double tau, int32_t max_products, double *dv, int32_t *di, int32_t *dn,
                        oracle_stats_t *st)
{
    stats_init(st);
    if (!hv || !hi || !hn || !dv || !di || !dn || NB <= 0 || MB < 1 || bs < 1 || n_occ <= 0 || n_occ >= NB * bs ||
        !(tol > 0) || !(tau >= 0) || max_products < 1 || max_products > ORACLE_LOG_LEN)
        return st->status = -1;
    for (int64_t I = 0; I < NB; ++I) if (hn[I] < 0 || hn[I] > MB) return st->status = -1;
    double emin, emax;
    oracle_gershgorin_ellblock(NB, MB, bs, hv, hi, hn, &emin, &emax);
    st->emin = emin; st->emax = emax;
    if (!(emax - emin > 0)) return st->status = -2;
    const size_t nm = (size_t)NB * (size_t)MB, nv = nm * (size_t)bs * (size_t)bs;
    double *xv = (double *)malloc(sizeof(double) * nv), *pv = (double *)malloc(sizeof(double) * nv),
           *yv = (double *)malloc(sizeof(double) * nv);
    int32_t *xi = (int32_t *)malloc(sizeof(int32_t) * nm), *pi = (int32_t *)malloc(sizeof(int32_t) * nm),
            *yi = (int32_t *)malloc(sizeof(int32_t) * nm);
    int32_t *xn = (int32_t *)malloc(sizeof(int32_t) * (size_t)NB), *pn = (int32_t *)malloc(sizeof(int32_t) * (size_t)NB),
            *yn = (int32_t *)malloc(sizeof(int32_t) * (size_t)NB);
    int status = 2, m = 0;
    int64_t bad = oracle_rescale_ellblock(NB, MB, bs, hv, hi, hn, emin, emax, xv, xi, xn);
    if (bad >= 0) { st->overflow_row = (int32_t)bad; status = -3; goto done; }
    for (m = 0;; ++m) {
        const double t = oracle_trace_ellblock(NB, MB, bs, xv, xi, xn);
        int32_t mxp = 0, mxu = 0;
        bad = oracle_x2_ellblock(NB, MB, bs, xv, xi, xn, tau, pv, pi, pn, &mxp);
        st->max_row_nnz[m] = mxp;
        st->trace[m] = t;
        if (bad >= 0) { st->overflow_row = (int32_t)bad; status = -3; break; }
        double e2, x2;
        ellblock_norms(NB, MB, bs, pv, pi, pn, xv, xi, xn, &e2, &x2);
        st->idem[m] = sqrt(e2) / sqrt(x2);
        const int s = stop_rule(m, st->idem, tol, max_products);
        if (s >= 0) { status = s; break; }
        const int b = (t - (double)n_occ <= 0.0);
        st->branch[m] = (uint8_t)b;
        if (b) {
            bad = oracle_update_ellblock(NB, MB, bs, xv, xi, xn, pv, pi, pn, tau, yv, yi, yn, &mxu);
            if (mxu > st->max_row_nnz[m]) st->max_row_nnz[m] = mxu;
            if (bad >= 0) { st->overflow_row = (int32_t)bad; status = -3; break; }
            memcpy(xv, yv, sizeof(double) * nv); memcpy(xi, yi, sizeof(int32_t) * nm);
            memcpy(xn, yn, sizeof(int32_t) * (size_t)NB);
        } else {
            memcpy(xv, pv, sizeof(double) * nv); memcpy(xi, pi, sizeof(int32_t) * nm);
            memcpy(xn, pn, sizeof(int32_t) * (size_t)NB);
        }
    }
    if (status >= 0) {
        memcpy(dv, xv, sizeof(double) * nv); memcpy(di, xi, sizeof(int32_t) * nm);
        memcpy(dn, xn, sizeof(int32_t) * (size_t)NB);
    }
done:
    st->m_star = m; st->n_products = m + 1;
    free(xv); free(pv); free(yv); free(xi); free(pi); free(yi); free(xn); free(pn); free(yn);
    return st->status = status;
}

int oracle_omp_threads(void)
{
    int n = 1;
#ifdef _OPENMP
#pragma omp parallel
    {
#pragma omp single
        n = omp_get_num_threads();
    }
#endif
    return n;
}
