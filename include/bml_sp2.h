/*
 * bml_sp2.h -- C ABI of libbmlsp2.so: the SP2 density-matrix hot path of arxiv 2401.13772 on one B200 (sm_100a).
 *
 * Citations are lines of the paper text PAPER.md ("P:<line>") with the section / equation / listing they fall in.
 *
 *   X_0 = (e_max I - H) / (e_max - e_min)                 Eq. 5, Listing 2
 *   X_{m+1} = X_m^2           if tr X_m >  N_occ          Eq. 6
 *   X_{m+1} = 2 X_m - X_m^2   if tr X_m <= N_occ          Eq. 7; "<=" from Listing 2
 *   D = X_n
 *
 * The library owns no device memory: every pointer in a bml_matrix_t and every workspace is a DEVICE pointer
 * owned by the caller (the Python binding uses torch tensors), borrowed for the duration of the call (the paper's
 * "persistent data allocation on the device", Listing 3, without its allocator).  All work is enqueued on
 * the CUDA stream passed as `cuda_stream` (a cudaStream_t cast to void*; NULL = legacy default stream).  There is no
 * CPU fallback: every entry point returns BML_ERR_CUDA if no sm_100 device / kernel image is usable.
 *
 * Return values (no exceptions, no abort, nothing printed):
 *    0  BML_OK                converged: e_m < idem_tol                                   (stop rule S1)
 *    1  BML_NOISE_FLOOR       stagnated on the truncation / round-off floor; D is valid   (stop rule S2)
 *    2  BML_MAX_PRODUCTS      max_products reached; D = last iterate, not converged       (stop rule S3)
 *   -1  BML_ERR_INVALID       bad argument (NULL, N <= 0, n_occ not in (0,N), tol <= 0, ld < N, M < 1, workspace
 *                             too small, D aliases H, max_products not in [1, BML_SP2_LOG_LEN], M > BML_ELL_MAX_M)
 *   -2  BML_ERR_DEGENERATE    e_max - e_min <= 0 (H = c I)
 *   -3  BML_ERR_ELL_OVERFLOW  an ELLPACK-R row needs more than M slots after thresholding; "may reach the limit M
 *                             and lead to a failure".  stats->overflow_row = lowest such row.
 *   -4  BML_ERR_CUDA          CUDA runtime error (launch failure, no device, ...)
 *   -5  BML_ERR_NOT_SYMMETRIC H is not bitwise symmetric (checked only with BML_SP2_FLAG_CHECK_SYMMETRY)
 *   -6  BML_ERR_ACC_CAPACITY  ELLPACK: a row of X*X touched more distinct columns BEFORE thresholding than the
 *                             on-chip accumulator holds (BML_ELL_ACC_SLOTS); stats->overflow_row = that row.
 * On a negative return D is undefined (bml_sp2_*: left untouched).
 */
#ifndef BML_SP2_H
#define BML_SP2_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#if defined(__GNUC__)
#define BML_API __attribute__((visibility("default")))
#else
#define BML_API
#endif

#define BML_SP2_LOG_LEN 128     /* max number of X^2 products per solve (length of the per-product logs)          */
#define BML_ELL_MAX_M 1024      /* largest ELLPACK-R row capacity M the sparse kernels are built for               */
#define BML_ELL_ACC_SLOTS 4096  /* per-row hash accumulator slots of the sparse X^2 kernel (pre-threshold fill)    */

enum {
    BML_OK = 0, BML_NOISE_FLOOR = 1, BML_MAX_PRODUCTS = 2,
    BML_ERR_INVALID = -1, BML_ERR_DEGENERATE = -2, BML_ERR_ELL_OVERFLOW = -3, BML_ERR_CUDA = -4,
    BML_ERR_NOT_SYMMETRIC = -5, BML_ERR_ACC_CAPACITY = -6
};

typedef enum { BML_DENSE = 0, BML_ELLPACK = 1 } bml_matrix_type_t;

/*
 * Matrix descriptor in the spirit of Listing 1 (`bml_matrix_ellpack_t`: N, M, value, index, nnz).
 * The struct itself lives on the HOST; the three arrays are DEVICE pointers, borrowed.
 *   dense  : value[i*ld + j], row-major, real double, ld >= N; index = nnz = NULL, M ignored.
 *   ellpack: ELLPACK-R: entry p (0 <= p < nnz[i]) of row i is value[i*M + p] at column index[i*M + p]
 *            (row-major, P:311 ROWMAJOR); slots p >= nnz[i] are ignored on input and written as (0.0, 0) on output.
 *            Input rows: column indices unique, in [0,N), in ANY order ("the ELLPACK-R format is unsorted").
 *            Output rows (D and every intermediate iterate): ascending column index.  ld ignored.
 */
typedef struct {
    int32_t  type;    /* bml_matrix_type_t */
    int32_t  M;       /* ellpack: slots per row (1 <= M <= BML_ELL_MAX_M)      */
    int64_t  N;       /* rows = columns                                         */
    int64_t  ld;      /* dense: leading dimension in elements                   */
    double  *value;   /* DEVICE                                                 */
    int32_t *index;   /* DEVICE, ellpack only                                   */
    int32_t *nnz;     /* DEVICE, ellpack only                                   */
} bml_matrix_t;

/* Problem statement of the paper: occupation (`nel`), tolerance ("check for convergence"),
 * drop threshold (`tau`; "discard small matrix elements"). */
typedef struct {
    int32_t  n_occ;         /* number of occupied orbitals, 0 < n_occ < N                                       */
    int32_t  max_products;  /* cap on X^2 products (Listing 2 `maxiter`), 1..BML_SP2_LOG_LEN             */
    double   idem_tol;      /* tolerance on e_m = ||X_m^2 - X_m||_F / ||X_m||_F                                 */
    double   drop_tol;      /* tau: keep |v| >= tau or the diagonal (ellpack only; 0 keeps everything)          */
    int32_t  precision;     /* dense only: 0 = FP64 DMMA products; 1, 2 = mixed precision: tcgen05 products of 16-bit
                               planes of X with FP32 TMEM accumulation promoted to FP64 every 512 columns of K, FP64
                               traces, norms and updates.  1 = two FP16 planes, X = Xh + 2^-11 Xl (3 cross terms);
                               2 = three BF16 planes, X = Xh + Xm + Xl (6 cross terms)                            */
    uint32_t flags;         /* BML_SP2_FLAG_* */
} bml_sp2_params_t;

#define BML_SP2_FLAG_CHECK_SYMMETRY 1u /* verify H == H^T bitwise first (one extra pass); else -5 is never returned */
/* Optional tighter spectral bounds for Eq. 5 (the paper's Eq. 5 uses the exact extreme eigenvalues; the
 * default here is Gershgorin): K steps (8..64) of the Lanczos recursion, see bml_lanczos_bounds below.
 * Usage: flags = BML_SP2_FLAG_LANCZOS_BOUNDS(24).  SP2 then needs fewer products (31 -> 24 on the long-range models). */
#define BML_SP2_FLAG_LANCZOS_BOUNDS(K) (((uint32_t)(K) & 0xffu) << 8)

/* Per-solve record, filled on the HOST when bml_sp2_* returns (the call synchronises the stream once, at the end). */
typedef struct {
    int32_t status;        /* = return value                                                                    */
    int32_t n_products;    /* number of X^2 products evaluated = m_star + 1                                     */
    int32_t m_star;        /* index of the returned iterate D = X_{m_star}; branch[0..m_star-1] are recorded    */
    int32_t overflow_row;  /* ellpack failures -3 / -6: the offending row, else -1                              */
    double  emin, emax;    /* Gershgorin bounds used in Eq. 5                                                   */
    uint8_t branch[BML_SP2_LOG_LEN];       /* b_m: 1 => X <- 2X - X^2 (Eq. 7), 0 => X <- X^2 (Eq. 6)            */
    double  trace[BML_SP2_LOG_LEN];        /* tr X_m                                                            */
    double  idem[BML_SP2_LOG_LEN];         /* e_m                                                               */
    int32_t max_row_nnz[BML_SP2_LOG_LEN];  /* ellpack: max stored row length of P_m and X_{m+1}; dense: 0       */
} bml_sp2_stats_t;

/*
 * Gershgorin circle bounds of a symmetric matrix (the BML op named at P:452; consumed as `emin`, `emax` by
 * Listing 2):  e_min = min_i (H_ii - sum_{j!=i} |H_ij|),  e_max = max_i (H_ii + sum_{j!=i} |H_ij|).
 * ellpack: over stored entries, a missing diagonal counts as 0.
 * d_bounds: DEVICE double[2] <- {e_min, e_max}.  d_workspace: DEVICE scratch of >= bml_gershgorin_workspace_bytes(N)
 * bytes.  Asynchronous on `cuda_stream`.  Returns 0, -1 or -4.
 */
BML_API size_t bml_gershgorin_workspace_bytes(int64_t N);
BML_API int bml_gershgorin(const bml_matrix_t *H, double *d_bounds, void *d_workspace, size_t workspace_bytes,
                   void *cuda_stream);

/*
 * Tighter spectral bounds (optional, readings B1-B3): `steps` steps of the Lanczos recursion on H from the
 * counter-based start vector u_i = 2 (splitmix64(seed + i) >> 11) 2^-53 - 1, Ritz values theta_i of the tridiagonal
 * matrix, e_max = min(Gershgorin, theta_max + |beta_K s_K,max| + pad), e_min = max(Gershgorin, theta_min - |beta_K
 * s_K,min| - pad), pad = 1% of the Ritz width.  Never looser than bml_gershgorin.  Enclosure of the spectrum is the
 * usual property of the safeguarded k-step Lanczos estimate, not a theorem: with steps >= 8 it held for every model and
 * seed tried (with 2-4 steps an outlying band can be missed, so steps < 8 is rejected); if it fails SP2 does not
 * converge and ends with BML_MAX_PRODUCTS.  steps in 8..64.  H dense or ellpack.
 * d_bounds: DEVICE double[2] <- {e_min, e_max}.  d_workspace >= bml_lanczos_bounds_workspace_bytes(N), 8-byte aligned.
 * One persistent cooperative launch (one CTA per SM) runs the whole recursion; the device must support cooperative
 * launches (else -4).  Asynchronous.  Returns 0, -1 or -4.
 */
BML_API size_t bml_lanczos_bounds_workspace_bytes(int64_t N);
BML_API int bml_lanczos_bounds(const bml_matrix_t *H, int32_t steps, uint64_t seed, double *d_bounds, void *d_workspace,
                       size_t workspace_bytes, void *cuda_stream);

/*
 * tr A = sum_i A_ii (`bml_trace`, Listing 2).  ellpack: sum of stored diagonal entries.
 * d_trace: DEVICE double[1].  Fixed summation order (bit-reproducible).  Asynchronous.  Returns 0, -1 or -4.
 */
BML_API int bml_trace(const bml_matrix_t *A, double *d_trace, void *cuda_stream);

/*
 * SP2 (Eq. 5-7, Listing 2) with the readings listed in DESIGN.md ("Readings of the paper"):
 *   bounds by bml_gershgorin; per product m: e_m = ||X_m^2 - X_m||_F / ||X_m||_F; stop rules S1 (e_m < idem_tol),
 *   S2 (m >= 2, e_m < 1e-2, e_m >= e_{m-2}), S3 (m + 1 == max_products); branch b_m = [tr X_m - n_occ <= 0];
 *   D = X_{m*}, the iterate that was tested.
 * H: input, never written.  D: output, same type (and for ellpack the same M) as H; must not alias H.
 * d_workspace: DEVICE scratch, >= bml_sp2_workspace_bytes(H, p) bytes, 1024-byte aligned.
 * stats: HOST.  Non-NULL: the call synchronises the stream once, at its end, to read the control block back, and returns
 *   the solve's status.  While it enqueues, the host also waits on an event behind every batch of 8 product launches, one
 *   batch BEHIND the one in flight (this only bounds how many launches are issued after the stop rule fired; the device
 *   never waits for the host).  NULL: the call is FULLY ASYNCHRONOUS -- all max_products launches are enqueued (those
 *   behind the device-side stop flag exit at once), the host never waits, nothing is copied back, and the return value
 *   is 0 / -1 / -4 for "enqueued" only; the verdict stays in the control block at the start of d_workspace and is read
 *   later with bml_sp2_read_stats (which synchronises).  On a negative status D is left untouched.
 * The whole solve is enqueued without any host round trip per product: the branch bit, the stop test and the
 * ping-pong buffer selection live in a device-resident control block.
 * Cached state.  Dense FP64, N <= 1024, not on the legacy default stream: the launches up to and including the first
 *   batch of products are captured once per argument set and replayed as a CUDA graph by later calls with the same
 *   device, pointers, shapes and parameters; results are identical.  The cache (4 graphs per host thread; the same
 *   holds for bml_chebyshev_dense) remembers the caller's H / workspace POINTERS as lookup keys -- they are compared,
 *   never dereferenced by the host, and a replay only touches the arrays of the call that replays it -- until
 *   bml_sp2_release_cached() is called on that thread.  Nothing else outlives a call.
 */
BML_API size_t bml_sp2_workspace_bytes(const bml_matrix_t *H, const bml_sp2_params_t *p);
BML_API int bml_sp2_dense(const bml_matrix_t *H, const bml_sp2_params_t *p, bml_matrix_t *D, void *d_workspace,
                  size_t workspace_bytes, bml_sp2_stats_t *stats, void *cuda_stream);
BML_API int bml_sp2_ellpack(const bml_matrix_t *H, const bml_sp2_params_t *p, bml_matrix_t *D, void *d_workspace,
                    size_t workspace_bytes, bml_sp2_stats_t *stats, void *cuda_stream);
/* Fill `stats` from the control block of the last bml_sp2_* call that used `d_workspace` (for calls made with
 * stats == NULL).  Synchronises `cuda_stream`.  Returns the solve's status, or -1 / -4. */
BML_API int bml_sp2_read_stats(const void *d_workspace, bml_sp2_stats_t *stats, void *cuda_stream);
/* Destroy the calling thread's cached CUDA graphs (see "Cached state" above).  Safe to call at any time. */
BML_API void bml_sp2_release_cached(void);

/*
 * One product of the hot loop, exported for per-kernel parity tests and per-kernel timing.
 *
 * bml_x2_dense: the fused symmetric-square kernel (steps D3 + D4 of DESIGN.md) on a caller-supplied iterate.
 *   X: dense N x N, bitwise symmetric, ld a multiple of 16 elements (precision 1, 2: ld == 16 * ceil(N / 16) exactly,
 *   the 16-bit planes in the workspace are sized for that pitch; anything else is -1), value 128-byte aligned.  Xnext: same shape/ld
 *   <- branch ? 2X - X*X : X*X  (Eq. 7 / Eq. 6), both triangles written.  d_sums: DEVICE double[4] <-
 *   { tr(X*X), ||X*X - X||_F^2, ||X||_F^2, tr(Xnext) }.  precision (0, 1, 2) as in bml_sp2_params_t.
 *   d_workspace >= bml_x2_dense_workspace_bytes(N, precision).
 * bml_x2_ellpack: the thresholded row-wise product + update (steps S3 + S4) on a caller-supplied iterate whose rows
 *   are in ascending column order.  Xnext <- branch ? thr(2X - thr(X*X)) : thr(X*X).  d_sums: DEVICE double[4] <-
 *   { tr thr(X*X), ||thr(X*X) - X||_F^2 over the union pattern, ||X||_F^2, tr(Xnext) };
 *   d_info: DEVICE int32[4] <- { lowest row with > M kept entries or INT32_MAX, lowest row exceeding the accumulator
 *   or INT32_MAX, max kept row length, 0 }.  d_workspace >= bml_x2_ellpack_workspace_bytes(N, M).
 *   X must be bitwise symmetric (X_ij == X_ji): row i is accumulated for the columns j >= i only and mirrored.
 * Asynchronous.  Return 0, -1 or -4.
 */
BML_API size_t bml_x2_dense_workspace_bytes(int64_t N, int32_t precision);
BML_API int bml_x2_dense(const bml_matrix_t *X, bml_matrix_t *Xnext, int32_t branch, int32_t precision, double *d_sums,
                 void *d_workspace, size_t workspace_bytes, void *cuda_stream);
BML_API size_t bml_x2_ellpack_workspace_bytes(int64_t N, int32_t M);
BML_API int bml_x2_ellpack(const bml_matrix_t *X, bml_matrix_t *Xnext, int32_t branch, double drop_tol, double *d_sums,
                   int32_t *d_info, void *d_workspace, size_t workspace_bytes, void *cuda_stream);

BML_API const char *bml_status_string(int status);
/* "major.minor.patch (sm_100a)" */
BML_API const char *bml_version(void);

#ifdef __cplusplus
}
#endif
#endif /* BML_SP2_H */
