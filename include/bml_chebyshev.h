/*
 * bml_chebyshev.h -- C ABI of libbmlsp2.so, part 2: the Chebyshev / Paterson-Stockmeyer Fermi-operator expansion of
 * arxiv 2401.13772 section IV.B on one B200 (sm_100a), dense FP64.
 *
 *   D = f_mu(H) ~ sum_{n=0}^{L} c_n T_n(H~)                                   Eq. 8
 *               = S_0 + T_k (S_1 + T_k (S_2 + ... + T_k S_{m-1}))             Eq. 10,  L + 1 = k m
 *   S_j = sum_{i<k} d_{i,j} T_i                                               Eq. 12
 *   T_i = 2 T_a T_b - T_{a-b},  a = ceil(i/2), b = floor(i/2)                 Eq. 11, 13, 14
 *
 * k + m - 2 matrix products instead of the L - 1 of the recursion Eq. 9.  Every product is of two polynomials of the
 * same symmetric H~, so it is symmetric: only the tiles on and above the diagonal are computed and mirrored, exactly
 * as in the SP2 kernels.  The T_i of one doubling level are independent ("can therefore be computed in parallel",
 * P:241); where the paper uses one stream per product, this library runs each level as ONE grouped launch.
 *
 * Conventions (pointers, streams, ownership, status codes) are those of bml_sp2.h.  Readings of the paper that this
 * interface fixes (items C1-C5): H~ maps the Gershgorin interval onto [-1, 1]; f_mu(eps) =
 * 1 / (1 + exp(beta (eps - mu))) with mu given by the caller (Fig. 3); c_n by Chebyshev-Gauss quadrature on
 * 2 (L + 1) nodes; d_{i,j} by repeated division of the series by T_k using Eq. 11.
 */
#ifndef BML_CHEBYSHEV_H
#define BML_CHEBYSHEV_H

#include "bml_sp2.h"

#ifdef __cplusplus
extern "C" {
#endif

#define BML_CHEB_MAX_K 32          /* 2 <= k <= 32                                              */
#define BML_CHEB_MAX_M 32          /* 1 <= m <= 32                                              */
#define BML_CHEB_MAX_TERMS 1024    /* k m = L + 1 <= 1024                                       */
#define BML_SYMM_MAX_JOBS 16       /* products per grouped launch                               */

typedef struct {
    double  mu;      /* chemical potential, in the units of H                                                     */
    double  beta;    /* 1 / (k_B T) > 0, in inverse units of H                                                    */
    int32_t k, m;    /* Eq. 10: L + 1 = k m; k polynomials T_0..T_{k-1} per partial sum S_j, m partial sums       */
    uint32_t flags;  /* BML_SP2_FLAG_CHECK_SYMMETRY                                                               */
    uint32_t pad;
} bml_cheb_params_t;

/* Filled on the HOST when bml_chebyshev_dense returns (it synchronises the stream once, at the end). */
typedef struct {
    int32_t status;        /* = return value                                                                      */
    int32_t n_products;    /* matrix products executed = (k - 1) + (m - 1)                                        */
    int32_t n_launches;    /* product-kernel launches (one per doubling level + one per nesting step of Eq. 10)   */
    int32_t L;             /* k m - 1                                                                             */
    double  emin, emax;    /* Gershgorin bounds used for H~                                                       */
    double  trace;         /* tr D = number of occupied states at (mu, beta)                                      */
    double  c[BML_CHEB_MAX_TERMS];   /* c_0..c_L of Eq. 8, as computed on the device                              */
    double  d[BML_CHEB_MAX_TERMS];   /* d_{i,j} of Eq. 10 at d[j * k + i]                                         */
} bml_cheb_stats_t;

/*
 * D <- sum_n c_n T_n(H~) ~ f_mu(H) by Eq. 10-14.
 * H: dense symmetric N x N, never written.  D: dense N x N (any ld >= N), must not alias H; both triangles written,
 * bitwise symmetric.  d_workspace: DEVICE scratch of >= bml_chebyshev_workspace_bytes(N, k, m) bytes, 1024-byte
 * aligned: (k + m) matrices of N x ld(N) doubles plus O(N) -- 8 GB at N = 8192, k = m = 8.
 * stats: HOST, may be NULL.  No host round trip inside the call: bounds, c_n and d_{i,j} are computed and consumed on
 * the device.  For N <= 2048 on a non-default stream the (static) launch sequence is captured once per argument set and
 * replayed as a CUDA graph by later calls with the same pointers, shapes and parameters; results are identical.
 * Returns BML_OK, -1 (also for k, m out of range or beta <= 0), -2, -4, -5.
 */
BML_API size_t bml_chebyshev_workspace_bytes(int64_t N, int32_t k, int32_t m);
BML_API int bml_chebyshev_dense(const bml_matrix_t *H, const bml_cheb_params_t *p, bml_matrix_t *D, void *d_workspace,
                                size_t workspace_bytes, bml_cheb_stats_t *stats, void *cuda_stream);

/*
 * The one matrix operation Eq. 10, 13 and 14 are made of, exported for per-kernel parity tests and timing:
 *     Out_q <- alpha_q A_q B_q + beta_q C_q + gamma_q I,   q = 0..n_jobs-1,   one grouped launch.
 * A_q, B_q: symmetric and COMMUTING (polynomials of one matrix), so that A_q B_q is symmetric; the kernel computes
 * tiles I <= J as A[I,:] B[J,:]^T and mirrors them.  C_q may be NULL (then beta_q is ignored) or equal to Out_q.
 * All matrices of the call: dense N x N, the same ld (a multiple of 16 elements), 128-byte aligned, and they must lie
 * at multiples of `slot_elems` (>= N ld, a multiple of 16) elements from `base` -- the kernel addresses operands as
 * slices of ONE 3-D tensor map (column, row, slot).  Out_q must differ from every A, B of the call.
 * a_slot[q], b_slot[q], c_slot[q] (-1 = none), out_slot[q]: slot numbers in [0, n_slots).
 * d_workspace >= bml_symm_ab_workspace_bytes() bytes, 1024-byte aligned.  Asynchronous.  Returns 0, -1 or -4.
 */
BML_API size_t bml_symm_ab_workspace_bytes(void);
BML_API int bml_symm_ab_dense(double *base, int64_t N, int64_t ld, int64_t slot_elems, int32_t n_slots, int32_t n_jobs,
                              const int32_t *a_slot, const int32_t *b_slot, const int32_t *c_slot,
                              const int32_t *out_slot, const double *alpha, const double *beta, const double *gamma,
                              void *d_workspace, size_t workspace_bytes, void *cuda_stream);

#ifdef __cplusplus
}
#endif
#endif /* BML_CHEBYSHEV_H */
