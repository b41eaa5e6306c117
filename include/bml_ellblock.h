/*
 * bml_ellblock.h -- C ABI of libbmlsp2.so, part 4: thresholded SP2 on ELLBLOCK, the block-sparse format of BML
 * ("ELLBLOCK is a generalization of ELLPACK-R where each element is a block"), with the block products
 * on the FP64 tensor cores.  Conventions (ownership, streams, statuses) as in bml_sp2.h.
 *
 * The paper gives the format one sentence; the readings this interface fixes (DESIGN.md "Readings" E1-E4):
 *   E1. one uniform block size bs in {4, 8, 16}; N = NB * bs (pad H with decoupled rows if N is not a multiple);
 *   E2. the threshold acts on BLOCKS: a block is kept iff its Frobenius norm >= drop_tol or it is a diagonal block
 *       (bs = 1 would be the scalar rule of bml_sp2_ellpack);
 *   E3. X must be symmetric as a matrix (block (J, I) = transpose of block (I, J), both stored or both absent);
 *   E4. everything else -- Gershgorin bounds over stored entries, Eq. 5 with a missing diagonal block inserted, the
 *       idempotency measure over the union of the block patterns, stop rules S1-S3, D = X_{m*}, more than MB blocks
 *       in a block row = failure -3 (stats->overflow_row = the BLOCK row) -- is bml_sp2_ellpack's, per element.
 * stats->max_row_nnz counts BLOCKS per block row.  Status -6 (BML_ERR_ACC_CAPACITY): the upper part (J >= I) of a block
 * row of X*X reaches more than 8 * MB (at most 8192) distinct block columns BEFORE thresholding, the capacity of the
 * candidate lists.
 */
#ifndef BML_ELLBLOCK_H
#define BML_ELLBLOCK_H

#include "bml_sp2.h"

#ifdef __cplusplus
extern "C" {
#endif

/*
 * ELLBLOCK descriptor (host struct, DEVICE arrays, borrowed): block p (0 <= p < nnz[I]) of block row I is the bs x bs
 * row-major array value[((I*MB + p)*bs + r)*bs + c] at block column index[I*MB + p].  Input block rows in any order;
 * every iterate and D in ascending block-column order, unused slots (0, zero block).  NB <= 2^19.
 */
typedef struct {
    int32_t  bs;      /* block edge: 4, 8 or 16                                  */
    int32_t  MB;      /* block slots per block row                               */
    int64_t  NB;      /* block rows = block columns; N = NB * bs                 */
    double  *value;   /* DEVICE, NB * MB * bs * bs                               */
    int32_t *index;   /* DEVICE, NB * MB                                         */
    int32_t *nnz;     /* DEVICE, NB                                              */
} bml_ellblock_t;

/* bml_gershgorin / bml_trace on ELLBLOCK (Listing 2).  Asynchronous.  Return 0, -1, -4. */
BML_API size_t bml_gershgorin_ellblock_workspace_bytes(int64_t NB, int32_t bs);
BML_API int bml_gershgorin_ellblock(const bml_ellblock_t *H, double *d_bounds, void *d_workspace, size_t workspace_bytes,
                                    void *cuda_stream);
BML_API int bml_trace_ellblock(const bml_ellblock_t *A, double *d_trace, void *cuda_stream);

/*
 * SP2 (Eq. 5-7, Listing 2) on ELLBLOCK.  p->drop_tol is the block threshold of E2; p->precision must be 0; of p->flags
 * only 0 is accepted.  D: same NB, MB, bs as H, must not alias H.  d_workspace >= bml_sp2_ellblock_workspace_bytes,
 * 1024-byte aligned.  stats as in bml_sp2_ellpack (NULL = fully asynchronous, read later with bml_sp2_read_stats).
 */
BML_API size_t bml_sp2_ellblock_workspace_bytes(int64_t NB, int32_t MB, int32_t bs);
BML_API int bml_sp2_ellblock(const bml_ellblock_t *H, const bml_sp2_params_t *p, bml_ellblock_t *D, void *d_workspace,
                             size_t workspace_bytes, bml_sp2_stats_t *stats, void *cuda_stream);

/*
 * One fused product on a caller-supplied iterate (block rows in ascending order, X symmetric as in E3), for per-kernel
 * parity tests and timing: Xnext <- branch ? thr(2X - thr(X X)) : thr(X X) (slots beyond nnz[I] are left untouched).  d_sums: DEVICE double[4] <-
 * { tr thr(X X), ||thr(X X) - X||_F^2 over the union block pattern, ||X||_F^2, tr Xnext }; d_info: DEVICE int32[4] <-
 * { lowest block row with more than MB kept blocks or INT32_MAX, INT32_MAX, max kept blocks per block row, that of
 * thr(X X) }.  Asynchronous.  Return 0, -1, -4.
 */
BML_API size_t bml_x2_ellblock_workspace_bytes(int64_t NB, int32_t MB, int32_t bs);
BML_API int bml_x2_ellblock(const bml_ellblock_t *X, bml_ellblock_t *Xnext, int32_t branch, double drop_tol, double *d_sums,
                            int32_t *d_info, void *d_workspace, size_t workspace_bytes, void *cuda_stream);

#ifdef __cplusplus
}
#endif
#endif /* BML_ELLBLOCK_H */
