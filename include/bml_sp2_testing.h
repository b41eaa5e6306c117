/*
 * bml_sp2_testing.h -- test and measurement hooks of libbmlsp2.so.  NOT part of the product interface: include/bml_sp2.h,
 * bml_chebyshev.h and bml_graph.h are the paper's problem statement; the calls below exist so that the host-computable
 * work partitions can be tested exhaustively without a GPU and so that bench.py can measure the FP64 tensor-pipe peak
 * of the box it runs on.  Only tests/ and bench.py use them.
 */
#ifndef BML_SP2_TESTING_H
#define BML_SP2_TESTING_H

#include "bml_sp2.h"

#ifdef __cplusplus
extern "C" {
#endif

/*
 * Measurement helper (not part of the method): issue `iters` back-to-back register-resident FP64 tensor-core
 * instructions (mma.sync m8n8k4 f64 = SASS DMMA.8x8x4) per warp on every SM and return the elapsed device time.
 * bench.py divides the flops by it to get the FP64 tensor-pipe peak at the clocks of the same run (the driver's
 * MEASURED_PEAKS.json has no FP64 entry).  *flops_out <- total flops issued, *ms_out <- CUDA-event milliseconds.
 * Synchronises the stream.  Returns 0 or -4.
 */
BML_API int bml_probe_fp64_tensor_peak(int32_t iters, double *flops_out, double *ms_out, void *cuda_stream);

/*
 * Introspection of the host-computable work distribution of the dense kernels (pure host functions, no GPU needed;
 * they run the same arithmetic as the kernels and exist so that the partition can be tested exhaustively on a CPU).
 * bml_dense_work_item: the it-th work item of CTA `cta` (of n_ctas) of the persistent FP64 kernel for an N x N product
 *   (N > 1024).  out5 <- { tile, I, J, kt_begin, kt_end }: tile (I, J), I <= J, of 128 x 128, k-slabs [kt_begin, kt_end)
 *   of ceil(N / 16).  Returns 0, 1 when the CTA's list has fewer than it + 1 items, or -1.
 * bml_dense_mixed_tile_count / bml_dense_mixed_tile_of_cta: grid size of the mixed kernel and the tile of a CTA
 *   (out2 <- { I, J }); returns 1 for the empty slots of the super-block order.
 */
BML_API int bml_dense_work_item(int64_t N, int32_t n_ctas, int32_t cta, int32_t it, int32_t *out5);
BML_API int bml_dense_mixed_tile_count(int64_t N);
BML_API int bml_dense_mixed_tile_of_cta(int64_t N, int32_t cta, int32_t *out2);

/*
 * Host-computable parts of the path, exported so that they can be tested exhaustively without a GPU:
 * bml_cheb_schedule: the doubling schedule of reading C5.  For i = 2..k: level[i-2] (1-based doubling level),
 *   a[i-2], b[i-2] with T_i = 2 T_a T_b - T_{a-b}.  Returns the number of levels, or -1.
 * bml_symm_work_item: the it-th work item of CTA `cta` (of n_ctas) of a grouped launch of n_jobs products of size N:
 *   out6 <- { job, I, J, kt_begin, kt_end, tile_edge }.  Returns 0, 1 when the list is exhausted, or -1.
 */
BML_API int bml_cheb_schedule(int32_t k, int32_t *level, int32_t *a, int32_t *b);
BML_API int bml_symm_work_item(int64_t N, int32_t n_jobs, int32_t n_ctas, int32_t cta, int32_t it, int32_t *out6);

/*
 * bml_dense_batch_work_item: the it-th work item of CTA `cta` (of n_ctas) of the batched symmetric-square kernel of the
 * graph-based SP2 solver, for parts of sizes n[0 .. n_jobs): out5 <- { part, tile (upper-triangle index of 128 x 128
 * tiles, column by column), kt_begin, kt_end, KT = ceil(n / 16) }.  Pure host arithmetic.  Returns 0, 1 past the end, -1.
 */
BML_API int bml_dense_batch_work_item(int32_t n_jobs, const int32_t *n, int32_t n_ctas, int32_t cta, int32_t it, int32_t *out5);

#ifdef __cplusplus
}
#endif
#endif /* BML_SP2_TESTING_H */
