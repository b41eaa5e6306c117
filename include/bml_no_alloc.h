/*
 * bml_no_alloc.h -- one entry point for callers that cannot allocate device memory (code under CUDA graph capture,
 * tight serving loops, harnesses that forbid cudaMalloc): the Gershgorin bounds of bml_sp2.h (the BML op named at
 * P:452; `emin`, `emax` of Listing 2) with their scratch in a static device array of the library instead
 * of a caller-supplied workspace.
 *
 *   bml_gershgorin_static(H, d_bounds, stream)  ==  bml_gershgorin(H, d_bounds, <library scratch>, ..., stream)
 *
 * Same kernels, same arithmetic and summation order as bml_gershgorin: d_bounds is bit-identical to that call's.
 *
 * The scratch (per row: lower and upper circle bound, 2 N doubles) is a file-scope `static __device__` array of
 * 2 * BML_GERSHGORIN_STATIC_MAX_N doubles = 1 MiB.  Every GPU on which the library is loaded holds it until the
 * process exits.  Consequences the caller must know:
 *   - N > BML_GERSHGORIN_STATIC_MAX_N is rejected with BML_ERR_STATIC_CAPACITY (-8); nothing is launched.  Use
 *     bml_gershgorin with a workspace of your own for larger matrices.
 *   - The call allocates nothing: no cudaMalloc / cudaFree / cudaMallocAsync, no allocating library routine.  The first
 *     call on a device resolves the array's device address (cudaGetSymbolAddress, once per device ordinal, with that
 *     device current); later calls only launch the two kernels.
 *   - ALL calls on one device share the one array, and it keeps the last call's contents.  Nothing in it has to start at
 *     zero (every element a call reads, rows 0 .. N-1, is written by that call first), so there is nothing to clear.
 *     Two calls that overlap on the GPU (different streams, or graphs replayed concurrently) RACE on it and both
 *     results are undefined: serialise them (one stream, or an event between them).
 * H: dense or ellpack (bml_matrix_t of bml_sp2.h), DEVICE arrays, never written.  d_bounds: DEVICE double[2] <-
 * {e_min, e_max}.  Asynchronous on `cuda_stream`.  Returns 0, BML_ERR_INVALID (-1), BML_ERR_CUDA (-4) or
 * BML_ERR_STATIC_CAPACITY (-8).
 */
#ifndef BML_NO_ALLOC_H
#define BML_NO_ALLOC_H

#include "bml_sp2.h"

#ifdef __cplusplus
extern "C" {
#endif

#define BML_GERSHGORIN_STATIC_MAX_N 65536   /* largest N bml_gershgorin_static serves (2 x 8 bytes of scratch per row) */
#define BML_ERR_STATIC_CAPACITY (-8)        /* N exceeds the static scratch of a no-allocation entry point             */

BML_API int bml_gershgorin_static(const bml_matrix_t *H, double *d_bounds, void *cuda_stream);
/* "N = ... exceeds ..." style message for -8, bml_status_string(status) for every other code */
BML_API const char *bml_no_alloc_status_string(int status);

#ifdef __cplusplus
}
#endif
#endif
