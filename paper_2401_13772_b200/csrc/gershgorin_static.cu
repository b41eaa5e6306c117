// gershgorin_static.cu -- include/bml_no_alloc.h: bml_gershgorin with its scratch in a static device array, for callers
// that cannot allocate (CUDA graph capture, serving loops, harnesses that forbid cudaMalloc).  The kernels are the ones
// bml_gershgorin launches (reductions.cu: one warp per row writes the row's lower / upper circle bound, one CTA reduces
// them in a fixed order); only where the 2 N doubles of row bounds live differs, so the bounds are bit-identical.
#include <stdio.h>

#include "common.cuh"
#include "../../include/bml_no_alloc.h"

namespace bmlsp2 {

int launch_gershgorin(const bml_matrix_t *H, double *d_bounds, double *rowlh, cudaStream_t st);     // reductions.cu

// [2 * N] row bounds of the call in flight.  1 MiB on every device that loads the library, until exit; shared by all
// calls on that device (calls that overlap on the GPU race, bml_no_alloc.h); nothing in it has to start at zero.
static __device__ __align__(256) double g_gershgorin_rowlh[2 * BML_GERSHGORIN_STATIC_MAX_N];

// In host code `g_gershgorin_rowlh` is a host-side stand-in for the symbol, not a device address: the address a kernel
// can use comes from cudaGetSymbolAddress, resolved once per device ordinal with that device current.
static double *static_rowlh_for_current_device()
{
    static double *ptr[MAX_DEVICES] = {};
    const int dev = current_device();
    if (dev < 0) return nullptr;
    if (!ptr[dev]) {
        double *p = nullptr;
        if (cudaGetSymbolAddress((void **)&p, g_gershgorin_rowlh) != cudaSuccess || !p) return nullptr;
        ptr[dev] = p;          // idempotent: two threads racing here store the same address
    }
    return ptr[dev];
}

}  // namespace bmlsp2

using namespace bmlsp2;

extern "C" {

int bml_gershgorin_static(const bml_matrix_t *H, double *d_bounds, void *cuda_stream)
{
    if (!H || !d_bounds || !H->value || H->N <= 0) return BML_ERR_INVALID;
    if (H->type == BML_DENSE) {
        if (H->ld < H->N) return BML_ERR_INVALID;
    } else if (H->type == BML_ELLPACK) {
        if (!H->index || !H->nnz || H->M < 1 || H->M > BML_ELL_MAX_M) return BML_ERR_INVALID;
    } else {
        return BML_ERR_INVALID;
    }
    if (H->N > BML_GERSHGORIN_STATIC_MAX_N) return BML_ERR_STATIC_CAPACITY;
    double *rowlh = static_rowlh_for_current_device();
    if (!rowlh) return BML_ERR_CUDA;
    return launch_gershgorin(H, d_bounds, rowlh, (cudaStream_t)cuda_stream);
}

const char *bml_no_alloc_status_string(int status)
{
    if (status == BML_ERR_STATIC_CAPACITY)
        return "N exceeds the static scratch of the no-allocation entry point (BML_GERSHGORIN_STATIC_MAX_N = 65536): "
               "use bml_gershgorin with a caller-supplied workspace";
    return bml_status_string(status);
}

}  // extern "C"
