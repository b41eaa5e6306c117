// symm_ab.cuh -- host-side interface of the grouped FP64 product kernel (symm_ab.cu), used by chebyshev.cu and api.cu.
#pragma once
#include "common.cuh"
#include "../../include/bml_chebyshev.h"

namespace bmlsp2 {

// one product of a grouped launch: Out = alpha A B + beta C + gamma I
struct SymmJob {
    int32_t a, b;            // operand slots in the 3-D tensor map of the slab
    const double *C;         // nullptr: no C term.  May equal Out (read and written by the same thread)
    double *Out;
    int64_t ldc, ldo;
    double alpha, beta, gamma;
};
struct SymmBatch {
    int32_t n_jobs, pad;
    SymmJob job[BML_SYMM_MAX_JOBS];
};

// 3-D map over a slab of n_slots matrices: dims { N columns, N rows, n_slots }, row pitch ld, slot pitch slot_elems
int make_slab_map(CUtensorMap *map, const double *base, int64_t N, int64_t ld, int64_t slot_elems, int n_slots);
// stream-K scratch (one partial-tile slot per CTA + hand-off flags); reset once, then epochs 1, 2, ... per launch
size_t symm_ab_sk_bytes();
int symm_ab_sk_reset(void *sk, cudaStream_t st);
int launch_symm_ab(const CUtensorMap &map, const SymmBatch &batch, int64_t N, void *sk, unsigned int epoch,
                   cudaStream_t stream);
int symm_ab_work_item(int64_t N, int n_jobs, int n_ctas, int cta, int it, int32_t out[6]);

}  // namespace bmlsp2
