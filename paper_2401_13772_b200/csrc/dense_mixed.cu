// dense_mixed.cu -- mixed-precision dense X^2 (split-BF16 tcgen05 products) -- NOT BUILT YET in this revision:
// precision = 1 returns BML_ERR_INVALID.
#include "common.cuh"

namespace bmlsp2 {

size_t dense_mixed_extra_bytes(int64_t, int64_t) { return 0; }

int sp2_dense_mixed_solve(const bml_matrix_t *, const bml_sp2_params_t *, double *, double *, int64_t, Sp2Ctl *,
                          double *, const double *, void *, cudaStream_t)
{
    return BML_ERR_INVALID;
}

int x2_dense_mixed_once(const bml_matrix_t *, bml_matrix_t *, Sp2Ctl *, double *, void *, cudaStream_t)
{
    return BML_ERR_INVALID;
}

}  // namespace bmlsp2
