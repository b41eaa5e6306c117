// reductions.cu -- the HBM-bound streaming steps of DESIGN.md: D0/S0 Gershgorin bounds, D1/S1 rescale
// (Eq. 5; Listing 2), bml_trace (Listing 2), control-block init, D6 output copy.
#include "common.cuh"

namespace bmlsp2 {

// ------------------------------------------------------------------------------------------------------------
// Gershgorin: one warp per row.  rowlh[2i] = H_ii - r_i, rowlh[2i+1] = H_ii + r_i, r_i = sum_{j != i} |H_ij|.
// ------------------------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256) gershgorin_rows_dense_kernel(const double *__restrict__ H, int64_t ld, int N,
                                                                    double *__restrict__ rowlh)
{
    const int lane = threadIdx.x & 31;
    const int row = blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5);
    if (row >= N) return;
    const double *__restrict__ h = H + (int64_t)row * ld;
    // Neumaier-compensated partial sums (4 independent chains per lane), combined by a compensated warp tree: the
    // radius is the exactly rounded sum of |H_ij| (to ~1e-32), so the bounds do not depend on the summation order
    double rs[4] = {0.0, 0.0, 0.0, 0.0}, rc[4] = {0.0, 0.0, 0.0, 0.0};
    int j = lane;
    for (; j + 96 < N; j += 128) {           // four independent 256-byte warp loads in flight
        const double v0 = h[j], v1 = h[j + 32], v2 = h[j + 64], v3 = h[j + 96];
        comp_add(rs[0], rc[0], (j == row) ? 0.0 : fabs(v0));
        comp_add(rs[1], rc[1], (j + 32 == row) ? 0.0 : fabs(v1));
        comp_add(rs[2], rc[2], (j + 64 == row) ? 0.0 : fabs(v2));
        comp_add(rs[3], rc[3], (j + 96 == row) ? 0.0 : fabs(v3));
    }
    for (; j < N; j += 32) comp_add(rs[0], rc[0], (j == row) ? 0.0 : fabs(h[j]));
    comp_merge(rs[0], rc[0], rs[1], rc[1]);
    comp_merge(rs[2], rc[2], rs[3], rc[3]);
    comp_merge(rs[0], rc[0], rs[2], rc[2]);
    const double rad = comp_warp_sum(rs[0], rc[0]);
    if (lane == 0) {
        const double d = h[row];
        rowlh[2 * (int64_t)row] = d - rad;
        rowlh[2 * (int64_t)row + 1] = d + rad;
    }
}

__global__ void __launch_bounds__(256) gershgorin_rows_ellpack_kernel(const double *__restrict__ value,
                                                                      const int32_t *__restrict__ index,
                                                                      const int32_t *__restrict__ nnz, int M, int N,
                                                                      double *__restrict__ rowlh)
{
    const int lane = threadIdx.x & 31;
    const int row = blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5);
    if (row >= N) return;
    const int n = nnz[row];
    const double *__restrict__ v = value + (int64_t)row * M;
    const int32_t *__restrict__ c = index + (int64_t)row * M;
    double rs = 0.0, rc = 0.0, d = 0.0;
    for (int p = lane; p < n; p += 32) {
        const double x = v[p];
        if (c[p] == row) d = x; else comp_add(rs, rc, fabs(x));
    }
    const double rad = comp_warp_sum(rs, rc);
    d = warp_sum(d);            // at most one lane holds the (unique) diagonal entry; a missing diagonal counts as 0
    if (lane == 0) {
        rowlh[2 * (int64_t)row] = d - rad;
        rowlh[2 * (int64_t)row + 1] = d + rad;
    }
}

// single CTA: bounds[0] = min_i rowlh[2i], bounds[1] = max_i rowlh[2i+1]
__global__ void __launch_bounds__(1024) gershgorin_reduce_kernel(const double *__restrict__ rowlh, int N,
                                                                 double *__restrict__ bounds)
{
    __shared__ double s_lo[32], s_hi[32];
    double lo = INFINITY, hi = -INFINITY;
    for (int i = threadIdx.x; i < N; i += blockDim.x) {
        lo = fmin(lo, rowlh[2 * (int64_t)i]);
        hi = fmax(hi, rowlh[2 * (int64_t)i + 1]);
    }
    lo = warp_min(lo); hi = warp_max(hi);
    if ((threadIdx.x & 31) == 0) { s_lo[threadIdx.x >> 5] = lo; s_hi[threadIdx.x >> 5] = hi; }
    __syncthreads();
    if (threadIdx.x < 32) {
        lo = threadIdx.x < (blockDim.x >> 5) ? s_lo[threadIdx.x] : INFINITY;
        hi = threadIdx.x < (blockDim.x >> 5) ? s_hi[threadIdx.x] : -INFINITY;
        lo = warp_min(lo); hi = warp_max(hi);
        if (threadIdx.x == 0) { bounds[0] = lo; bounds[1] = hi; }
    }
}

// ------------------------------------------------------------------------------------------------------------
// Trace: single CTA, fixed order (thread-strided partials, then a fixed tree) -> bit-reproducible.
// ------------------------------------------------------------------------------------------------------------
__device__ __forceinline__ double block_sum_1024(double v)
{
    __shared__ double s_w[32];
    v = warp_sum(v);
    if ((threadIdx.x & 31) == 0) s_w[threadIdx.x >> 5] = v;
    __syncthreads();
    double r = 0.0;
    if (threadIdx.x < 32) {
        r = threadIdx.x < (blockDim.x >> 5) ? s_w[threadIdx.x] : 0.0;
        r = warp_sum(r);
    }
    return r;   // valid in thread 0
}

__global__ void __launch_bounds__(1024) trace_dense_kernel(const double *__restrict__ A, int64_t ld, int N,
                                                           double *__restrict__ out)
{
    double v = 0.0;
    for (int i = threadIdx.x; i < N; i += blockDim.x) v += A[(int64_t)i * ld + i];
    v = block_sum_1024(v);
    if (threadIdx.x == 0) *out = v;
}

// ------------------------------------------------------------------------------------------------------------
// Rescale (Eq. 5 with Gershgorin bounds): X_ij = -s H_ij (i != j), X_ii = s (e_max - H_ii), s = 1/(e_max - e_min).
// Writes the padded workspace iterate (leading dimension ldx >= N, pad columns zeroed).
// ------------------------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256) rescale_dense_kernel(const double *__restrict__ H, int64_t ldh, int N,
                                                            const double *__restrict__ bounds,
                                                            double *__restrict__ X, int64_t ldx)
{
    const double emin = bounds[0], emax = bounds[1];
    const double s = 1.0 / (emax - emin);
    const int row = blockIdx.x;
    const double *__restrict__ h = H + (int64_t)row * ldh;
    double *__restrict__ x = X + (int64_t)row * ldx;
    for (int j = blockIdx.y * blockDim.x + threadIdx.x; j < ldx; j += gridDim.y * blockDim.x) {
        double v = 0.0;
        if (j < N) {
            const double hv = h[j];
            v = (j == row) ? s * (emax - hv) : -s * hv;
        }
        x[j] = v;
    }
}

// ------------------------------------------------------------------------------------------------------------
// Control block init: runs after Gershgorin + rescale + trace(X_0).  Degenerate bounds -> status -2.
// ------------------------------------------------------------------------------------------------------------
__global__ void sp2_init_ctl_kernel(Sp2Ctl *ctl, const double *__restrict__ bounds, const double *__restrict__ tr0,
                                    int n_occ, int max_products, double idem_tol, int loop_mode, int branch0,
                                    const int *__restrict__ fail_flag)
{
    if (threadIdx.x != 0 || blockIdx.x != 0) return;
    ctl->m = 0; ctl->done = 0; ctl->status = BML_MAX_PRODUCTS; ctl->parity = 0;
    ctl->overflow_row = INT32_MAX; ctl->overflow_upd = INT32_MAX; ctl->acc_row = INT32_MAX;
    ctl->nnz_max_p = 0; ctl->nnz_max_upd = 0; ctl->fail_row = -1; ctl->arrivals = 0; ctl->n_done = 0; ctl->epoch = 1u;
    ctl->n_occ = n_occ; ctl->max_products = max_products; ctl->loop_mode = loop_mode; ctl->idem_tol = idem_tol;
    for (int q = 0; q < 4; ++q) ctl->sums[q] = 0.0;
    if (loop_mode) {
        const double emin = bounds[0], emax = bounds[1];
        ctl->emin = emin; ctl->emax = emax;
        const double t = *tr0;
        ctl->tr_cur = t;
        ctl->branch_cur = (t - (double)n_occ <= 0.0) ? 1 : 0;
        if (!(emax - emin > 0.0)) { ctl->done = 1; ctl->status = BML_ERR_DEGENERATE; }
        if (fail_flag) {
            // fail_flag[0]: symmetry violation (-5); fail_flag[1]: INT32_MAX - lowest ELLPACK rescale overflow row (-3)
            if (fail_flag[0]) { ctl->done = 1; ctl->status = BML_ERR_NOT_SYMMETRIC; }
            else if (fail_flag[1]) { ctl->done = 1; ctl->status = BML_ERR_ELL_OVERFLOW; ctl->fail_row = INT32_MAX - fail_flag[1]; }
        }
    } else {
        ctl->emin = 0.0; ctl->emax = 0.0; ctl->tr_cur = 0.0;
        ctl->branch_cur = branch0;
    }
    for (int q = 0; q < BML_SP2_LOG_LEN; ++q) { ctl->branch[q] = 0; ctl->trace[q] = 0.0; ctl->idem[q] = 0.0; ctl->max_row_nnz[q] = 0; }
}

// symmetry check (flag BML_SP2_FLAG_CHECK_SYMMETRY): H_ij == H_ji bitwise
__global__ void __launch_bounds__(256) check_symmetry_kernel(const double *__restrict__ H, int64_t ld, int N,
                                                             int *__restrict__ flag)
{
    const int i = blockIdx.x;
    for (int j = blockIdx.y * blockDim.x + threadIdx.x; j < i; j += gridDim.y * blockDim.x)
        if (H[(int64_t)i * ld + j] != H[(int64_t)j * ld + i]) atomicExch(flag, 1);
}

// D6: D <- X_{m*} (buffer `parity`), dense.
__global__ void __launch_bounds__(256) copy_out_dense_kernel(const double *__restrict__ buf0,
                                                             const double *__restrict__ buf1, int64_t ldx, int N,
                                                             const Sp2Ctl *__restrict__ ctl, double *__restrict__ D,
                                                             int64_t ldd)
{
    if (ctl->done && ctl->status < 0) return;       // failed solve: D is left untouched (X_0 may hold Inf / NaN)
    const double *__restrict__ X = ctl->parity ? buf1 : buf0;
    const int row = blockIdx.x;
    for (int j = blockIdx.y * blockDim.x + threadIdx.x; j < N; j += gridDim.y * blockDim.x)
        D[(int64_t)row * ldd + j] = X[(int64_t)row * ldx + j];
}

// ------------------------------------------------------------------------------------------------------------
// host launchers
// ------------------------------------------------------------------------------------------------------------
#define BML_CHECK_LAUNCH() do { if (cudaGetLastError() != cudaSuccess) return BML_ERR_CUDA; } while (0)

int launch_gershgorin(const bml_matrix_t *H, double *d_bounds, double *rowlh, cudaStream_t st)
{
    const int N = (int)H->N;
    const int rows_per_cta = 8;
    const int grid = (N + rows_per_cta - 1) / rows_per_cta;
    if (H->type == BML_DENSE)
        gershgorin_rows_dense_kernel<<<grid, 256, 0, st>>>(H->value, H->ld, N, rowlh);
    else
        gershgorin_rows_ellpack_kernel<<<grid, 256, 0, st>>>(H->value, H->index, H->nnz, H->M, N, rowlh);
    BML_CHECK_LAUNCH();
    gershgorin_reduce_kernel<<<1, 1024, 0, st>>>(rowlh, N, d_bounds);
    BML_CHECK_LAUNCH();
    return 0;
}

int launch_gershgorin_reduce(const double *rowlh, int N, double *d_bounds, cudaStream_t st)
{
    gershgorin_reduce_kernel<<<1, 1024, 0, st>>>(rowlh, N, d_bounds);
    BML_CHECK_LAUNCH();
    return 0;
}

int launch_trace_dense(const double *A, int64_t ld, int N, double *d_out, cudaStream_t st)
{
    trace_dense_kernel<<<1, 1024, 0, st>>>(A, ld, N, d_out);
    BML_CHECK_LAUNCH();
    return 0;
}

// ELLPACK trace needs N doubles of scratch; bml_trace has no workspace argument, so it is computed by one CTA that
// walks the rows itself (N*nnz reads, single CTA: fine for the diagnostic entry point; the SP2 loop never calls it).
__global__ void __launch_bounds__(1024) trace_ellpack_kernel(const double *__restrict__ value,
                                                             const int32_t *__restrict__ index,
                                                             const int32_t *__restrict__ nnz, int M, int N,
                                                             double *__restrict__ out)
{
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5, nw = blockDim.x >> 5;
    double acc = 0.0;   // lane 0 of each warp accumulates its rows in ascending order
    for (int row = warp; row < N; row += nw) {
        const int n = nnz[row];
        double d = 0.0;
        for (int p = lane; p < n; p += 32)
            if (index[(int64_t)row * M + p] == row) d = value[(int64_t)row * M + p];
        d = warp_sum(d);
        acc += d;
    }
    __shared__ double s_w[32];
    if (lane == 0) s_w[warp] = acc;
    __syncthreads();
    if (threadIdx.x < 32) {
        double r = threadIdx.x < nw ? s_w[threadIdx.x] : 0.0;
        r = warp_sum(r);
        if (threadIdx.x == 0) *out = r;
    }
}

int launch_trace_ellpack(const bml_matrix_t *A, double *d_out, cudaStream_t st)
{
    trace_ellpack_kernel<<<1, 1024, 0, st>>>(A->value, A->index, A->nnz, A->M, (int)A->N, d_out);
    BML_CHECK_LAUNCH();
    return 0;
}

int launch_rescale_dense(const bml_matrix_t *H, const double *d_bounds, double *X, int64_t ldx, cudaStream_t st)
{
    const int N = (int)H->N;
    dim3 grid((unsigned)N, (unsigned)((ldx + 1023) / 1024));
    if (grid.y > 8) grid.y = 8;
    rescale_dense_kernel<<<grid, 256, 0, st>>>(H->value, H->ld, N, d_bounds, X, ldx);
    BML_CHECK_LAUNCH();
    return 0;
}

int launch_check_symmetry(const bml_matrix_t *H, int *d_flag, cudaStream_t st)
{
    const int N = (int)H->N;
    dim3 grid((unsigned)N, (unsigned)((N + 1023) / 1024));
    if (grid.y > 8) grid.y = 8;
    check_symmetry_kernel<<<grid, 256, 0, st>>>(H->value, H->ld, N, d_flag);
    BML_CHECK_LAUNCH();
    return 0;
}

int launch_init_ctl(Sp2Ctl *ctl, const double *d_bounds, const double *d_tr0, int n_occ, int max_products,
                    double idem_tol, int loop_mode, int branch0, const int *fail_flag, cudaStream_t st)
{
    sp2_init_ctl_kernel<<<1, 32, 0, st>>>(ctl, d_bounds, d_tr0, n_occ, max_products, idem_tol, loop_mode, branch0,
                                          fail_flag);
    BML_CHECK_LAUNCH();
    return 0;
}

int launch_copy_out_dense(const double *buf0, const double *buf1, int64_t ldx, int N, const Sp2Ctl *ctl, double *D,
                          int64_t ldd, cudaStream_t st)
{
    dim3 grid((unsigned)N, (unsigned)((N + 1023) / 1024));
    if (grid.y > 8) grid.y = 8;
    copy_out_dense_kernel<<<grid, 256, 0, st>>>(buf0, buf1, ldx, N, ctl, D, ldd);
    BML_CHECK_LAUNCH();
    return 0;
}

}  // namespace bmlsp2
