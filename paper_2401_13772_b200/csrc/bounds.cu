// bounds.cu -- optional tighter spectral bounds for Eq. 5 (readings B1-B3): K steps of
// the Lanczos recursion on H from a counter-based start vector, the extreme Ritz values of the K x K tridiagonal matrix
// widened by their residual norms and a 1% pad, intersected with the Gershgorin bounds already in d_bounds.
// Two launches per step (matrix-vector product; one-CTA vector update with full reorthogonalisation and fixed-order
// reductions), one finishing
// thread for the tridiagonal eigenproblem.  Everything stays on the device.
#include "common.cuh"

namespace bmlsp2 {

constexpr int LZ_MAX_STEPS = 64;
constexpr int LZ_THREADS = 1024;

struct LanczosCtl {
    double alpha[LZ_MAX_STEPS];
    double beta[LZ_MAX_STEPS + 1];     // beta[0] = 0; beta[j + 1] = norm of the residual of step j
    int32_t steps;                     // steps taken so far
    int32_t stopped;                   // exact breakdown: beta = 0
};

// SplitMix64 (Steele, Lea, Flood 2014) on a counter: the oracle draws the same start vector without sharing code
__device__ __forceinline__ double lz_uniform(uint64_t x)
{
    x += 0x9E3779B97F4A7C15ull;
    uint64_t z = x;
    z = (z ^ (z >> 30)) * 0xBF58476D1CE4E5B9ull;
    z = (z ^ (z >> 27)) * 0x94D049BB133111EBull;
    z ^= z >> 31;
    return 2.0 * ((double)(z >> 11) * 0x1.0p-53) - 1.0;
}

// fixed-order block sum (all threads get the result)
__device__ __forceinline__ double lz_block_sum(double v, double *s_part)
{
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    v = warp_sum(v);
    __syncthreads();
    if (lane == 0) s_part[warp] = v;
    __syncthreads();
    double t = 0.0;
#pragma unroll
    for (int w = 0; w < LZ_THREADS / 32; ++w) t += s_part[w];
    return t;
}

__global__ void __launch_bounds__(LZ_THREADS) lanczos_start_kernel(double *__restrict__ v, int N, uint64_t seed,
                                                                   LanczosCtl *__restrict__ ctl)
{
    __shared__ double s_part[LZ_THREADS / 32];
    double acc = 0.0;
    for (int i = threadIdx.x; i < N; i += LZ_THREADS) {
        const double u = lz_uniform(seed + (uint64_t)i);
        v[i] = u;
        acc += u * u;
    }
    const double inv = 1.0 / sqrt(lz_block_sum(acc, s_part));
    for (int i = threadIdx.x; i < N; i += LZ_THREADS) v[i] *= inv;
    if (threadIdx.x == 0) { ctl->steps = 0; ctl->stopped = 0; ctl->beta[0] = 0.0; }
}

// w = H v, one warp per row
__global__ void __launch_bounds__(256) lanczos_matvec_dense_kernel(const double *__restrict__ H, int64_t ld, int N,
                                                                   const double *__restrict__ V, double *__restrict__ w,
                                                                   const LanczosCtl *__restrict__ ctl)
{
    if (ctl->stopped) return;
    const int r = (blockIdx.x * blockDim.x + threadIdx.x) >> 5, lane = threadIdx.x & 31;
    if (r >= N) return;
    const double *__restrict__ v = V + (size_t)ctl->steps * N;
    const double *row = H + (int64_t)r * ld;
    double acc = 0.0;
    for (int j = lane; j < N; j += 32) acc = fma(row[j], v[j], acc);
    acc = warp_sum(acc);
    if (lane == 0) w[r] = acc;
}
__global__ void __launch_bounds__(256) lanczos_matvec_ellpack_kernel(const double *__restrict__ hv,
                                                                     const int32_t *__restrict__ hi,
                                                                     const int32_t *__restrict__ hn, int N, int M,
                                                                     const double *__restrict__ V, double *__restrict__ w,
                                                                     const LanczosCtl *__restrict__ ctl)
{
    if (ctl->stopped) return;
    const int r = (blockIdx.x * blockDim.x + threadIdx.x) >> 5, lane = threadIdx.x & 31;
    if (r >= N) return;
    const double *__restrict__ v = V + (size_t)ctl->steps * N;
    const int n = hn[r];
    double acc = 0.0;
    for (int p = lane; p < n; p += 32) acc = fma(hv[(size_t)r * M + p], v[hi[(size_t)r * M + p]], acc);
    acc = warp_sum(acc);
    if (lane == 0) w[r] = acc;
}

// alpha_j = v_j.w;  w -= alpha_j v_j + beta_j v_{j-1};  two passes of classical Gram-Schmidt against v_0 .. v_j (reading
// B3: without them the recursion loses orthogonality once an extreme Ritz value converges and the residual term of the
// other end is reproducible to two digits only);  beta_{j+1} = ||w||;  v_{j+1} = w / beta_{j+1}.
// V holds the Lanczos vectors, row j = v_j.  One CTA; every reduction in a fixed order.
__global__ void __launch_bounds__(LZ_THREADS) lanczos_update_kernel(double *__restrict__ V, double *__restrict__ w, int N,
                                                                    LanczosCtl *__restrict__ ctl)
{
    __shared__ double s_part[LZ_THREADS / 32];
    __shared__ double s_c[LZ_MAX_STEPS];
    if (ctl->stopped) return;
    const int j = ctl->steps;
    const double beta_j = ctl->beta[j];
    const double *v = V + (size_t)j * N, *v_prev = V + (size_t)(j > 0 ? j - 1 : 0) * N;
    double acc = 0.0;
    for (int i = threadIdx.x; i < N; i += LZ_THREADS) acc = fma(v[i], w[i], acc);
    const double alpha = lz_block_sum(acc, s_part);
    for (int i = threadIdx.x; i < N; i += LZ_THREADS) w[i] = w[i] - alpha * v[i] - (j > 0 ? beta_j * v_prev[i] : 0.0);
    for (int pass = 0; pass < 2; ++pass) {
        __syncthreads();
        // one warp per previous vector: c_q = v_q . w (lane-strided partial sums, then the shuffle tree: fixed order)
        for (int q = threadIdx.x >> 5; q <= j; q += LZ_THREADS / 32) {
            const double *vq = V + (size_t)q * N;
            double a = 0.0;
            for (int i = threadIdx.x & 31; i < N; i += 32) a = fma(vq[i], w[i], a);
            a = warp_sum(a);
            if ((threadIdx.x & 31) == 0) s_c[q] = a;
        }
        __syncthreads();
        for (int i = threadIdx.x; i < N; i += LZ_THREADS) {
            double x = w[i];
            for (int q = 0; q <= j; ++q) x -= s_c[q] * V[(size_t)q * N + i];
            w[i] = x;
        }
    }
    acc = 0.0;
    for (int i = threadIdx.x; i < N; i += LZ_THREADS) acc = fma(w[i], w[i], acc);
    const double beta = sqrt(lz_block_sum(acc, s_part));
    if (beta > 0.0 && j + 1 < LZ_MAX_STEPS) {
        const double inv = 1.0 / beta;
        double *vn = V + (size_t)(j + 1) * N;
        for (int i = threadIdx.x; i < N; i += LZ_THREADS) vn[i] = w[i] * inv;
    }
    if (threadIdx.x == 0) {
        ctl->alpha[j] = alpha;
        ctl->beta[j + 1] = beta;
        ctl->steps = j + 1;
        if (!(beta > 0.0)) ctl->stopped = 1;
    }
}

// Eigenvalues of the K x K tridiagonal matrix by the implicit-shift QL iteration, carrying along the LAST ROW of the
// eigenvector matrix (all that the residual norms |beta_K s_{K-1,i}| need).  Then tighten d_bounds in place.
__global__ void lanczos_finish_kernel(const LanczosCtl *__restrict__ ctl, double *__restrict__ d_bounds)
{
    if (threadIdx.x != 0 || blockIdx.x != 0) return;
    const int n = ctl->steps;
    if (n < 1) return;
    double d[LZ_MAX_STEPS], e[LZ_MAX_STEPS], z[LZ_MAX_STEPS];
    for (int i = 0; i < n; ++i) { d[i] = ctl->alpha[i]; e[i] = (i + 1 < n) ? ctl->beta[i + 1] : 0.0; z[i] = (i == n - 1) ? 1.0 : 0.0; }
    const double beta_n = ctl->beta[n];
    bool ok = true;
    for (int l = 0; l < n && ok; ++l) {
        int iter = 0, m;
        do {
            for (m = l; m < n - 1; ++m) {
                const double dd = fabs(d[m]) + fabs(d[m + 1]);
                if (fabs(e[m]) <= 2.220446049250313e-16 * dd) break;
            }
            if (m != l) {
                if (iter++ == 80) { ok = false; break; }
                double g = (d[l + 1] - d[l]) / (2.0 * e[l]);
                double r = hypot(g, 1.0);
                g = d[m] - d[l] + e[l] / (g + copysign(r, g));
                double s = 1.0, c = 1.0, p = 0.0;
                int i;
                for (i = m - 1; i >= l; --i) {
                    double f = s * e[i];
                    const double b = c * e[i];
                    r = hypot(f, g);
                    e[i + 1] = r;
                    if (r == 0.0) { d[i + 1] -= p; e[m] = 0.0; break; }
                    s = f / r; c = g / r;
                    g = d[i + 1] - p;
                    r = (d[i] - g) * s + 2.0 * c * b;
                    p = s * r;
                    d[i + 1] = g + p;
                    g = c * r - b;
                    f = z[i + 1];
                    z[i + 1] = s * z[i] + c * f;
                    z[i] = c * z[i] - s * f;
                }
                if (r == 0.0 && i >= l) continue;
                d[l] -= p; e[l] = g; e[m] = 0.0;
            }
        } while (m != l);
    }
    if (!ok) return;                    // keep the Gershgorin bounds
    int imin = 0, imax = 0;
    for (int i = 1; i < n; ++i) { if (d[i] < d[imin]) imin = i; if (d[i] > d[imax]) imax = i; }
    const double pad = 0.01 * (d[imax] - d[imin]);
    const double lo = d[imin] - fabs(beta_n * z[imin]) - pad, hi = d[imax] + fabs(beta_n * z[imax]) + pad;
    d_bounds[0] = fmax(d_bounds[0], lo);
    d_bounds[1] = fmin(d_bounds[1], hi);
}

// ------------------------------------------------------------------------------------------------------------
// host side
// ------------------------------------------------------------------------------------------------------------
// V (LZ_MAX_STEPS Lanczos vectors), w, the control block
size_t lanczos_workspace_doubles(int64_t N)
{
    return (size_t)(LZ_MAX_STEPS + 1) * (size_t)N + (sizeof(LanczosCtl) + 7) / 8 + 16;
}

// d_bounds: IN the Gershgorin bounds, OUT the tightened ones.  work: lanczos_workspace_doubles(N) doubles.
int launch_lanczos_bounds(const bml_matrix_t *H, int steps, uint64_t seed, double *d_bounds, double *work, cudaStream_t st)
{
    if (steps < 8 || steps > LZ_MAX_STEPS) return BML_ERR_INVALID;      // fewer steps do not see outlying bands
    const int N = (int)H->N;
    double *V = work, *w = work + (size_t)LZ_MAX_STEPS * N;
    LanczosCtl *ctl = (LanczosCtl *)(work + (size_t)(LZ_MAX_STEPS + 1) * N + 8);
    if (steps > N) steps = N;
    lanczos_start_kernel<<<1, LZ_THREADS, 0, st>>>(V, N, seed, ctl);
    const unsigned grid = (unsigned)(((size_t)N * 32 + 255) / 256);
    for (int j = 0; j < steps; ++j) {
        if (H->type == BML_DENSE)
            lanczos_matvec_dense_kernel<<<grid, 256, 0, st>>>(H->value, H->ld, N, V, w, ctl);
        else
            lanczos_matvec_ellpack_kernel<<<grid, 256, 0, st>>>(H->value, H->index, H->nnz, N, H->M, V, w, ctl);
        lanczos_update_kernel<<<1, LZ_THREADS, 0, st>>>(V, w, N, ctl);
    }
    lanczos_finish_kernel<<<1, 32, 0, st>>>(ctl, d_bounds);
    return cudaGetLastError() == cudaSuccess ? 0 : BML_ERR_CUDA;
}

}  // namespace bmlsp2
