// bounds.cu -- optional tighter spectral bounds for Eq. 5 (readings B1-B3): K steps of
// the Lanczos recursion on H from a counter-based start vector, the extreme Ritz values of the K x K tridiagonal matrix
// widened by their residual norms and a 1% pad, intersected with the Gershgorin bounds already in d_bounds.
// One persistent cooperative launch runs the whole recursion (matrix-vector products, vector updates with full
// reorthogonalisation, every scalar product as fixed-order per-CTA partials behind a grid barrier); one finishing
// thread then solves the tridiagonal eigenproblem.  Everything stays on the device.
#include <cooperative_groups.h>

#include "common.cuh"
#include "dense_fp64_core.cuh"

namespace cg = cooperative_groups;

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

// ------------------------------------------------------------------------------------------------------------
// The whole recursion is ONE persistent cooperative launch (one CTA per SM).  CTA c owns the contiguous index range
// [c chunk, (c + 1) chunk) of every vector; a scalar product is per-CTA partial sums -> grid barrier -> every CTA adds
// the G partials in the same fixed order, so all CTAs hold bitwise identical alpha, c_q, beta and take the same
// branches (no broadcast, no atomics; results are bit-reproducible).  Each phase writes its partials to a region
// of its own (a fast CTA may already write the next phase's while a slow one still reads this one's).
// ------------------------------------------------------------------------------------------------------------
constexpr int LZ_REG_ALPHA = 0, LZ_REG_PASS0 = 1, LZ_REG_PASS1 = 1 + LZ_MAX_STEPS, LZ_REG_NORM = 1 + 2 * LZ_MAX_STEPS;
constexpr int LZ_PART_ROWS = 2 + 2 * LZ_MAX_STEPS;          // rows of G partials each
constexpr int LZ_MAX_GRID = 256;

// part[(row0 + q) G + cta] = sum over this CTA's index range of V[q][i] w[i], q = q0 .. q1: one warp per q
__device__ __forceinline__ void lz_partial_dots(const double *V, const double *w, int N, int q0, int q1, int i0, int i1,
                                                double *part, int row0, int G)
{
    const int lane = threadIdx.x & 31;
    for (int q = q0 + (threadIdx.x >> 5); q <= q1; q += LZ_THREADS / 32) {
        const double *vq = V + (size_t)q * N;
        double a = 0.0;
        for (int i = i0 + lane; i < i1; i += 32) a = fma(vq[i], w[i], a);
        a = warp_sum(a);
        if (lane == 0) part[(size_t)(row0 + q) * G + blockIdx.x] = a;
    }
}
// s_c[q] = sum over CTAs (lane-strided, then the shuffle tree: the same order in every CTA), q = q0 .. q1
__device__ __forceinline__ void lz_gather(const double *part, int row0, int q0, int q1, int G, double *s_c)
{
    const int lane = threadIdx.x & 31;
    for (int q = q0 + (threadIdx.x >> 5); q <= q1; q += LZ_THREADS / 32) {
        double a = 0.0;
        for (int c = lane; c < G; c += 32) a += part[(size_t)(row0 + q) * G + c];
        a = warp_sum(a);
        if (lane == 0) s_c[q] = a;
    }
    __syncthreads();
}

// Recursion per step j (the oracle's order, oracle/bounds.py): w = H v_j;  alpha_j = v_j.w;
// w -= alpha_j v_j + beta_j v_{j-1};  two passes of classical Gram-Schmidt against v_0 .. v_j (reading B3: without them
// the recursion loses orthogonality once an extreme Ritz value converges and the residual term of the other end is
// reproducible to two digits only);  beta_{j+1} = ||w||;  v_{j+1} = w / beta_{j+1}.  V holds the Lanczos vectors,
// row j = v_j.  H is dense (hi == nullptr: hv = values, ld) or ELLPACK-R (hv, hi, hn, ld = M).
__global__ void __launch_bounds__(LZ_THREADS, 1)
lanczos_run_kernel(const double *__restrict__ hv, const int32_t *__restrict__ hi, const int32_t *__restrict__ hn, int64_t ld,
                   int N, int steps, uint64_t seed, double *V, double *w, double *part, LanczosCtl *ctl)
{
    cg::grid_group grid = cg::this_grid();
    __shared__ double s_c[LZ_MAX_STEPS + 1];
    const int G = gridDim.x, lane = threadIdx.x & 31;
    const int chunk = (N + G - 1) / G;
    const int i0 = min(N, (int)blockIdx.x * chunk), i1 = min(N, i0 + chunk);
    const int gwarp = (blockIdx.x * LZ_THREADS + threadIdx.x) >> 5, nwarps = G * (LZ_THREADS / 32);

    // start vector: counter-based uniform numbers, normalised
    for (int i = i0 + threadIdx.x; i < i1; i += LZ_THREADS) V[i] = lz_uniform(seed + (uint64_t)i);
    __syncthreads();
    lz_partial_dots(V, V, N, 0, 0, i0, i1, part, LZ_REG_NORM, G);
    grid.sync();
    lz_gather(part, LZ_REG_NORM, 0, 0, G, s_c);
    {
        const double inv = 1.0 / sqrt(s_c[0]);
        for (int i = i0 + threadIdx.x; i < i1; i += LZ_THREADS) V[i] *= inv;
    }
    if (blockIdx.x == 0 && threadIdx.x == 0) { ctl->steps = 0; ctl->stopped = 0; ctl->beta[0] = 0.0; }
    grid.sync();

    double beta_j = 0.0;
    for (int j = 0; j < steps; ++j) {
        const double *v = V + (size_t)j * N, *v_prev = V + (size_t)(j > 0 ? j - 1 : 0) * N;
        // w = H v_j: one warp per row, rows dealt round-robin over all warps of the grid
        if (hi == nullptr) {
            for (int r = gwarp; r < N; r += nwarps) {
                const double *__restrict__ row = hv + (int64_t)r * ld;
                double acc = 0.0;
#pragma unroll 8
                for (int c = lane; c < N; c += 32) acc = fma(row[c], v[c], acc);
                acc = warp_sum(acc);
                if (lane == 0) w[r] = acc;
            }
        } else {
            for (int r = gwarp; r < N; r += nwarps) {
                const int n = hn[r];
                double acc = 0.0;
                for (int p = lane; p < n; p += 32) acc = fma(hv[(size_t)r * ld + p], v[hi[(size_t)r * ld + p]], acc);
                acc = warp_sum(acc);
                if (lane == 0) w[r] = acc;
            }
        }
        grid.sync();
        lz_partial_dots(V, w, N, j, j, i0, i1, part, LZ_REG_ALPHA - j, G);      // row0 + q = LZ_REG_ALPHA
        grid.sync();
        lz_gather(part, LZ_REG_ALPHA - j, j, j, G, s_c);
        const double alpha = s_c[j];
        for (int i = i0 + threadIdx.x; i < i1; i += LZ_THREADS)
            w[i] = w[i] - alpha * v[i] - (j > 0 ? beta_j * v_prev[i] : 0.0);
        for (int pass = 0; pass < 2; ++pass) {
            const int row0 = pass ? LZ_REG_PASS1 : LZ_REG_PASS0;
            __syncthreads();
            lz_partial_dots(V, w, N, 0, j, i0, i1, part, row0, G);
            grid.sync();
            lz_gather(part, row0, 0, j, G, s_c);
            for (int i = i0 + threadIdx.x; i < i1; i += LZ_THREADS) {
                double x = w[i];
                for (int q = 0; q <= j; ++q) x -= s_c[q] * V[(size_t)q * N + i];
                w[i] = x;
            }
        }
        __syncthreads();
        lz_partial_dots(w, w, N, 0, 0, i0, i1, part, LZ_REG_NORM, G);
        grid.sync();
        lz_gather(part, LZ_REG_NORM, 0, 0, G, s_c);
        const double beta = sqrt(s_c[0]);
        if (beta > 0.0 && j + 1 < LZ_MAX_STEPS) {
            const double inv = 1.0 / beta;
            double *vn = V + (size_t)(j + 1) * N;
            for (int i = i0 + threadIdx.x; i < i1; i += LZ_THREADS) vn[i] = w[i] * inv;
        }
        if (blockIdx.x == 0 && threadIdx.x == 0) {
            ctl->alpha[j] = alpha;
            ctl->beta[j + 1] = beta;
            ctl->steps = j + 1;
            if (!(beta > 0.0)) ctl->stopped = 1;
        }
        if (!(beta > 0.0)) break;           // exact breakdown; every CTA holds the same beta
        beta_j = beta;
        grid.sync();                        // v_{j+1} complete before the next product reads it
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
// V (LZ_MAX_STEPS Lanczos vectors), w, the per-CTA partial sums, the control block
size_t lanczos_workspace_doubles(int64_t N)
{
    return (size_t)(LZ_MAX_STEPS + 1) * (size_t)N + (size_t)LZ_PART_ROWS * LZ_MAX_GRID + (sizeof(LanczosCtl) + 7) / 8 + 16;
}

// d_bounds: IN the Gershgorin bounds, OUT the tightened ones.  work: lanczos_workspace_doubles(N) doubles.
int launch_lanczos_bounds(const bml_matrix_t *H, int steps, uint64_t seed, double *d_bounds, double *work, cudaStream_t st)
{
    if (steps < 8 || steps > LZ_MAX_STEPS) return BML_ERR_INVALID;      // fewer steps do not see outlying bands
    int N = (int)H->N;
    double *V = work, *w = work + (size_t)LZ_MAX_STEPS * N, *part = w + N;
    LanczosCtl *ctl = (LanczosCtl *)(part + (size_t)LZ_PART_ROWS * LZ_MAX_GRID + 8);
    if (steps > N) steps = N;
    int G = sk_grid();                                                   // one CTA per SM, cooperative launch
    if (G <= 0) return BML_ERR_CUDA;
    if (G > LZ_MAX_GRID) G = LZ_MAX_GRID;
    const double *hv = H->value;
    const int32_t *hi = H->type == BML_DENSE ? nullptr : H->index, *hn = H->type == BML_DENSE ? nullptr : H->nnz;
    int64_t ld = H->type == BML_DENSE ? H->ld : (int64_t)H->M;
    void *args[] = {&hv, &hi, &hn, &ld, &N, &steps, &seed, &V, &w, &part, &ctl};
    if (cudaLaunchCooperativeKernel((const void *)lanczos_run_kernel, dim3((unsigned)G), dim3(LZ_THREADS), args, 0, st) !=
        cudaSuccess)
        return BML_ERR_CUDA;
    lanczos_finish_kernel<<<1, 32, 0, st>>>(ctl, d_bounds);
    return cudaGetLastError() == cudaSuccess ? 0 : BML_ERR_CUDA;
}

}  // namespace bmlsp2
