// ellpack.cu -- the sparse path of DESIGN.md on ELLPACK-R (Listing 1): S1 rescale, S3 thresholded row-wise
// SpGEMM X*X, S4 fused update / norms / canonical (ascending-column) write-back, S5 finaliser.
//
// One warp owns one output row at a time (Gustavson row merge, "sparse-sparse matrix multiply").  The row's
// accumulator is a per-warp open-addressing hash table in shared memory (BML_ELL_ACC_SLOTS keys + FP64 values).
// Contributions to one output entry are added in order of increasing slot p of row i, each as fma(x_ik, x_kj, acc):
// the p loop is sequential, the 32 lanes take different j of row k (unique within the row), so no two lanes ever
// update the same entry in the same step and the accumulation order is the canonical one of the oracle
// (readings item 11) -- values are bit-identical to it, not merely close.
#include "common.cuh"

namespace bmlsp2 {

constexpr int E_SLOTS = BML_ELL_ACC_SLOTS;
constexpr int E_MASK = E_SLOTS - 1;
constexpr int E_EMPTY = -1;
constexpr int E_DROPPED = 1 << 30;    // P entry fell below tau (value zeroed)
constexpr int E_INX = 1 << 29;        // column also present in row i of X
constexpr int E_KEY = (1 << 29) - 1;
constexpr int E_MAX_WARPS = 4;
constexpr int E_MAX_GRID = 1024;

__device__ __forceinline__ int e_hash(int j) { return (int)(((uint32_t)j * 2654435761u) >> 20) & E_MASK; }

static inline int next_pow2(int x) { int p = 1; while (p < x) p <<= 1; return p; }
// row stage sa[M] f64, sk[M] int, sn[M] int; later aliased by the (column, slot) sort buffer of >= 32 entries
static inline size_t e_scratch_bytes(int M) { return M >= 16 ? (size_t)16 * (size_t)M : 256; }
static inline size_t e_warp_bytes(int M) { return (size_t)E_SLOTS * 12 + e_scratch_bytes(M); }

size_t ellpack_rowstats_bytes(int64_t) { return (size_t)E_MAX_GRID * 4 * sizeof(double); }

// bitonic sort of n (power of two) 64-bit keys in shared memory by one warp, ascending
__device__ __forceinline__ void warp_bitonic_sort(unsigned long long *buf, int n, int lane)
{
    for (int k = 2; k <= n; k <<= 1) {
        for (int j = k >> 1; j > 0; j >>= 1) {
            for (int t = lane; t < (n >> 1); t += 32) {
                const int i = ((t & ~(j - 1)) << 1) | (t & (j - 1));
                const int l = i | j;
                const bool up = (i & k) == 0;
                const unsigned long long a = buf[i], b = buf[l];
                if ((a > b) == up) { buf[i] = b; buf[l] = a; }
            }
            __syncwarp();
        }
    }
}

// ------------------------------------------------------------------------------------------------------------
// S3 + S4: thresholded row product, fused update, norms, sorted write-back.
// ------------------------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(E_MAX_WARPS * 32, 1)
x2_ellpack_kernel(double *__restrict__ v0, int32_t *__restrict__ i0, int32_t *__restrict__ n0,
                  double *__restrict__ v1, int32_t *__restrict__ i1, int32_t *__restrict__ n1, int N, int M,
                  double tau, int sort_cap, Sp2Ctl *__restrict__ ctl, double *__restrict__ partials)
{
    if (ctl->done) return;
    const int parity = ctl->parity;
    const int branch = ctl->branch_cur;
    const double *__restrict__ xv = parity ? v1 : v0;
    const int32_t *__restrict__ xi = parity ? i1 : i0;
    const int32_t *__restrict__ xn = parity ? n1 : n0;
    double *__restrict__ ov = parity ? v0 : v1;
    int32_t *__restrict__ oi = parity ? i0 : i1;
    int32_t *__restrict__ on = parity ? n0 : n1;

    extern __shared__ __align__(16) uint8_t smem[];
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31, nwarps = blockDim.x >> 5;
    uint8_t *wbase = smem + (size_t)warp * ((size_t)E_SLOTS * 12 + (size_t)sort_cap * 8);
    double *vals = (double *)wbase;                                  // [E_SLOTS]
    int *keys = (int *)(wbase + (size_t)E_SLOTS * 8);                // [E_SLOTS]
    uint8_t *scratch = wbase + (size_t)E_SLOTS * 12;
    double *sa = (double *)scratch;                                  // [M] values of row i
    int *sk = (int *)(scratch + (size_t)8 * M);                      // [M] columns of row i (= rows k to merge)
    int *sn = sk + M;                                                // [M] nnz of those rows
    unsigned long long *sortbuf = (unsigned long long *)scratch;     // aliases sa/sk/sn after phase B
    __shared__ double s_part[E_MAX_WARPS][4];
    __shared__ int s_last;

    double w_trp = 0.0, w_e = 0.0, w_x = 0.0, w_trn = 0.0;          // this warp's running sums over its rows
    int w_ovf_p = INT32_MAX, w_ovf_u = INT32_MAX, w_acc = INT32_MAX, w_max_p = 0, w_max_u = 0;

    for (int64_t row64 = (int64_t)blockIdx.x * nwarps + warp; row64 < N; row64 += (int64_t)gridDim.x * nwarps) {
        const int row = (int)row64;
        const int64_t rbase = (int64_t)row * M;
        const int n_i = min(xn[row], M);
        // clear the key table; stage row i
        for (int s = lane; s < E_SLOTS; s += 32) keys[s] = E_EMPTY;
        for (int p = lane; p < n_i; p += 32) {
            const int k = xi[rbase + p];
            sk[p] = k;
            sa[p] = xv[rbase + p];
            sn[p] = xn[k];
        }
        __syncwarp();

        // ---------------- accumulate: acc[j] = fma(x_ik, x_kj, acc[j]), p ascending ----------------
        bool full = false;
        for (int p = 0; p < n_i; ++p) {
            const int k = sk[p];
            const double a = sa[p];
            const int n_k = sn[p];
            const int64_t kbase = (int64_t)k * M;
            for (int q0 = 0; q0 < n_k; q0 += 128) {
                int jj[4]; double vv[4];
#pragma unroll
                for (int u = 0; u < 4; ++u) {
                    const int q = q0 + u * 32 + lane;
                    jj[u] = -1; vv[u] = 0.0;
                    if (q < n_k) { jj[u] = __ldg(xi + kbase + q); vv[u] = __ldg(xv + kbase + q); }
                }
#pragma unroll
                for (int u = 0; u < 4; ++u) {
                    const int j = jj[u];
                    if (j >= 0) {
                        int slot = e_hash(j);
                        int tries = 0;
                        while (true) {
                            const int key = keys[slot];
                            if (key == j) { vals[slot] = fma(a, vv[u], vals[slot]); break; }
                            if (key == E_EMPTY) {
                                const int old = atomicCAS(&keys[slot], E_EMPTY, j);
                                if (old == E_EMPTY) { vals[slot] = a * vv[u]; break; }   // = fma(a, v, 0.0)
                                if (old == j) { vals[slot] = fma(a, vv[u], vals[slot]); break; }
                            }
                            slot = (slot + 1) & E_MASK;
                            if (++tries > E_SLOTS) { full = true; break; }
                        }
                    }
                }
            }
            __syncwarp();
            if (__any_sync(0xffffffffu, full)) { full = true; break; }
        }
        if (full) {                       // accumulator capacity exceeded: status -6
            w_acc = min(w_acc, row);
            if (lane == 0) on[row] = 0;
            __syncwarp();
            continue;
        }

        // ---------------- phase A: threshold P = thr_tau(X X) (keep |p| >= tau or the diagonal) ----------------
        double r_trp = 0.0, r_e = 0.0, r_x = 0.0, r_trn = 0.0;
        int cnt_p = 0;
        for (int s = lane; s < E_SLOTS; s += 32) {
            const int key = keys[s];
            if (key != E_EMPTY) {
                const double pv = vals[s];
                if (fabs(pv) >= tau || key == row) {
                    ++cnt_p;
                    if (key == row) r_trp += pv;
                } else {
                    keys[s] = key | E_DROPPED;
                    vals[s] = 0.0;
                }
            }
        }
        __syncwarp();
        // ---------------- phase B: entries of row i of X: norms, update value, mark ----------------
        for (int p = lane; p < n_i; p += 32) {
            const int j = sk[p];
            const double x = sa[p];
            // normally present (x_ii * x_ij touched it); a row stored without its diagonal may miss it: then P_ij is
            // absent and the column enters the union pattern as an X-only entry (value 0, dropped)
            int slot = e_hash(j);
            for (int tries = 0; tries <= E_SLOTS; ++tries) {
                const int key = keys[slot];
                if (key != E_EMPTY && (key & E_KEY) == j) break;
                if (key == E_EMPTY) {
                    const int old = atomicCAS(&keys[slot], E_EMPTY, j | E_DROPPED);
                    if (old == E_EMPTY) { vals[slot] = 0.0; break; }
                    if ((old & E_KEY) == j) break;
                }
                slot = (slot + 1) & E_MASK;
            }
            const double pk = vals[slot];                                   // 0 if dropped
            const double d = pk - x;
            r_e += d * d;
            r_x += x * x;
            keys[slot] |= E_INX;
            if (branch) vals[slot] = 2.0 * x - pk;                          // Eq. 7 on the union pattern
        }
        __syncwarp();
        cnt_p = __reduce_add_sync(0xffffffffu, cnt_p);
        // ---------------- phase C: select X' entries, compact (j, slot) into the sort buffer ----------------
        int kept = 0;   // warp-uniform
        for (int s0 = 0; s0 < E_SLOTS; s0 += 32) {
            const int s = s0 + lane;
            const int key = keys[s];
            bool keep = false;
            int j = 0;
            if (key != E_EMPTY) {
                j = key & E_KEY;
                const double v = vals[s];
                const bool inx = (key & E_INX) != 0, dropped = (key & E_DROPPED) != 0;
                if (!inx) {
                    // column only in P: P - X = p; X' = -p (branch) or p, kept iff P kept it
                    if (!dropped) {
                        r_e += v * v;
                        keep = true;
                        if (branch) vals[s] = -v;
                    }
                } else if (branch) {
                    keep = (fabs(v) >= tau) || (j == row);
                } else {
                    keep = !dropped;
                }
                if (keep && j == row) r_trn += vals[s];
            }
            const unsigned bal = __ballot_sync(0xffffffffu, keep);
            if (keep) {
                const int pos = kept + __popc(bal & ((1u << lane) - 1u));
                if (pos < sort_cap) sortbuf[pos] = ((unsigned long long)(unsigned)j << 32) | (unsigned)s;
            }
            kept += __popc(bal);
        }
        __syncwarp();
        w_max_p = max(w_max_p, cnt_p);
        w_max_u = max(w_max_u, kept);
        if (cnt_p > M) w_ovf_p = min(w_ovf_p, row);
        if (kept > M) {
            w_ovf_u = min(w_ovf_u, row);
            if (lane == 0) on[row] = 0;
        } else {
            // ---------------- sort ascending by column, write the row, zero-fill unused slots ----------------
            int n2 = 32;
            while (n2 < kept) n2 <<= 1;
            for (int q = kept + lane; q < n2; q += 32) sortbuf[q] = ~0ull;
            __syncwarp();
            warp_bitonic_sort(sortbuf, n2, lane);
            for (int q = lane; q < M; q += 32) {
                int j = 0; double v = 0.0;
                if (q < kept) {
                    const unsigned long long e = sortbuf[q];
                    j = (int)(e >> 32);
                    v = vals[(int)(e & 0xffffffffu)];
                }
                oi[rbase + q] = j;
                ov[rbase + q] = v;
            }
            if (lane == 0) on[row] = kept;
        }
        w_trp += warp_sum(r_trp); w_e += warp_sum(r_e); w_x += warp_sum(r_x); w_trn += warp_sum(r_trn);
        __syncwarp();
    }

    // ---------------- per-CTA partials (fixed order), flags, last-CTA finaliser (S5) ----------------
    if (lane == 0) {
        s_part[warp][0] = w_trp; s_part[warp][1] = w_e; s_part[warp][2] = w_x; s_part[warp][3] = w_trn;
        if (w_ovf_p != INT32_MAX) atomicMin(&ctl->overflow_row, w_ovf_p);
        if (w_ovf_u != INT32_MAX) atomicMin(&ctl->overflow_upd, w_ovf_u);
        if (w_acc != INT32_MAX) atomicMin(&ctl->acc_row, w_acc);
        atomicMax(&ctl->nnz_max_p, w_max_p);
        atomicMax(&ctl->nnz_max_upd, w_max_u);
    }
    __syncthreads();
    if (threadIdx.x < 4) {
        double v = 0.0;
        for (int w = 0; w < nwarps; ++w) v += s_part[w][threadIdx.x];
        partials[(size_t)blockIdx.x * 4 + threadIdx.x] = v;
    }
    __threadfence();
    __syncthreads();
    if (threadIdx.x == 0) {
        const uint32_t prev = atomicAdd(&ctl->arrivals, 1u);
        s_last = (prev + 1u == gridDim.x);
    }
    __syncthreads();
    if (s_last && warp == 0) {
        __threadfence();
        double s[4] = {0.0, 0.0, 0.0, 0.0};
        const volatile double *vp = partials;
        for (int b = lane; b < (int)gridDim.x; b += 32) {
#pragma unroll
            for (int q = 0; q < 4; ++q) s[q] += vp[(size_t)b * 4 + q];
        }
#pragma unroll
        for (int q = 0; q < 4; ++q) s[q] = warp_sum(s[q]);
        if (lane == 0) sp2_finalise(ctl, s);
    }
}

// ------------------------------------------------------------------------------------------------------------
// S1: rescale on ELLPACK-R (Eq. 5; the paper's Listing 4, is this kind of kernel) + canonical row order.
// One warp per row: X_ij = -s H_ij (i != j), X_ii = s (e_max - H_ii); a missing diagonal is inserted (H_ii = 0).
// diag[row] <- X_ii for the trace.  fail_flag[1] <- max over overflowing rows of (INT32_MAX - row) (0 = none).
// ------------------------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(128)
rescale_ellpack_kernel(const double *__restrict__ hv, const int32_t *__restrict__ hi, const int32_t *__restrict__ hn,
                       int N, int M, const double *__restrict__ bounds, double *__restrict__ xv,
                       int32_t *__restrict__ xi, int32_t *__restrict__ xn, double *__restrict__ diag,
                       int *__restrict__ fail_flag, int sort_cap)
{
    extern __shared__ __align__(16) uint8_t smem[];
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31, nwarps = blockDim.x >> 5;
    unsigned long long *sortbuf = (unsigned long long *)(smem + (size_t)warp * sort_cap * 8);
    const double emin = bounds[0], emax = bounds[1];
    const double s = 1.0 / (emax - emin);
    const int row = blockIdx.x * nwarps + warp;
    if (row >= N) return;
    const int64_t rbase = (int64_t)row * M;
    const int n = min(hn[row], M);
    int has = 0;
    for (int p = lane; p < n; p += 32) {
        const int j = hi[rbase + p];
        has |= (j == row);
        sortbuf[p] = ((unsigned long long)(unsigned)j << 32) | (unsigned)p;
    }
    has = __any_sync(0xffffffffu, has);
    const int total = n + (has ? 0 : 1);
    if (total > M) {
        if (lane == 0) { atomicMax(&fail_flag[1], INT32_MAX - row); xn[row] = 0; diag[row] = 0.0; }
        return;
    }
    if (!has && lane == 0) sortbuf[n] = ((unsigned long long)(unsigned)row << 32) | 0xffffffffu;   // inserted diagonal
    int n2 = 32;
    while (n2 < total) n2 <<= 1;
    __syncwarp();
    for (int q = total + lane; q < n2; q += 32) sortbuf[q] = ~0ull;
    __syncwarp();
    warp_bitonic_sort(sortbuf, n2, lane);
    for (int q = lane; q < M; q += 32) {
        int j = 0; double v = 0.0;
        if (q < total) {
            const unsigned long long e = sortbuf[q];
            j = (int)(e >> 32);
            const unsigned p = (unsigned)(e & 0xffffffffu);
            const double h = (p == 0xffffffffu) ? 0.0 : hv[rbase + p];
            v = (j == row) ? s * (emax - h) : -s * h;
            if (j == row) diag[row] = v;
        }
        xi[rbase + q] = j;
        xv[rbase + q] = v;
    }
    if (lane == 0) xn[row] = total;
}

__global__ void __launch_bounds__(1024) sum_vector_kernel(const double *__restrict__ v, int N, double *__restrict__ out)
{
    __shared__ double s_w[32];
    double s = 0.0;
    for (int i = threadIdx.x; i < N; i += blockDim.x) s += v[i];
    s = warp_sum(s);
    if ((threadIdx.x & 31) == 0) s_w[threadIdx.x >> 5] = s;
    __syncthreads();
    if (threadIdx.x < 32) {
        double r = threadIdx.x < (blockDim.x >> 5) ? s_w[threadIdx.x] : 0.0;
        r = warp_sum(r);
        if (threadIdx.x == 0) *out = r;
    }
}

// S6: D <- X_{m*}
__global__ void __launch_bounds__(256)
copy_out_ellpack_kernel(const double *__restrict__ v0, const int32_t *__restrict__ i0, const int32_t *__restrict__ n0,
                        const double *__restrict__ v1, const int32_t *__restrict__ i1, const int32_t *__restrict__ n1,
                        int64_t N, int M, const Sp2Ctl *__restrict__ ctl, double *__restrict__ dv,
                        int32_t *__restrict__ di, int32_t *__restrict__ dn)
{
    const int parity = ctl->parity;
    const double *__restrict__ sv = parity ? v1 : v0;
    const int32_t *__restrict__ si = parity ? i1 : i0;
    const int32_t *__restrict__ sn = parity ? n1 : n0;
    const int64_t nm = N * (int64_t)M;
    for (int64_t e = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; e < nm; e += (int64_t)gridDim.x * blockDim.x) {
        dv[e] = sv[e];
        di[e] = si[e];
    }
    for (int64_t r = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; r < N; r += (int64_t)gridDim.x * blockDim.x)
        dn[r] = sn[r];
}

__global__ void x2_ellpack_info_kernel(const Sp2Ctl *__restrict__ ctl, int32_t *__restrict__ info)
{
    if (threadIdx.x == 0 && blockIdx.x == 0) {
        info[0] = min(ctl->overflow_row, ctl->overflow_upd);
        info[1] = ctl->acc_row;
        info[2] = max(ctl->nnz_max_p, ctl->nnz_max_upd);
        info[3] = ctl->nnz_max_p;
    }
}

// ------------------------------------------------------------------------------------------------------------
// host launchers
// ------------------------------------------------------------------------------------------------------------
#define BML_CHECK_LAUNCH() do { if (cudaGetLastError() != cudaSuccess) return BML_ERR_CUDA; } while (0)

static int sm_count()
{
    static int sms = 0;
    if (!sms) {
        int dev = 0;
        if (cudaGetDevice(&dev) != cudaSuccess || cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess)
            sms = 0;
    }
    return sms;
}

int launch_x2_ellpack(const double *v0, const int32_t *i0, const int32_t *n0, double *v1, int32_t *i1, int32_t *n1,
                      int64_t N, int M, double tau, Sp2Ctl *ctl, double *partials, cudaStream_t st)
{
    const int sms = sm_count();
    if (sms <= 0) return BML_ERR_CUDA;
    const size_t smem_cap = 227 * 1024 - 256;
    int nwarps = (int)(smem_cap / e_warp_bytes(M));
    if (nwarps > E_MAX_WARPS) nwarps = E_MAX_WARPS;
    if (nwarps < 1) return BML_ERR_INVALID;
    const size_t smem = (size_t)nwarps * e_warp_bytes(M);
    static size_t attr_smem = 0;
    if (smem > attr_smem) {
        if (cudaFuncSetAttribute(x2_ellpack_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem) != cudaSuccess)
            return BML_ERR_CUDA;
        attr_smem = smem;
    }
    int64_t grid = (N + nwarps - 1) / nwarps;
    if (grid > sms) grid = sms;
    if (grid > E_MAX_GRID) grid = E_MAX_GRID;
    // the (j, slot) sort buffer aliases the row stage: e_scratch_bytes(M) / 8 entries
    // buffer 0 is only read while parity == 0 (the standalone entry point passes a const X there)
    x2_ellpack_kernel<<<(unsigned)grid, nwarps * 32, smem, st>>>((double *)v0, (int32_t *)i0, (int32_t *)n0, v1, i1, n1,
                                                                 (int)N, M, tau, (int)(e_scratch_bytes(M) / 8), ctl, partials);
    BML_CHECK_LAUNCH();
    return 0;
}

int launch_rescale_ellpack(const bml_matrix_t *H, const double *d_bounds, double *xv, int32_t *xi, int32_t *xn,
                           double *diag, double *d_tr0, int *fail_flag, cudaStream_t st)
{
    const int N = (int)H->N, M = H->M;
    const int cap = next_pow2(M + 1) < 32 ? 32 : next_pow2(M + 1);
    const int nwarps = 4;
    const size_t smem = (size_t)nwarps * cap * 8;
    static size_t attr_smem = 48 * 1024;
    if (smem > attr_smem) {
        if (cudaFuncSetAttribute(rescale_ellpack_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem) != cudaSuccess)
            return BML_ERR_CUDA;
        attr_smem = smem;
    }
    rescale_ellpack_kernel<<<(N + nwarps - 1) / nwarps, nwarps * 32, smem, st>>>(H->value, H->index, H->nnz, N, M,
                                                                                  d_bounds, xv, xi, xn, diag,
                                                                                  fail_flag, cap);
    BML_CHECK_LAUNCH();
    sum_vector_kernel<<<1, 1024, 0, st>>>(diag, N, d_tr0);
    BML_CHECK_LAUNCH();
    return 0;
}

int launch_copy_out_ellpack(const double *v0, const int32_t *i0, const int32_t *n0, const double *v1,
                            const int32_t *i1, const int32_t *n1, int64_t N, int M, const Sp2Ctl *ctl, double *dv,
                            int32_t *di, int32_t *dn, cudaStream_t st)
{
    const int sms = sm_count();
    if (sms <= 0) return BML_ERR_CUDA;
    copy_out_ellpack_kernel<<<sms * 8, 256, 0, st>>>(v0, i0, n0, v1, i1, n1, N, M, ctl, dv, di, dn);
    BML_CHECK_LAUNCH();
    return 0;
}

int launch_x2_ellpack_info(const Sp2Ctl *ctl, int32_t *d_info, cudaStream_t st)
{
    x2_ellpack_info_kernel<<<1, 32, 0, st>>>(ctl, d_info);
    BML_CHECK_LAUNCH();
    return 0;
}

}  // namespace bmlsp2
