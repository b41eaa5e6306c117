// common.cuh -- shared device helpers of libbmlsp2 (sm_100a only): the device-resident SP2 control block,
// mbarrier / TMA / DMMA PTX wrappers, deterministic reductions.
#pragma once
#include <cuda.h>
#include <cuda_runtime.h>
#include <stdint.h>

#include "../../include/bml_sp2.h"

namespace bmlsp2 {

// ------------------------------------------------------------------------------------------------------------
// Device-resident control block of one SP2 solve.  Written only by the finaliser
// (the last CTA of each product kernel) and by the init kernel; read by every CTA at kernel start.  The host
// copies it back once, at the end of the solve.
// ------------------------------------------------------------------------------------------------------------
struct Sp2Ctl {
    int32_t m;             // index of the product that runs next (X_m is in buffer `parity`)
    int32_t done;          // 0 = running, 1 = stop rule fired or failure: later product launches exit at once
    int32_t status;        // BML_* once done
    int32_t parity;        // which ping-pong buffer holds X_m
    int32_t branch_cur;    // b_m = [tr X_m - n_occ <= 0], decided by the previous finaliser (Eq. 6-7)
    int32_t overflow_row;  // ellpack: lowest row of P_m = thr(X_m^2) with > M kept entries (INT32_MAX = none)
    int32_t overflow_upd;  // ellpack: lowest row of X_{m+1} with > M kept entries (INT32_MAX = none)
    int32_t acc_row;       // ellpack: lowest row that overflowed the hash accumulator (INT32_MAX = none)
    int32_t nnz_max_p;     // ellpack: max kept row length of P_m within the current product
    int32_t nnz_max_upd;   // ellpack: max kept row length of X_{m+1} within the current product
    int32_t fail_row;      // row reported to the host with status -3 / -6
    uint32_t arrivals;     // last-CTA-done counter of the current product
    int32_t n_occ;
    int32_t max_products;
    int32_t loop_mode;     // 1 = inside bml_sp2_* (apply stop rules), 0 = standalone bml_x2_* call
    int32_t n_done;        // number of X^2 products evaluated so far
    uint32_t epoch;        // launch counter of this solve (>= 1): tags the split-tile hand-off flags of the FP64 kernel
    double idem_tol;
    double tr_cur;         // tr X_m
    double emin, emax;
    double sums[4];        // { tr P, ||P - X||_F^2, ||X||_F^2, tr X' } of the last finished product
    uint8_t branch[BML_SP2_LOG_LEN];
    double trace[BML_SP2_LOG_LEN];
    double idem[BML_SP2_LOG_LEN];
    int32_t max_row_nnz[BML_SP2_LOG_LEN];
};

// Stop rules S1 / S2 / S3 and the next branch bit (DESIGN.md "Readings" items 3-7).  Called by ONE thread after the
// four sums of product m are final.  s = { tr P_m, ||P_m - X_m||^2, ||X_m||^2, tr X_{m+1} }.
__device__ __forceinline__ void sp2_finalise(Sp2Ctl *ctl, const double s[4])
{
    ctl->sums[0] = s[0]; ctl->sums[1] = s[1]; ctl->sums[2] = s[2]; ctl->sums[3] = s[3];
    ctl->arrivals = 0;
    ctl->epoch += 1u;
    if (!ctl->loop_mode) return;
    const int m = ctl->m;
    ctl->n_done = m + 1;
    const double e = sqrt(s[1]) / sqrt(s[2]);
    ctl->trace[m] = ctl->tr_cur;
    ctl->idem[m] = e;
    const int nnz_p = ctl->nnz_max_p, nnz_u = ctl->nnz_max_upd;
    ctl->max_row_nnz[m] = nnz_p;
    ctl->nnz_max_p = 0; ctl->nnz_max_upd = 0;
    int status = -100;
    // ELLPACK failures of the product itself come before the stop test (readings item 9; same order as the oracle)
    if (ctl->acc_row != INT32_MAX) { status = BML_ERR_ACC_CAPACITY; ctl->fail_row = ctl->acc_row; }
    else if (ctl->overflow_row != INT32_MAX) { status = BML_ERR_ELL_OVERFLOW; ctl->fail_row = ctl->overflow_row; }
    else if (e < ctl->idem_tol) status = BML_OK;                                               // S1
    else if (m >= 2 && e < 1e-2 && e >= ctl->idem[m - 2]) status = BML_NOISE_FLOOR;             // S2
    else if (m + 1 == ctl->max_products) status = BML_MAX_PRODUCTS;                             // S3
    else if (ctl->overflow_upd != INT32_MAX) {            // the update X_{m+1} is only needed when SP2 goes on
        status = BML_ERR_ELL_OVERFLOW; ctl->fail_row = ctl->overflow_upd;
        ctl->branch[m] = (uint8_t)ctl->branch_cur;
        if (nnz_u > nnz_p) ctl->max_row_nnz[m] = nnz_u;
    }
    if (status != -100) { ctl->done = 1; ctl->status = status; return; }   // D = X_m: `parity` is NOT flipped
    if (nnz_u > nnz_p) ctl->max_row_nnz[m] = nnz_u;
    ctl->branch[m] = (uint8_t)ctl->branch_cur;
    ctl->parity ^= 1;
    ctl->m = m + 1;
    ctl->tr_cur = s[3];
    ctl->branch_cur = (s[3] - (double)ctl->n_occ <= 0.0) ? 1 : 0;          // Eq. 6-7, "<=" of Listing 2
}

// ------------------------------------------------------------------------------------------------------------
// PTX wrappers
// ------------------------------------------------------------------------------------------------------------
__device__ __forceinline__ uint32_t smem_u32(const void *p) { return (uint32_t)__cvta_generic_to_shared(p); }

__device__ __forceinline__ void mbar_init(uint64_t *bar, uint32_t count)
{
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count));
}
__device__ __forceinline__ void mbar_fence_init()
{
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
}
__device__ __forceinline__ void fence_proxy_async()
{
    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
}
__device__ __forceinline__ void mbar_expect_tx(uint64_t *bar, uint32_t bytes)
{
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_arrive(uint64_t *bar)
{
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(smem_u32(bar)) : "memory");
}
__device__ __forceinline__ bool mbar_try_wait(uint64_t *bar, uint32_t parity)
{
    uint32_t ok;
    asm volatile(
        "{\n\t.reg .pred p;\n\t"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\t"
        "selp.u32 %0, 1, 0, p;\n\t}"
        : "=r"(ok)
        : "r"(smem_u32(bar)), "r"(parity)
        : "memory");
    return ok != 0;
}
__device__ __forceinline__ void mbar_wait(uint64_t *bar, uint32_t parity)
{
    while (!mbar_try_wait(bar, parity)) { }
}

// 2D tiled TMA load global -> shared, completion on an mbarrier (SASS UTMALDG).  c0 = innermost coordinate.
__device__ __forceinline__ void tma_load_2d(void *smem_dst, const CUtensorMap *map, int32_t c0, int32_t c1, uint64_t *bar)
{
    asm volatile(
        "cp.async.bulk.tensor.2d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%3, %4}], [%2];"
        ::"r"(smem_u32(smem_dst)), "l"(map), "r"(smem_u32(bar)), "r"(c0), "r"(c1)
        : "memory");
}
__device__ __forceinline__ void tma_prefetch_desc(const CUtensorMap *map)
{
    asm volatile("prefetch.tensormap [%0];" ::"l"(map) : "memory");
}

// FP64 tensor-core MMA, D(8x8) += A(8x4, row) * B(4x8, col).  SASS: DMMA.8x8x4.
// lane = 4*g + t:  a = A[g][t],  b = B[t][g],  c0/c1 = C[g][2t], C[g][2t+1].
__device__ __forceinline__ void dmma884(double &c0, double &c1, double a, double b)
{
    asm("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0, %1}, {%2}, {%3}, {%0, %1};"
                 : "+d"(c0), "+d"(c1)
                 : "d"(a), "d"(b));
}

__device__ __forceinline__ double warp_sum(double v)
{
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    return v;
}
__device__ __forceinline__ double warp_min(double v)
{
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v = fmin(v, __shfl_xor_sync(0xffffffffu, v, o));
    return v;
}
__device__ __forceinline__ double warp_max(double v)
{
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v = fmax(v, __shfl_xor_sync(0xffffffffu, v, o));
    return v;
}

// Neumaier-compensated accumulation: (s, c) represents s + c with ~2x the working precision
__device__ __forceinline__ void comp_add(double &s, double &c, double x)
{
    const double t = s + x;
    c += (fabs(s) >= fabs(x)) ? ((s - t) + x) : ((x - t) + s);
    s = t;
}
__device__ __forceinline__ void comp_merge(double &s, double &c, double s2, double c2)
{
    comp_add(s, c, s2);
    c += c2;
}
// all lanes return the same fixed-order compensated sum
__device__ __forceinline__ double comp_warp_sum(double s, double c)
{
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        const double s2 = __shfl_xor_sync(0xffffffffu, s, o), c2 = __shfl_xor_sync(0xffffffffu, c, o);
        // both partners must compute the same value: add in a symmetric order (larger |.| first is what
        // comp_add's branch does, so the result is independent of which lane is "s" and which is "s2")
        comp_merge(s, c, s2, c2);
    }
    return s + c;
}

// ------------------------------------------------------------------------------------------------------------
// Tile order of the symmetric-square kernels.  Upper-triangle tiles (I <= J) of a T x T tile grid are visited in
// super-blocks of G x G tiles (super-blocks column by column, tiles row by row inside one): the ~148 CTAs resident at
// any time then share 2 G row panels of X instead of ~150, so panels are re-read from L2, not from HBM.  Every
// super-block is launched with all G*G slots; slots below the diagonal or outside the grid exit at once (they still
// take part in the last-CTA count).
// ------------------------------------------------------------------------------------------------------------
constexpr int TILE_SB = 12;         // 12 x 12 = 144 tiles per super-block, about one wave of 148 SMs
// small grids (the whole iterate sits in L2 anyway) keep the plain triangular order, which has no empty slots
__host__ __device__ __forceinline__ bool tile_sb_plain(int T) { return T <= 2 * TILE_SB; }
__host__ __device__ __forceinline__ int tile_sb_grid(int T)
{
    if (tile_sb_plain(T)) return T * (T + 1) / 2;
    const int S = (T + TILE_SB - 1) / TILE_SB;
    return S * (S + 1) / 2 * TILE_SB * TILE_SB;
}
// t -> (i, j), i <= j, column by column: t = j (j + 1) / 2 + i
__host__ __device__ __forceinline__ void tri_decode(int t, int &i, int &j)
{
    j = (int)((sqrt(8.0 * (double)t + 1.0) - 1.0) * 0.5);
    while ((j + 1) * (j + 2) / 2 <= t) ++j;
    while (j * (j + 1) / 2 > t) --j;
    i = t - j * (j + 1) / 2;
}
__host__ __device__ __forceinline__ bool tile_sb_decode(int bid, int T, int &I, int &J)
{
    if (tile_sb_plain(T)) { tri_decode(bid, I, J); return true; }
    constexpr int GG = TILE_SB * TILE_SB;
    const int sb = bid / GG, w = bid - sb * GG;
    int bi, bj;
    tri_decode(sb, bi, bj);
    I = bi * TILE_SB + w / TILE_SB;
    J = bj * TILE_SB + w % TILE_SB;
    return I <= J && J < T;
}

// One-time host state (kernel attributes, SM counts, cooperative grid sizes) is kept PER DEVICE ORDINAL: a process may
// drive several GPUs, and cudaFuncSetAttribute / the SM count belong to the device that is current at the call.
constexpr int MAX_DEVICES = 64;
static inline int current_device()
{
    int d = -1;
    if (cudaGetDevice(&d) != cudaSuccess || d < 0 || d >= MAX_DEVICES) return -1;
    return d;
}
// raise a kernel's dynamic shared-memory limit to `bytes` once per device (`have` = per-device high-water mark)
template <class Kernel>
static inline int ensure_smem_attr(Kernel kernel, size_t bytes, size_t (&have)[MAX_DEVICES], size_t floor_bytes = 0)
{
    const int dev = current_device();
    if (dev < 0) return BML_ERR_CUDA;
    if (have[dev] < floor_bytes) have[dev] = floor_bytes;
    if (bytes > have[dev]) {
        if (cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)bytes) != cudaSuccess)
            return BML_ERR_CUDA;
        have[dev] = bytes;
    }
    return 0;
}
static inline int device_sm_count()
{
    static int sms[MAX_DEVICES] = {};
    const int dev = current_device();
    if (dev < 0) return 0;
    if (!sms[dev] && cudaDeviceGetAttribute(&sms[dev], cudaDevAttrMultiProcessorCount, dev) != cudaSuccess) sms[dev] = 0;
    return sms[dev];
}

// The same super-block order WITHOUT empty slots, for the persistent kernels that walk a dense list of tile numbers:
// t in [0, T (T + 1) / 2) -> (I, J), I <= J.  Super-blocks column by column; inside an off-diagonal super-block row by
// row, inside a diagonal one the triangular order.  At most S (S + 1) / 2 (~20) steps per work item of ~1 ms.
__host__ __device__ __forceinline__ void tri_sb_decode(int t, int T, int &I, int &J)
{
    if (tile_sb_plain(T)) { tri_decode(t, I, J); return; }
    const int S = (T + TILE_SB - 1) / TILE_SB;
    for (int bj = 0; bj < S; ++bj) {
        const int c0 = bj * TILE_SB, nc = (T - c0 < TILE_SB) ? T - c0 : TILE_SB;
        for (int bi = 0; bi <= bj; ++bi) {
            const int r0 = bi * TILE_SB, nr = (T - r0 < TILE_SB) ? T - r0 : TILE_SB;
            const int cnt = (bi == bj) ? nr * (nr + 1) / 2 : nr * nc;
            if (t < cnt) {
                if (bi == bj) { int i, j; tri_decode(t, i, j); I = r0 + i; J = c0 + j; }
                else { I = r0 + t / nc; J = c0 + t % nc; }
                return;
            }
            t -= cnt;
        }
    }
    I = J = T - 1;      // not reached for t < T (T + 1) / 2
}

// Host-side helpers (api.cu)
typedef CUresult (*PFN_encodeTiled)(CUtensorMap *, CUtensorMapDataType, cuuint32_t, void *, const cuuint64_t *,
                                    const cuuint64_t *, const cuuint32_t *, const cuuint32_t *, CUtensorMapInterleave,
                                    CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);
PFN_encodeTiled get_encode_tiled();

// Enqueue the product launches of one solve without ever letting the GPU wait for the host: the first batch and one
// batch AHEAD are always queued; after each batch the device-side stop flag is copied to pinned host memory and the
// host waits on an event recorded behind the batch BEFORE the one in flight.  Launches behind the stop flag exit at
// once on the device, so correctness never depends on the host seeing the flag; batching only bounds how many of
// them are issued (at most two batches instead of max_products - n_products).  These event waits are the only host
// synchronisation of a solve besides the final read of the control block, and they trail the device by a batch.
constexpr int ENQ_FIRST = 16, ENQ_BATCH = 8, ENQ_RING = 4;
struct EnqueueState {
    int32_t *h_done = nullptr;          // pinned, ENQ_RING slots
    cudaEvent_t ev[ENQ_RING] = {};
    bool ok = false;
    EnqueueState()
    {
        if (cudaHostAlloc((void **)&h_done, ENQ_RING * sizeof(int32_t), cudaHostAllocDefault) != cudaSuccess) return;
        for (int i = 0; i < ENQ_RING; ++i)
            if (cudaEventCreateWithFlags(&ev[i], cudaEventDisableTiming) != cudaSuccess) return;
        ok = true;
    }
};

EnqueueState &enqueue_state();      // api.cu: one per host thread

// `already`: product launches of the first batch that are in the stream already (a replayed CUDA graph, api.cu).
// `no_host_wait`: the caller asked for a fully asynchronous solve (stats == NULL): every one of the max_products
// launches is enqueued and the host never waits; the launches behind the stop flag cost a few microseconds each.
template <class LaunchFn>
static int enqueue_products(LaunchFn &&launch_one, Sp2Ctl *d_ctl, int max_products, cudaStream_t st, int already = 0,
                            bool no_host_wait = false)
{
    EnqueueState &es = enqueue_state();
    if (!es.ok || no_host_wait) {       // (or no pinned memory / events): plain enqueue of everything
        for (int l = already; l < max_products; ++l) { int r = launch_one(); if (r) return r; }
        return 0;
    }
    int enq = already, batch = 0;
    auto enqueue_batch = [&](int n) -> int {
        for (int l = 0; l < n && enq < max_products; ++l, ++enq) { int r = launch_one(); if (r) return r; }
        const int slot = batch % ENQ_RING;
        if (cudaMemcpyAsync(&es.h_done[slot], &d_ctl->done, sizeof(int32_t), cudaMemcpyDeviceToHost, st) != cudaSuccess ||
            cudaEventRecord(es.ev[slot], st) != cudaSuccess)
            return BML_ERR_CUDA;
        ++batch;
        return 0;
    };
    int r = enqueue_batch(ENQ_FIRST - already);
    if (r) return r;
    while (enq < max_products) {
        if ((r = enqueue_batch(ENQ_BATCH))) return r;          // one batch ahead ...
        const int prev = (batch - 2) % ENQ_RING;               // ... then look at the batch before it
        if (cudaEventSynchronize(es.ev[prev]) != cudaSuccess) return BML_ERR_CUDA;
        if (es.h_done[prev]) break;
    }
    return 0;
}


}  // namespace bmlsp2
