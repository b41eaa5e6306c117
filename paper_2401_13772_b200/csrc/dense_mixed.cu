// dense_mixed.cu -- mixed-precision dense X^2 (BASELINE.json configs[3]; not in the paper, readings item 17).
//
// X (FP64 master) is kept next to a split into 16-bit planes; one product tile P_IJ = sum_K X_IK X_JK^T is evaluated on
// the 5th-gen tensor cores (tcgen05.mma.kind::f16, operands staged by TMA, FP32 accumulators in TMEM) as a sum of
// plane cross terms.  The FP32 accumulator only ever holds a K-chunk of M_KC columns; every chunk is read back with
// tcgen05.ld and added to FP64 accumulators held in registers by the eight epilogue warps (two TMEM accumulator
// buffers: the next chunk's MMAs run while the previous chunk is promoted).  The FP64 epilogue is the one of the FP64
// kernel (Eq. 6 / Eq. 7, tr P, ||P - X||^2, ||X||^2, tr X', mirrored write, last-CTA finaliser) and additionally writes
// the planes of X' for the next product.  Two splits are built (bml_sp2_params_t::precision):
//
//   precision 1, FP16 x 2 (default):  X = Xh + 2^-11 Xl,  Xh = fp16(X), Xl = fp16(2^11 (X - Xh))   (2 x 11 bits; the
//       scaling keeps the residual plane out of the FP16 subnormal range).  Three cross terms per 16 columns of K:
//       Xh Xh^T into accumulator columns 0..127, Xh Xl^T and Xl Xh^T into columns 128..255.
//       Promotion:  acc += double(big + 2^-11 small).  The dropped Xl Xl^T term is <= 2^-22.
//       The large term hh has the accumulator to itself: 8 FP32 updates per chunk instead of 48.
//   precision 2, BF16 x 3:  X = Xh + Xm + Xl (bf16 each, 3 x 8 bits); the six cross terms of weight <= 2,
//       Xh Xl^T + Xl Xh^T + Xm Xm^T + Xh Xm^T + Xm Xh^T + Xh Xh^T, 12 MMAs (N = 128) per 32 columns, one accumulator.
//
// CTA pairs (round 2): a cluster of two CTAs (one TPC) computes a 256 x 128 tile with tcgen05.mma.cta_group::2 (M = 256,
// N = 128): CTA r of the pair holds the 128 rows 2 Ip + r of the A operand and HALF of the B operand (64 of the 128 rows
// of block row J); the tensor cores of both SMs read both halves.  Per k-slab a CTA therefore stages 1.5 operand tiles
// instead of 2: -25% of the L2 -> SM operand stream that bounds this kernel, and -25% shared-memory
// reads per MMA.  Each CTA keeps its own 128 x 128 accumulator tile (TMEM lanes of its own SM) and runs its own
// promotion and epilogue, exactly as a single CTA did.
//
// Roles (384 threads per CTA): warp 0 = TMA producer (one lane; both CTAs, completing on the LEADER's full barrier),
// warp 1 = MMA issuer (one lane, leader CTA only; tcgen05.commit multicasts to the barriers of both CTAs), warp 2 = TMEM
// allocator, warps 4..11 = epilogue (thread <-> one accumulator row, 64 columns).  Shared memory: STAGES x { A planes
// (128 rows) ; B half planes (64 rows) } x BK elements (K-major UMMA canonical layout; 128-byte rows / SWIZZLE_128B for
// the two-plane split, 64-byte rows / SWIZZLE_64B for the three-plane split).
#include <cuda_bf16.h>
#include <cuda_fp16.h>

#include "common.cuh"

namespace bmlsp2 {

constexpr int M_BM = 128;
constexpr int M_BN = 128;
constexpr int M_KC = 512;                      // K-chunk of the leading term promoted to FP64 (columns)
constexpr int M_EPI_WARPS = 8;
constexpr int M_CTRL_WARPS = 4;
constexpr int M_THREADS = (M_CTRL_WARPS + M_EPI_WARPS) * 32;
constexpr int M_REGS_CTRL = 56;
constexpr int M_REGS_EPI = 224;                // 128 x 56 + 256 x 224 = 64512
constexpr int M_MAX_PLANES = 3;

enum { MV_F16X2 = 1, MV_BF16X3 = 2 };          // = bml_sp2_params_t::precision

template <int V> struct MixedCfg;
// BK = 16-bit elements per k-slab: one shared-memory row of the K-major operand tile.  128-byte rows (SWIZZLE_128B)
// make every TMA request a full L2 line; the three-plane variant only has room for 64-byte rows (SWIZZLE_64B).
template <> struct MixedCfg<MV_F16X2> {
    // TMEM (512 columns): one accumulator S for hl + lh over the WHOLE K range (weight 2^-11: 2 N / 16 truncating
    // updates cost 2^-11 N / 8 ulp, 6e-8 relative at N = 16384), then three buffers of 128 columns for the chunks of hh
    static constexpr int PLANES = 2, BK = 64, STAGES = 4, NSBUF = 1, NBUF = 3;
    static constexpr int S_CHUNKS = 1 << 20;                                 // chunks per S period: never drained early
    static constexpr double S_WEIGHT = 0x1p-11;
    static constexpr uint32_t FMT = 0;                                       // F16
};
template <> struct MixedCfg<MV_BF16X3> {
    // TMEM: two accumulators S for the five terms of weight <= 2^-8, drained every S_CHUNKS chunks (2048 columns: 640
    // updates at 2^-7 of the leading term's magnitude), and two buffers for the chunks of hh
    static constexpr int PLANES = 3, BK = 32, STAGES = 6, NSBUF = 2, NBUF = 2;
    static constexpr int S_CHUNKS = 2048 / M_KC;
    static constexpr double S_WEIGHT = 1.0;
    static constexpr uint32_t FMT = 1;                                       // BF16
};

// tcgen05 instruction descriptor (kind::f16): D = F32, A/B format, both K-major, N, M = 256 (the CTA pair's tile)
__host__ __device__ constexpr uint32_t m_idesc(uint32_t fmt, int n)
{
    return (1u << 4) | (fmt << 7) | (fmt << 10) | ((uint32_t)(n >> 3) << 17) | ((uint32_t)((2 * M_BM) >> 4) << 24);
}

// shared-memory matrix descriptor: K-major, rows of ROW_BYTES (64: SWIZZLE_64B, 128: SWIZZLE_128B), 8-row groups
// 8 * ROW_BYTES apart, sm_100 descriptor version 1
template <int ROW_BYTES>
__device__ __forceinline__ uint64_t umma_desc(uint32_t saddr)
{
    constexpr uint64_t layout = ROW_BYTES == 128 ? 2ull : 4ull;
    return (uint64_t)((saddr >> 4) & 0x3FFFu) | ((uint64_t)((8u * ROW_BYTES) >> 4) << 32) | (1ull << 46) | (layout << 61);
}

__device__ __forceinline__ void umma_f16(uint32_t tmem_d, uint64_t adesc, uint64_t bdesc, uint32_t idesc,
                                         uint32_t accumulate)
{
    asm volatile(
        "{\n\t.reg .pred p;\n\t"
        "setp.ne.b32 p, %4, 0;\n\t"
        "tcgen05.mma.cta_group::2.kind::f16 [%0], %1, %2, %3, p;\n\t}"
        ::"r"(tmem_d), "l"(adesc), "l"(bdesc), "r"(idesc), "r"(accumulate)
        : "memory");
}
// arrives on the barrier at this shared-memory offset in BOTH CTAs of the pair when the MMAs issued so far are complete
__device__ __forceinline__ void umma_commit(uint64_t *bar)
{
    asm volatile("tcgen05.commit.cta_group::2.mbarrier::arrive::one.shared::cluster.multicast::cluster.b64 [%0], %1;"
                 ::"r"(smem_u32(bar)), "h"((uint16_t)3)
                 : "memory");
}
__device__ __forceinline__ uint32_t cluster_ctarank()
{
    uint32_t r;
    asm volatile("mov.u32 %0, %%cluster_ctarank;" : "=r"(r));
    return r;
}
// shared::cluster address of the same shared-memory location in CTA `rank` of the cluster
__device__ __forceinline__ uint32_t mapa_u32(uint32_t saddr, uint32_t rank)
{
    uint32_t r;
    asm volatile("mapa.shared::cluster.u32 %0, %1, %2;" : "=r"(r) : "r"(saddr), "r"(rank));
    return r;
}
__device__ __forceinline__ void mbar_arrive_cluster(uint32_t cluster_addr)
{
    // what the waiter needs ordered before this arrive is the completion of this warp's tcgen05.ld (tcgen05.wait::ld +
    // tcgen05.fence::before_thread_sync), not generic memory: the .release.cluster form costs a MEMBAR.ALL.GPU per
    // arrive (measured: 18.7 instead of 15.0 ms per product)
    asm volatile("mbarrier.arrive.shared::cluster.b64 _, [%0];" ::"r"(cluster_addr) : "memory");
}
__device__ __forceinline__ void cluster_sync_all()
{
    asm volatile("barrier.cluster.arrive.release.aligned;" ::: "memory");
    asm volatile("barrier.cluster.wait.acquire.aligned;" ::: "memory");
}
// TMA load of a CTA of the pair into its OWN shared memory, completing on a barrier given by its shared::cluster
// address (the leader's full barrier)
__device__ __forceinline__ void tma_load_2d_pair(void *smem_dst, const CUtensorMap *map, int32_t c0, int32_t c1,
                                                 uint32_t bar_cluster_addr)
{
    asm volatile(
        "cp.async.bulk.tensor.2d.cta_group::2.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%3, %4}], [%2];"
        ::"r"(smem_u32(smem_dst)), "l"(map), "r"(bar_cluster_addr), "r"(c0), "r"(c1)
        : "memory");
}

// Pair -> (Ip, J): the pair computes tiles (2 Ip, J) and (2 Ip + 1, J) of the upper triangle, J >= 2 Ip.  Large grids
// are visited in super-blocks of 6 pair rows x 12 columns (the 12 x 12 tile footprint of tile_sb_decode: the ~74
// resident pairs share 24 row panels); small ones column by column without empty slots.
constexpr int PAIR_SBI = TILE_SB / 2;
__host__ __device__ __forceinline__ int pair_grid(int T)
{
    if (tile_sb_plain(T)) {
        int n = 0;
        for (int j = 0; j < T; ++j) n += j / 2 + 1;
        return n;
    }
    const int S = (T + TILE_SB - 1) / TILE_SB;
    return S * (S + 1) / 2 * PAIR_SBI * TILE_SB;
}
__host__ __device__ __forceinline__ bool pair_decode(int pid, int T, int &Ip, int &J)
{
    if (tile_sb_plain(T)) {
        int j = 0, base = 0;
        while (base + j / 2 + 1 <= pid) { base += j / 2 + 1; ++j; }
        J = j; Ip = pid - base;
        return true;
    }
    constexpr int GG = PAIR_SBI * TILE_SB;
    const int sb = pid / GG, w = pid - sb * GG;
    int bi, bj;
    tri_decode(sb, bi, bj);
    Ip = bi * PAIR_SBI + w / TILE_SB;
    J = bj * TILE_SB + w % TILE_SB;
    return 2 * Ip <= J && J < T;
}
__device__ __forceinline__ void tc_fence_before() { asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory"); }
__device__ __forceinline__ void tc_fence_after() { asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory"); }

// 32 lanes x 16 consecutive FP32 columns of TMEM -> 16 registers per thread (thread = its own lane)
__device__ __forceinline__ void tmem_ld16(uint32_t taddr, uint32_t (&v)[16])
{
    asm volatile(
        "tcgen05.ld.sync.aligned.32x32b.x16.b32 "
        "{%0, %1, %2, %3, %4, %5, %6, %7, %8, %9, %10, %11, %12, %13, %14, %15}, [%16];"
        : "=r"(v[0]), "=r"(v[1]), "=r"(v[2]), "=r"(v[3]), "=r"(v[4]), "=r"(v[5]), "=r"(v[6]), "=r"(v[7]), "=r"(v[8]),
          "=r"(v[9]), "=r"(v[10]), "=r"(v[11]), "=r"(v[12]), "=r"(v[13]), "=r"(v[14]), "=r"(v[15])
        : "r"(taddr)
        : "memory");
}
__device__ __forceinline__ void tmem_ld_wait() { asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory"); }

// split of one FP64 value into the raw 16-bit patterns of the planes (round to nearest at every level)
template <int V>
__device__ __forceinline__ void split_planes(double x, uint16_t (&pl)[M_MAX_PLANES])
{
    if (V == MV_F16X2) {
        const __half h = __double2half(x);
        const double r1 = x - (double)__half2float(h);
        pl[0] = __half_as_ushort(h);
        pl[1] = __half_as_ushort(__double2half(r1 * 2048.0));
        pl[2] = 0;
    } else {
        const __nv_bfloat16 h = __double2bfloat16(x);
        const double r1 = x - (double)__bfloat162float(h);
        const __nv_bfloat16 m = __double2bfloat16(r1);
        const double r2 = r1 - (double)__bfloat162float(m);
        pl[0] = __bfloat16_as_ushort(h);
        pl[1] = __bfloat16_as_ushort(m);
        pl[2] = __bfloat16_as_ushort(__double2bfloat16(r2));
    }
}

// planes[p][r][c], p = 0 .. PLANES-1; leading dimension ldp elements
template <int V>
__global__ void __launch_bounds__(256)
split_planes_kernel(const double *__restrict__ X, int64_t ld, int N, uint16_t *__restrict__ planes, int64_t ldp)
{
    const int64_t plane = (int64_t)N * ldp;
    const int64_t total = (int64_t)N * N;
    for (int64_t e = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; e < total; e += (int64_t)gridDim.x * blockDim.x) {
        const int64_t r = e / N, c = e - r * N;
        uint16_t pl[M_MAX_PLANES];
        split_planes<V>(X[r * ld + c], pl);
#pragma unroll
        for (int p = 0; p < MixedCfg<V>::PLANES; ++p) planes[p * plane + r * ldp + c] = pl[p];
    }
}

// "FP64 traces" (BASELINE.json configs[3]): the diagonal of X^2 in full FP64 from the master iterate,
// dsq[i] = sum_k X_ik^2 (X symmetric), one warp per row, fixed summation order.  The product kernel writes these values on
// the diagonal instead of its mixed-precision ones, so tr(X^2) -- and with it tr X_{m+1}, which decides the next branch
// -- carries FP64 round-off only (the mixed products' one-sided truncation bias would otherwise sit in the trace:
// 4.5e-3 at N = 16384).  One extra read of X per product (HBM-bound, ~2% of the product time).
__global__ void __launch_bounds__(256)
diag_x2_fp64_kernel(const double *__restrict__ buf0, const double *__restrict__ buf1, int64_t ld, int N,
                    const Sp2Ctl *__restrict__ ctl, double *__restrict__ dsq)
{
    if (ctl->done) return;
    const double *__restrict__ X = ctl->parity ? buf1 : buf0;
    const int lane = threadIdx.x & 31;
    const int row = blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5);
    if (row >= N) return;
    const double *__restrict__ xr = X + (int64_t)row * ld;
    double s0 = 0.0, s1 = 0.0, s2 = 0.0, s3 = 0.0;
    int k = lane;
    for (; k + 96 < N; k += 128) {
        const double a = xr[k], b = xr[k + 32], c = xr[k + 64], d = xr[k + 96];
        s0 = fma(a, a, s0); s1 = fma(b, b, s1); s2 = fma(c, c, s2); s3 = fma(d, d, s3);
    }
    for (; k < N; k += 32) { const double a = xr[k]; s0 = fma(a, a, s0); }
    const double s = warp_sum((s0 + s1) + (s2 + s3));
    if (lane == 0) dsq[row] = s;
}

template <int V>
__global__ void __cluster_dims__(2, 1, 1) __launch_bounds__(M_THREADS, 1)
x2_dense_mixed_kernel(const __grid_constant__ CUtensorMap map0, const __grid_constant__ CUtensorMap map1,
                      double *__restrict__ buf0, double *__restrict__ buf1, uint16_t *__restrict__ pl0,
                      uint16_t *__restrict__ pl1, int64_t ld, int N, Sp2Ctl *__restrict__ ctl,
                      double *__restrict__ partials, const double *__restrict__ dsq)
{
    using Cfg = MixedCfg<V>;
    constexpr int PLANES = Cfg::PLANES, STAGES = Cfg::STAGES, NBUF = Cfg::NBUF, NSBUF = Cfg::NSBUF, M_BK = Cfg::BK;
    constexpr int BUF0 = NSBUF * M_BN, S_CHUNKS = Cfg::S_CHUNKS;
    constexpr int TMEM_COLS = 512;
    static_assert(BUF0 + NBUF * M_BN <= TMEM_COLS && 2048 % M_KC == 0, "TMEM plan");
    constexpr int M_PLANE_TILE = M_BM * M_BK * 2, M_KC_SLABS = M_KC / M_BK, ROWB = M_BK * 2;
    constexpr int M_HALF_TILE = M_PLANE_TILE / 2;                    // 64 rows of one plane
    constexpr int STAGE_BYTES = PLANES * (M_PLANE_TILE + M_HALF_TILE);
    if (ctl->done) return;
    const int parity = ctl->parity;
    const int branch = ctl->branch_cur;
    const CUtensorMap *map = parity ? &map1 : &map0;
    const double *__restrict__ X = parity ? buf1 : buf0;
    double *__restrict__ Xn = parity ? buf0 : buf1;
    uint16_t *__restrict__ Pn = parity ? pl0 : pl1;

    extern __shared__ uint8_t smem_raw[];
    uint8_t *smem = smem_raw + ((1024u - (smem_u32(smem_raw) & 1023u)) & 1023u);
    uint64_t *full_bar = (uint64_t *)(smem + (size_t)STAGES * STAGE_BYTES);   // used in the leader CTA only
    uint64_t *empty_bar = full_bar + STAGES;
    uint64_t *tfull_bar = empty_bar + STAGES;         // [NBUF] accumulator buffer ready for the epilogue
    uint64_t *tempty_bar = tfull_bar + NBUF;          // [NBUF] accumulator buffer drained by BOTH CTAs (leader's copy)
    uint64_t *sempty_bar = tempty_bar + NBUF;         // [NSBUF] S accumulator drained by both CTAs (leader's copy)
    double (*s_red)[4] = (double (*)[4])(sempty_bar + NSBUF);  // [M_EPI_WARPS][4]
    uint32_t *s_tmem = (uint32_t *)(s_red + M_EPI_WARPS);
    int *s_last = (int *)(s_tmem + 1);

    const int warp_all = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const uint32_t rank = cluster_ctarank();          // 0 = leader (issues the MMAs)
    const int T = (N + M_BM - 1) / M_BM;
    int Ip, J;
    const bool pvalid = pair_decode((int)(blockIdx.x >> 1), T, Ip, J);                  // cluster-uniform
    const int I = 2 * Ip + (int)rank;
    const bool valid = pvalid && I <= J && I < T;     // this CTA's tile is an upper-triangle tile (CTA-uniform)
    const bool diag = (I == J);
    const int nslabs = (N + M_BK - 1) / M_BK;
    const int nchunks = (nslabs + M_KC_SLABS - 1) / M_KC_SLABS;

    if (threadIdx.x == 0) {
        for (int s = 0; s < STAGES; ++s) { mbar_init(&full_bar[s], 1); mbar_init(&empty_bar[s], 1); }
        for (int b = 0; b < NBUF; ++b) { mbar_init(&tfull_bar[b], 1); mbar_init(&tempty_bar[b], 2 * M_EPI_WARPS); }
        for (int b = 0; b < NSBUF; ++b) mbar_init(&sempty_bar[b], 2 * M_EPI_WARPS);
        mbar_fence_init();
        fence_proxy_async();
    }
    if (threadIdx.x < M_EPI_WARPS * 4) ((double *)s_red)[threadIdx.x] = 0.0;     // empty slots contribute zero
    if (pvalid && warp_all == 2) {
        // the same warp of both CTAs allocates the pair's columns (same address in both SMs)
        asm volatile("tcgen05.alloc.cta_group::2.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(smem_u32(s_tmem)),
                     "n"(TMEM_COLS)
                     : "memory");
        asm volatile("tcgen05.relinquish_alloc_permit.cta_group::2.sync.aligned;" ::: "memory");
    }
    tc_fence_before();
    __syncthreads();
    cluster_sync_all();          // the peer's barriers are initialised before anything arrives on them
    tc_fence_after();
    const uint32_t tmem_base = *(volatile uint32_t *)s_tmem;

    if (!pvalid) {
        // pair slot below the diagonal / outside the tile grid: nothing to compute
    } else if (warp_all < M_CTRL_WARPS) {
        asm volatile("setmaxnreg.dec.sync.aligned.u32 %0;" ::"n"(M_REGS_CTRL));
        if (warp_all == 0 && lane == 0) {
            // ===================== TMA producer (both CTAs) =====================
            tma_prefetch_desc(map);
            // every load of the pair completes on the leader's full barrier, which expects the bytes of both CTAs
            uint32_t full_leader[STAGES];
#pragma unroll
            for (int s = 0; s < STAGES; ++s) full_leader[s] = mapa_u32(smem_u32(&full_bar[s]), 0);
            for (int slab = 0; slab < nslabs; ++slab) {
                const int s = slab % STAGES;
                const uint32_t ph = (uint32_t)(slab / STAGES) & 1u;
                mbar_wait(&empty_bar[s], ph ^ 1u);
                if (rank == 0) mbar_expect_tx(&full_bar[s], 2u * STAGE_BYTES);
                uint8_t *dst = smem + (size_t)s * STAGE_BYTES;
                uint32_t fl = full_leader[0];
#pragma unroll
                for (int q = 1; q < STAGES; ++q) fl = (s == q) ? full_leader[q] : fl;
#pragma unroll
                for (int p = 0; p < PLANES; ++p) {
                    // own 128 rows of the A operand (two boxes of 64 rows: one tensor map serves A and the B halves)
                    tma_load_2d_pair(dst + p * M_PLANE_TILE, map, slab * M_BK, p * N + I * M_BM, fl);
                    tma_load_2d_pair(dst + p * M_PLANE_TILE + M_HALF_TILE, map, slab * M_BK, p * N + I * M_BM + 64, fl);
                }
#pragma unroll
                for (int p = 0; p < PLANES; ++p)          // own half of the B operand: rows 64 rank .. 64 rank + 63 of block row J
                    tma_load_2d_pair(dst + PLANES * M_PLANE_TILE + p * M_HALF_TILE, map, slab * M_BK,
                                     p * N + J * M_BN + 64 * (int)rank, fl);
            }
        } else if (warp_all == 1 && lane == 0 && rank == 0) {
            // ===================== MMA issuer (leader CTA) =====================
            for (int slab = 0; slab < nslabs; ++slab) {
                const int s = slab % STAGES;
                const uint32_t ph = (uint32_t)(slab / STAGES) & 1u;
                const int chunk = slab / M_KC_SLABS, within = slab % M_KC_SLABS;
                const int buf = chunk % NBUF;
                const int period = chunk / S_CHUNKS, sbuf = period % NSBUF;
                const bool s_first = within == 0 && chunk % S_CHUNKS == 0;        // first slab of an S period
                if (within == 0) {
                    mbar_wait(&tempty_bar[buf], ((uint32_t)(chunk / NBUF) & 1u) ^ 1u);
                    if (s_first) mbar_wait(&sempty_bar[sbuf], ((uint32_t)(period / NSBUF) & 1u) ^ 1u);
                    tc_fence_after();
                }
                mbar_wait(&full_bar[s], ph);
                tc_fence_after();
                // descriptors are shared-memory OFFSETS: every CTA of the pair reads its own A rows and B half there
                const uint32_t a_base = smem_u32(smem + (size_t)s * STAGE_BYTES);
                const uint32_t b_base = a_base + PLANES * M_PLANE_TILE;
                const uint32_t d_tmem = tmem_base + (uint32_t)(BUF0 + buf * M_BN);      // chunk of the leading term
                const uint32_t s_tmem_acc = tmem_base + (uint32_t)(sbuf * M_BN);        // the small terms
                constexpr uint32_t IDESC = m_idesc(Cfg::FMT, M_BN);
                if (V == MV_F16X2) {
                    const uint64_t ah = umma_desc<ROWB>(a_base), al = umma_desc<ROWB>(a_base + M_PLANE_TILE);
                    const uint64_t bh = umma_desc<ROWB>(b_base), bl = umma_desc<ROWB>(b_base + M_HALF_TILE);
#pragma unroll
                    for (int ks = 0; ks < M_BK / 16; ++ks) {   // UMMA_K = 16 elements = 32 bytes = 2 descriptor units
                        umma_f16(s_tmem_acc, ah + 2 * ks, bl + 2 * ks, IDESC, (s_first && ks == 0) ? 0u : 1u);     // hl
                        umma_f16(s_tmem_acc, al + 2 * ks, bh + 2 * ks, IDESC, 1u);                                 // lh
                        umma_f16(d_tmem, ah + 2 * ks, bh + 2 * ks, IDESC, (within | ks) != 0 ? 1u : 0u);           // hh
                    }
                } else {
                    // cross terms of weight <= 2^-8, smallest first: (A plane, B plane)
                    const int ta[5] = {0, 2, 1, 0, 1};
                    const int tb[5] = {2, 0, 1, 1, 0};
#pragma unroll
                    for (int t = 0; t < 5; ++t) {
                        const uint64_t ad = umma_desc<ROWB>(a_base + ta[t] * M_PLANE_TILE);
                        const uint64_t bd = umma_desc<ROWB>(b_base + tb[t] * M_HALF_TILE);
#pragma unroll
                        for (int ks = 0; ks < M_BK / 16; ++ks)
                            umma_f16(s_tmem_acc, ad + 2 * ks, bd + 2 * ks, IDESC, (s_first && t == 0 && ks == 0) ? 0u : 1u);
                    }
                    const uint64_t ah = umma_desc<ROWB>(a_base), bh = umma_desc<ROWB>(b_base);
#pragma unroll
                    for (int ks = 0; ks < M_BK / 16; ++ks)
                        umma_f16(d_tmem, ah + 2 * ks, bh + 2 * ks, IDESC, (within | ks) != 0 ? 1u : 0u);           // hh
                }
                umma_commit(&empty_bar[s]);                   // frees the stage in both CTAs when these MMAs have read it
                if (within == M_KC_SLABS - 1 || slab == nslabs - 1) umma_commit(&tfull_bar[buf]);
            }
        }
    } else {
        // ===================== epilogue warps: promote every K-chunk to FP64, then the fused SP2 epilogue ============
        asm volatile("setmaxnreg.inc.sync.aligned.u32 %0;" ::"n"(M_REGS_EPI));
        const int e = warp_all - M_CTRL_WARPS;          // 0..7; TMEM lane quarter = warp_all % 4 = e % 4
        const int q = e & 3, half = e >> 2;
        double acc[64];
#pragma unroll
        for (int i = 0; i < 64; ++i) acc[i] = 0.0;
        const uint32_t t_lane = tmem_base + ((uint32_t)(q * 32) << 16) + (uint32_t)(half * 64);
        for (int chunk = 0; chunk < nchunks; ++chunk) {
            const int buf = chunk % NBUF;
            mbar_wait(&tfull_bar[buf], (uint32_t)(chunk / NBUF) & 1u);
            tc_fence_after();
#pragma unroll
            for (int g = 0; g < 4; g += 2) {
                uint32_t v[16], w[16];
                tmem_ld16(t_lane + (uint32_t)(BUF0 + buf * M_BN + g * 16), v);
                tmem_ld16(t_lane + (uint32_t)(BUF0 + buf * M_BN + g * 16 + 16), w);
                tmem_ld_wait();
#pragma unroll
                for (int i = 0; i < 16; ++i) acc[g * 16 + i] += (double)__uint_as_float(v[i]);
#pragma unroll
                for (int i = 0; i < 16; ++i) acc[g * 16 + 16 + i] += (double)__uint_as_float(w[i]);
            }
            tc_fence_before();
            __syncwarp();
            if (lane == 0) {      // the buffer is free when the epilogue warps of BOTH CTAs have drained it: leader's barrier
                if (rank == 0) mbar_arrive(&tempty_bar[buf]);
                else mbar_arrive_cluster(mapa_u32(smem_u32(&tempty_bar[buf]), 0));
            }
            if ((chunk + 1) % S_CHUNKS == 0 || chunk == nchunks - 1) {
                // end of an S period (the chunk's commit covers every earlier MMA): the small terms, weighted
                const int sbuf = (chunk / S_CHUNKS) % NSBUF;
#pragma unroll
                for (int g = 0; g < 4; g += 2) {
                    uint32_t v[16], w[16];
                    tmem_ld16(t_lane + (uint32_t)(sbuf * M_BN + g * 16), v);
                    tmem_ld16(t_lane + (uint32_t)(sbuf * M_BN + g * 16 + 16), w);
                    tmem_ld_wait();
#pragma unroll
                    for (int i = 0; i < 16; ++i) acc[g * 16 + i] += (double)__uint_as_float(v[i]) * Cfg::S_WEIGHT;
#pragma unroll
                    for (int i = 0; i < 16; ++i) acc[g * 16 + 16 + i] += (double)__uint_as_float(w[i]) * Cfg::S_WEIGHT;
                }
                tc_fence_before();
                __syncwarp();
                if (lane == 0) {
                    if (rank == 0) mbar_arrive(&sempty_bar[sbuf]);
                    else mbar_arrive_cluster(mapa_u32(smem_u32(&sempty_bar[sbuf]), 0));
                }
            }
        }

        // fused epilogue (D4), staged through shared memory so that every global access is a full row segment.  A
        // thread owns accumulator row r and 64 columns, i.e. a warp-wide access by accumulator ownership touches 32
        // different rows (8- and 2-byte scattered stores: measured 5 ms of a 17 ms product).  Instead: (1) the X tile
        // is read row by row into the (now idle) pipeline stages, (2) every thread updates its elements in place,
        // (3) the X' tile, its mirror and the planes are written row by row, 1 KB / 256 B contiguous per warp access.
        double s_trp = 0.0, s_e = 0.0, s_x = 0.0, s_trn = 0.0;
        // the second CTA of a pair on the diagonal (tile (2 Ip + 1, 2 Ip)) and rows beyond the grid took part in the MMAs
        // only: their tile is the mirror image of one computed elsewhere / does not exist
        if (valid) {
            constexpr int SS = M_BN + 1;                       // padded row stride (doubles): conflict-free column reads
            static_assert((size_t)M_BM * SS * 8 <= (size_t)STAGES * STAGE_BYTES, "tile staging must fit the stage ring");
            double *S = (double *)smem;
            const int rl = q * 32 + lane;                      // accumulator row inside the tile
            const int r = I * M_BM + rl;
            const int64_t plane = (int64_t)N * ld;
            // (1) rows e, e + 8, ... of the X tile; lane covers 4 consecutive columns (ld is a multiple of 16: in bounds)
            if (I * M_BM + M_BM <= N && J * M_BN + M_BN <= N) {
                // tile entirely inside the matrix: no bounds test, so the reads of 8 rows are in flight together (with the
                // loads inside the condition below, each of a warp's 16 rows costs one L2 round trip)
                constexpr int RA = 8;
                static_assert((M_BM / M_EPI_WARPS) % RA == 0, "read-ahead depth must divide the rows per warp");
                const double *xt = X + (int64_t)(I * M_BM + e) * ld + J * M_BN + lane * 4;
    #pragma unroll
                for (int k = 0; k < M_BM / M_EPI_WARPS; k += RA) {
                    double2 a[RA], bb[RA];
    #pragma unroll
                    for (int u = 0; u < RA; ++u) {
                        const double2 *src = (const double2 *)(xt + (int64_t)((k + u) * M_EPI_WARPS) * ld);
                        a[u] = src[0]; bb[u] = src[1];
                    }
    #pragma unroll
                    for (int u = 0; u < RA; ++u) {
                        double *dst = S + (e + (k + u) * M_EPI_WARPS) * SS + lane * 4;
                        dst[0] = a[u].x; dst[1] = a[u].y; dst[2] = bb[u].x; dst[3] = bb[u].y;
                    }
                }
            } else {
                for (int rr = e; rr < M_BM; rr += M_EPI_WARPS) {
                    const int gr = I * M_BM + rr, gc = J * M_BN + lane * 4;
                    if (gr < N && gc < N) {
                        const double2 *src = (const double2 *)(X + (int64_t)gr * ld + gc);
                        const double2 a = src[0], bb = src[1];
                        double *dst = S + rr * SS + lane * 4;
                        dst[0] = a.x; dst[1] = a.y; dst[2] = bb.x; dst[3] = bb.y;
                    }
                }
            }
            asm volatile("bar.sync 1, %0;" ::"n"(M_EPI_WARPS * 32) : "memory");
            // (2) update in place
            if (r < N) {
    #pragma unroll
                for (int i = 0; i < 64; ++i) {
                    const int cl = half * 64 + i, c = J * M_BN + cl;
                    if (c < N && (!diag || r <= c)) {
                        const double p = (r == c) ? dsq[r] : acc[i];       // FP64 diagonal (diag_x2_fp64_kernel)
                        const double x = S[rl * SS + cl];
                        const double d = p - x;
                        const double xn = branch ? (2.0 * x - p) : p;     // Eq. 7 : Eq. 6
                        S[rl * SS + cl] = xn;
                        if (r == c) { s_trp += p; s_trn += xn; s_e += d * d; s_x += x * x; }
                        else { s_e += 2.0 * (d * d); s_x += 2.0 * (x * x); }
                    }
                }
            }
            asm volatile("bar.sync 1, %0;" ::"n"(M_EPI_WARPS * 32) : "memory");
            // (3) write-out.  Diagonal tiles hold X' only for row <= column: the other half is read transposed, which
            // also makes X' bitwise symmetric; off-diagonal tiles are written twice, directly and mirrored.
            for (int pass = 0; pass < (diag ? 1 : 2); ++pass) {
                for (int rr = e; rr < M_BM; rr += M_EPI_WARPS) {
                    const int gr = (pass ? J : I) * M_BM + rr, gc = (pass ? I : J) * M_BN + lane * 4;
                    if (gr >= N || gc >= N) continue;
                    double v[4];
    #pragma unroll
                    for (int u = 0; u < 4; ++u) {
                        const int cl = lane * 4 + u;
                        v[u] = pass ? S[cl * SS + rr] : ((!diag || cl >= rr) ? S[rr * SS + cl] : S[cl * SS + rr]);
                    }
                    const int64_t o = (int64_t)gr * ld + gc;
                    uint16_t pl[4][M_MAX_PLANES];
    #pragma unroll
                    for (int u = 0; u < 4; ++u) split_planes<V>(v[u], pl[u]);
                    if (gc + 3 < N) {
                        double2 *dst = (double2 *)(Xn + o);
                        dst[0] = make_double2(v[0], v[1]);
                        dst[1] = make_double2(v[2], v[3]);
    #pragma unroll
                        for (int k = 0; k < PLANES; ++k) {
                            uint2 w;
                            w.x = (uint32_t)pl[0][k] | ((uint32_t)pl[1][k] << 16);
                            w.y = (uint32_t)pl[2][k] | ((uint32_t)pl[3][k] << 16);
                            *(uint2 *)(Pn + k * plane + o) = w;
                        }
                    } else {
    #pragma unroll
                        for (int u = 0; u < 4; ++u) {
                            if (gc + u < N) {
                                Xn[o + u] = v[u];
    #pragma unroll
                                for (int k = 0; k < PLANES; ++k) Pn[k * plane + o + u] = pl[u][k];
                            }
                        }
                    }
                }
            }
        }
        s_trp = warp_sum(s_trp); s_e = warp_sum(s_e); s_x = warp_sum(s_x); s_trn = warp_sum(s_trn);
        if (lane == 0) { s_red[e][0] = s_trp; s_red[e][1] = s_e; s_red[e][2] = s_x; s_red[e][3] = s_trn; }
    }
    tc_fence_before();
    __syncthreads();
    cluster_sync_all();          // nothing of the peer (remote arrives, multicast commits, its MMAs' reads) is still on its way
    if (pvalid && warp_all == 2) {
        tc_fence_after();
        asm volatile("tcgen05.dealloc.cta_group::2.sync.aligned.b32 %0, %1;" ::"r"(tmem_base), "n"(TMEM_COLS) : "memory");
    }

    // ===================== per-tile partials, last-CTA finaliser (D5) =====================
    if (threadIdx.x < 4) {
        double v = 0.0;
#pragma unroll
        for (int w = 0; w < M_EPI_WARPS; ++w) v += s_red[w][threadIdx.x];
        partials[(size_t)blockIdx.x * 4 + threadIdx.x] = v;
        __threadfence();
    }
    __syncthreads();
    if (threadIdx.x == 0) {
        __threadfence();      // release: cumulative over the partial sums the barrier above ordered before this thread
        const uint32_t prev = atomicAdd(&ctl->arrivals, 1u);
        __threadfence();      // acquire, before the barrier below hands the verdict to the finalising warp
        *s_last = (prev + 1u == gridDim.x);
    }
    __syncthreads();
    if (*s_last && warp_all == 0) {
        __threadfence();
        double s[4] = {0.0, 0.0, 0.0, 0.0};
        const volatile double *vp = partials;
        for (int tI = lane; tI < (int)gridDim.x; tI += 32) {
#pragma unroll
            for (int k = 0; k < 4; ++k) s[k] += vp[(size_t)tI * 4 + k];
        }
#pragma unroll
        for (int k = 0; k < 4; ++k) s[k] = warp_sum(s[k]);
        if (lane == 0) sp2_finalise(ctl, s);
    }
}

// ------------------------------------------------------------------------------------------------------------
// host side
// ------------------------------------------------------------------------------------------------------------
// number of CTAs (= per-CTA partial-sum slots) of one mixed product: two per pair slot (128 x 128 tile per CTA)
int dense_mixed_num_tiles(int64_t N) { return 2 * pair_grid((int)((N + M_BM - 1) / M_BM)); }

// host-side view of the CTA -> tile map of the mixed kernel (the same pair_decode() the device runs); 1 = this CTA
// writes no tile (empty pair slot, the below-diagonal half of a pair on the diagonal, or a row beyond the grid)
int dense_mixed_tile_of_cta(int64_t N, int cta, int32_t out[2])
{
    const int T = (int)((N + M_BM - 1) / M_BM);
    if (N < 1 || cta < 0 || cta >= 2 * pair_grid(T)) return BML_ERR_INVALID;
    int Ip, J;
    if (!pair_decode(cta >> 1, T, Ip, J)) return 1;
    const int I = 2 * Ip + (cta & 1);
    if (I > J || I >= T) return 1;
    out[0] = I; out[1] = J;
    return 0;
}

// the planes of one iterate, stacked: rows p * N + r, leading dimension ldp (= the FP64 iterate's ld)
template <int V>
static int make_plane_map(CUtensorMap *map, const uint16_t *base, int64_t N, int64_t ldp)
{
    PFN_encodeTiled enc = get_encode_tiled();
    if (!enc) return BML_ERR_CUDA;
    const cuuint64_t dims[2] = {(cuuint64_t)N, (cuuint64_t)(MixedCfg<V>::PLANES * N)};
    const cuuint64_t strides[1] = {(cuuint64_t)ldp * sizeof(uint16_t)};
    const cuuint32_t box[2] = {(cuuint32_t)MixedCfg<V>::BK, 64u};      // half a tile: A = two boxes, B half = one
    const cuuint32_t estr[2] = {1, 1};
    CUresult r = enc(map, V == MV_F16X2 ? CU_TENSOR_MAP_DATA_TYPE_FLOAT16 : CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, 2,
                     (void *)base, dims, strides, box, estr, CU_TENSOR_MAP_INTERLEAVE_NONE,
                     MixedCfg<V>::BK == 64 ? CU_TENSOR_MAP_SWIZZLE_128B : CU_TENSOR_MAP_SWIZZLE_64B,
                     CU_TENSOR_MAP_L2_PROMOTION_L2_256B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    return r == CUDA_SUCCESS ? 0 : BML_ERR_CUDA;
}

// room for the larger split (3 planes) so that the workspace size does not depend on the variant
static inline size_t plane_set_bytes(int64_t N, int64_t ldx)
{
    return ((size_t)M_MAX_PLANES * (size_t)N * (size_t)ldx * sizeof(uint16_t) + 1023) / 1024 * 1024;
}

size_t dense_mixed_extra_bytes(int64_t N, int64_t ldx)
{
    return 2 * plane_set_bytes(N, ldx) + ((size_t)N * sizeof(double) + 1023) / 1024 * 1024;     // + dsq[N]
}

template <int V>
static int launch_split(const double *X, int64_t ld, int64_t N, uint16_t *planes, cudaStream_t st)
{
    int64_t blocks = (N * N + 255) / 256;
    if (blocks > 148 * 16) blocks = 148 * 16;
    split_planes_kernel<V><<<(unsigned)blocks, 256, 0, st>>>(X, ld, (int)N, planes, ld);
    return cudaGetLastError() == cudaSuccess ? 0 : BML_ERR_CUDA;
}

template <int V>
static int launch_x2_mixed(const CUtensorMap &m0, const CUtensorMap &m1, double *b0, double *b1, uint16_t *p0,
                           uint16_t *p1, int64_t ld, int64_t N, Sp2Ctl *ctl, double *partials, double *dsq,
                           cudaStream_t st)
{
    constexpr size_t smem = (size_t)MixedCfg<V>::STAGES * MixedCfg<V>::PLANES * (M_BM * MixedCfg<V>::BK * 2) * 3 / 2 +
                            1024 /*align*/ + 1024 /*barriers, scratch*/;
    static size_t have[MAX_DEVICES] = {};
    if (ensure_smem_attr(x2_dense_mixed_kernel<V>, smem, have)) return BML_ERR_CUDA;
    diag_x2_fp64_kernel<<<(unsigned)((N + 7) / 8), 256, 0, st>>>(b0, b1, ld, (int)N, ctl, dsq);
    x2_dense_mixed_kernel<V><<<dense_mixed_num_tiles(N), M_THREADS, smem, st>>>(m0, m1, b0, b1, p0, p1, ld, (int)N, ctl,
                                                                                partials, dsq);
    return cudaGetLastError() == cudaSuccess ? 0 : BML_ERR_CUDA;
}

template <int V>
static int solve_v(int64_t N, int max_products, double *X0, double *X1, int64_t ldx, Sp2Ctl *ctl, double *partials,
                   void *extra, cudaStream_t st, bool no_host_wait = false)
{
    uint16_t *p0 = (uint16_t *)extra;
    uint16_t *p1 = (uint16_t *)((uint8_t *)extra + plane_set_bytes(N, ldx));
    double *dsq = (double *)((uint8_t *)extra + 2 * plane_set_bytes(N, ldx));
    CUtensorMap m0, m1;
    int r;
    if ((r = make_plane_map<V>(&m0, p0, N, ldx))) return r;
    if ((r = make_plane_map<V>(&m1, p1, N, ldx))) return r;
    if ((r = launch_split<V>(X0, ldx, N, p0, st))) return r;
    if (max_products == 1) return launch_x2_mixed<V>(m0, m1, X0, X1, p0, p1, ldx, N, ctl, partials, dsq, st);
    return enqueue_products([&]() { return launch_x2_mixed<V>(m0, m1, X0, X1, p0, p1, ldx, N, ctl, partials, dsq, st); },
                            ctl, max_products, st, 0, no_host_wait);
}

// X0 (already rescaled, in buffer 0) -> planes of buffer 0, then the fused products
int sp2_dense_mixed_solve(const bml_matrix_t *H, const bml_sp2_params_t *p, double *X0, double *X1, int64_t ldx,
                          Sp2Ctl *ctl, double *partials, const double *, void *extra, cudaStream_t st, bool no_host_wait)
{
    if (p->precision == MV_BF16X3)
        return solve_v<MV_BF16X3>(H->N, p->max_products, X0, X1, ldx, ctl, partials, extra, st, no_host_wait);
    return solve_v<MV_F16X2>(H->N, p->max_products, X0, X1, ldx, ctl, partials, extra, st, no_host_wait);
}

// one product on a caller-supplied iterate (the control block was initialised in standalone mode)
int x2_dense_mixed_once(const bml_matrix_t *X, bml_matrix_t *Xn, int precision, Sp2Ctl *ctl, double *partials,
                        void *extra, cudaStream_t st)
{
    if (precision == MV_BF16X3) return solve_v<MV_BF16X3>(X->N, 1, X->value, Xn->value, X->ld, ctl, partials, extra, st);
    return solve_v<MV_F16X2>(X->N, 1, X->value, Xn->value, X->ld, ctl, partials, extra, st);
}

}  // namespace bmlsp2
