// dense_fp64.cu -- steps D3 + D4 + D5 of DESIGN.md: the fused FP64 symmetric-square kernel.
//
//   P_IJ = sum_K X_IK * X_JK^T      (X symmetric, so X^2 = X X^T: both operands are ROW panels of X, K-contiguous)
//   only tiles I <= J are computed; the epilogue applies Eq. 6 / Eq. 7, accumulates tr P, ||P - X||_F^2,
//   ||X||_F^2, tr X', and writes X'_IJ and its mirror X'_JI.  The last CTA reduces the per-tile partial sums in a
//   fixed order and runs the stop rules / next branch bit on the device (no host round trip, P:201-208 done on-chip).
//
// Pipeline: one producer thread issues TMA (cp.async.bulk.tensor, 128B swizzle, FP64 tensor map) into a STAGES-deep
// ring of { A panel 128 x 16, B panel 128 x 16 } tiles guarded by full/empty mbarriers; 8 consumer warps (2 x 4, warp
// tile 64 x 32) read fragments with conflict-free LDS.64 and issue mma.sync m8n8k4 f64 (SASS DMMA.8x8x4).
#include <cooperative_groups.h>

#include "dense_fp64_core.cuh"

namespace cg = cooperative_groups;

namespace bmlsp2 {


template <int BT>
__global__ void __launch_bounds__(D_THREADS, 1)
x2_dense_fp64_kernel(const __grid_constant__ CUtensorMap map0, const __grid_constant__ CUtensorMap map1,
                     double *__restrict__ buf0, double *__restrict__ buf1, int64_t ld, int N,
                     Sp2Ctl *__restrict__ ctl, double *__restrict__ partials)
{
    constexpr int D_BM = BT, D_BN = BT, D_PANEL_BYTES = d_panel_bytes(BT), D_STAGE_BYTES = d_stage_bytes(BT);
    constexpr int MI = BT / 16, NI = BT / 32;        // 8 x 8 fragments per warp tile (BT/2) x (BT/4)
    // every CTA sees the control block written by the previous product's finaliser (kernel boundary orders it)
    if (ctl->done) return;
    const int parity = ctl->parity;
    const int branch = ctl->branch_cur;
    const CUtensorMap *map = parity ? &map1 : &map0;
    const double *__restrict__ X = parity ? buf1 : buf0;
    double *__restrict__ Xn = parity ? buf0 : buf1;

    extern __shared__ uint8_t smem_raw[];
    // SWIZZLE_128B tiles need 1024-byte alignment; pointer arithmetic (no integer round trip) keeps the shared
    // address space visible to the compiler so fragment loads stay LDS
    uint8_t *smem = smem_raw + ((1024u - (smem_u32(smem_raw) & 1023u)) & 1023u);
    uint64_t *full_bar = (uint64_t *)(smem + (size_t)D_STAGES * D_STAGE_BYTES);
    uint64_t *empty_bar = full_bar + D_STAGES;
    double (*s_red)[4] = (double (*)[4])(empty_bar + D_STAGES);          // [D_CONSUMER_WARPS][4]
    int *s_last = (int *)(s_red + D_CONSUMER_WARPS);

    const int warp_all = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int warp = warp_all - D_PRODUCER_WARPS;      // consumer warp index 0..7 (negative: producer warpgroup)
    int I, J;
    const bool valid = tile_sb_decode((int)blockIdx.x, (N + D_BM - 1) / D_BM, I, J);    // CTA-uniform
    const bool diag = (I == J);
    const int KT = (N + D_BK - 1) / D_BK;

    if (threadIdx.x == 0) {
        for (int s = 0; s < D_STAGES; ++s) { mbar_init(&full_bar[s], 1); mbar_init(&empty_bar[s], D_CONSUMER_WARPS); }
        mbar_fence_init();
        fence_proxy_async();
    }
    if (threadIdx.x < D_CONSUMER_WARPS * 4) ((double *)s_red)[threadIdx.x] = 0.0;     // empty slots contribute zero
    __syncthreads();

    if (!valid) {
        // slot below the diagonal / outside the tile grid: nothing to compute
    } else if (warp < 0) {
        // ===================== TMA producer warpgroup (one elected lane works) =====================
        asm volatile("setmaxnreg.dec.sync.aligned.u32 %0;" ::"n"(D_REGS_PRODUCER));
        if (warp_all == 0 && lane == 0) {
            tma_prefetch_desc(map);
            const uint32_t tx = diag ? D_PANEL_BYTES : D_STAGE_BYTES;
            for (int kt = 0; kt < KT; ++kt) {
                const int s = kt % D_STAGES;
                const uint32_t ph = (uint32_t)(kt / D_STAGES) & 1u;
                mbar_wait(&empty_bar[s], ph ^ 1u);   // first pass over the ring: passes immediately
                mbar_expect_tx(&full_bar[s], tx);
                uint8_t *dst = smem + (size_t)s * D_STAGE_BYTES;
                tma_load_2d(dst, map, kt * D_BK, I * D_BM, &full_bar[s]);
                if (!diag) tma_load_2d(dst + D_PANEL_BYTES, map, kt * D_BK, J * D_BN, &full_bar[s]);
            }
        }
        // producer warp falls through to the final reduction barrier
    } else {
        // ===================== DMMA consumers =====================
        asm volatile("setmaxnreg.inc.sync.aligned.u32 %0;" ::"n"(D_REGS_CONSUMER));
        const int wm = warp >> 2, wn = warp & 3;     // 2 x 4 warps; warp tile 64 x 32
        double acc[MI][NI][2];
#pragma unroll
        for (int i = 0; i < MI; ++i)
#pragma unroll
            for (int j = 0; j < NI; ++j) { acc[i][j][0] = 0.0; acc[i][j][1] = 0.0; }

        uint32_t koff[4];
        dmma_koff(lane, koff);
        const uint8_t *a_base = smem + wm * (D_BM / 2) * 128;
        const uint8_t *b_base = smem + (diag ? 0 : D_PANEL_BYTES) + wn * (D_BN / 4) * 128;

        StageRelease release;   // stages go back to the producer one slab late (dense_fp64_core.cuh)
        for (int kt = 0; kt < KT; ++kt) {
            const int s = kt % D_STAGES;
            const uint32_t ph = (uint32_t)(kt / D_STAGES) & 1u;
            mbar_wait(&full_bar[s], ph);
            const uint8_t *sa = a_base + (size_t)s * D_STAGE_BYTES, *sb = b_base + (size_t)s * D_STAGE_BYTES;
            dmma_slab<MI, NI>(acc, sa, sb, koff);
            release.after_slab(empty_bar, s, lane);
        }

        // ===================== fused epilogue (D4) =====================
        double s_trp = 0.0, s_e = 0.0, s_x = 0.0, s_trn = 0.0;
        sp2_tile_epilogue<MI, NI, BT>(acc, X, Xn, ld, N, I, J, wm, wn, lane, branch, s_trp, s_e, s_x, s_trn);
        s_trp = warp_sum(s_trp); s_e = warp_sum(s_e); s_x = warp_sum(s_x); s_trn = warp_sum(s_trn);
        if (lane == 0) { s_red[warp][0] = s_trp; s_red[warp][1] = s_e; s_red[warp][2] = s_x; s_red[warp][3] = s_trn; }
    }
    __syncthreads();

    // ===================== per-tile partials, last-CTA finaliser (D5) =====================
    if (threadIdx.x < 4) {
        double v = 0.0;
#pragma unroll
        for (int w = 0; w < D_CONSUMER_WARPS; ++w) v += s_red[w][threadIdx.x];
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
            for (int q = 0; q < 4; ++q) s[q] += vp[(size_t)tI * 4 + q];
        }
#pragma unroll
        for (int q = 0; q < 4; ++q) s[q] = warp_sum(s[q]);
        if (lane == 0) sp2_finalise(ctl, s);
    }
}

// ------------------------------------------------------------------------------------------------------------
// Whole-solve variant for small matrices (N <= 1024: one CTA per tile fits one wave of co-resident CTAs): ALL products of
// an SP2 solve in ONE cooperative launch.  A product there is 5-40 us of work against ~18 us per kernel launch + drain, so
// the launch sequence, not the arithmetic, set time-to-D (0.27 ms at N = 256 for 15 products; "fast
// time-to-solution" at about a thousand orbitals is the paper's use case).  Between products: the last CTA's finaliser
// (stop rules, next branch bit), then a grid barrier; the epilogue's global writes are fenced for the async proxy because
// the next product's TMA loads read them.  The TMA ring and its mbarrier phases run on across products.
// ------------------------------------------------------------------------------------------------------------
// ring depth of the whole-solve kernel: small tiles have small stages (8 KB at BT = 32, 16 KB at BT = 64)
constexpr int loop_stages(int BT) { return BT == 32 ? 16 : 12; }
constexpr size_t loop_smem_bytes(int BT) { return (size_t)loop_stages(BT) * d_stage_bytes(BT) + 1024 + 1024; }

template <int BT>
__global__ void __launch_bounds__(D_THREADS, 1)
sp2_dense_fp64_loop_kernel(const __grid_constant__ CUtensorMap map0, const __grid_constant__ CUtensorMap map1,
                           double *__restrict__ buf0, double *__restrict__ buf1, int64_t ld, int N,
                           Sp2Ctl *__restrict__ ctl, double *__restrict__ partials, int max_products)
{
    constexpr int D_BM = BT, D_BN = BT, D_PANEL_BYTES = d_panel_bytes(BT), D_STAGE_BYTES = d_stage_bytes(BT);
    constexpr int MI = BT / 16, NI = BT / 32;
    constexpr int ST = loop_stages(BT);          // deep ring: (almost) a whole row panel pair in flight
    cg::grid_group grid = cg::this_grid();

    extern __shared__ uint8_t smem_raw[];
    uint8_t *smem = smem_raw + ((1024u - (smem_u32(smem_raw) & 1023u)) & 1023u);
    uint64_t *full_bar = (uint64_t *)(smem + (size_t)ST * D_STAGE_BYTES);
    uint64_t *empty_bar = full_bar + ST;
    double (*s_red)[4] = (double (*)[4])(empty_bar + ST);
    int *s_last = (int *)(s_red + D_CONSUMER_WARPS);

    const int warp_all = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int warp = warp_all - D_PRODUCER_WARPS;
    int I, J;
    const bool valid = tile_sb_decode((int)blockIdx.x, (N + D_BM - 1) / D_BM, I, J);
    const bool diag = (I == J);
    const int KT = (N + D_BK - 1) / D_BK;

    if (threadIdx.x == 0) {
        for (int s = 0; s < ST; ++s) { mbar_init(&full_bar[s], 1); mbar_init(&empty_bar[s], D_CONSUMER_WARPS); }
        mbar_fence_init();
        fence_proxy_async();
    }
    __syncthreads();
    if (warp < 0) asm volatile("setmaxnreg.dec.sync.aligned.u32 %0;" ::"n"(D_REGS_PRODUCER));
    else asm volatile("setmaxnreg.inc.sync.aligned.u32 %0;" ::"n"(D_REGS_CONSUMER));

    int slab = 0;                       // runs on across products (both roles count the same slabs)
    StageRelease release;
    uint32_t koff[4];
    dmma_koff(lane, koff);
    // Every CTA keeps its own copy of the loop state and takes the stop / branch decision itself from the same per-CTA
    // partial sums added in the same order (bitwise identical in every CTA), so a product costs ONE grid barrier and one
    // read of the partials; CTA 0 alone writes the control block (logs, parity, status) for the host and the copy-out.
    int m = ctl->m, parity = ctl->parity, branch = ctl->branch_cur;
    bool done = ctl->done != 0;
    const int loop_mode = ctl->loop_mode, n_occ = ctl->n_occ;
    const double idem_tol = ctl->idem_tol;
    double e_prev1 = 0.0, e_prev2 = 0.0;          // e_{m-1}, e_{m-2}
    for (int it = 0; it < max_products && !done; ++it) {
        const CUtensorMap *map = parity ? &map1 : &map0;
        const double *__restrict__ X = parity ? buf1 : buf0;
        double *__restrict__ Xn = parity ? buf0 : buf1;
        double *part = partials + (size_t)(it & 1) * gridDim.x * 4;      // two sets: a fast CTA may already write the next
        if (threadIdx.x < D_CONSUMER_WARPS * 4) ((double *)s_red)[threadIdx.x] = 0.0;
        __syncthreads();
        if (!valid) {
        } else if (warp < 0) {
            if (warp_all == 0 && lane == 0) {
                const uint32_t tx = diag ? D_PANEL_BYTES : D_STAGE_BYTES;
                for (int kt = 0; kt < KT; ++kt, ++slab) {
                    const int s = slab % ST;
                    const uint32_t ph = (uint32_t)(slab / ST) & 1u;
                    mbar_wait(&empty_bar[s], ph ^ 1u);
                    mbar_expect_tx(&full_bar[s], tx);
                    uint8_t *dst = smem + (size_t)s * D_STAGE_BYTES;
                    tma_load_2d(dst, map, kt * D_BK, I * D_BM, &full_bar[s]);
                    if (!diag) tma_load_2d(dst + D_PANEL_BYTES, map, kt * D_BK, J * D_BN, &full_bar[s]);
                }
            }
        } else {
            const int wm = warp >> 2, wn = warp & 3;
            double acc[MI][NI][2];
#pragma unroll
            for (int i = 0; i < MI; ++i)
#pragma unroll
                for (int j = 0; j < NI; ++j) { acc[i][j][0] = 0.0; acc[i][j][1] = 0.0; }
            const uint8_t *a_base = smem + wm * (D_BM / 2) * 128;
            const uint8_t *b_base = smem + (diag ? 0 : D_PANEL_BYTES) + wn * (D_BN / 4) * 128;
            for (int kt = 0; kt < KT; ++kt, ++slab) {
                const int s = slab % ST;
                const uint32_t ph = (uint32_t)(slab / ST) & 1u;
                mbar_wait(&full_bar[s], ph);
                const uint8_t *sa = a_base + (size_t)s * D_STAGE_BYTES, *sb = b_base + (size_t)s * D_STAGE_BYTES;
                dmma_slab<MI, NI>(acc, sa, sb, koff);
                release.after_slab(empty_bar, s, lane);
            }
            double s_trp = 0.0, s_e = 0.0, s_x = 0.0, s_trn = 0.0;
            sp2_tile_epilogue<MI, NI, BT>(acc, X, Xn, ld, N, I, J, wm, wn, lane, branch, s_trp, s_e, s_x, s_trn);
            s_trp = warp_sum(s_trp); s_e = warp_sum(s_e); s_x = warp_sum(s_x); s_trn = warp_sum(s_trn);
            if (lane == 0) { s_red[warp][0] = s_trp; s_red[warp][1] = s_e; s_red[warp][2] = s_x; s_red[warp][3] = s_trn; }
            // X' is read by the next product's TMA loads (async proxy): order this thread's global writes before them
            asm volatile("fence.proxy.async;" ::: "memory");
        }
        __syncthreads();
        if (threadIdx.x < 4) {
            double v = 0.0;
#pragma unroll
            for (int w = 0; w < D_CONSUMER_WARPS; ++w) v += s_red[w][threadIdx.x];
            __stcg(&part[(size_t)blockIdx.x * 4 + threadIdx.x], v);
        }
        // no __threadfence() here: grid.sync() orders every thread's earlier global writes (X', the partial sums) before
        // every thread's later reads; a fence per thread on top of it cost 3.9 us per product (measured, N = 256)
        grid.sync();
        // every warp adds the partials in the same fixed order: all threads of all CTAs hold identical sums
        double sm[4] = {0.0, 0.0, 0.0, 0.0};
        for (int tI = lane; tI < (int)gridDim.x; tI += 32) {
#pragma unroll
            for (int q = 0; q < 4; ++q) sm[q] += __ldcg(&part[(size_t)tI * 4 + q]);
        }
#pragma unroll
        for (int q = 0; q < 4; ++q) sm[q] = warp_sum(sm[q]);
        // the record (same rules, same numbers), written by a warp that has no role in the next product's pipeline
        // (thread 0 is the TMA producer: the record on its path delayed CTA 0, and with it every grid barrier)
        if (blockIdx.x == 0 && warp_all == D_PRODUCER_WARPS - 1 && lane == 0) sp2_finalise(ctl, sm);
        if (!loop_mode) { done = true; break; }
        // the decision of sp2_finalise (common.cuh), taken locally
        const double e = sqrt(sm[1]) / sqrt(sm[2]);
        if (e < idem_tol || (m >= 2 && e < 1e-2 && e >= e_prev2) || m + 1 == max_products) { done = true; break; }
        e_prev2 = e_prev1; e_prev1 = e;
        parity ^= 1;
        m += 1;
        branch = (sm[3] - (double)n_occ <= 0.0) ? 1 : 0;
    }
}

// ------------------------------------------------------------------------------------------------------------
// Persistent variant for the roofline regime (128 x 128 tiles): one CTA per SM walks a fixed work list.
//   * tiles (upper triangle, t = J (J + 1) / 2 + I) are dealt out in full waves of G = gridDim.x: CTA c takes tile
//     w G + c of wave w and runs the whole K loop of it;
//   * the R = tiles mod G tiles of the last, partial wave are split along K ("stream-K"): their R KT k-slabs are cut
//     into G equal contiguous ranges, one per CTA, so that every SM works until the end instead of R of them doing a
//     whole tile while G - R idle (N = 2048: 136 tiles on 148 SMs; N = 8192: 2080 = 14 x 148 + 8).
//     The CTA whose range holds k-slab 0 of a tile owns the tile: the others store their FP64 partial accumulators to
//     global scratch (one 128 KB slot per CTA, thread-major so the stores coalesce) and raise a flag tagged with the
//     launch epoch; the owner adds the partials in ascending CTA order (fixed order: bit-reproducible) and runs the
//     fused epilogue.  Launched cooperatively, so all CTAs are resident and the flag waits cannot starve.
// The TMA ring and the mbarrier phases run on across work items; the fused epilogue (D4) and the finaliser (D5) are
// those of the kernel above.
// ------------------------------------------------------------------------------------------------------------

__global__ void __launch_bounds__(D_THREADS, 1)
x2_dense_fp64_sk_kernel(const __grid_constant__ CUtensorMap map0, const __grid_constant__ CUtensorMap map1,
                        double *__restrict__ buf0, double *__restrict__ buf1, int64_t ld, int N,
                        Sp2Ctl *__restrict__ ctl, double *__restrict__ partials, double *__restrict__ sk_scratch,
                        unsigned int *__restrict__ sk_flags)
{
    constexpr int BT = 128, D_BM = BT, D_BN = BT, D_PANEL_BYTES = d_panel_bytes(BT), D_STAGE_BYTES = d_stage_bytes(BT);
    constexpr int MI = BT / 16, NI = BT / 32;
    if (ctl->done) return;
    const int parity = ctl->parity;
    const int branch = ctl->branch_cur;
    const unsigned int epoch = ctl->epoch;
    const CUtensorMap *map = parity ? &map1 : &map0;
    const double *__restrict__ X = parity ? buf1 : buf0;
    double *__restrict__ Xn = parity ? buf0 : buf1;

    extern __shared__ uint8_t smem_raw[];
    uint8_t *smem = smem_raw + ((1024u - (smem_u32(smem_raw) & 1023u)) & 1023u);
    uint64_t *full_bar = (uint64_t *)(smem + (size_t)D_STAGES * D_STAGE_BYTES);
    uint64_t *empty_bar = full_bar + D_STAGES;
    double (*s_red)[4] = (double (*)[4])(empty_bar + D_STAGES);          // [D_CONSUMER_WARPS][4]
    int *s_last = (int *)(s_red + D_CONSUMER_WARPS);

    const int warp_all = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int warp = warp_all - D_PRODUCER_WARPS;
    const int T = (N + D_BM - 1) / D_BM, tiles = T * (T + 1) / 2;
    const int KT = (N + D_BK - 1) / D_BK;
    const int G = (int)gridDim.x, c = (int)blockIdx.x;

    if (threadIdx.x == 0) {
        for (int s = 0; s < D_STAGES; ++s) { mbar_init(&full_bar[s], 1); mbar_init(&empty_bar[s], D_CONSUMER_WARPS); }
        mbar_fence_init();
        fence_proxy_async();
    }
    if (threadIdx.x < D_CONSUMER_WARPS * 4) ((double *)s_red)[threadIdx.x] = 0.0;
    __syncthreads();

    if (warp < 0) {
        // ===================== TMA producer warpgroup (one elected lane works) =====================
        asm volatile("setmaxnreg.dec.sync.aligned.u32 %0;" ::"n"(D_REGS_PRODUCER));
        if (warp_all == 0 && lane == 0) {
            tma_prefetch_desc(map);
            int slab = 0;
            SkItem w;
            for (int it = 0; sk_item(it, c, G, tiles, KT, sk_handoff_slabs(128), w); ++it) {
                int I, J;
                tri_sb_decode(w.tile, T, I, J);
                const bool diag = (I == J);
                const uint32_t tx = diag ? D_PANEL_BYTES : D_STAGE_BYTES;
                for (int kt = w.kt0; kt < w.kt1; ++kt, ++slab) {
                    const int s = slab % D_STAGES;
                    const uint32_t ph = (uint32_t)(slab / D_STAGES) & 1u;
                    mbar_wait(&empty_bar[s], ph ^ 1u);
                    mbar_expect_tx(&full_bar[s], tx);
                    uint8_t *dst = smem + (size_t)s * D_STAGE_BYTES;
                    tma_load_2d(dst, map, kt * D_BK, I * D_BM, &full_bar[s]);
                    if (!diag) tma_load_2d(dst + D_PANEL_BYTES, map, kt * D_BK, J * D_BN, &full_bar[s]);
                }
            }
        }
    } else {
        // ===================== DMMA consumers =====================
        asm volatile("setmaxnreg.inc.sync.aligned.u32 %0;" ::"n"(D_REGS_CONSUMER));
        const int wm = warp >> 2, wn = warp & 3;     // 2 x 4 warps; warp tile 64 x 32
        const int ctid = warp * 32 + lane;           // consumer thread id 0..255
        uint32_t koff[4];
        dmma_koff(lane, koff);
        double s_trp = 0.0, s_e = 0.0, s_x = 0.0, s_trn = 0.0;
        int slab = 0;
        StageRelease release;   // stages go back to the producer one slab late (dense_fp64_core.cuh)
        SkItem w;
        for (int it = 0; sk_item(it, c, G, tiles, KT, sk_handoff_slabs(128), w); ++it) {
            int I, J;
            tri_sb_decode(w.tile, T, I, J);
            const bool diag = (I == J);
            double acc[MI][NI][2];
#pragma unroll
            for (int i = 0; i < MI; ++i)
#pragma unroll
                for (int j = 0; j < NI; ++j) { acc[i][j][0] = 0.0; acc[i][j][1] = 0.0; }
            const uint8_t *a_base = smem + wm * (D_BM / 2) * 128;
            const uint8_t *b_base = smem + (diag ? 0 : D_PANEL_BYTES) + wn * (D_BN / 4) * 128;
            for (int kt = w.kt0; kt < w.kt1; ++kt, ++slab) {
                const int s = slab % D_STAGES;
                const uint32_t ph = (uint32_t)(slab / D_STAGES) & 1u;
                mbar_wait(&full_bar[s], ph);
                const uint8_t *sa = a_base + (size_t)s * D_STAGE_BYTES, *sb = b_base + (size_t)s * D_STAGE_BYTES;
                dmma_slab<MI, NI>(acc, sa, sb, koff);
                release.after_slab(empty_bar, s, lane);
            }

            if (w.kt0 > 0) {
                // ---------- contributor: hand the partial accumulators to the tile's owner ----------
                double *slot = sk_scratch + (size_t)c * SK_SLOT_DOUBLES + ctid;
#pragma unroll
                for (int i = 0; i < MI; ++i)
#pragma unroll
                    for (int j = 0; j < NI; ++j) {
                        __stcg(slot + (size_t)((i * NI + j) * 2 + 0) * 256, acc[i][j][0]);
                        __stcg(slot + (size_t)((i * NI + j) * 2 + 1) * 256, acc[i][j][1]);
                    }
                __threadfence();
                consumers_bar();
                if (ctid == 0) {
                    // release by the thread that raises the flag, AFTER the barrier: cumulative over every consumer
                    // thread's stores (a fence before the barrier alone does not order them before this write)
                    __threadfence();
                    atomicExch(&sk_flags[c], epoch);
                }
                continue;
            }
            if (w.kt1 < KT) {
                // ---------- owner of a split tile: add the other CTAs' partials in ascending CTA order ----------
                const int W = tiles / G, R = tiles - W * G;
                const int64_t UT = (int64_t)R * KT;
                const int64_t tile_end = (int64_t)(w.tile - W * G + 1) * KT;
                for (int c2 = c + 1; c2 < G; ++c2) {
                    const int64_t v0 = (int64_t)c2 * UT / G, v1 = (int64_t)(c2 + 1) * UT / G;
                    if (v0 >= tile_end) break;
                    if (v1 <= v0) continue;
                    if (ctid == 0) {
                        while (atomicAdd(&sk_flags[c2], 0u) != epoch) __nanosleep(64);
                        __threadfence();
                    }
                    consumers_bar();
                    const double *slot = sk_scratch + (size_t)c2 * SK_SLOT_DOUBLES + ctid;
#pragma unroll
                    for (int i = 0; i < MI; ++i)
#pragma unroll
                        for (int j = 0; j < NI; ++j) {
                            acc[i][j][0] += __ldcg(slot + (size_t)((i * NI + j) * 2 + 0) * 256);
                            acc[i][j][1] += __ldcg(slot + (size_t)((i * NI + j) * 2 + 1) * 256);
                        }
                }
            }

            // ===================== fused epilogue (D4) =====================
            sp2_tile_epilogue<MI, NI, BT>(acc, X, Xn, ld, N, I, J, wm, wn, lane, branch, s_trp, s_e, s_x, s_trn);
        }
        s_trp = warp_sum(s_trp); s_e = warp_sum(s_e); s_x = warp_sum(s_x); s_trn = warp_sum(s_trn);
        if (lane == 0) { s_red[warp][0] = s_trp; s_red[warp][1] = s_e; s_red[warp][2] = s_x; s_red[warp][3] = s_trn; }
    }
    __syncthreads();

    // ===================== per-CTA partial sums, last-CTA finaliser (D5) =====================
    if (threadIdx.x < 4) {
        double v = 0.0;
#pragma unroll
        for (int w2 = 0; w2 < D_CONSUMER_WARPS; ++w2) v += s_red[w2][threadIdx.x];
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
            for (int q = 0; q < 4; ++q) s[q] += vp[(size_t)tI * 4 + q];
        }
#pragma unroll
        for (int q = 0; q < 4; ++q) s[q] = warp_sum(s[q]);
        if (lane == 0) sp2_finalise(ctl, s);
    }
}

// ------------------------------------------------------------------------------------------------------------
// host side
// ------------------------------------------------------------------------------------------------------------
// tile edge for an N x N product: the roofline tile unless that leaves most of the chip idle
int dense_fp64_tile(int64_t N) { return N <= 512 ? 32 : (N <= 1024 ? 64 : 128); }

int make_dense_map(CUtensorMap *map, const double *base, int64_t N, int64_t ld)
{
    PFN_encodeTiled enc = get_encode_tiled();
    if (!enc) return BML_ERR_CUDA;
    const cuuint64_t dims[2] = {(cuuint64_t)N, (cuuint64_t)N};           // innermost first: columns (k), rows
    const cuuint64_t strides[1] = {(cuuint64_t)ld * sizeof(double)};     // bytes, dims 1..rank-1
    const cuuint32_t box[2] = {(cuuint32_t)D_BK, (cuuint32_t)dense_fp64_tile(N)};
    const cuuint32_t estr[2] = {1, 1};
    CUresult r = enc(map, CU_TENSOR_MAP_DATA_TYPE_FLOAT64, 2, (void *)base, dims, strides, box, estr,
                     CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
                     CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    return r == CUDA_SUCCESS ? 0 : BML_ERR_CUDA;
}

int sk_grid()
{
    static int g[MAX_DEVICES] = {};
    const int dev = current_device();
    if (dev < 0) return 0;
    if (!g[dev]) {
        int sms = 0, coop = 0;
        if (cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess ||
            cudaDeviceGetAttribute(&coop, cudaDevAttrCooperativeLaunch, dev) != cudaSuccess || !coop)
            return 0;
        g[dev] = sms < SK_MAX_GRID ? sms : SK_MAX_GRID;      // one CTA per SM (198 KB of shared memory each)
    }
    return g[dev];
}

// number of CTAs (= per-CTA partial-sum slots) of one product
int dense_fp64_num_tiles(int64_t N)
{
    const int bt = dense_fp64_tile(N);
    if (bt == 128) return SK_MAX_GRID;
    return tile_sb_grid((int)((N + bt - 1) / bt));
}

// global scratch of the persistent kernel: one partial-tile slot per CTA + the hand-off flags
size_t dense_fp64_sk_bytes(int64_t N)
{
    if (dense_fp64_tile(N) != 128) return 0;
    return (size_t)SK_MAX_GRID * SK_SLOT_DOUBLES * sizeof(double) + 1024;
}

// flags must not hold a tag from an earlier solve in the same workspace: zero them when a solve starts
int dense_fp64_sk_reset(void *sk, int64_t N, cudaStream_t st)
{
    if (dense_fp64_tile(N) != 128) return 0;
    unsigned int *flags = (unsigned int *)((uint8_t *)sk + (size_t)SK_MAX_GRID * SK_SLOT_DOUBLES * sizeof(double));
    return cudaMemsetAsync(flags, 0, 1024, st) == cudaSuccess ? 0 : BML_ERR_CUDA;
}

static int launch_x2_dense_fp64_sk(const CUtensorMap &map0, const CUtensorMap &map1, double *buf0, double *buf1,
                                   int64_t ld, int64_t N, Sp2Ctl *ctl, double *partials, void *sk, cudaStream_t stream)
{
    const int G = sk_grid();
    if (G <= 0 || !sk) return BML_ERR_CUDA;
    static size_t have[MAX_DEVICES] = {};
    if (ensure_smem_attr(x2_dense_fp64_sk_kernel, d_smem_bytes(128), have)) return BML_ERR_CUDA;
    double *scratch = (double *)sk;
    unsigned int *flags = (unsigned int *)((uint8_t *)sk + (size_t)SK_MAX_GRID * SK_SLOT_DOUBLES * sizeof(double));
    int n = (int)N;
    CUtensorMap m0 = map0, m1 = map1;
    void *args[] = {&m0, &m1, &buf0, &buf1, &ld, &n, &ctl, &partials, &scratch, &flags};
    if (cudaLaunchCooperativeKernel((const void *)x2_dense_fp64_sk_kernel, dim3((unsigned)G), dim3(D_THREADS), args,
                                    d_smem_bytes(128), stream) != cudaSuccess)
        return BML_ERR_CUDA;
    return cudaGetLastError() == cudaSuccess ? 0 : BML_ERR_CUDA;
}

template <int BT>
static int launch_x2_dense_fp64_t(const CUtensorMap &map0, const CUtensorMap &map1, double *buf0, double *buf1,
                                  int64_t ld, int64_t N, Sp2Ctl *ctl, double *partials, cudaStream_t stream)
{
    static size_t have[MAX_DEVICES] = {};
    if (ensure_smem_attr(x2_dense_fp64_kernel<BT>, d_smem_bytes(BT), have)) return BML_ERR_CUDA;
    x2_dense_fp64_kernel<BT><<<dense_fp64_num_tiles(N), D_THREADS, d_smem_bytes(BT), stream>>>(map0, map1, buf0, buf1, ld,
                                                                                              (int)N, ctl, partials);
    return cudaGetLastError() == cudaSuccess ? 0 : BML_ERR_CUDA;
}

// The whole product loop of a small solve in one cooperative launch.  Returns 1 if this device / size cannot run it (the
// caller then enqueues the products one launch each), 0 when enqueued, or a negative status.
template <int BT>
static int launch_sp2_loop_t(const CUtensorMap &map0, const CUtensorMap &map1, double *buf0, double *buf1, int64_t ld,
                             int64_t N, Sp2Ctl *ctl, double *partials, int max_products, cudaStream_t stream)
{
    static size_t have[MAX_DEVICES] = {};
    if (ensure_smem_attr(sp2_dense_fp64_loop_kernel<BT>, loop_smem_bytes(BT), have)) return BML_ERR_CUDA;
    const int tiles = dense_fp64_num_tiles(N);
    if (sk_grid() <= 0 || tiles > sk_grid()) return 1;          // all CTAs must be co-resident (one per SM)
    int n = (int)N;
    CUtensorMap m0 = map0, m1 = map1;
    void *args[] = {&m0, &m1, &buf0, &buf1, &ld, &n, &ctl, &partials, &max_products};
    if (cudaLaunchCooperativeKernel((const void *)sp2_dense_fp64_loop_kernel<BT>, dim3((unsigned)tiles), dim3(D_THREADS), args,
                                    loop_smem_bytes(BT), stream) != cudaSuccess)
        return BML_ERR_CUDA;
    return cudaGetLastError() == cudaSuccess ? 0 : BML_ERR_CUDA;
}

// one CTA per tile, all co-resident (one per SM): N <= 1024 on a device with cooperative launch and enough SMs
bool dense_fp64_loop_available(int64_t N)
{
    return dense_fp64_tile(N) != 128 && sk_grid() > 0 && dense_fp64_num_tiles(N) <= sk_grid();
}

int launch_sp2_dense_fp64_loop(const CUtensorMap &map0, const CUtensorMap &map1, double *buf0, double *buf1, int64_t ld,
                               int64_t N, Sp2Ctl *ctl, double *partials, int max_products, cudaStream_t stream)
{
    switch (dense_fp64_tile(N)) {
        case 32: return launch_sp2_loop_t<32>(map0, map1, buf0, buf1, ld, N, ctl, partials, max_products, stream);
        case 64: return launch_sp2_loop_t<64>(map0, map1, buf0, buf1, ld, N, ctl, partials, max_products, stream);
        default: return 1;
    }
}

// Enqueue one product.  buf0/buf1: ping-pong iterates (leading dimension ld, multiple of 16, 128-byte aligned).
// host-side view of the persistent kernel's work list (the same sk_item() the device runs): bml_dense_work_item
int dense_fp64_work_item(int64_t N, int n_ctas, int cta, int it, int32_t out[5])
{
    if (N <= 1024 || n_ctas < 1 || cta < 0 || cta >= n_ctas || it < 0) return BML_ERR_INVALID;
    const int T = (int)((N + 127) / 128), tiles = T * (T + 1) / 2, KT = (int)((N + D_BK - 1) / D_BK);
    SkItem w;
    if (!sk_item(it, cta, n_ctas, tiles, KT, sk_handoff_slabs(128), w)) return 1;
    int I, J;
    tri_sb_decode(w.tile, T, I, J);
    out[0] = w.tile; out[1] = I; out[2] = J; out[3] = w.kt0; out[4] = w.kt1;
    return 0;
}

// sk: the scratch of dense_fp64_sk_bytes(N) bytes (used by the persistent 128 x 128 kernel only)
int launch_x2_dense_fp64(const CUtensorMap &map0, const CUtensorMap &map1, double *buf0, double *buf1, int64_t ld,
                         int64_t N, Sp2Ctl *ctl, double *partials, void *sk, cudaStream_t stream)
{
    switch (dense_fp64_tile(N)) {
        case 32: return launch_x2_dense_fp64_t<32>(map0, map1, buf0, buf1, ld, N, ctl, partials, stream);
        case 64: return launch_x2_dense_fp64_t<64>(map0, map1, buf0, buf1, ld, N, ctl, partials, stream);
        default: return launch_x2_dense_fp64_sk(map0, map1, buf0, buf1, ld, N, ctl, partials, sk, stream);
    }
}

}  // namespace bmlsp2
