// dense_batch.cu -- the fused FP64 symmetric square (steps D3 + D4 + D5 of DESIGN.md) over a BATCH of independent
// matrices of unequal sizes that share ONE SP2 control block: the local solver of the graph-based construction with SP2
// (bml_graph.h, bml_graph_sp2_ellpack; PAPER.md VIII.B Listing 11 with prg_build_DM = SP2 of IV.A; reading G3').
//
// All parts take the same branch b_m, run the same number of products and stop together (one polynomial for every
// part), so a product of the whole batch is ONE persistent cooperative launch:
//   * work unit = one 16-column k-slab of one upper-triangle 128 x 128 tile of one part; the U = sum_p tiles_p KT_p
//     units, ordered part by part, tile by tile, slab by slab, are cut into G equal contiguous ranges, one per CTA
//     (pure stream-K: parts of 5,600 and of 900 orbitals mix without any wave quantisation, and a batch of small parts
//     fills the machine where one of them alone cannot);
//   * a tile whose slabs straddle a range boundary is owned by the CTA that holds its slab 0; the others hand their
//     FP64 partial accumulators over through the global scratch slots of dense_fp64.cu, added in ascending CTA order
//     (fixed order: bit-reproducible).  A contributor's part of a tile comes FIRST in its range and the owner's LAST,
//     so the chain c -> c + 1 cannot cycle;
//   * the fused epilogue (sp2_tile_epilogue) applies Eq. 6 / Eq. 7 and sums tr P and tr X' over the CORE rows of each
//     part only, the two norms over the whole part; the last CTA reduces the per-CTA partials in a fixed order and runs
//     the shared stop rules / next branch bit (sp2_finalise).
// TMA descriptors live in a job table in global memory (written by the host before the first launch of a solve).
#include "dense_fp64_core.cuh"

namespace bmlsp2 {

struct BatchJob {
    double *buf0, *buf1;     // ping-pong iterates of the part (leading dimension ld, multiple of 16, 128-byte aligned)
    const uint8_t *core;     // [N] 1 = core orbital (its diagonal counts in the traces); NULL = every row
    int64_t ld;
    int64_t unit0;           // index of the part's first work unit in the batch's unit list
    int32_t N, KT, tiles, tile0;   // tile0: index of the part's first tile in the batch's tile list
};
constexpr int BATCH_MAX_JOBS = 256;
struct alignas(128) BatchTable {
    CUtensorMap map[2][BATCH_MAX_JOBS];      // [buffer][job]: FP64 tensor map of that iterate buffer (box 16 x 128)
    BatchJob job[BATCH_MAX_JOBS];
    int64_t units;
    int32_t n_jobs, tiles_total;
};
size_t dense_batch_table_bytes() { return sizeof(BatchTable); }

struct BatchItem {
    int job, tile, kt0, kt1;
};
// Work list of CTA c: first W = tiles_total / G WHOLE tiles, dealt in waves (tile w G + c of wave w: the CTAs resident
// at any time work on ~G consecutive tiles of one part, i.e. on one super-block, and share its row panels in L2 -- with
// contiguous ranges per CTA every tile pulled both its panels from HBM: 42.5 GB per product at 4 x 5600 against 2 GB
// algorithmic); then the units of the remaining tiles_total - W G tiles are cut into G equal contiguous ranges
// (stream-K with unequal KT).  Identical arithmetic in the producer, the consumers and the host-side test hook.
struct BatchWalk {
    int wv, W, job;
    int64_t u, u1;
};
__host__ __device__ __forceinline__ void batch_walk_init(BatchWalk &k, const BatchJob *jobs, int n_jobs, int tiles_total,
                                                         int64_t units, int G, int c, int64_t &tail_unit0)
{
    k.W = tiles_total / G;
    k.wv = 0;
    k.job = 0;
    const int t_tail = k.W * G;                       // first tile of the split tail
    tail_unit0 = units;
    for (int p = 0; p < n_jobs; ++p)
        if (t_tail < jobs[p].tile0 + jobs[p].tiles) { tail_unit0 = jobs[p].unit0 + (int64_t)(t_tail - jobs[p].tile0) * jobs[p].KT; break; }
    const int64_t UT = units - tail_unit0;
    k.u = tail_unit0 + (int64_t)c * UT / G;
    k.u1 = tail_unit0 + (int64_t)(c + 1) * UT / G;
}
// next item; u_item = first unit of the item (meaningful for tail items); false when the list is exhausted
__host__ __device__ __forceinline__ bool batch_walk_next(BatchWalk &k, const BatchJob *jobs, int G, int c, BatchItem &w,
                                                         int64_t &u_item)
{
    if (k.wv < k.W) {
        const int q = k.wv * G + c;
        ++k.wv;
        while (q >= jobs[k.job].tile0 + jobs[k.job].tiles) ++k.job;
        w.job = k.job; w.tile = q - jobs[k.job].tile0; w.kt0 = 0; w.kt1 = jobs[k.job].KT;
        u_item = jobs[k.job].unit0 + (int64_t)w.tile * w.kt1;
        return true;
    }
    if (k.u >= k.u1) return false;
    while (k.u >= jobs[k.job].unit0 + (int64_t)jobs[k.job].tiles * jobs[k.job].KT) ++k.job;
    const int KT = jobs[k.job].KT;
    const int64_t rel = k.u - jobs[k.job].unit0;
    u_item = k.u;
    w.job = k.job;
    w.tile = (int)(rel / KT);
    w.kt0 = (int)(rel - (int64_t)w.tile * KT);
    const int64_t left = k.u1 - k.u;
    w.kt1 = (int64_t)(KT - w.kt0) <= left ? KT : w.kt0 + (int)left;
    k.u += w.kt1 - w.kt0;
    return true;
}

__global__ void __launch_bounds__(D_THREADS, 1)
x2_dense_fp64_batch_kernel(const BatchTable *__restrict__ tb, Sp2Ctl *__restrict__ ctl, double *__restrict__ partials,
                           double *__restrict__ sk_scratch, unsigned int *__restrict__ sk_flags)
{
    constexpr int BT = 128, D_BM = BT, D_BN = BT, D_PANEL_BYTES = d_panel_bytes(BT), D_STAGE_BYTES = d_stage_bytes(BT);
    constexpr int MI = BT / 16, NI = BT / 32;
    if (ctl->done) return;
    const int parity = ctl->parity;
    const int branch = ctl->branch_cur;
    const unsigned int epoch = ctl->epoch;

    extern __shared__ uint8_t smem_raw[];
    uint8_t *smem = smem_raw + ((1024u - (smem_u32(smem_raw) & 1023u)) & 1023u);
    uint64_t *full_bar = (uint64_t *)(smem + (size_t)D_STAGES * D_STAGE_BYTES);
    uint64_t *empty_bar = full_bar + D_STAGES;
    double (*s_red)[4] = (double (*)[4])(empty_bar + D_STAGES);          // [D_CONSUMER_WARPS][4]
    int *s_last = (int *)(s_red + D_CONSUMER_WARPS);

    const int warp_all = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int warp = warp_all - D_PRODUCER_WARPS;
    const int G = (int)gridDim.x, c = (int)blockIdx.x;
    const int64_t U = tb->units;

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
            int slab = 0;
            BatchItem w;
            BatchWalk walk;
            int64_t tail0, u_item;
            batch_walk_init(walk, tb->job, tb->n_jobs, tb->tiles_total, U, G, c, tail0);
            while (batch_walk_next(walk, tb->job, G, c, w, u_item)) {
                const CUtensorMap *map = &tb->map[parity][w.job];
                int I, J;
                tri_sb_decode(w.tile, (tb->job[w.job].N + 127) / 128, I, J);
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
        StageRelease release;
        BatchItem w;
        BatchWalk walk;
        int64_t tail0, u_item;
        batch_walk_init(walk, tb->job, tb->n_jobs, tb->tiles_total, U, G, c, tail0);
        const int64_t UT = U - tail0;
        while (batch_walk_next(walk, tb->job, G, c, w, u_item)) {
            const BatchJob &jb = tb->job[w.job];
            const int KT = jb.KT;
            int I, J;
            tri_sb_decode(w.tile, (jb.N + 127) / 128, I, J);
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
                    __threadfence();                 // release, cumulative over every consumer's stores (after the barrier)
                    atomicExch(&sk_flags[c], epoch);
                }
                continue;
            }
            if (w.kt1 < KT) {
                // ---------- owner of a split tile: add the following CTAs' partials in ascending CTA order ----------
                const int64_t tile_end = u_item + KT;        // kt0 == 0: the tile's units are [u_item, u_item + KT)
                for (int c2 = c + 1; c2 < G; ++c2) {
                    const int64_t v0 = tail0 + (int64_t)c2 * UT / G, v1 = tail0 + (int64_t)(c2 + 1) * UT / G;
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
            // ===================== fused epilogue (D4), traces over the core rows =====================
            const double *__restrict__ X = parity ? jb.buf1 : jb.buf0;
            double *__restrict__ Xn = parity ? jb.buf0 : jb.buf1;
            sp2_tile_epilogue<MI, NI, BT>(acc, X, Xn, jb.ld, jb.N, I, J, wm, wn, lane, branch, s_trp, s_e, s_x, s_trn, jb.core);
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
        __threadfence();
        const uint32_t prev = atomicAdd(&ctl->arrivals, 1u);
        __threadfence();
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

// tr over the core rows of every part's X_0 (fixed order: one CTA, parts one after the other)
__global__ void __launch_bounds__(1024) batch_core_trace_kernel(const BatchTable *__restrict__ tb, double *__restrict__ out)
{
    __shared__ double s_w[32];
    double v = 0.0;
    for (int p = 0; p < tb->n_jobs; ++p) {
        const BatchJob &jb = tb->job[p];
        for (int i = threadIdx.x; i < jb.N; i += blockDim.x)
            if (!jb.core || jb.core[i]) v += jb.buf0[(int64_t)i * jb.ld + i];
    }
    v = warp_sum(v);
    if ((threadIdx.x & 31) == 0) s_w[threadIdx.x >> 5] = v;
    __syncthreads();
    if (threadIdx.x < 32) {
        double r = s_w[threadIdx.x];
        r = warp_sum(r);
        if (threadIdx.x == 0) *out = r;
    }
}

// D6 helper: which buffer holds X_{m*}
__global__ void batch_final_buffers_kernel(const BatchTable *__restrict__ tb, const Sp2Ctl *__restrict__ ctl,
                                           const double **__restrict__ out)
{
    const int p = blockIdx.x * blockDim.x + threadIdx.x;
    if (p < tb->n_jobs) out[p] = ctl->parity ? tb->job[p].buf1 : tb->job[p].buf0;
}

// ------------------------------------------------------------------------------------------------------------
// host side
// ------------------------------------------------------------------------------------------------------------
int make_dense_map128(CUtensorMap *map, const double *base, int64_t N, int64_t ld)
{
    PFN_encodeTiled enc = get_encode_tiled();
    if (!enc) return BML_ERR_CUDA;
    const cuuint64_t dims[2] = {(cuuint64_t)N, (cuuint64_t)N};
    const cuuint64_t strides[1] = {(cuuint64_t)ld * sizeof(double)};
    const cuuint32_t box[2] = {(cuuint32_t)D_BK, 128u};
    const cuuint32_t estr[2] = {1, 1};
    CUresult r = enc(map, CU_TENSOR_MAP_DATA_TYPE_FLOAT64, 2, (void *)base, dims, strides, box, estr,
                     CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
                     CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    return r == CUDA_SUCCESS ? 0 : BML_ERR_CUDA;
}

// Fill the HOST copy of a job table: parts of sizes n[p] with iterate buffers buf0[p], buf1[p] (pitch ld[p]) and core
// flags core[p] (device pointers).  Returns 0 or a negative status.
int dense_batch_fill(void *h_table, int n_jobs, const int32_t *n, double *const *buf0, double *const *buf1,
                     const int64_t *ld, const uint8_t *const *core)
{
    if (n_jobs < 1 || n_jobs > BATCH_MAX_JOBS) return BML_ERR_INVALID;
    BatchTable *tb = (BatchTable *)h_table;
    memset(tb, 0, sizeof(*tb));
    tb->n_jobs = n_jobs;
    int64_t units = 0, tiles = 0;
    for (int p = 0; p < n_jobs; ++p) {
        if (n[p] < 1 || (ld[p] % 16) != 0 || ld[p] < n[p] || ((uintptr_t)buf0[p] & 127) || ((uintptr_t)buf1[p] & 127))
            return BML_ERR_INVALID;
        BatchJob &jb = tb->job[p];
        const int T = (n[p] + 127) / 128;
        jb.buf0 = buf0[p]; jb.buf1 = buf1[p]; jb.core = core ? core[p] : nullptr; jb.ld = ld[p];
        jb.N = n[p]; jb.KT = (n[p] + D_BK - 1) / D_BK; jb.tiles = T * (T + 1) / 2; jb.unit0 = units; jb.tile0 = (int32_t)tiles;
        units += (int64_t)jb.tiles * jb.KT;
        tiles += jb.tiles;
        if (tiles > 0x3fffffff) return BML_ERR_INVALID;
        int r;
        if ((r = make_dense_map128(&tb->map[0][p], buf0[p], n[p], ld[p]))) return r;
        if ((r = make_dense_map128(&tb->map[1][p], buf1[p], n[p], ld[p]))) return r;
    }
    tb->units = units;
    tb->tiles_total = (int32_t)tiles;
    return 0;
}

// host view of the work list (the arithmetic of batch_next): item `it` of CTA `cta`; out5 <- { job, tile, kt0, kt1, KT }
int dense_batch_work_item(int n_jobs, const int32_t *n, int n_ctas, int cta, int it, int32_t out[5])
{
    if (n_jobs < 1 || n_jobs > BATCH_MAX_JOBS || n_ctas < 1 || cta < 0 || cta >= n_ctas || it < 0) return BML_ERR_INVALID;
    static thread_local BatchJob jobs[BATCH_MAX_JOBS];
    int64_t units = 0;
    int tiles = 0;
    for (int p = 0; p < n_jobs; ++p) {
        if (n[p] < 1) return BML_ERR_INVALID;
        const int T = (n[p] + 127) / 128;
        jobs[p].N = n[p]; jobs[p].KT = (n[p] + D_BK - 1) / D_BK; jobs[p].tiles = T * (T + 1) / 2;
        jobs[p].unit0 = units; jobs[p].tile0 = tiles;
        units += (int64_t)jobs[p].tiles * jobs[p].KT;
        tiles += jobs[p].tiles;
    }
    BatchWalk walk;
    BatchItem w;
    int64_t tail0, u_item;
    batch_walk_init(walk, jobs, n_jobs, tiles, units, n_ctas, cta, tail0);
    for (int q = 0; batch_walk_next(walk, jobs, n_ctas, cta, w, u_item); ++q)
        if (q == it) { out[0] = w.job; out[1] = w.tile; out[2] = w.kt0; out[3] = w.kt1; out[4] = jobs[w.job].KT; return 0; }
    return 1;
}

int launch_x2_dense_fp64_batch(const void *d_table, Sp2Ctl *ctl, double *partials, void *sk, cudaStream_t stream)
{
    const int G = sk_grid();
    if (G <= 0 || !sk) return BML_ERR_CUDA;
    static size_t have[MAX_DEVICES] = {};
    if (ensure_smem_attr(x2_dense_fp64_batch_kernel, d_smem_bytes(128), have)) return BML_ERR_CUDA;
    double *scratch = (double *)sk;
    unsigned int *flags = (unsigned int *)((uint8_t *)sk + (size_t)SK_MAX_GRID * SK_SLOT_DOUBLES * sizeof(double));
    const BatchTable *tb = (const BatchTable *)d_table;
    void *args[] = {&tb, &ctl, &partials, &scratch, &flags};
    if (cudaLaunchCooperativeKernel((const void *)x2_dense_fp64_batch_kernel, dim3((unsigned)G), dim3(D_THREADS), args,
                                    d_smem_bytes(128), stream) != cudaSuccess)
        return BML_ERR_CUDA;
    return cudaGetLastError() == cudaSuccess ? 0 : BML_ERR_CUDA;
}

int launch_batch_core_trace(const void *d_table, double *d_out, cudaStream_t st)
{
    batch_core_trace_kernel<<<1, 1024, 0, st>>>((const BatchTable *)d_table, d_out);
    return cudaGetLastError() == cudaSuccess ? 0 : BML_ERR_CUDA;
}

int launch_batch_final_buffers(const void *d_table, const Sp2Ctl *ctl, const double **d_out, int n_jobs, cudaStream_t st)
{
    batch_final_buffers_kernel<<<(n_jobs + 255) / 256, 256, 0, st>>>((const BatchTable *)d_table, ctl, d_out);
    return cudaGetLastError() == cudaSuccess ? 0 : BML_ERR_CUDA;
}

}  // namespace bmlsp2
