// symm_ab.cu -- the grouped FP64 product kernel of the Chebyshev path (Eq. 10, 13, 14):
//
//   Out_q = alpha_q A_q B_q + beta_q C_q + gamma_q I,   q = 0 .. n_jobs - 1,   ONE launch
//
// A_q, B_q are polynomials of the same symmetric matrix: symmetric and commuting, so A B = A B^T is symmetric and
// tile (I, J), I <= J, is sum_K A[I, K] B[J, K]^T -- two K-contiguous ROW panels, as in the SP2 square (dense_fp64.cu),
// computed once and mirrored.  The jobs of one launch are the T_i of one doubling level (Eq. 13-14: "can therefore be
// computed in parallel", P:241 -- the paper uses one stream per product) or one nesting step of Eq. 10.
//
// One persistent CTA per SM walks the list { job x upper-triangle tile } in full waves and splits the last, partial
// wave along K (the stream-K scheme of dense_fp64.cu; the list and its hand-off are the same sk_item()).  Operands are
// slices of ONE 3-D tensor map (column, row, slot) over the caller's slab of matrices, so a launch needs no per-job
// descriptors.  Pipeline, fragment layout and MMA step: dense_fp64_core.cuh.
#include "dense_fp64_core.cuh"
#include "symm_ab.cuh"

namespace bmlsp2 {

__device__ __forceinline__ void tma_load_3d(void *smem_dst, const CUtensorMap *map, int32_t c0, int32_t c1, int32_t c2,
                                            uint64_t *bar)
{
    asm volatile(
        "cp.async.bulk.tensor.3d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%3, %4, %5}], [%2];"
        ::"r"(smem_u32(smem_dst)), "l"(map), "r"(smem_u32(bar)), "r"(c0), "r"(c1), "r"(c2)
        : "memory");
}

template <int BT>
__global__ void __launch_bounds__(D_THREADS, 1)
symm_ab_fp64_kernel(const __grid_constant__ CUtensorMap map, const __grid_constant__ SymmBatch batch, int N,
                    double *__restrict__ sk_scratch, unsigned int *__restrict__ sk_flags, unsigned int epoch)
{
    constexpr int PANEL_BYTES = d_panel_bytes(BT), STAGE_BYTES = d_stage_bytes(BT);
    constexpr int MI = BT / 16, NI = BT / 32;        // 8 x 8 fragments per warp tile (BT/2) x (BT/4)

    extern __shared__ uint8_t smem_raw[];
    uint8_t *smem = smem_raw + ((1024u - (smem_u32(smem_raw) & 1023u)) & 1023u);
    uint64_t *full_bar = (uint64_t *)(smem + (size_t)D_STAGES * STAGE_BYTES);
    uint64_t *empty_bar = full_bar + D_STAGES;

    const int warp_all = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int warp = warp_all - D_PRODUCER_WARPS;
    const int T = (N + BT - 1) / BT, tiles = T * (T + 1) / 2, total = tiles * batch.n_jobs;
    const int KT = (N + D_BK - 1) / D_BK;
    const int G = (int)gridDim.x, c = (int)blockIdx.x;

    if (threadIdx.x == 0) {
        for (int s = 0; s < D_STAGES; ++s) { mbar_init(&full_bar[s], 1); mbar_init(&empty_bar[s], D_CONSUMER_WARPS); }
        mbar_fence_init();
        fence_proxy_async();
    }
    __syncthreads();

    if (warp < 0) {
        // ===================== TMA producer warpgroup (one elected lane works) =====================
        asm volatile("setmaxnreg.dec.sync.aligned.u32 %0;" ::"n"(D_REGS_PRODUCER));
        if (warp_all == 0 && lane == 0) {
            tma_prefetch_desc(&map);
            int slab = 0;
            SkItem w;
            for (int it = 0; sk_item(it, c, G, total, KT, sk_handoff_slabs(BT), w); ++it) {
                const int q = w.tile / tiles;
                int I, J;
                tri_decode(w.tile - q * tiles, I, J);
                const int sa = batch.job[q].a, sb = batch.job[q].b;
                const bool one_panel = (I == J) && (sa == sb);
                const uint32_t tx = one_panel ? PANEL_BYTES : STAGE_BYTES;
                for (int kt = w.kt0; kt < w.kt1; ++kt, ++slab) {
                    const int s = slab % D_STAGES;
                    const uint32_t ph = (uint32_t)(slab / D_STAGES) & 1u;
                    mbar_wait(&empty_bar[s], ph ^ 1u);
                    mbar_expect_tx(&full_bar[s], tx);
                    uint8_t *dst = smem + (size_t)s * STAGE_BYTES;
                    tma_load_3d(dst, &map, kt * D_BK, I * BT, sa, &full_bar[s]);
                    if (!one_panel) tma_load_3d(dst + PANEL_BYTES, &map, kt * D_BK, J * BT, sb, &full_bar[s]);
                }
            }
        }
        return;
    }

    // ===================== DMMA consumers =====================
    asm volatile("setmaxnreg.inc.sync.aligned.u32 %0;" ::"n"(D_REGS_CONSUMER));
    const int wm = warp >> 2, wn = warp & 3;         // 2 x 4 warps
    const int g = lane >> 2, t = lane & 3;
    const int pg = perm8(g);
    const int ctid = warp * 32 + lane;               // consumer thread id 0..255
    uint32_t koff[4];
    dmma_koff(lane, koff);
    int slab = 0;
    StageRelease release;   // stages go back to the producer one slab late (dense_fp64_core.cuh)
    SkItem w;
    for (int it = 0; sk_item(it, c, G, total, KT, sk_handoff_slabs(BT), w); ++it) {
        const int q = w.tile / tiles;
        int I, J;
        tri_decode(w.tile - q * tiles, I, J);
        const bool diag = (I == J);
        const bool one_panel = diag && (batch.job[q].a == batch.job[q].b);
        double acc[MI][NI][2];
#pragma unroll
        for (int i = 0; i < MI; ++i)
#pragma unroll
            for (int j = 0; j < NI; ++j) { acc[i][j][0] = 0.0; acc[i][j][1] = 0.0; }
        const uint8_t *a_base = smem + wm * (BT / 2) * 128;
        const uint8_t *b_base = smem + (one_panel ? 0 : PANEL_BYTES) + wn * (BT / 4) * 128;
        for (int kt = w.kt0; kt < w.kt1; ++kt, ++slab) {
            const int s = slab % D_STAGES;
            const uint32_t ph = (uint32_t)(slab / D_STAGES) & 1u;
            mbar_wait(&full_bar[s], ph);
            dmma_slab<MI, NI>(acc, a_base + (size_t)s * STAGE_BYTES, b_base + (size_t)s * STAGE_BYTES, koff);
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
            const int W = total / G, R = total - W * G;
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

        // ===================== fused epilogue: alpha P + beta C + gamma I, mirrored =====================
        const SymmJob &jb = batch.job[q];
        const double *__restrict__ C = jb.C;
        double *__restrict__ Out = jb.Out;
        const int64_t ldc = jb.ldc, ldo = jb.ldo;
        const double alpha = jb.alpha, beta = jb.beta, gamma = jb.gamma;
        const int row0 = I * BT + wm * (BT / 2) + pg;
        const int col0 = J * BT + wn * (BT / 4);
        // 16-byte accesses need even leading dimensions and 16-byte aligned bases (the slab always is; a caller's D may
        // not be): CTA-uniform choice per job
        const bool vec = (((ldo | ldc) & 1) == 0) && ((((uintptr_t)Out | (uintptr_t)C) & 15) == 0);
        auto one = [&](int r, int cc, double p) {
            // diagonal tiles: only r <= cc is used and mirrored -> Out is bitwise symmetric
            if (r < N && cc < N && (!diag || r <= cc)) {
                double v = alpha * p;
                if (C) v = fma(beta, C[(int64_t)r * ldc + cc], v);
                if (r == cc) v += gamma;
                Out[(int64_t)r * ldo + cc] = v;
                if (r != cc) Out[(int64_t)cc * ldo + r] = v;
            }
        };
        if (vec && C != nullptr && I * BT + BT <= N && J * BT + BT <= N) {
            // Tile entirely inside the matrix (CTA-uniform): C is read RB fragment rows ahead of its use instead of
            // inside the per-element conditions below (one L2 round trip per step, see sp2_tile_epilogue).  Same
            // arithmetic, element by element.
            const int cadj = (t < 2) ? 4 * t : 4 * (t - 2) + 2;               // frag_adjacent's column of this lane
            auto one_c = [&](int r, int cc, double p, double cv) {
                if (r <= cc) {                                                // only reached on diagonal tiles
                    double v = fma(beta, cv, alpha * p);
                    if (r == cc) v += gamma;
                    Out[(int64_t)r * ldo + cc] = v;
                    if (r != cc) Out[(int64_t)cc * ldo + r] = v;
                }
            };
            constexpr int RB = MI >= 4 ? 4 : 2;
#pragma unroll
            for (int i = 0; i < MI; i += RB) {
                double2 cv[RB][NI];
#pragma unroll
                for (int ii = 0; ii < RB; ++ii)
#pragma unroll
                    for (int j = 0; j < NI; ++j)
                        cv[ii][j] = *(const double2 *)(C + (int64_t)(row0 + (i + ii) * 8) * ldc + col0 + j * 8 + cadj);
#pragma unroll
                for (int ii = 0; ii < RB; ++ii) {
                    const int r = row0 + (i + ii) * 8;
#pragma unroll
                    for (int j = 0; j < NI; ++j) {
                        double p0 = acc[i + ii][j][0], p1 = acc[i + ii][j][1];
                        const int cc = col0 + j * 8 + frag_adjacent(p0, p1, t);
                        const double2 c2 = cv[ii][j];
                        if (!diag || r < cc) {
                            const double v0 = fma(beta, c2.x, alpha * p0), v1 = fma(beta, c2.y, alpha * p1);
                            *(double2 *)(Out + (int64_t)r * ldo + cc) = make_double2(v0, v1);
                            Out[(int64_t)cc * ldo + r] = v0;
                            Out[(int64_t)(cc + 1) * ldo + r] = v1;
                        } else {
                            one_c(r, cc, p0, c2.x);
                            one_c(r, cc + 1, p1, c2.y);
                        }
                    }
                }
            }
            continue;
        }
#pragma unroll
        for (int i = 0; i < MI; ++i) {
            const int r = row0 + i * 8;
#pragma unroll
            for (int j = 0; j < NI; ++j) {
                double p0 = acc[i][j][0], p1 = acc[i][j][1];
                const int cc = col0 + j * 8 + frag_adjacent(p0, p1, t);       // columns cc, cc + 1 (cc even)
                if (vec && r < N && cc + 1 < N && (!diag || r < cc)) {
                    double v0 = alpha * p0, v1 = alpha * p1;
                    if (C) {
                        const double2 c2 = *(const double2 *)(C + (int64_t)r * ldc + cc);
                        v0 = fma(beta, c2.x, v0);
                        v1 = fma(beta, c2.y, v1);
                    }
                    *(double2 *)(Out + (int64_t)r * ldo + cc) = make_double2(v0, v1);
                    Out[(int64_t)cc * ldo + r] = v0;
                    Out[(int64_t)(cc + 1) * ldo + r] = v1;
                } else {
                    one(r, cc, p0);
                    one(r, cc + 1, p1);
                }
            }
        }
    }
}

// ------------------------------------------------------------------------------------------------------------
// host side
// ------------------------------------------------------------------------------------------------------------
int dense_fp64_tile(int64_t N);        // dense_fp64.cu: 32 / 64 / 128

int make_slab_map(CUtensorMap *map, const double *base, int64_t N, int64_t ld, int64_t slot_elems, int n_slots)
{
    PFN_encodeTiled enc = get_encode_tiled();
    if (!enc) return BML_ERR_CUDA;
    const cuuint64_t dims[3] = {(cuuint64_t)N, (cuuint64_t)N, (cuuint64_t)n_slots};
    const cuuint64_t strides[2] = {(cuuint64_t)ld * sizeof(double), (cuuint64_t)slot_elems * sizeof(double)};
    const cuuint32_t box[3] = {(cuuint32_t)D_BK, (cuuint32_t)dense_fp64_tile(N), 1};
    const cuuint32_t estr[3] = {1, 1, 1};
    CUresult r = enc(map, CU_TENSOR_MAP_DATA_TYPE_FLOAT64, 3, (void *)base, dims, strides, box, estr,
                     CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
                     CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    return r == CUDA_SUCCESS ? 0 : BML_ERR_CUDA;
}

// stream-K scratch of the grouped kernel: one partial-tile slot per CTA + the hand-off flags
size_t symm_ab_sk_bytes() { return (size_t)SK_MAX_GRID * SK_SLOT_DOUBLES * sizeof(double) + 1024; }

static unsigned int *symm_flags(void *sk)
{
    return (unsigned int *)((uint8_t *)sk + (size_t)SK_MAX_GRID * SK_SLOT_DOUBLES * sizeof(double));
}

// a workspace may hold tags of an earlier call: zero the flags, then count epochs from 1
int symm_ab_sk_reset(void *sk, cudaStream_t st)
{
    return cudaMemsetAsync(symm_flags(sk), 0, 1024, st) == cudaSuccess ? 0 : BML_ERR_CUDA;
}

template <int BT>
static int launch_symm_t(const CUtensorMap &map, const SymmBatch &batch, int64_t N, void *sk, unsigned int epoch,
                         cudaStream_t stream)
{
    const int G = sk_grid();
    if (G <= 0 || !sk) return BML_ERR_CUDA;
    static size_t have[MAX_DEVICES] = {};
    if (ensure_smem_attr(symm_ab_fp64_kernel<BT>, d_smem_bytes(BT), have)) return BML_ERR_CUDA;
    double *scratch = (double *)sk;
    unsigned int *flags = symm_flags(sk);
    int n = (int)N;
    CUtensorMap m = map;
    SymmBatch b = batch;
    void *args[] = {&m, &b, &n, &scratch, &flags, &epoch};
    if (cudaLaunchCooperativeKernel((const void *)symm_ab_fp64_kernel<BT>, dim3((unsigned)G), dim3(D_THREADS), args,
                                    d_smem_bytes(BT), stream) != cudaSuccess)
        return BML_ERR_CUDA;
    return cudaGetLastError() == cudaSuccess ? 0 : BML_ERR_CUDA;
}

// Enqueue one grouped launch.  epoch: 1, 2, ... since the last symm_ab_sk_reset() of `sk`.
int launch_symm_ab(const CUtensorMap &map, const SymmBatch &batch, int64_t N, void *sk, unsigned int epoch,
                   cudaStream_t stream)
{
    if (batch.n_jobs < 1 || batch.n_jobs > BML_SYMM_MAX_JOBS) return BML_ERR_INVALID;
    switch (dense_fp64_tile(N)) {
        case 32: return launch_symm_t<32>(map, batch, N, sk, epoch, stream);
        case 64: return launch_symm_t<64>(map, batch, N, sk, epoch, stream);
        default: return launch_symm_t<128>(map, batch, N, sk, epoch, stream);
    }
}

// host-side view of the work list (the same sk_item() the device runs): bml_symm_work_item
int symm_ab_work_item(int64_t N, int n_jobs, int n_ctas, int cta, int it, int32_t out[6])
{
    if (N < 1 || n_jobs < 1 || n_jobs > BML_SYMM_MAX_JOBS || n_ctas < 1 || cta < 0 || cta >= n_ctas || it < 0)
        return BML_ERR_INVALID;
    const int bt = dense_fp64_tile(N);
    const int T = (int)((N + bt - 1) / bt), tiles = T * (T + 1) / 2, KT = (int)((N + D_BK - 1) / D_BK);
    SkItem w;
    if (!sk_item(it, cta, n_ctas, tiles * n_jobs, KT, sk_handoff_slabs(bt), w)) return 1;
    const int q = w.tile / tiles;
    int I, J;
    tri_decode(w.tile - q * tiles, I, J);
    out[0] = q; out[1] = I; out[2] = J; out[3] = w.kt0; out[4] = w.kt1; out[5] = bt;
    return 0;
}

}  // namespace bmlsp2
