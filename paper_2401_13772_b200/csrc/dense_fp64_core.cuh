// dense_fp64_core.cuh -- what the FP64 DMMA product kernels share (dense_fp64.cu: SP2's fused symmetric square;
// symm_ab.cu: the grouped alpha A B + beta C + gamma I products of the Chebyshev path): tile geometry, the swizzled
// fragment addressing, the k-slab MMA step and the work list of the persistent stream-K kernels.
#pragma once
#include "common.cuh"

namespace bmlsp2 {

// Tile edge BT (tile = BT x BT): 128 for the roofline regime; 64 / 32 for small matrices, where 128 x 128 tiles would
// leave most SMs idle (N = 256 has 3 tiles of 128 but 36 of 32) and a product is pure latency.  The 8 consumer warps
// always form a 2 x 4 grid: warp tile (BT/2) x (BT/4).
constexpr int D_BK = 16;           // k-slab: 16 doubles = 128 B = one SWIZZLE_128B row
constexpr int D_STAGES = 6;        // 6 x 32 KB = 192 KB at BT = 128
constexpr int D_CONSUMER_WARPS = 8;
constexpr int D_PRODUCER_WARPS = 4;     // one warpgroup, so that setmaxnreg can hand its registers to the consumers
constexpr int D_THREADS = (D_PRODUCER_WARPS + D_CONSUMER_WARPS) * 32;   // 384: ptxas caps at 168 regs/thread ...
constexpr int D_REGS_PRODUCER = 40;     // ... re-split by setmaxnreg: 128 x 40 + 256 x 232 = 64512 = 384 x 168
constexpr int D_REGS_CONSUMER = 232;
constexpr int d_panel_bytes(int BT) { return BT * D_BK * 8; }       // 16 KB at BT = 128
constexpr int d_stage_bytes(int BT) { return 2 * d_panel_bytes(BT); }
constexpr size_t d_smem_bytes(int BT)
{
    return (size_t)D_STAGES * d_stage_bytes(BT) + 1024 /*align*/ + 512 /*barriers + reduction scratch*/;
}

// MMA row/col index g (0..7) -> physical row inside an 8-row group.  With the 128B TMA swizzle (16-byte chunk c of
// row r stored at chunk c ^ (r & 7)) the four rows touched by one half-warp of an LDS.64 fragment load must have
// distinct (r >> 1) & 3 to hit 32 distinct banks: g = 0..3 -> rows 0,2,4,6 and g = 4..7 -> rows 1,3,5,7.
__device__ __forceinline__ int perm8(int g) { return ((g & 3) << 1) | (g >> 2); }

// byte offset of this lane's fragment element inside a panel for k-step kk of a 16-column slab (row perm8(g), plus
// 8-row groups via immediates): lane = 4 g + t reads column 4 kk + t of row perm8(g) through the 128B swizzle
__device__ __forceinline__ void dmma_koff(int lane, uint32_t koff[4])
{
    const int pg = perm8(lane >> 2), t = lane & 3;
#pragma unroll
    for (int kk = 0; kk < 4; ++kk)
        koff[kk] = (uint32_t)(pg * 128 + ((((kk * 2 + (t >> 1)) ^ pg) << 4) | ((t & 1) << 3)));
}

// one 16-column k-slab of a warp tile: 4 k-steps of MI x NI m8n8k4 FP64 MMAs, fragments straight from shared memory
template <int MI, int NI>
__device__ __forceinline__ void dmma_slab(double (&acc)[MI][NI][2], const uint8_t *sa, const uint8_t *sb,
                                          const uint32_t (&koff)[4])
{
#pragma unroll
    for (int kk = 0; kk < 4; ++kk) {
        double a[MI], b[NI];
#pragma unroll
        for (int i = 0; i < MI; ++i) a[i] = *(const double *)(sa + koff[kk] + i * 8 * 128);
#pragma unroll
        for (int j = 0; j < NI; ++j) b[j] = *(const double *)(sb + koff[kk] + j * 8 * 128);
#pragma unroll
        for (int i = 0; i < MI; ++i)
#pragma unroll
            for (int j = 0; j < NI; ++j) dmma884(acc[i][j][0], acc[i][j][1], a[i], b[j]);
    }
}

// Exchange inside the lane pairs (t, t ^ 2) of a fragment row so that every lane ends up with two ADJACENT columns:
// the m8n8k4 accumulator layout gives lane t the physical columns perm8(2t), perm8(2t+1) = {0,2} {4,6} {1,3} {5,7};
// afterwards the lanes hold {0,1} {4,5} {2,3} {6,7} and the epilogues can use 16-byte loads and stores.
// Returns the first (even) column of the pair.  Must be called by all 32 lanes.
__device__ __forceinline__ int frag_adjacent(double &v0, double &v1, int t)
{
    const bool lo = t < 2;
    const double recv = __shfl_xor_sync(0xffffffffu, lo ? v1 : v0, 2);
    if (lo) v1 = recv; else v0 = recv;
    return lo ? 4 * t : 4 * (t - 2) + 2;
}

// Fused epilogue (D4) of one tile held in the consumers' accumulators: X' = b ? 2X - P : P with its mirror, and this
// thread's share of { tr P, ||P - X||^2, ||X||^2, tr X' }.  `core` (may be NULL): per-row flags; the two TRACES then
// count only the rows whose flag is set (the graph-based solver's occupation is counted over core orbitals, bml_graph.h);
// the norms always run over the whole tile.  Fragment columns are first made adjacent (frag_adjacent) so
// that X is read and X' written 16 bytes at a time; the iterates live in the workspace (ld a multiple of 16 doubles,
// 128-byte aligned), so every pair is aligned.  Diagonal tiles use only r <= c and mirror it: X' is bitwise symmetric.
template <int MI, int NI, int BT>
__device__ __forceinline__ void sp2_tile_epilogue(double (&acc)[MI][NI][2], const double *__restrict__ X,
                                                  double *__restrict__ Xn, int64_t ld, int N, int I, int J, int wm, int wn,
                                                  int lane, int branch, double &s_trp, double &s_e, double &s_x,
                                                  double &s_trn, const uint8_t *__restrict__ core = nullptr)
{
    const int g = lane >> 2, t = lane & 3;
    const bool diag = (I == J);
    const int row0 = I * BT + wm * (BT / 2) + perm8(g);
    const int col0 = J * BT + wn * (BT / 4);
    auto one = [&](int r, int c, double p) {
        if (r < N && c < N && (!diag || r <= c)) {
            const double x = X[(int64_t)r * ld + c];
            const double d = p - x;
            const double xn = branch ? (2.0 * x - p) : p;             // Eq. 7 : Eq. 6
            Xn[(int64_t)r * ld + c] = xn;
            if (r == c) {
                if (!core || core[r]) { s_trp += p; s_trn += xn; }
                s_e += d * d; s_x += x * x;
            } else {
                Xn[(int64_t)c * ld + r] = xn;                         // mirror
                s_e += 2.0 * (d * d); s_x += 2.0 * (x * x);
            }
        }
    };
    if (I * BT + BT <= N && J * BT + BT <= N) {
        // Tile entirely inside the matrix (CTA-uniform): the reads of X need no bounds test, so they are issued two
        // fragment rows (2 x NI 16-byte loads) ahead of their use.  With the loads inside the per-element conditions
        // below every (i, j) step costs one L2 round trip (8 warps per SM: nothing else hides it).  Same arithmetic in
        // the same order as the general path: the sums are bitwise the same.
        const int cadj = (t < 2) ? 4 * t : 4 * (t - 2) + 2;             // frag_adjacent's column of this lane
        auto one_x = [&](int r, int c, double p, double x) {
            if (r <= c) {                                               // only reached on diagonal tiles
                const double d = p - x;
                const double xn = branch ? (2.0 * x - p) : p;
                Xn[(int64_t)r * ld + c] = xn;
                if (r == c) {
                    if (!core || core[r]) { s_trp += p; s_trn += xn; }
                    s_e += d * d; s_x += x * x;
                } else {
                    Xn[(int64_t)c * ld + r] = xn;
                    s_e += 2.0 * (d * d); s_x += 2.0 * (x * x);
                }
            }
        };
#pragma unroll
        constexpr int RB = MI >= 4 ? 4 : 2;                            // fragment rows read ahead
#pragma unroll
        for (int i = 0; i < MI; i += RB) {
            double2 xv[RB][NI];
#pragma unroll
            for (int ii = 0; ii < RB; ++ii)
#pragma unroll
                for (int j = 0; j < NI; ++j)
                    xv[ii][j] = *(const double2 *)(X + (int64_t)(row0 + (i + ii) * 8) * ld + col0 + j * 8 + cadj);
#pragma unroll
            for (int ii = 0; ii < RB; ++ii) {
                const int r = row0 + (i + ii) * 8;
#pragma unroll
                for (int j = 0; j < NI; ++j) {
                    double p0 = acc[i + ii][j][0], p1 = acc[i + ii][j][1];
                    const int c = col0 + j * 8 + frag_adjacent(p0, p1, t);
                    const double2 x = xv[ii][j];
                    if (!diag || r < c) {
                        const double d0 = p0 - x.x, d1 = p1 - x.y;
                        const double xn0 = branch ? (2.0 * x.x - p0) : p0, xn1 = branch ? (2.0 * x.y - p1) : p1;
                        *(double2 *)(Xn + (int64_t)r * ld + c) = make_double2(xn0, xn1);
                        Xn[(int64_t)c * ld + r] = xn0;
                        Xn[(int64_t)(c + 1) * ld + r] = xn1;
                        s_e += 2.0 * (d0 * d0) + 2.0 * (d1 * d1);
                        s_x += 2.0 * (x.x * x.x) + 2.0 * (x.y * x.y);
                    } else {
                        one_x(r, c, p0, x.x);
                        one_x(r, c + 1, p1, x.y);
                    }
                }
            }
        }
        return;
    }
#pragma unroll
    for (int i = 0; i < MI; ++i) {
        const int r = row0 + i * 8;
#pragma unroll
        for (int j = 0; j < NI; ++j) {
            double p0 = acc[i][j][0], p1 = acc[i][j][1];
            const int c = col0 + j * 8 + frag_adjacent(p0, p1, t);
            if (r < N && c + 1 < N && (!diag || r < c)) {
                // both elements strictly above the diagonal: one 16-byte read of X, one 16-byte write of X'
                const double2 x = *(const double2 *)(X + (int64_t)r * ld + c);
                const double d0 = p0 - x.x, d1 = p1 - x.y;
                const double xn0 = branch ? (2.0 * x.x - p0) : p0, xn1 = branch ? (2.0 * x.y - p1) : p1;
                *(double2 *)(Xn + (int64_t)r * ld + c) = make_double2(xn0, xn1);
                Xn[(int64_t)c * ld + r] = xn0;
                Xn[(int64_t)(c + 1) * ld + r] = xn1;
                s_e += 2.0 * (d0 * d0) + 2.0 * (d1 * d1);
                s_x += 2.0 * (x.x * x.x) + 2.0 * (x.y * x.y);
            } else {
                one(r, c, p0);
                one(r, c + 1, p1);
            }
        }
    }
}

// Release of a ring stage back to the TMA producer, ONE SLAB LATE.  ptxas schedules a stage's mbarrier.arrive right
// behind the ISSUE of the slab's last fragment loads (the MMAs that consume them follow it), and the arrive does not
// wait for those loads to have read shared memory: when the consumers run close behind the producer (short, store-only
// epilogues; measured on the grouped Chebyshev launches, ~1 wrong 32-byte fragment chunk per 40000 tiles) the refill of
// the stage could land under the last k-step's loads.  Releasing stage n only after the loads of slab n + 1 were issued
// closes that: shared-memory loads of one warp complete in order, and slab n + 1's first MMAs -- issued before that
// point -- already needed its own first loads, hence every load of slab n, to have completed.  Costs one of the
// D_STAGES stages of look-ahead.
struct StageRelease {
    int owed = -1;          // stage read by the previous slab, not yet released
    __device__ __forceinline__ void after_slab(uint64_t *empty_bar, int s, int lane)
    {
        __syncwarp();
        if (lane == 0 && owed >= 0) mbar_arrive(&empty_bar[owed]);
        owed = s;
    }
};

// ------------------------------------------------------------------------------------------------------------
// Work list of the persistent kernels (see dense_fp64.cu): full waves of tiles, then a K-split last wave.
// ------------------------------------------------------------------------------------------------------------
struct SkItem {
    int tile, kt0, kt1;
};
// Cost of one split-tile hand-off (partials to global memory, fence, flag, the owner's poll and reload) in units of
// one k-slab of the tile's mainloop: small tiles have short slabs, so the same ~2-3 us weigh more.
__host__ __device__ constexpr int sk_handoff_slabs(int bt) { return bt >= 128 ? 2 : (bt >= 64 ? 8 : 20); }

// it-th work item of CTA c (identical arithmetic in every role); false when the list is exhausted.
// The last, partial wave of R tiles is split along K over all G CTAs only if that is shorter than running the R tiles
// whole on R CTAs: R KT / G + hs < KT (hs = sk_handoff_slabs).  Otherwise CTA c < R takes tile W G + c whole.
__host__ __device__ __forceinline__ bool sk_item(int it, int c, int G, int tiles, int KT, int hs, SkItem &w)
{
    const int W = tiles / G, R = tiles - W * G;
    if (it < W) { w.tile = it * G + c; w.kt0 = 0; w.kt1 = KT; return true; }
    if (R == 0) return false;
    if ((int64_t)R * KT + (int64_t)hs * G >= (int64_t)KT * G) {
        if (it > W || c >= R) return false;
        w.tile = W * G + c; w.kt0 = 0; w.kt1 = KT;
        return true;
    }
    const int64_t UT = (int64_t)R * KT;
    const int64_t u0 = (int64_t)c * UT / G, u1 = (int64_t)(c + 1) * UT / G;
    const int64_t tl = u0 / KT + (it - W);
    const int64_t b = tl * KT;
    const int64_t s = u0 > b ? u0 : b, f = u1 < b + KT ? u1 : b + KT;
    if (s >= f) return false;
    w.tile = W * G + (int)tl; w.kt0 = (int)(s - b); w.kt1 = (int)(f - b);
    return true;
}
__device__ __forceinline__ void consumers_bar()
{
    asm volatile("bar.sync 1, %0;" ::"n"(D_CONSUMER_WARPS * 32) : "memory");
}

constexpr int SK_ACC = 64;                                             // FP64 accumulators per consumer thread
constexpr size_t SK_SLOT_DOUBLES = (size_t)SK_ACC * D_CONSUMER_WARPS * 32;   // 128 x 128

constexpr int SK_MAX_GRID = 256;      // scratch slots / flags provisioned for a persistent kernel
int sk_grid();                        // dense_fp64.cu: CTAs of a persistent launch (one per SM), 0 if unsupported

}  // namespace bmlsp2
