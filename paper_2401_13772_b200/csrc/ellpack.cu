// ellpack.cu -- the sparse path of DESIGN.md on ELLPACK-R (Listing 1): S1 rescale, S3 thresholded row-wise
// SpGEMM X*X, S4 fused update / norms / canonical (ascending-column) write-back, S5 finaliser.
//
// Gustavson row merge ("sparse-sparse matrix multiply"), per product:
//   ell_block_summary_kernel   per row of X: its 32-column blocks and the largest |x| in each (input of the pre-screen)
//   x2_ellpack_upper_kernel    row i of thr(X X) for the columns j >= i only (X is bitwise symmetric, so P_ij and P_ji
//                              are the same chain of fma's); every kept entry is also appended to the list of row j.
//                              Instance <small table, pre-screen, 7 groups> over all rows, then instance <large table,
//                              no screen, 4 groups> over the rows the first one passed on (or over all rows when the
//                              pre-screen does not apply: tau = 0, M > 512, N > 131072)
//   x2_ellpack_assemble_kernel full row = sorted(appended entries) ++ upper part; update, threshold, norms, write-back
// Kernel 1: a GROUP of E_GW warps owns one output row at a time; several groups share a CTA (one CTA per SM), each
// with its own open-addressing hash accumulator in shared memory (2048 or BML_ELL_ACC_SLOTS keys + FP64 values).  For
// every stored entry p of row i (ascending p) the group's 128 threads take the entries of row k = index[i][p] with
// column >= i (a suffix found by binary search while row i is staged) and do acc[j] = fma(x_ik, x_kj, acc[j]); a
// group barrier separates step p from step p+1.  Contributions to one output entry are therefore added in order of
// increasing p, each as one fma: the canonical order of the oracle (readings item 11) -- values are
// bit-identical to it, not merely close.
//
// The gathers of rows k are issued two p-steps ahead into registers (coalesced: a warp reads 32 consecutive slots of
// row k), so their L2 latency is hidden behind the hash updates of the current step.  The hash keeps 32 consecutive
// columns in 32 distinct banks (slot = bucket(j >> 5) * 32 + ((j + rot(j >> 5)) & 31), collisions step to the next
// bucket): runs of consecutive columns, which is what rows of a short-range matrix consist of, are conflict-free.
#include "common.cuh"

namespace bmlsp2 {

constexpr int E_SLOTS = BML_ELL_ACC_SLOTS;      // the large table: the documented capacity (status -6 beyond it)
#ifndef BML_ELL_BUCKET_LOG2
#define BML_ELL_BUCKET_LOG2 5          // columns per bucket = 32
#endif
constexpr int E_BL = BML_ELL_BUCKET_LOG2;
constexpr int E_BW = 1 << E_BL;                 // bucket width (consecutive columns that stay consecutive slots)
static_assert(E_SLOTS == 4096, "the large table is written for 4096 slots");
constexpr int E_SL2_BIG = 12;                   // log2 of the large table
constexpr int E_SL2_SMALL = 11;                 // log2 of the small table of the pre-screened kernel (2048 slots)
constexpr int E_EMPTY = -1;
constexpr int E_GW = 4;               // warps per row group
constexpr int E_GT = E_GW * 32;       // threads per row group
constexpr int E_MAX_GROUPS = 4;       // row groups (= rows in flight) per CTA with the large table
constexpr int E_MAX_GROUPS_SMALL = 7; // ... with the small table
constexpr int E_NBUF_SMALL = 2;       // rotating gather buffers of the small-table instance (28 warps per SM hide the
                                      // L2 latency of a one-step look-ahead; a third buffer spills at 72 registers)
constexpr int E_MAX_GRID = 1024;
constexpr int E_SCREEN_MAX_N = 32 * 2 * (1 << E_SL2_SMALL);     // one FP32 bound per 32-column block, aliased on the values

// bucket and in-bucket rotation from the column-block id: the rotation spreads columns that sit at the same position of
// many blocks (the centre of a stencil) over all positions, while E_BW consecutive columns still map to E_BW consecutive
// (rotated) slots of one bucket.  SL2 = log2 of the table size.
template <int SL2>
__device__ __forceinline__ int e_hash(int j)
{
    constexpr int SHIFT = 32 - (SL2 - E_BL);
    const uint32_t h = (uint32_t)(j >> E_BL) * 2654435761u;
    return (int)((h >> SHIFT) << E_BL) | (int)((j + (h >> (SHIFT - E_BL))) & (uint32_t)(E_BW - 1));
}
// probe sequence (double hashing on the bucket): same position, `stride` buckets further (stride odd, so all buckets
// are visited); after a full cycle over the buckets, the next position
template <int SL2>
__device__ __forceinline__ int e_stride(int j)
{
    constexpr int BUCKETS = 1 << (SL2 - E_BL);
    const uint32_t h = (uint32_t)(j >> E_BL) * 2654435761u;
    return (int)((((h >> 8) & (BUCKETS - 1)) | 1u) << E_BL);
}
template <int SL2>
__device__ __forceinline__ int e_next(int slot, int tries, int stride)
{
    constexpr int BUCKETS = 1 << (SL2 - E_BL);
    slot = (slot + stride) & ((1 << SL2) - 1);
    if ((tries & (BUCKETS - 1)) == 0) slot = (slot & ~(E_BW - 1)) | ((slot + 1) & (E_BW - 1));
    return slot;
}

static inline int next_pow2(int x) { int p = 1; while (p < x) p <<= 1; return p; }
// row stage sa[M] f64, sk[M] int, sn[M] int; later aliased by the (column, slot) sort buffer of >= 32 entries
static inline size_t e_scratch_bytes(int M) { return M >= 16 ? (size_t)16 * (size_t)M : 256; }
static inline size_t e_group_bytes(int M, int slots = E_SLOTS) { return (size_t)slots * 12 + e_scratch_bytes(M); }

size_t ellpack_rowstats_bytes(int64_t) { return (size_t)E_MAX_GRID * 4 * sizeof(double); }

__device__ __forceinline__ void group_bar(int grp)
{
    asm volatile("bar.sync %0, %1;" ::"r"(grp + 1), "n"(E_GT) : "memory");
}
// group barrier that also ORs a per-thread flag over the group (every thread gets the same answer)
__device__ __forceinline__ bool group_bar_or(int grp, bool flag)
{
    int r;
    asm volatile(
        "{\n\t.reg .pred p, q;\n\t"
        "setp.ne.s32 q, %3, 0;\n\t"
        "bar.red.or.pred p, %1, %2, q;\n\t"
        "selp.s32 %0, 1, 0, p;\n\t}"
        : "=r"(r)
        : "r"(grp + 1), "n"(E_GT), "r"((int)flag)
        : "memory");
    return r != 0;
}

// bitonic sort of n (power of two, >= 64 or handled by one warp's worth of pairs) 64-bit keys in shared memory by one
// row group, ascending.  Sub-steps whose partner distance is < 64 stay inside the 64-element region one warp owns, so
// they only need a warp barrier; the group barrier is taken when data crosses warps.
__device__ __forceinline__ void group_bitonic_sort(unsigned long long *buf, int n, int tg, int grp)
{
    bool cross = true;      // the buffer was filled by arbitrary threads
    for (int k = 2; k <= n; k <<= 1) {
        for (int j = k >> 1; j > 0; j >>= 1) {
            if (cross || j >= 64) group_bar(grp); else __syncwarp();
            cross = (j >= 64);
            for (int t = tg; t < (n >> 1); t += E_GT) {
                const int i = ((t & ~(j - 1)) << 1) | (t & (j - 1));
                const int l = i | j;
                const bool up = (i & k) == 0;
                const unsigned long long a = buf[i], b = buf[l];
                if ((a > b) == up) { buf[i] = b; buf[l] = a; }
            }
        }
    }
    group_bar(grp);
}

// warp bitonic sort (rescale kernel)
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
// S3: accumulate one output row, acc[j] = fma(x_ik, x_kj, acc[j]) for p ascending.  CC = E_GT-entry chunks of a
// gathered row per step (CC * E_GT >= the longest row k merged into this row i; chosen per row).
// Returns true if the accumulator ran out of slots (group-uniform).
// ------------------------------------------------------------------------------------------------------------
template <int CC>
struct Gather {
    int j[CC];
    double v[CC];
};

// slow path of the accumulator lookup: the home slot of column j holds another key or is empty.  Walks the probe
// sequence, inserting j (value 0) if it is not there yet.  Returns the slot, or -1 when the table is full.
template <int SL2>
__device__ __forceinline__ int e_probe_insert(int *keys, double *vals, int j, int s, int kk)
{
    const int stride = e_stride<SL2>(j);
    int tries = 0;
    while (true) {
        if (kk == E_EMPTY) {
            const int old = atomicCAS(&keys[s], E_EMPTY, j);
            if (old == E_EMPTY) { vals[s] = 0.0; return s; }
            kk = old;
        }
        if (kk == j) return s;
        if (++tries > (1 << SL2)) return -1;
        s = e_next<SL2>(s, tries, stride);
        kk = keys[s];
    }
}

// ============================================================================================================
// Symmetric evaluation (the default path).  X is bitwise symmetric, so P_ij and P_ji are the same chain of fma's
// (same products x_ik x_kj = x_jk x_ki, same ascending k): bit-identical.  Kernel 1 therefore accumulates, for row i,
// only the columns j >= i: of every gathered row k it takes the SUFFIX starting at the first column >= i (found by
// binary search while row i is staged), which halves the multiply-adds.  It thresholds and sorts that upper part,
// stores it, and appends a copy (i, P_ij) to the "lower list" of every row j > i.  Kernel 2 assembles each full row of
// P = sorted(lower list) ++ upper part and runs the fused update / threshold / norms / write-back against row i of X.
// ============================================================================================================

// gather of the suffix of row k = sk[p]: sn[p] = (first slot << 16) | count.  Only the lanes that have an entry load;
// the others keep what an earlier step left in g (the structs are zeroed once per row), and every use is guarded by the
// lane's position against `cnt`.  Unsigned 32 x 32 -> 64-bit offset arithmetic: one IMAD.WIDE.U32.
template <int CC>
__device__ __forceinline__ void s_gather(Gather<CC> &g, int &cnt, int p, int n_i, const double *__restrict__ xv,
                                         const int32_t *__restrict__ xi, unsigned M, const int *sk, const int *sn, int tg)
{
    cnt = 0;
    if (p < n_i) {
        const unsigned pk = (unsigned)sn[p];
        const int n_k = (int)(pk & 0xffffu);
        cnt = n_k;
        const uint64_t off = (uint64_t)(unsigned)sk[p] * M + ((pk >> 16) + (unsigned)tg);
        const int32_t *pi = xi + off;
        const double *pv = xv + off;
#pragma unroll
        for (int c = 0; c < CC; ++c) {
            if (c * E_GT + tg < n_k) { g.j[c] = __ldg(pi + c * E_GT); g.v[c] = __ldg(pv + c * E_GT); }
        }
    }
}

// column j passed the pre-screen of this row (one bit per 32-column block)
__device__ __forceinline__ bool e_allowed(const unsigned *allow, int j)
{
    return (allow[(unsigned)j >> 10] >> (((unsigned)j >> 5) & 31u)) & 1u;
}

// hash update of the first NC chunks of a gathered suffix (straight-line: the NC lookups are independent).
// SCREEN: entries whose 32-column block failed the row's pre-screen are skipped (they would be dropped anyway).
// Returns true when the table is full.
template <int SL2, bool SCREEN, int NC, int CC>
__device__ __forceinline__ bool s_accumulate(const Gather<CC> &g, int cnt, int tg, double a, int *keys, double *vals,
                                             const unsigned *allow)
{
    static_assert(NC <= CC, "chunk count");
    int slot[NC], key[NC];
    bool ok[NC];
    bool full = false;
#pragma unroll
    for (int c = 0; c < NC; ++c) {
        ok[c] = c * E_GT + tg < cnt && (!SCREEN || e_allowed(allow, g.j[c]));      // g.j is a valid column on every lane
        slot[c] = e_hash<SL2>(g.j[c]);
    }
#pragma unroll
    for (int c = 0; c < NC; ++c) key[c] = keys[slot[c]];
#pragma unroll
    for (int c = 0; c < NC; ++c) {
        if (ok[c] && key[c] != g.j[c]) {
            slot[c] = e_probe_insert<SL2>(keys, vals, g.j[c], slot[c], key[c]);
            if (slot[c] < 0) { full = true; slot[c] = 0; }
        }
    }
    double acc[NC];
#pragma unroll
    for (int c = 0; c < NC; ++c) acc[c] = vals[slot[c]];
#pragma unroll
    for (int c = 0; c < NC; ++c)
        if (ok[c] && !full) vals[slot[c]] = fma(a, g.v[c], acc[c]);
    return full;
}

// one p-step: a warp dispatches on the number of E_GT-entry chunks in which IT has lanes (warp-uniform; a warp beyond
// the end of a short suffix goes straight to the barrier), then the group barrier that orders step p before step
// p + 1; an empty suffix costs nothing.  REDUCE: the barrier also ORs the table-full flag over the group into `stop`
// (every third step: the flag only has to stop a failing row early).  Returns the thread's own flag.
template <int SL2, bool SCREEN, int CC>
__device__ __forceinline__ bool s_step(const Gather<CC> &g, int cnt, double a, int *keys, double *vals, const unsigned *allow,
                                       int grp, int tg, bool full, bool &stop, const bool REDUCE)
{
    if (cnt <= 0) return full;          // group-uniform; `stop` is only ever set group-uniformly
    const int mine = cnt - (tg & ~31);  // entries at or beyond this warp's first lane, chunk 0
    if (mine > 0) {
        const int nc = (mine + E_GT - 1) / E_GT;
        if (nc == 1) full |= s_accumulate<SL2, SCREEN, 1, CC>(g, cnt, tg, a, keys, vals, allow);
        else if (CC >= 2 && nc == 2) full |= s_accumulate<SL2, SCREEN, (CC >= 2 ? 2 : CC), CC>(g, cnt, tg, a, keys, vals, allow);
        else if (CC >= 3 && nc == 3) full |= s_accumulate<SL2, SCREEN, (CC >= 3 ? 3 : CC), CC>(g, cnt, tg, a, keys, vals, allow);
        else if (CC >= 4 && nc == 4) full |= s_accumulate<SL2, SCREEN, (CC >= 4 ? 4 : CC), CC>(g, cnt, tg, a, keys, vals, allow);
        else full |= s_accumulate<SL2, SCREEN, CC, CC>(g, cnt, tg, a, keys, vals, allow);
    }
    if (REDUCE) { stop = group_bar_or(grp, full); return full; }
    group_bar(grp);
    return full;
}

// returns true (group-uniform) when the accumulator ran out of slots.  The gathers run NB - 1 p-steps ahead of the
// accumulation in NB rotating register buffers.
template <int SL2, bool SCREEN, int CC, int NB>
__device__ __forceinline__ bool s_accumulate_row(const double *__restrict__ xv, const int32_t *__restrict__ xi, int M,
                                                 int n_i, const double *sa, const int *sk, const int *sn, int *keys,
                                                 double *vals, const unsigned *allow, int row, int tg, int grp)
{
    bool full = false, stop = false;
    Gather<CC> g[NB];
    int n[NB];
#pragma unroll
    for (int u = 0; u < NB; ++u)
#pragma unroll
        for (int c = 0; c < CC; ++c) { g[u].j[c] = row; g[u].v[c] = 0.0; }
#pragma unroll
    for (int u = 0; u < NB - 1; ++u) s_gather<CC>(g[u], n[u], u, n_i, xv, xi, (unsigned)M, sk, sn, tg);
    for (int p = 0; p < n_i; p += NB) {
#pragma unroll
        for (int u = 0; u < NB; ++u) {
            if (p + u < n_i) {             // group-uniform
                s_gather<CC>(g[(u + NB - 1) % NB], n[(u + NB - 1) % NB], p + u + NB - 1, n_i, xv, xi, (unsigned)M, sk, sn, tg);
                full = s_step<SL2, SCREEN, CC>(g[u], n[u], sa[p + u], keys, vals, allow, grp, tg, full, stop, u == NB - 1);
            }
        }
        if (stop) break;                   // group-uniform: the OR came with the last step's barrier
    }
    return group_bar_or(grp, full);        // flags raised in steps whose barrier did not carry them
}

// the same with three buffers rotated by name (the large-table instance: the indexed form above costs it registers)
template <int SL2, bool SCREEN, int CC>
__device__ __forceinline__ bool s_accumulate_row3(const double *__restrict__ xv, const int32_t *__restrict__ xi, int M,
                                                  int n_i, const double *sa, const int *sk, const int *sn, int *keys,
                                                  double *vals, const unsigned *allow, int row, int tg, int grp)
{
    bool full = false, stop = false;
    Gather<CC> gA, gB, gC;
#pragma unroll
    for (int c = 0; c < CC; ++c) { gA.j[c] = gB.j[c] = gC.j[c] = row; gA.v[c] = gB.v[c] = gC.v[c] = 0.0; }
    int nA, nB, nC;
    s_gather<CC>(gA, nA, 0, n_i, xv, xi, (unsigned)M, sk, sn, tg);
    s_gather<CC>(gB, nB, 1, n_i, xv, xi, (unsigned)M, sk, sn, tg);
    for (int p = 0; p < n_i; p += 3) {
        s_gather<CC>(gC, nC, p + 2, n_i, xv, xi, (unsigned)M, sk, sn, tg);
        full = s_step<SL2, SCREEN, CC>(gA, nA, sa[p], keys, vals, allow, grp, tg, full, stop, false);
        if (p + 1 < n_i) {
            s_gather<CC>(gA, nA, p + 3, n_i, xv, xi, (unsigned)M, sk, sn, tg);
            full = s_step<SL2, SCREEN, CC>(gB, nB, sa[p + 1], keys, vals, allow, grp, tg, full, stop, false);
        }
        if (p + 2 < n_i) {
            s_gather<CC>(gB, nB, p + 4, n_i, xv, xi, (unsigned)M, sk, sn, tg);
            full = s_step<SL2, SCREEN, CC>(gC, nC, sa[p + 2], keys, vals, allow, grp, tg, full, stop, true);
            if (stop) break;               // group-uniform: the OR came with the barrier
        }
    }
    return group_bar_or(grp, full);        // flags raised in steps whose barrier did not carry them
}

// ------------------------------------------------------------------------------------------------------------
// Exact pre-screen of one output row (small-table kernel).  |P_ij| <= sum_k |x_ik| |x_kj| <= sum_k |x_ik| max_{j' in
// block(j)} |x_kj'| =: bound(block(j)), with block = 32 consecutive columns.  The per-row block maxima of X come from
// ell_block_summary_kernel (one (block id, max) list per row).  A block whose bound is below tau holds only entries the
// threshold drops, so the numeric pass neither inserts nor accumulates them: the accumulator shrinks from the two-hop
// candidate set (up to ~2300 columns of the upper half on the 5' model) to about the kept set (<= ~1000), which is
// what lets a 2048-slot table -- and seven rows in flight per SM instead of four -- do.  The bounds are summed in FP32
// with shared-memory atomics (order-free: no barrier per k); |x| is rounded up, and the 1e-3 margin on tau covers the
// rounding of the sum, so every skipped entry is one the oracle drops as well.  The bound array aliases the values of
// the (not yet initialised) table.
// ------------------------------------------------------------------------------------------------------------
constexpr int E_PS_U = 8;      // rows k whose block lists are in flight per warp
__device__ __forceinline__ void s_prescreen(int row, int n_i, int N, int SB, const double *sa, const int *sk,
                                            const int32_t *__restrict__ sb_id, const float *__restrict__ sb_mx,
                                            const int32_t *__restrict__ sb_n, float *bnd, unsigned *allow, double tau,
                                            int tg, int grp)
{
    const int lane = tg & 31, wg = tg >> 5;
    const int NBK = (N + 31) >> 5, rb = row >> 5;
    for (int b = tg; b < NBK; b += E_GT) bnd[b] = 0.0f;
    group_bar(grp);
    for (int p0 = wg * 32; p0 < n_i; p0 += E_GW * 32) {
        const int pl = p0 + lane;
        int kl = 0, cl = 0;
        float al = 0.0f;
        if (pl < n_i) { kl = sk[pl]; cl = __ldg(sb_n + kl); al = __double2float_ru(fabs(sa[pl])); }
        const int nu = min(32, n_i - p0);
        for (int u0 = 0; u0 < nu; u0 += E_PS_U) {
            int id[E_PS_U][2];
            float mx[E_PS_U][2], au[E_PS_U];
#pragma unroll
            for (int u = 0; u < E_PS_U; ++u) {
                const int src = min(u0 + u, 31);
                const int k = __shfl_sync(0xffffffffu, kl, src);
                const int c = (u0 + u < nu) ? __shfl_sync(0xffffffffu, cl, src) : 0;
                au[u] = __shfl_sync(0xffffffffu, al, src);
                const int64_t base = (int64_t)k * SB;
#pragma unroll
                for (int h = 0; h < 2; ++h) {
                    const int e = h * 32 + lane;
                    id[u][h] = e < c ? __ldg(sb_id + base + e) : -1;
                    mx[u][h] = e < c ? __ldg(sb_mx + base + e) : 0.0f;
                }
                for (int e = 64 + lane; e < c; e += 32) {          // a row with more than 64 column blocks: rare
                    const int b = __ldg(sb_id + base + e);
                    if (b >= rb) atomicAdd(&bnd[b], au[u] * __ldg(sb_mx + base + e));
                }
            }
#pragma unroll
            for (int u = 0; u < E_PS_U; ++u)
#pragma unroll
                for (int h = 0; h < 2; ++h)
                    if (id[u][h] >= rb) atomicAdd(&bnd[id[u][h]], au[u] * mx[u][h]);
        }
    }
    group_bar(grp);
    const float thr = (float)(tau * (1.0 - 1e-3));
    for (int w = tg; w < ((NBK + 31) >> 5); w += E_GT) {
        unsigned bits = 0u;
        for (int b = 0; b < 32; ++b) {
            const int bb = (w << 5) + b;
            if (bb < NBK && bnd[bb] >= thr) bits |= 1u << b;
        }
        if (w == (rb >> 5)) bits |= 1u << (rb & 31);          // the diagonal is kept whatever its value
        allow[w] = bits;
    }
    group_bar(grp);
}

// ------------------------------------------------------------------------------------------------------------
// Kernel 1 (S3, upper half): P_ij for j >= i, thresholded, sorted; lower copies appended to the rows j > i.
//   tv/ti/tn : upper part of thr(X X), row-major ELLPACK-R (ascending columns)
//   lv/li/lcnt : per row j, the entries (i, P_ji = P_ij) with i < j, in arrival order; lcnt[j] counts ALL arrivals
//                (slots beyond M are not written: the row has overflowed then anyway)
// ------------------------------------------------------------------------------------------------------------
// Two instances.  <E_SL2_SMALL, true, 7>: 2048-slot tables behind the exact pre-screen (s_prescreen), seven rows in
// flight per SM; a row whose screened fill still does not fit (or whose gathered rows need more than four chunks) goes
// to fail_list.  <E_SL2_BIG, false, 4>: the 4096-slot tables without a screen, over all rows (tau = 0, large N or M) or
// over row_list[0 .. *row_count) -- the rows the first instance passed on; a table that overflows here is status -6.
template <int SL2, bool SCREEN, int MAXG, int NBUF>
__global__ void __launch_bounds__(MAXG * E_GT, 1)
x2_ellpack_upper_kernel(const double *__restrict__ v0, const int32_t *__restrict__ i0, const int32_t *__restrict__ n0,
                        const double *__restrict__ v1, const int32_t *__restrict__ i1, const int32_t *__restrict__ n1,
                        int N, int M, double tau, int sort_cap, Sp2Ctl *__restrict__ ctl, double *__restrict__ tv,
                        int32_t *__restrict__ ti, int32_t *__restrict__ tn, double *__restrict__ lv,
                        int32_t *__restrict__ li, int32_t *__restrict__ lcnt, const int32_t *__restrict__ sb_id,
                        const float *__restrict__ sb_mx, const int32_t *__restrict__ sb_n, int32_t *__restrict__ fail_list,
                        int32_t *__restrict__ fail_count, const int32_t *__restrict__ row_list,
                        const int32_t *__restrict__ row_count, int allow_off)
{
    constexpr int SLOTS = 1 << SL2;
    if (ctl->done) return;
    const int parity = ctl->parity;
    const double *__restrict__ xv = parity ? v1 : v0;
    const int32_t *__restrict__ xi = parity ? i1 : i0;
    const int32_t *__restrict__ xn = parity ? n1 : n0;

    extern __shared__ __align__(16) uint8_t smem[];
    const int ngroups = blockDim.x / E_GT;
    const int grp = threadIdx.x / E_GT, tg = threadIdx.x % E_GT, lane = threadIdx.x & 31;
    uint8_t *gbase = smem + (size_t)grp * ((size_t)SLOTS * 12 + (size_t)sort_cap * 8);
    double *vals = (double *)gbase;
    int *keys = (int *)(gbase + (size_t)SLOTS * 8);
    uint8_t *scratch = gbase + (size_t)SLOTS * 12;
    double *sa = (double *)scratch;
    int *sk = (int *)(scratch + (size_t)8 * M);
    int *sn = sk + M;
    unsigned long long *sortbuf = (unsigned long long *)scratch;     // aliases sa/sk/sn after the accumulation
    // [(N / 32 + 31) / 32] words per group: the 32-column blocks of the row in hand that passed the pre-screen
    unsigned *allow = SCREEN ? (unsigned *)(smem + allow_off) + (size_t)grp * ((((N + 31) >> 5) + 31) >> 5) : nullptr;
    __shared__ int s_kept[MAXG], s_nkmax[MAXG][2];

    int w_acc = INT32_MAX;
    if (tg == 0) { s_nkmax[grp][0] = 0; s_nkmax[grp][1] = 0; }
    group_bar(grp);
    int it = 0;
    const int nrows = row_list ? *row_count : N;
    for (int64_t row64 = (int64_t)blockIdx.x * ngroups + grp; row64 < nrows; row64 += (int64_t)gridDim.x * ngroups) {
        const int row = row_list ? row_list[row64] : (int)row64;
        const int64_t rbase = (int64_t)row * M;
        const int n_i = min(xn[row], M);
        {
            int4 *k4 = (int4 *)keys;
            const int4 e4 = make_int4(E_EMPTY, E_EMPTY, E_EMPTY, E_EMPTY);
            for (int s = tg; s < SLOTS / 4; s += E_GT) k4[s] = e4;
        }
        int nk_max = 0;
        // Four entries of row i per thread at a time (one pass for n_i <= 4 E_GT): their binary searches -- about
        // log2(n_k) dependent L2 loads each -- advance in lock step with unconditional loads, so a round costs one
        // round trip for all four instead of one each.
        constexpr int SU = 4;
        for (int p0 = tg; p0 < n_i; p0 += SU * E_GT) {
            int k[SU], nk[SU], lo[SU], hi[SU];
#pragma unroll
            for (int u = 0; u < SU; ++u) k[u] = (p0 + u * E_GT < n_i) ? xi[rbase + p0 + u * E_GT] : row;
#pragma unroll
            for (int u = 0; u < SU; ++u) {
                nk[u] = (p0 + u * E_GT < n_i) ? min(xn[k[u]], M) : 0;
                lo[u] = 0; hi[u] = nk[u];
            }
            // first slot of row k whose column is >= row (rows are in ascending column order)
            bool more = true;
            while (more) {
                int v[SU], mid[SU];
#pragma unroll
                for (int u = 0; u < SU; ++u) {
                    mid[u] = (lo[u] < hi[u]) ? ((lo[u] + hi[u]) >> 1) : 0;      // slot 0 always exists: a safe read
                    v[u] = __ldg(xi + (int64_t)k[u] * M + mid[u]);
                }
                more = false;
#pragma unroll
                for (int u = 0; u < SU; ++u) {
                    if (lo[u] < hi[u]) {
                        if (v[u] < row) lo[u] = mid[u] + 1; else hi[u] = mid[u];
                    }
                    more |= lo[u] < hi[u];
                }
            }
#pragma unroll
            for (int u = 0; u < SU; ++u) {
                const int p = p0 + u * E_GT;
                if (p < n_i) {
                    sk[p] = k[u];
                    sa[p] = xv[rbase + p];
                    sn[p] = (lo[u] << 16) | (nk[u] - lo[u]);
                    nk_max = max(nk_max, nk[u] - lo[u]);
                }
            }
        }
        nk_max = __reduce_max_sync(0xffffffffu, nk_max);
        if (lane == 0) atomicMax(&s_nkmax[grp][it & 1], nk_max);
        if (tg == 0) { s_kept[grp] = 0; s_nkmax[grp][(it + 1) & 1] = 0; }
        group_bar(grp);
        const int chunks = (s_nkmax[grp][it & 1] + E_GT - 1) / E_GT;
        ++it;

        if (SCREEN) s_prescreen(row, n_i, N, M, sa, sk, sb_id, sb_mx, sb_n, (float *)vals, allow, tau, tg, grp);

        bool full = false;
#define S_ACC(CC)                                                                                                      \
    full = (NBUF == 3) ? s_accumulate_row3<SL2, SCREEN, CC>(xv, xi, M, n_i, sa, sk, sn, keys, vals, allow, row, tg, grp)   \
                       : s_accumulate_row<SL2, SCREEN, CC, (NBUF == 3 ? 2 : NBUF)>(xv, xi, M, n_i, sa, sk, sn, keys, vals, \
                                                                                  allow, row, tg, grp)
        if (chunks <= 1) S_ACC(1);
        else if (chunks == 2) S_ACC(2);
        else if (chunks == 3) S_ACC(3);
        else if (chunks == 4) S_ACC(4);
        else if (SCREEN) full = true;     // longer gathered rows need more registers than seven groups leave: large table
        else if (chunks <= 6) S_ACC(6);
        else S_ACC(8);
#undef S_ACC
        if (full) {
            if (SCREEN) {                 // passed on to the large-table instance
                if (tg == 0) fail_list[atomicAdd(fail_count, 1)] = row;
            } else {                      // accumulator capacity exceeded: status -6
                w_acc = min(w_acc, row);
                if (tg == 0) tn[row] = 0;
            }
            group_bar(grp);
            continue;
        }

        // threshold (keep |p| >= tau or the diagonal) and compact (column, slot) into the sort buffer
        for (int s0 = 0; s0 < SLOTS; s0 += E_GT) {
            const int s = s0 + tg;
            const int key = s < SLOTS ? keys[s] : E_EMPTY;
            const bool keep = key != E_EMPTY && (fabs(vals[s]) >= tau || key == row);
            if (keep && key != row) {         // mirror: P_ji = P_ij, appended to row j = key (j > row); counts are exact
                const int pos = atomicAdd(&lcnt[key], 1);
                if (pos < M) { li[(int64_t)key * M + pos] = row; lv[(int64_t)key * M + pos] = vals[s]; }
            }
            const unsigned bal = __ballot_sync(0xffffffffu, keep);
            if (bal) {
                int base = 0;
                if (lane == 0) base = atomicAdd(&s_kept[grp], __popc(bal));
                base = __shfl_sync(0xffffffffu, base, 0);
                if (keep) {
                    const int pos = base + __popc(bal & ((1u << lane) - 1u));
                    if (pos < sort_cap) sortbuf[pos] = ((unsigned long long)(unsigned)key << 32) | (unsigned)s;
                }
            }
        }
        group_bar(grp);
        const int kept = s_kept[grp];
        if (tg == 0) tn[row] = kept;          // may exceed M: kernel 2 turns that into the overflow status
        const int nw = min(kept, min(M, sort_cap));
        int n2 = 32;
        while (n2 < nw) n2 <<= 1;
        for (int q = nw + tg; q < n2; q += E_GT) sortbuf[q] = ~0ull;
        // (entries beyond nw only exist when the row has overflowed; they are not needed then)
        group_bitonic_sort(sortbuf, n2, tg, grp);
        for (int q = tg; q < nw; q += E_GT) {
            const unsigned long long e = sortbuf[q];
            const int j = (int)(e >> 32);
            const double v = vals[(int)(e & 0xffffffffu)];
            ti[rbase + q] = j;
            tv[rbase + q] = v;
        }
        group_bar(grp);
    }
    if (w_acc != INT32_MAX && tg == 0) atomicMin(&ctl->acc_row, w_acc);
}

// ------------------------------------------------------------------------------------------------------------
// Kernel 2 (S4 + S5): one warp per row.  P_i = sorted(lower list) ++ upper part; then, against row i of X:
// ||P - X||^2 over the union pattern, ||X||^2, X' = b ? thr(2X - P) : P, tr P, tr X', sorted write-back, and the
// last-CTA finaliser.  All sums run over sorted lists in a fixed lane-strided order: bit-reproducible.
// Per-warp shared memory: pc[M] int, pf[M] uint8, pv[M] double, ec[M] int, ev[M] double, sortbuf[pow2(M)] u64 (a row
// of P longer than M is an overflow and is not assembled).
// ------------------------------------------------------------------------------------------------------------
constexpr int A_MAX_WARPS = 6;
static inline size_t a_warp_bytes(int M)
{
    const size_t m = M < 16 ? 16 : M;
    const size_t b = m * 4 + m + m * 8 + m * 4 + m * 8 + (size_t)next_pow2((int)m) * 8;
    return (b + 63) / 64 * 64;
}

// first index q in [0, n) with c[q] >= key (c ascending)
__device__ __forceinline__ int a_lower_bound(const int *c, int n, int key)
{
    int lo = 0, hi = n;
    while (lo < hi) {
        const int mid = (lo + hi) >> 1;
        if (c[mid] < key) lo = mid + 1; else hi = mid;
    }
    return lo;
}

__global__ void __launch_bounds__(A_MAX_WARPS * 32)
x2_ellpack_assemble_kernel(double *__restrict__ v0, int32_t *__restrict__ i0, int32_t *__restrict__ n0,
                           double *__restrict__ v1, int32_t *__restrict__ i1, int32_t *__restrict__ n1, int N, int M,
                           double tau, Sp2Ctl *__restrict__ ctl, double *__restrict__ partials,
                           const double *__restrict__ tv, const int32_t *__restrict__ ti,
                           const int32_t *__restrict__ tn, const double *__restrict__ lv,
                           const int32_t *__restrict__ li, int32_t *__restrict__ lcnt, int warp_bytes)
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
    const int m = M < 16 ? 16 : M;
    int cap2 = 1;
    while (cap2 < m) cap2 <<= 1;
    uint8_t *wb = smem + (size_t)warp * warp_bytes;
    double *pv = (double *)wb;                                           // [m] values of P_i, later of X'_i
    double *ev = pv + m;                                                 // [m] kept X-only entries
    unsigned long long *sortbuf = (unsigned long long *)(ev + m);        // [cap2]
    int *pc = (int *)(sortbuf + cap2);                                   // [m] columns of P_i
    int *ec = pc + m;                                                    // [m]
    uint8_t *pf = (uint8_t *)(ec + m);                                   // [m] 0 = P only, 1 = in X and kept, 2 = in X, dropped
    __shared__ double s_part[A_MAX_WARPS][4];
    __shared__ int s_last;

    double w_trp = 0.0, w_e = 0.0, w_x = 0.0, w_trn = 0.0;
    int w_ovf_p = INT32_MAX, w_ovf_u = INT32_MAX, w_max_p = 0, w_max_u = 0;

    for (int64_t row64 = (int64_t)blockIdx.x * nwarps + warp; row64 < N; row64 += (int64_t)gridDim.x * nwarps) {
        const int row = (int)row64;
        const int64_t rbase = (int64_t)row * M;
        const int n_i = min(xn[row], M);
        const int u_all = tn[row], l_all = lcnt[row];
        __syncwarp();
        if (lane == 0) lcnt[row] = 0;                 // ready for the next product
        const int cnt_p = u_all + l_all;              // stored length of row i of P = thr(X X)
        w_max_p = max(w_max_p, cnt_p);
        if (cnt_p > M) {                              // ELLPACK-R overflow of P: status -3 in the finaliser
            w_ovf_p = min(w_ovf_p, row);
            if (lane == 0) on[row] = 0;
            continue;
        }
        const int n_l = l_all, u = u_all, np = n_l + u;
        // ---- lower part: sort the appended (row j, value) pairs by column
        int n2 = 32;
        while (n2 < n_l) n2 <<= 1;
#pragma unroll 4
        for (int q = lane; q < n2; q += 32)
            sortbuf[q] = q < n_l ? (((unsigned long long)(unsigned)li[rbase + q] << 32) | (unsigned)q) : ~0ull;
        __syncwarp();
        if (n_l > 1) warp_bitonic_sort(sortbuf, n2, lane);
#pragma unroll 4
        for (int q = lane; q < n_l; q += 32) {
            const unsigned long long e = sortbuf[q];
            pc[q] = (int)(e >> 32);
            pv[q] = lv[rbase + (int)(e & 0xffffffffu)];
            pf[q] = 0;
        }
#pragma unroll 4
        for (int q = lane; q < u; q += 32) {
            pc[n_l + q] = ti[rbase + q];
            pv[n_l + q] = tv[rbase + q];
            pf[n_l + q] = 0;
        }
        __syncwarp();
        // ---- entries of row i of X: match against P_i (binary search in the sorted columns), norms, update
        double r_trp = 0.0, r_e = 0.0, r_x = 0.0, r_trn = 0.0;
        int ne = 0;                                   // kept X-only entries (warp-uniform)
        for (int p0 = 0; p0 < n_i; p0 += 32) {
            const int p = p0 + lane;
            bool keepx = false;
            int j = 0;
            double xnew = 0.0;
            if (p < n_i) {
                j = xi[rbase + p];
                const double x = xv[rbase + p];
                const int q = a_lower_bound(pc, np, j);
                const bool found = q < np && pc[q] == j;
                const double pk = found ? pv[q] : 0.0;            // absent from thr(X X): 0
                const double d = pk - x;
                r_e += d * d;
                r_x += x * x;
                xnew = branch ? (2.0 * x - pk) : pk;              // Eq. 7 on the union pattern : Eq. 6
                if (found) {
                    if (j == row) r_trp += pk;
                    const bool keep = branch ? (fabs(xnew) >= tau || j == row) : true;
                    pv[q] = xnew;
                    pf[q] = keep ? 1 : 2;
                    if (keep && j == row) r_trn += xnew;
                } else {
                    keepx = branch && (fabs(xnew) >= tau || j == row);
                    if (keepx && j == row) r_trn += xnew;
                }
            }
            const unsigned bal = __ballot_sync(0xffffffffu, keepx);
            if (keepx) {
                const int pos = ne + __popc(bal & ((1u << lane) - 1u));
                ec[pos] = j;
                ev[pos] = xnew;
            }
            ne += __popc(bal);
        }
        __syncwarp();
        // ---- columns only in P: (P - X)^2 = p^2, X' = -p (Eq. 7) or p, always kept; then compact the kept entries
        int kept = 0;
        for (int q0 = 0; q0 < np; q0 += 32) {
            const int q = q0 + lane;
            bool keep = false;
            if (q < np) {
                if (pf[q] == 0) {
                    const double pk = pv[q];
                    r_e += pk * pk;
                    const double xnew = branch ? -pk : pk;
                    pv[q] = xnew;
                    if (pc[q] == row) { r_trp += pk; r_trn += xnew; }
                    keep = true;
                } else {
                    keep = pf[q] == 1;
                }
            }
            const unsigned bal = __ballot_sync(0xffffffffu, keep);
            if (keep) {
                const int pos = kept + __popc(bal & ((1u << lane) - 1u));
                if (pos < cap2) sortbuf[pos] = ((unsigned long long)(unsigned)pc[q] << 32) | (unsigned)q;
            }
            kept += __popc(bal);
        }
        for (int q = lane; q < ne; q += 32) {
            const int pos = kept + q;
            if (pos < cap2) sortbuf[pos] = ((unsigned long long)(unsigned)ec[q] << 32) | (0x80000000u | (unsigned)q);
        }
        kept += ne;
        __syncwarp();
        w_max_u = max(w_max_u, kept);
        if (kept > M) {
            w_ovf_u = min(w_ovf_u, row);
            if (lane == 0) on[row] = 0;
        } else {
            int k2 = 32;
            while (k2 < kept) k2 <<= 1;
            for (int q = kept + lane; q < k2; q += 32) sortbuf[q] = ~0ull;
            __syncwarp();
            warp_bitonic_sort(sortbuf, k2, lane);
            for (int q = lane; q < M; q += 32) {
                int j = 0; double v = 0.0;
                if (q < kept) {
                    const unsigned long long e = sortbuf[q];
                    const unsigned src = (unsigned)(e & 0xffffffffu);
                    j = (int)(e >> 32);
                    v = (src & 0x80000000u) ? ev[src & 0x7fffffffu] : pv[src];
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
        __threadfence();      // release: cumulative over the partial sums the barrier above ordered before this thread
        const uint32_t prev = atomicAdd(&ctl->arrivals, 1u);
        __threadfence();      // acquire, before the barrier below hands the verdict to the finalising warp
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
    if (ctl->done && ctl->status < 0) return;       // failed solve: D is left untouched
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
// Per-row column-block summary of the iterate X (input of s_prescreen): for every row, the 32-column blocks it has
// entries in (ascending, rows are sorted) and the largest |x| in each, rounded up to FP32.  One warp per row; the
// entries of one block are contiguous, so a block is a run of equal (column >> 5).
// ------------------------------------------------------------------------------------------------------------
constexpr int E_SUM_WARPS = 8;
__global__ void __launch_bounds__(E_SUM_WARPS * 32)
ell_block_summary_kernel(const double *__restrict__ v0, const int32_t *__restrict__ i0, const int32_t *__restrict__ n0,
                         const double *__restrict__ v1, const int32_t *__restrict__ i1, const int32_t *__restrict__ n1,
                         int N, int M, const Sp2Ctl *__restrict__ ctl, int32_t *__restrict__ sb_id,
                         float *__restrict__ sb_mx, int32_t *__restrict__ sb_n)
{
    if (ctl->done) return;
    const int parity = ctl->parity;
    const double *__restrict__ xv = parity ? v1 : v0;
    const int32_t *__restrict__ xi = parity ? i1 : i0;
    const int32_t *__restrict__ xn = parity ? n1 : n0;
    extern __shared__ __align__(16) uint8_t smem[];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    int *s_id = (int *)smem + (size_t)warp * 2 * M;
    unsigned *s_mx = (unsigned *)(s_id + M);
    for (int row = blockIdx.x * E_SUM_WARPS + warp; row < N; row += gridDim.x * E_SUM_WARPS) {
        const int n = min(xn[row], M);
        const int64_t rbase = (int64_t)row * M;
        for (int q = lane; q < n; q += 32) s_mx[q] = 0u;
        __syncwarp();
        int nseg = 0, last_b = -1;
        for (int c0 = 0; c0 < n; c0 += 32) {
            const int e = c0 + lane;
            const bool valid = e < n;
            const int b = valid ? (xi[rbase + e] >> E_BL) : -2;
            int pb = __shfl_up_sync(0xffffffffu, b, 1);
            if (lane == 0) pb = last_b;
            const bool head = valid && b != pb;
            const unsigned hb = __ballot_sync(0xffffffffu, head);
            const int seg = nseg + __popc(hb & (0xffffffffu >> (31 - lane))) - 1;       // heads at or before this lane
            if (head) s_id[seg] = b;
            // non-negative floats order like their bit patterns
            if (valid) atomicMax(&s_mx[seg], __float_as_uint(__double2float_ru(fabs(xv[rbase + e]))));
            nseg += __popc(hb);
            last_b = __shfl_sync(0xffffffffu, b, min(31, n - 1 - c0));
        }
        __syncwarp();
        for (int q = lane; q < nseg; q += 32) {
            sb_id[rbase + q] = s_id[q];
            sb_mx[rbase + q] = __uint_as_float(s_mx[q]);
        }
        if (lane == 0) sb_n[row] = nseg;
        __syncwarp();
    }
}

// ------------------------------------------------------------------------------------------------------------
// host launchers
// ------------------------------------------------------------------------------------------------------------
#define BML_CHECK_LAUNCH() do { if (cudaGetLastError() != cudaSuccess) return BML_ERR_CUDA; } while (0)

static int sm_count() { return device_sm_count(); }

// bytes of the scratch the symmetric product needs: upper parts (tv, ti, tn) and lower lists (lv, li, lcnt)
size_t ellpack_sym_bytes(int64_t N, int M)
{
    const size_t nm = (size_t)N * (size_t)M;
    auto up = [](size_t x) { return (x + 1023) / 1024 * 1024; };
    // + the column-block summaries of the iterate (ids, maxima, counts), the list of rows passed on to the large
    //   tables and its counter
    return 2 * up(nm * 8) + 2 * up(nm * 4) + 2 * up((size_t)N * 4) + 2 * up(nm * 4) + 2 * up((size_t)N * 4) + 1024;
}

// the lower-list counters must be zero when a solve starts (kernel 2 re-zeroes them after every product)
int ellpack_sym_reset(void *sym, int64_t N, int M, cudaStream_t st)
{
    const size_t nm = (size_t)N * (size_t)M;
    auto up = [](size_t x) { return (x + 1023) / 1024 * 1024; };
    uint8_t *p = (uint8_t *)sym + 2 * up(nm * 8) + 2 * up(nm * 4) + up((size_t)N * 4);
    return cudaMemsetAsync(p, 0, (size_t)N * 4, st) == cudaSuccess ? 0 : BML_ERR_CUDA;
}

// One product = kernel 1 (upper half of thr(X X) + mirror append) followed by kernel 2 (assemble, update, finalise).
int launch_x2_ellpack(const double *v0, const int32_t *i0, const int32_t *n0, double *v1, int32_t *i1, int32_t *n1,
                      int64_t N, int M, double tau, Sp2Ctl *ctl, double *partials, void *sym, cudaStream_t st)
{
    const int sms = sm_count();
    if (sms <= 0 || !sym) return BML_ERR_CUDA;
    const size_t nm = (size_t)N * (size_t)M;
    auto up = [](size_t x) { return (x + 1023) / 1024 * 1024; };
    uint8_t *p = (uint8_t *)sym;
    double *tv = (double *)p; p += up(nm * 8);
    double *lv = (double *)p; p += up(nm * 8);
    int32_t *ti = (int32_t *)p; p += up(nm * 4);
    int32_t *li = (int32_t *)p; p += up(nm * 4);
    int32_t *tn = (int32_t *)p; p += up((size_t)N * 4);
    int32_t *lcnt = (int32_t *)p; p += up((size_t)N * 4);
    int32_t *sb_id = (int32_t *)p; p += up(nm * 4);
    float *sb_mx = (float *)p; p += up(nm * 4);
    int32_t *sb_n = (int32_t *)p; p += up((size_t)N * 4);
    int32_t *fail_list = (int32_t *)p; p += up((size_t)N * 4);
    int32_t *fail_count = (int32_t *)p;

    // ---- kernel 1
    const size_t smem_cap = 227 * 1024 - 1024;
    const int sort_cap = (int)(e_scratch_bytes(M) / 8);
    if (M > 8 * E_GT) return BML_ERR_INVALID;
    // (a) small tables behind the pre-screen, when it applies: tau > 0, rows gathered in <= 4 chunks, one FP32 bound per
    //     32-column block fits the values of a small table
    const size_t allow_bytes = (size_t)((((N + 31) / 32) + 31) / 32) * 4;
    int ng_small = (int)(smem_cap / (e_group_bytes(M, 1 << E_SL2_SMALL) + allow_bytes));
    if (ng_small > E_MAX_GROUPS_SMALL) ng_small = E_MAX_GROUPS_SMALL;
    const bool screened = tau > 0.0 && M <= 4 * E_GT && N <= E_SCREEN_MAX_N && ng_small > E_MAX_GROUPS;
    if (screened) {
        if (cudaMemsetAsync(fail_count, 0, sizeof(int32_t), st) != cudaSuccess) return BML_ERR_CUDA;
        const size_t sum_smem = (size_t)E_SUM_WARPS * 2 * M * 4;
        static size_t attr_s[MAX_DEVICES] = {};
        if (ensure_smem_attr(ell_block_summary_kernel, sum_smem, attr_s, 48 * 1024)) return BML_ERR_CUDA;
        int64_t grid_s = (N + E_SUM_WARPS - 1) / E_SUM_WARPS;
        if (grid_s > (int64_t)sms * 8) grid_s = (int64_t)sms * 8;
        ell_block_summary_kernel<<<(unsigned)grid_s, E_SUM_WARPS * 32, sum_smem, st>>>(v0, i0, n0, v1, i1, n1, (int)N, M, ctl,
                                                                                       sb_id, sb_mx, sb_n);
        BML_CHECK_LAUNCH();
        const size_t gb = e_group_bytes(M, 1 << E_SL2_SMALL);
        const size_t allow_off = (size_t)ng_small * gb;
        const size_t smem_a = allow_off + (size_t)ng_small * allow_bytes;
        auto ka = x2_ellpack_upper_kernel<E_SL2_SMALL, true, E_MAX_GROUPS_SMALL, E_NBUF_SMALL>;
        static size_t attr_a[MAX_DEVICES] = {};
        if (ensure_smem_attr(ka, smem_a, attr_a)) return BML_ERR_CUDA;
        int64_t grid_a = (N + ng_small - 1) / ng_small;
        if (grid_a > sms) grid_a = sms;
        ka<<<(unsigned)grid_a, ng_small * E_GT, smem_a, st>>>(v0, i0, n0, v1, i1, n1, (int)N, M, tau, sort_cap, ctl, tv, ti, tn,
                                                             lv, li, lcnt, sb_id, sb_mx, sb_n, fail_list, fail_count, nullptr,
                                                             nullptr, (int)allow_off);
        BML_CHECK_LAUNCH();
    }
    // (b) the large tables: every row, or the rows (a) passed on
    {
        int ngroups = (int)(smem_cap / e_group_bytes(M));
        if (ngroups > E_MAX_GROUPS) ngroups = E_MAX_GROUPS;
        if (ngroups < 1) return BML_ERR_INVALID;
        const size_t smem1 = (size_t)ngroups * e_group_bytes(M);
        auto kb = x2_ellpack_upper_kernel<E_SL2_BIG, false, E_MAX_GROUPS, 3>;
        static size_t attr1[MAX_DEVICES] = {};
        if (ensure_smem_attr(kb, smem1, attr1)) return BML_ERR_CUDA;
        int64_t grid1 = (N + ngroups - 1) / ngroups;
        if (grid1 > sms) grid1 = sms;
        kb<<<(unsigned)grid1, ngroups * E_GT, smem1, st>>>(v0, i0, n0, v1, i1, n1, (int)N, M, tau, sort_cap, ctl, tv, ti, tn, lv,
                                                          li, lcnt, nullptr, nullptr, nullptr, nullptr, nullptr,
                                                          screened ? fail_list : nullptr, screened ? fail_count : nullptr, 0);
        BML_CHECK_LAUNCH();
    }

    // ---- kernel 2
    const size_t wbytes = a_warp_bytes(M);
    int nwarps = (int)(smem_cap / wbytes);
    if (nwarps > A_MAX_WARPS) nwarps = A_MAX_WARPS;
    if (nwarps < 1) return BML_ERR_INVALID;
    const size_t smem2 = (size_t)nwarps * wbytes;
    static size_t attr2[MAX_DEVICES] = {};
    if (ensure_smem_attr(x2_ellpack_assemble_kernel, smem2, attr2, 48 * 1024)) return BML_ERR_CUDA;
    int64_t grid2 = (N + nwarps - 1) / nwarps;
    const int64_t per_sm = (int64_t)(smem_cap / smem2) > 0 ? (int64_t)(smem_cap / smem2) : 1;
    if (grid2 > sms * per_sm) grid2 = sms * per_sm;
    if (grid2 > E_MAX_GRID) grid2 = E_MAX_GRID;
    // buffer 0 is only read while parity == 0 (the standalone entry point passes a const X there)
    x2_ellpack_assemble_kernel<<<(unsigned)grid2, nwarps * 32, smem2, st>>>(
        (double *)v0, (int32_t *)i0, (int32_t *)n0, v1, i1, n1, (int)N, M, tau, ctl, partials, tv, ti, tn, lv, li, lcnt,
        (int)wbytes);
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
    static size_t attr_smem[MAX_DEVICES] = {};
    if (ensure_smem_attr(rescale_ellpack_kernel, smem, attr_smem, 48 * 1024)) return BML_ERR_CUDA;
    rescale_ellpack_kernel<<<(N + nwarps - 1) / nwarps, nwarps * 32, smem, st>>>(H->value, H->index, H->nnz, N, M,
                                                                                  d_bounds, xv, xi, xn, diag,
                                                                                  fail_flag, cap);
    BML_CHECK_LAUNCH();
    sum_vector_kernel<<<1, 1024, 0, st>>>(diag, N, d_tr0);
    BML_CHECK_LAUNCH();
    return 0;
}

int launch_sum_vector(const double *v, int N, double *d_out, cudaStream_t st)
{
    sum_vector_kernel<<<1, 1024, 0, st>>>(v, N, d_out);
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
