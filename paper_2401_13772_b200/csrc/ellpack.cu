// ellpack.cu -- the sparse path of DESIGN.md on ELLPACK-R (Listing 1): S1 rescale, S3 thresholded row-wise
// SpGEMM X*X, S4 fused update / norms / canonical (ascending-column) write-back, S5 finaliser.
//
// Gustavson row merge ("sparse-sparse matrix multiply").  A GROUP of E_GW warps owns one output row at a time;
// E_MAX_GROUPS groups share a CTA (one CTA per SM), each with its own open-addressing hash accumulator in shared
// memory (BML_ELL_ACC_SLOTS keys + FP64 values).  For every stored entry p of row i (ascending p) the group's 128
// threads take the entries of row k = index[i][p] (unique columns, one or more per thread) and do
// acc[j] = fma(x_ik, x_kj, acc[j]); a group barrier separates step p from step p+1.  Contributions to one output
// entry are therefore added in order of increasing p, each as one fma: the canonical order of the oracle (DESIGN.md
// readings item 11) -- values are bit-identical to it, not merely close.
//
// The gathers of rows k are issued two p-steps ahead into registers (coalesced: a warp reads 32 consecutive slots of
// row k), so their L2 latency is hidden behind the hash updates of the current step.  The hash keeps 32 consecutive
// columns in 32 distinct banks (slot = bucket(j >> 5) * 32 + ((j + rot(j >> 5)) & 31), collisions step to the next
// bucket): runs of consecutive columns, which is what rows of a short-range matrix consist of, are conflict-free.
#include "common.cuh"

namespace bmlsp2 {

constexpr int E_SLOTS = BML_ELL_ACC_SLOTS;
constexpr int E_MASK = E_SLOTS - 1;
constexpr int E_BUCKETS = E_SLOTS / 32;
constexpr int E_BUCKET_SHIFT = 32 - 7;  // log2(E_BUCKETS) = 7
static_assert(E_BUCKETS == 128, "bucket hash is written for 4096 slots");
constexpr int E_EMPTY = -1;
constexpr int E_DROPPED = 1 << 30;    // P entry fell below tau (value zeroed)
constexpr int E_INX = 1 << 29;        // column also present in row i of X
constexpr int E_KEY = (1 << 29) - 1;
constexpr int E_GW = 4;               // warps per row group
constexpr int E_GT = E_GW * 32;       // threads per row group
constexpr int E_MAX_GROUPS = 4;       // row groups (= rows in flight) per CTA
constexpr int E_MAX_GRID = 1024;

// bucket and in-bucket rotation from the 32-column block id: the rotation spreads columns that sit at the same
// position of many blocks (the centre of a stencil) over all 32 positions, while 32 consecutive columns still map
// to 32 distinct banks
__device__ __forceinline__ int e_hash(int j)
{
    const uint32_t h = (uint32_t)(j >> 5) * 2654435761u;
    return (int)((h >> E_BUCKET_SHIFT) << 5) | (int)((j + (h >> (E_BUCKET_SHIFT - 5))) & 31u);
}
// probe sequence (double hashing on the bucket): same position, `stride` buckets further (stride odd, so all buckets
// are visited); after a full cycle over the buckets, the next position
__device__ __forceinline__ int e_stride(int j)
{
    const uint32_t h = (uint32_t)(j >> 5) * 2654435761u;
    return (int)((((h >> 8) & (E_BUCKETS - 1)) | 1u) << 5);
}
__device__ __forceinline__ int e_next(int slot, int tries, int stride)
{
    slot = (slot + stride) & E_MASK;
    if ((tries & (E_BUCKETS - 1)) == 0) slot = (slot + 1) & E_MASK;
    return slot;
}

static inline int next_pow2(int x) { int p = 1; while (p < x) p <<= 1; return p; }
// row stage sa[M] f64, sk[M] int, sn[M] int; later aliased by the (column, slot) sort buffer of >= 32 entries
static inline size_t e_scratch_bytes(int M) { return M >= 16 ? (size_t)16 * (size_t)M : 256; }
static inline size_t e_group_bytes(int M) { return (size_t)E_SLOTS * 12 + e_scratch_bytes(M); }

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
__device__ __forceinline__ int e_probe_insert(int *keys, double *vals, int j, int s, int kk)
{
    const int stride = e_stride(j);
    int tries = 0;
    while (true) {
        if (kk == E_EMPTY) {
            const int old = atomicCAS(&keys[s], E_EMPTY, j);
            if (old == E_EMPTY) { vals[s] = 0.0; return s; }
            kk = old;
        }
        if (kk == j) return s;
        if (++tries > E_SLOTS) return -1;
        s = e_next(s, tries, stride);
        kk = keys[s];
    }
}

template <int CC>
__device__ __forceinline__ void e_gather(Gather<CC> &g, int p, int n_i, const double *__restrict__ xv,
                                         const int32_t *__restrict__ xi, int M, const int *sk, const int *sn, int tg)
{
#pragma unroll
    for (int c = 0; c < CC; ++c) { g.j[c] = -1; g.v[c] = 0.0; }
    if (p < n_i) {
        const int n_k = sn[p];
        const int32_t *pi = xi + (int64_t)sk[p] * M + tg;
        const double *pv = xv + (int64_t)sk[p] * M + tg;
#pragma unroll
        for (int c = 0; c < CC; ++c) {
            if (c * E_GT + tg < n_k) { g.j[c] = __ldg(pi + c * E_GT); g.v[c] = __ldg(pv + c * E_GT); }
        }
    }
}

template <int CC>
__device__ __forceinline__ bool e_accumulate(const Gather<CC> &g, double a, int *keys, double *vals)
{
    int slot[CC], key[CC];
    bool full = false;
#pragma unroll
    for (int c = 0; c < CC; ++c) slot[c] = e_hash(g.j[c]);
#pragma unroll
    for (int c = 0; c < CC; ++c) key[c] = keys[slot[c]];
#pragma unroll
    for (int c = 0; c < CC; ++c) {
        if (g.j[c] >= 0 && key[c] != g.j[c]) {
            slot[c] = e_probe_insert(keys, vals, g.j[c], slot[c], key[c]);
            if (slot[c] < 0) { full = true; slot[c] = 0; }
        }
    }
    double acc[CC];
#pragma unroll
    for (int c = 0; c < CC; ++c) acc[c] = vals[slot[c]];
#pragma unroll
    for (int c = 0; c < CC; ++c)
        if (g.j[c] >= 0 && !full) vals[slot[c]] = fma(a, g.v[c], acc[c]);
    return full;
}

// gathers run two p-steps ahead of the accumulation (three register buffers, rotated by unrolling)
template <int CC>
__device__ __forceinline__ bool accumulate_row(const double *__restrict__ xv, const int32_t *__restrict__ xi, int M,
                                               int n_i, const double *sa, const int *sk, const int *sn, int *keys,
                                               double *vals, int tg, int grp)
{
    bool full = false;      // this thread ran out of accumulator slots
    Gather<CC> gA, gB, gC;
    e_gather<CC>(gA, 0, n_i, xv, xi, M, sk, sn, tg);
    e_gather<CC>(gB, 1, n_i, xv, xi, M, sk, sn, tg);
    for (int p = 0; p < n_i; p += 3) {
        e_gather<CC>(gC, p + 2, n_i, xv, xi, M, sk, sn, tg);
        full |= e_accumulate<CC>(gA, sa[p], keys, vals);
        full = group_bar_or(grp, full);
        if (p + 1 < n_i) {
            e_gather<CC>(gA, p + 3, n_i, xv, xi, M, sk, sn, tg);
            full |= e_accumulate<CC>(gB, sa[p + 1], keys, vals);
            full = group_bar_or(grp, full);
        }
        if (p + 2 < n_i) {
            e_gather<CC>(gB, p + 4, n_i, xv, xi, M, sk, sn, tg);
            full |= e_accumulate<CC>(gC, sa[p + 2], keys, vals);
            full = group_bar_or(grp, full);
        }
        if (full) break;     // group-uniform: every thread got the same OR at the same barrier
    }
    return full;
}

// ------------------------------------------------------------------------------------------------------------
// S3 + S4: thresholded row product, fused update, norms, sorted write-back.
// ------------------------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(E_MAX_GROUPS * E_GT, 1)
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
    const int ngroups = blockDim.x / E_GT;
    const int grp = threadIdx.x / E_GT, tg = threadIdx.x % E_GT, wg = tg >> 5, lane = threadIdx.x & 31;
    uint8_t *gbase = smem + (size_t)grp * ((size_t)E_SLOTS * 12 + (size_t)sort_cap * 8);
    double *vals = (double *)gbase;                                  // [E_SLOTS]
    int *keys = (int *)(gbase + (size_t)E_SLOTS * 8);                // [E_SLOTS]
    uint8_t *scratch = gbase + (size_t)E_SLOTS * 12;
    double *sa = (double *)scratch;                                  // [M] values of row i
    int *sk = (int *)(scratch + (size_t)8 * M);                      // [M] columns of row i (= rows k to merge)
    int *sn = sk + M;                                                // [M] nnz of those rows
    unsigned long long *sortbuf = (unsigned long long *)scratch;     // aliases sa/sk/sn after phase B
    __shared__ double s_part[E_MAX_GROUPS * E_GW][4];
    __shared__ int s_cntp[E_MAX_GROUPS], s_kept[E_MAX_GROUPS], s_nkmax[E_MAX_GROUPS][2];
    __shared__ int s_last;

    double w_trp = 0.0, w_e = 0.0, w_x = 0.0, w_trn = 0.0;          // this thread's running sums over its rows
    int w_ovf_p = INT32_MAX, w_ovf_u = INT32_MAX, w_acc = INT32_MAX, w_max_p = 0, w_max_u = 0;   // group-uniform

    if (tg == 0) { s_nkmax[grp][0] = 0; s_nkmax[grp][1] = 0; }
    group_bar(grp);
    int it = 0;
    for (int64_t row64 = (int64_t)blockIdx.x * ngroups + grp; row64 < N; row64 += (int64_t)gridDim.x * ngroups) {
        const int row = (int)row64;
        const int64_t rbase = (int64_t)row * M;
        const int n_i = min(xn[row], M);
        // clear the key table; stage row i
        {
            int4 *k4 = (int4 *)keys;
            const int4 e4 = make_int4(E_EMPTY, E_EMPTY, E_EMPTY, E_EMPTY);
            for (int s = tg; s < E_SLOTS / 4; s += E_GT) k4[s] = e4;
        }
        int nk_max = 0;
        for (int p = tg; p < n_i; p += E_GT) {
            const int k = xi[rbase + p];
            const int n_k = min(xn[k], M);
            sk[p] = k;
            sa[p] = xv[rbase + p];
            sn[p] = n_k;
            nk_max = max(nk_max, n_k);
        }
        nk_max = __reduce_max_sync(0xffffffffu, nk_max);
        if (lane == 0) atomicMax(&s_nkmax[grp][it & 1], nk_max);
        // per-row counters: the previous row's readers are behind its closing barrier
        if (tg == 0) { s_cntp[grp] = 0; s_kept[grp] = 0; s_nkmax[grp][(it + 1) & 1] = 0; }
        group_bar(grp);
        const int chunks = (s_nkmax[grp][it & 1] + E_GT - 1) / E_GT;     // group-uniform
        ++it;

        // ---------------- accumulate: acc[j] = fma(x_ik, x_kj, acc[j]), p ascending ----------------
        bool full;
#define E_ACC(CC) full = accumulate_row<CC>(xv, xi, M, n_i, sa, sk, sn, keys, vals, tg, grp)
        if (chunks <= 1) E_ACC(1);
        else if (chunks == 2) E_ACC(2);
        else if (chunks == 3) E_ACC(3);
        else if (chunks == 4) E_ACC(4);
        else if (chunks <= 6) E_ACC(6);
        else E_ACC(8);
#undef E_ACC
        if (full) {                       // accumulator capacity exceeded: status -6
            w_acc = min(w_acc, row);
            if (tg == 0) on[row] = 0;
            group_bar(grp);
            continue;
        }

        // ---------------- phase A: threshold P = thr_tau(X X) (keep |p| >= tau or the diagonal) ----------------
        double r_trp = 0.0, r_e = 0.0, r_x = 0.0, r_trn = 0.0;
        int cnt_p = 0;
        for (int s = tg; s < E_SLOTS; s += E_GT) {
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
        cnt_p = __reduce_add_sync(0xffffffffu, cnt_p);
        if (lane == 0 && cnt_p) atomicAdd(&s_cntp[grp], cnt_p);
        group_bar(grp);
        // ---------------- phase B: entries of row i of X: norms, update value, mark ----------------
        for (int p = tg; p < n_i; p += E_GT) {
            const int j = sk[p];
            const double x = sa[p];
            // normally present (x_ii * x_ij touched it); a row stored without its diagonal may miss it: then P_ij is
            // absent and the column enters the union pattern as an X-only entry (value 0, dropped)
            int slot = e_hash(j), tries = 0;
            const int stride = e_stride(j);
            while (true) {
                const int key = keys[slot];
                if (key != E_EMPTY && (key & E_KEY) == j) break;
                if (key == E_EMPTY) {
                    const int old = atomicCAS(&keys[slot], E_EMPTY, j | E_DROPPED);
                    if (old == E_EMPTY) { vals[slot] = 0.0; break; }
                    if ((old & E_KEY) == j) break;
                }
                if (++tries > E_SLOTS) { full = true; slot = -1; break; }
                slot = e_next(slot, tries, stride);
            }
            if (slot >= 0) {
                const double pk = vals[slot];                                   // 0 if dropped
                const double d = pk - x;
                r_e += d * d;
                r_x += x * x;
                keys[slot] |= E_INX;
                if (branch) vals[slot] = 2.0 * x - pk;                          // Eq. 7 on the union pattern
            }
        }
        if (group_bar_or(grp, full)) {
            w_acc = min(w_acc, row);
            if (tg == 0) on[row] = 0;
            group_bar(grp);
            continue;
        }
        cnt_p = s_cntp[grp];
        // ---------------- phase C: select X' entries, compact (j, slot) into the sort buffer ----------------
        for (int s0 = 0; s0 < E_SLOTS; s0 += E_GT) {
            const int s = s0 + tg;
            const int key = s < E_SLOTS ? keys[s] : E_EMPTY;
            bool keep = false;
            int j = 0;
            if (key != E_EMPTY) {
                j = key & E_KEY;
                const double v = vals[s];
                const bool inx = (key & E_INX) != 0, dropped = (key & E_DROPPED) != 0;
                if (!inx) {
                    // column only in P: X' = -p (branch) or p, kept iff P kept it; its (P - X)^2 = p^2 is added in
                    // the sorted write-back pass so that the sum does not depend on which slot the key landed in
                    if (!dropped) {
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
            if (bal) {
                int base = 0;
                if (lane == 0) base = atomicAdd(&s_kept[grp], __popc(bal));
                base = __shfl_sync(0xffffffffu, base, 0);
                if (keep) {
                    const int pos = base + __popc(bal & ((1u << lane) - 1u));
                    if (pos < sort_cap) sortbuf[pos] = ((unsigned long long)(unsigned)j << 32) | (unsigned)s;
                }
            }
        }
        group_bar(grp);
        const int kept = s_kept[grp];
        w_max_p = max(w_max_p, cnt_p);
        w_max_u = max(w_max_u, kept);
        if (cnt_p > M) w_ovf_p = min(w_ovf_p, row);
        if (kept > M) {
            w_ovf_u = min(w_ovf_u, row);
            if (tg == 0) on[row] = 0;
        } else {
            // ---------------- sort ascending by column, write the row, zero-fill unused slots ----------------
            int n2 = 32;
            while (n2 < kept) n2 <<= 1;
            for (int q = kept + tg; q < n2; q += E_GT) sortbuf[q] = ~0ull;
            group_bitonic_sort(sortbuf, n2, tg, grp);
            for (int q = tg; q < M; q += E_GT) {
                int j = 0; double v = 0.0;
                if (q < kept) {
                    const unsigned long long e = sortbuf[q];
                    j = (int)(e >> 32);
                    const int s = (int)(e & 0xffffffffu);
                    v = vals[s];
                    if (!(keys[s] & E_INX)) r_e += v * v;            // P-only column: (P - X)^2 = p^2
                }
                oi[rbase + q] = j;
                ov[rbase + q] = v;
            }
            if (tg == 0) on[row] = kept;
        }
        w_trp += r_trp; w_e += r_e; w_x += r_x; w_trn += r_trn;
        group_bar(grp);     // the scratch / table are reused by the next row
    }

    // ---------------- per-CTA partials (fixed order), flags, last-CTA finaliser (S5) ----------------
    w_trp = warp_sum(w_trp); w_e = warp_sum(w_e); w_x = warp_sum(w_x); w_trn = warp_sum(w_trn);
    if (lane == 0) {
        double *sp = s_part[grp * E_GW + wg];
        sp[0] = w_trp; sp[1] = w_e; sp[2] = w_x; sp[3] = w_trn;
    }
    if (tg == 0) {
        if (w_ovf_p != INT32_MAX) atomicMin(&ctl->overflow_row, w_ovf_p);
        if (w_ovf_u != INT32_MAX) atomicMin(&ctl->overflow_upd, w_ovf_u);
        if (w_acc != INT32_MAX) atomicMin(&ctl->acc_row, w_acc);
        atomicMax(&ctl->nnz_max_p, w_max_p);
        atomicMax(&ctl->nnz_max_upd, w_max_u);
    }
    __syncthreads();
    if (threadIdx.x < 4) {
        double v = 0.0;
        for (int w = 0; w < ngroups * E_GW; ++w) v += s_part[w][threadIdx.x];
        partials[(size_t)blockIdx.x * 4 + threadIdx.x] = v;
    }
    __threadfence();
    __syncthreads();
    if (threadIdx.x == 0) {
        const uint32_t prev = atomicAdd(&ctl->arrivals, 1u);
        s_last = (prev + 1u == gridDim.x);
    }
    __syncthreads();
    if (s_last && threadIdx.x < 32) {
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
    const size_t smem_cap = 227 * 1024 - 1024;      // static shared memory of the kernel stays below 1 KB
    int ngroups = (int)(smem_cap / e_group_bytes(M));
    if (ngroups > E_MAX_GROUPS) ngroups = E_MAX_GROUPS;
    if (ngroups < 1 || M > 8 * E_GT) return BML_ERR_INVALID;
    const size_t smem = (size_t)ngroups * e_group_bytes(M);
    static size_t attr_smem = 0;
    if (smem > attr_smem) {
        if (cudaFuncSetAttribute(x2_ellpack_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem) != cudaSuccess)
            return BML_ERR_CUDA;
        attr_smem = smem;
    }
    int64_t grid = (N + ngroups - 1) / ngroups;
    if (grid > sms) grid = sms;
    if (grid > E_MAX_GRID) grid = E_MAX_GRID;
    // the (j, slot) sort buffer aliases the row stage: e_scratch_bytes(M) / 8 entries
    // buffer 0 is only read while parity == 0 (the standalone entry point passes a const X there)
    x2_ellpack_kernel<<<(unsigned)grid, ngroups * E_GT, smem, st>>>((double *)v0, (int32_t *)i0, (int32_t *)n0, v1, i1,
                                                                     n1, (int)N, M, tau, (int)(e_scratch_bytes(M) / 8),
                                                                     ctl, partials);
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
