// ellblock.cu -- thresholded SP2 on ELLBLOCK ("a generalization of ELLPACK-R where each element is a
// block"): block-sparse X*X on the FP64 tensor cores (mma.sync m8n8k4 f64 = SASS DMMA.8x8x4), with the
// block threshold, the update, the norms and the stop rules fused as in the scalar path (ellpack.cu).
//
// Layout (readings E1-E4 of DESIGN.md): N = NB * bs; block p of block row I is value[((I*MB + p)*bs + r)*bs + c] at block
// column index[I*MB + p]; nnz[I] blocks; block columns ascending in every iterate.  A block of thr(A) is kept iff its
// Frobenius norm >= tau or it is a diagonal block.
//
// X is symmetric (X_KJ = X_JK^T bit for bit: both triangles are always written from one computed block), so
//     P_IJ = sum_{K in row I and in row J} X_IK * X_JK^T ,          K ascending,
// an INNER product of two block rows: both operands are read with the same "row block" addressing (the dense kernel's
// X X^T trick), the accumulators of one output block live in the registers of ONE warp from the first K to the last, and
// no accumulator table, hash or atomic is needed -- which matters because the pre-threshold block fill (several hundred
// 8 x 8 blocks per block row) does not fit shared memory.  Two kernels per product:
//   kernel 1 (upper): block row I per CTA; the candidate block columns J >= I (those reachable through some K) are
//     enumerated in ascending order from a bitmap over the block columns; a warp intersects the sorted block lists of
//     rows I and J, chains the DMMAs, takes the block norm, and the kept blocks are written in arrival order (kernel 2
//     looks them up with a whole-warp scan; every iterate it writes is in ascending order again).
//   kernel 2 (assemble): block row J per CTA; for every candidate column C (both triangles) the block of thr(X X) is
//     read from its own upper list (C >= J) or transposed from row C's upper list (C < J); update against X on the
//     union of the patterns, block threshold, norms, traces, ascending write-back, last-CTA finaliser.
#include <string.h>

#include "common.cuh"
#include "../../include/bml_ellblock.h"

namespace bmlsp2 {

constexpr int EB_THREADS = 512;
constexpr int EB_WARPS = EB_THREADS / 32;
constexpr int EB_MAX_GRID = 1024;
constexpr int EB_CHUNKS = 8;             // 32-entry chunks of a block row's index list fetched together (kernel 1)
constexpr int EB_REF_SHIFT = 13;         // reference to a stored block: (block row << 13) | slot; NB <= 2^19, MB < 2^13 - 1
constexpr uint32_t EB_REF_NONE = 0xFFFFFFFFu;
constexpr int EB_PIPE_MAX = 8;               // block pairs whose operand loads are in flight together (kernel 1)

__device__ __forceinline__ int eb_find(const int *__restrict__ list, int n, int key)
{
    int lo = 0, hi = n;
    while (lo < hi) { const int mid = (lo + hi) >> 1; if (list[mid] < key) lo = mid + 1; else hi = mid; }
    return (lo < n && list[lo] == key) ? lo : -1;
}

// the same search done by a whole warp on a list in GLOBAL memory: every lane tests the slots lane, lane + 32, ... (one
// round of independent, coalesced loads instead of log2(n) dependent ones); all lanes return the position or -1
__device__ __forceinline__ int eb_find_warp(const int *__restrict__ list, int n, int key, int lane)
{
    int hit = -1;
    for (int q0 = 0; q0 < n; q0 += 128) {
        int v[4];
#pragma unroll
        for (int u = 0; u < 4; ++u) { const int q = q0 + u * 32 + lane; v[u] = q < n ? __ldg(list + q) : -1; }
#pragma unroll
        for (int u = 0; u < 4; ++u) if (v[u] == key) hit = q0 + u * 32 + lane;
    }
    const unsigned bal = __ballot_sync(0xffffffffu, hit >= 0);
    return bal ? __shfl_sync(0xffffffffu, hit, __ffs(bal) - 1) : -1;
}

// The set bits of the bitmap as the ascending list cand[0 .. n) (clearing the bitmap on the way); returns n, which may
// exceed cand_cap (entries beyond it are not written).  All threads of the CTA take part; the caller has synchronised
// after setting the bits.
__device__ __forceinline__ int eb_scan_bitmap(unsigned *bitmap, int NBW, int *cand, int cand_cap, int *s_scan)
{
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    int base = 0;
    for (int w0 = 0; w0 < NBW; w0 += EB_THREADS) {
        const int w = w0 + tid;
        const unsigned bits = w < NBW ? bitmap[w] : 0u;
        if (w < NBW) bitmap[w] = 0u;
        const int cnt = __popc(bits);
        int inc = cnt;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) { const int t = __shfl_up_sync(0xffffffffu, inc, o); if (lane >= o) inc += t; }
        if (lane == 31) s_scan[warp] = inc;
        __syncthreads();
        int wbase = 0, total = 0;
#pragma unroll
        for (int w2 = 0; w2 < EB_WARPS; ++w2) { const int t = s_scan[w2]; if (w2 < warp) wbase += t; total += t; }
        int pos = base + wbase + inc - cnt;
        unsigned b = bits;
        while (b) {
            const int bit = __ffs(b) - 1;
            b &= b - 1;
            if (pos < cand_cap) cand[pos] = (w << 5) | bit;
            ++pos;
        }
        base += total;
        __syncthreads();
    }
    return base;
}

// Candidate block columns of block row I: every J (>= jmin) stored in some row K with K stored in row I.  Sets the bits,
// then writes the ascending list cand[0 .. ncand).  All threads of the CTA take part.
__device__ __forceinline__ int eb_candidates(const int32_t *__restrict__ xi, const int32_t *__restrict__ xn, int MB, int NB,
                                             const int *sI, int nI, int jmin, unsigned *bitmap, int *cand, int cand_cap,
                                             int *s_scan)
{
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    for (int p = warp; p < nI; p += EB_WARPS) {
        const int K = sI[p];
        const int nK = min(xn[K], MB);
        const int32_t *row = xi + (int64_t)K * MB;
        for (int q = lane; q < nK; q += 32) {
            const int J = row[q];
            if (J >= jmin) atomicOr(&bitmap[J >> 5], 1u << (J & 31));
        }
    }
    __syncthreads();
    return eb_scan_bitmap(bitmap, (NB + 31) >> 5, cand, cand_cap, s_scan);
}

// The same enumeration with the pre-screen folded in: while the two-hop neighbours J of row I are marked, the bound
// sum_K ||X_IK||_F ||X_KJ||_F >= ||P_IJ||_F is accumulated per block column (FP32 atomics in shared memory; X is symmetric,
// so ||X_KJ|| = ||X_JK||), and only the columns whose bound reaches tau (or J = I) enter the list -- the others would be
// dropped whatever their entries are.  The 1e-4 margin covers the FP32 rounding of up to MB positive terms; which side
// of the margin a borderline column falls on does not change any result (kernel 1 repeats the test in FP64).
__device__ __forceinline__ int eb_candidates_bounded(const int32_t *__restrict__ xi, const int32_t *__restrict__ xn,
                                                     const double *__restrict__ bnX, int MB, int NB, const int *sI,
                                                     const double *snrm, int nI, int I, double tau, unsigned *bitmap,
                                                     float *sbound, int *cand, int cand_cap, int *s_scan)
{
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int NBW = (NB + 31) >> 5;
    for (int p = warp; p < nI; p += EB_WARPS) {
        const int K = sI[p];
        const double nIK = snrm[p];
        const int nK = min(xn[K], MB);
        const int32_t *row = xi + (int64_t)K * MB;
        const double *nrow = bnX + (int64_t)K * MB;
        for (int q = lane; q < nK; q += 32) {
            const int J = row[q];
            if (J >= I) {
                atomicOr(&bitmap[J >> 5], 1u << (J & 31));
                atomicAdd(&sbound[J], (float)(nIK * nrow[q]));
            }
        }
    }
    __syncthreads();
    const float thr = (float)(tau * (1.0 - 1e-4));
    int base = 0;
    for (int w0 = 0; w0 < NBW; w0 += EB_THREADS) {
        const int w = w0 + tid;
        unsigned b = w < NBW ? bitmap[w] : 0u;
        if (w < NBW) bitmap[w] = 0u;
        unsigned bits = 0u;
        while (b) {
            const int bit = __ffs(b) - 1;
            b &= b - 1;
            const int J = (w << 5) | bit;
            const float v = sbound[J];
            sbound[J] = 0.0f;
            if (J == I || v >= thr) bits |= 1u << bit;
        }
        const int cnt = __popc(bits);
        int inc = cnt;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) { const int t = __shfl_up_sync(0xffffffffu, inc, o); if (lane >= o) inc += t; }
        if (lane == 31) s_scan[warp] = inc;
        __syncthreads();
        int wbase = 0, total = 0;
#pragma unroll
        for (int w2 = 0; w2 < EB_WARPS; ++w2) { const int t = s_scan[w2]; if (w2 < warp) wbase += t; total += t; }
        int pos = base + wbase + inc - cnt;
        while (bits) {
            const int bit = __ffs(bits) - 1;
            bits &= bits - 1;
            if (pos < cand_cap) cand[pos] = (w << 5) | bit;
            ++pos;
        }
        base += total;
        __syncthreads();
    }
    return base;
}

__device__ __forceinline__ double lds_f64(uint32_t saddr)
{
    double v;
    asm("ld.shared.f64 %0, [%1];" : "=d"(v) : "r"(saddr));
    return v;
}

// PIPE block pairs of one candidate: acc += X_IK * X_JK^T for the matches list[0 .. nm), in order.  The operand blocks
// of row J (global memory: L2) are all requested before the first DMMA; row I's blocks come from shared memory (32-bit
// address sA_u32).  FULL: nm == PIPE, no predicates.
template <int BS, int PIPE, bool FULL>
__device__ __forceinline__ void eb_group(double (&acc)[(BS + 7) / 8][(BS + 7) / 8][2], const unsigned *list, int nm,
                                         uint32_t sA_u32, const double *__restrict__ valJ, int g, int t)
{
    constexpr int MT = (BS + 7) / 8, KS = (BS + 3) / 4, BB = BS * BS;
    uint32_t aoff[PIPE];
    double bq[PIPE][KS][MT];
#pragma unroll
    for (int u = 0; u < PIPE; ++u) {
        const unsigned e = (FULL || u < nm) ? list[u] : 0u;                       // broadcast
        aoff[u] = sA_u32 + (e >> 16) * (uint32_t)(BB * 8);
        const double *Bp = valJ + (size_t)(e & 0xffffu) * BB;
#pragma unroll
        for (int s = 0; s < KS; ++s)
#pragma unroll
            for (int m = 0; m < MT; ++m) {
                const int r = m * 8 + g, col = 4 * s + t;
                bq[u][s][m] = ((FULL || u < nm) && r < BS && col < BS) ? __ldg(Bp + r * BS + col) : 0.0;
            }
    }
#pragma unroll
    for (int u = 0; u < PIPE; ++u) {
        if (FULL || u < nm) {                      // warp-uniform
#pragma unroll
            for (int s = 0; s < KS; ++s) {
                double a[MT];
#pragma unroll
                for (int m = 0; m < MT; ++m) {
                    const int r = m * 8 + g, col = 4 * s + t;
                    a[m] = (r < BS && col < BS) ? lds_f64(aoff[u] + (uint32_t)(r * BS + col) * 8u) : 0.0;
                }
#pragma unroll
                for (int m = 0; m < MT; ++m)
#pragma unroll
                    for (int n = 0; n < MT; ++n) dmma884(acc[m][n][0], acc[m][n][1], a[m], bq[u][s][n]);
            }
        }
    }
}

// ------------------------------------------------------------------------------------------------------------
// Kernel 1: upper blocks of thr(X X)
// ------------------------------------------------------------------------------------------------------------
template <int BS>
__global__ void __launch_bounds__(EB_THREADS, 1)
x2_ellblock_upper_kernel(const double *__restrict__ v0, const int32_t *__restrict__ i0, const int32_t *__restrict__ n0,
                         const double *__restrict__ v1, const int32_t *__restrict__ i1, const int32_t *__restrict__ n1,
                         int NB, int MB, double tau, int cand_cap, int use_map, int match_off, int bound_off,
                         Sp2Ctl *__restrict__ ctl,
                         double *__restrict__ tv, int32_t *__restrict__ ti, int32_t *__restrict__ tn,
                         uint32_t *__restrict__ lref, int32_t *__restrict__ lcnt, const double *__restrict__ bn0,
                         const double *__restrict__ bn1)
{
    constexpr int MT = (BS + 7) / 8, KS = (BS + 3) / 4, BB = BS * BS;
    constexpr int EB_PIPE = BS == 16 ? 4 : EB_PIPE_MAX;        // bs = 16: 16 operand registers per block pair
    if (ctl->done) return;
    const int parity = ctl->parity;
    const double *__restrict__ xv = parity ? v1 : v0;
    const int32_t *__restrict__ xi = parity ? i1 : i0;
    const int32_t *__restrict__ xn = parity ? n1 : n0;
    const double *__restrict__ bnX = parity ? bn1 : bn0;             // Frobenius norms of the blocks of X

    extern __shared__ __align__(16) uint8_t smem[];
    const int NBW = (NB + 31) >> 5;
    double *sA = (double *)smem;                                     // [MB][BS*BS] blocks of block row I
    const uint32_t sA_u32 = smem_u32(sA);
    int *sI = (int *)(sA + (size_t)MB * BB);                         // [MB] their block columns
    int *cand = sI + MB;                                             // [cand_cap]
    unsigned *bitmap = (unsigned *)(cand + cand_cap);                // [NBW]
    // direct map block column -> 1 + position in row I (0 = absent), when NB is small enough to afford 2 NB bytes: one
    // shared-memory load per entry of row J instead of a binary search in row I's list
    unsigned short *spos = use_map ? (unsigned short *)(bitmap + NBW) : nullptr;
    // per warp: the matches of the candidate in hand, [MB] entries (after the map, 4-byte aligned: NB * 2 + 16 bytes)
    unsigned *mlist = (unsigned *)(smem + match_off) + (size_t)(threadIdx.x >> 5) * MB;
    double *snrm = (double *)(smem + match_off + (size_t)EB_WARPS * MB * 4);      // [MB] norms of the blocks of row I
    float *sbound = bound_off ? (float *)(smem + bound_off) : nullptr;            // [NB] pre-screen bound per block column
    __shared__ int s_scan[EB_WARPS];
    __shared__ int s_ticket, s_kept;

    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int g = lane >> 2, t = lane & 3;
    for (int w = tid; w < NBW; w += EB_THREADS) bitmap[w] = 0u;
    if (use_map) for (int w = tid; w < NB; w += EB_THREADS) spos[w] = 0;
    if (sbound) for (int w = tid; w < NB; w += EB_THREADS) sbound[w] = 0.0f;

    for (int I = blockIdx.x; I < NB; I += gridDim.x) {
        const int nI = min(xn[I], MB);
        __syncthreads();
        for (int p = tid; p < nI; p += EB_THREADS) {
            const int K = xi[(int64_t)I * MB + p];
            sI[p] = K;
            snrm[p] = bnX[(int64_t)I * MB + p];
            if (use_map) spos[K] = (unsigned short)(p + 1);
        }
        if (tid == 0) { s_ticket = 0; s_kept = 0; }
        {
            const double2 *src = (const double2 *)(xv + (int64_t)I * MB * BB);
            double2 *dst = (double2 *)sA;
            for (int e = tid; e < nI * BB / 2; e += EB_THREADS) dst[e] = src[e];
        }
        __syncthreads();
        const int ncand_all = sbound ? eb_candidates_bounded(xi, xn, bnX, MB, NB, sI, snrm, nI, I, tau, bitmap, sbound, cand,
                                                             cand_cap, s_scan)
                                     : eb_candidates(xi, xn, MB, NB, sI, nI, I, bitmap, cand, cand_cap, s_scan);
        const int ncand = min(ncand_all, cand_cap);
        // more candidate blocks (before thresholding) than the list holds: the capacity failure -6, like the scalar
        // path's accumulator table
        if (ncand_all > cand_cap && tid == 0) atomicMin(&ctl->acc_row, I);
        // Candidates are handed out by a ticket counter: a warp that drew a candidate with few matches takes the next
        // one instead of waiting at a batch barrier.
        while (true) {
            int c = 0;
            if (lane == 0) c = atomicAdd(&s_ticket, 1);
            c = __shfl_sync(0xffffffffu, c, 0);
            if (c >= ncand) break;
            bool keep = false;
            double acc[MT][MT][2];
#pragma unroll
            for (int a = 0; a < MT; ++a)
#pragma unroll
                for (int b = 0; b < MT; ++b) { acc[a][b][0] = 0.0; acc[a][b][1] = 0.0; }
            int J = -1;
            {
                J = cand[c];
                const int nJ = min(xn[J], MB);
                const int32_t *rowJ = xi + (int64_t)J * MB;
                const double *valJ = xv + (int64_t)J * MB * BB;
                // (1) intersection of the block lists of rows I and J, written to the warp's match list in ascending K
                // (row J is in ascending order): entry = (position in row I << 16) | position in row J
                // The block norms of row J travel with its block columns (same round trip): the pre-screen below needs
                // those of the matches, and a second, dependent load would cost the skipped candidates as much again.
                int nmatch = 0;
                double bound = 0.0;
                const double *bnJ = bnX + (int64_t)J * MB;
                for (int qg = 0; qg < nJ; qg += 32 * EB_CHUNKS) {
                    int kq[EB_CHUNKS];                     // block columns of row J, EB_CHUNKS x 32 at a time (one round trip)
                    double nq[EB_CHUNKS];
#pragma unroll
                    for (int u = 0; u < EB_CHUNKS; ++u) {
                        const int q = qg + u * 32 + lane;
                        kq[u] = q < nJ ? __ldg(rowJ + q) : -1;
                        nq[u] = q < nJ ? __ldg(bnJ + q) : 0.0;
                    }
#pragma unroll
                    for (int u = 0; u < EB_CHUNKS; ++u) {
                        const int q0 = qg + u * 32;
                        if (q0 >= nJ) break;
                        const int pI = kq[u] < 0 ? -1 : (use_map ? (int)spos[kq[u]] - 1 : eb_find(sI, nI, kq[u]));
                        const unsigned bal = __ballot_sync(0xffffffffu, pI >= 0);
                        if (pI >= 0) {
                            mlist[nmatch + __popc(bal & ((1u << lane) - 1u))] = ((unsigned)pI << 16) | (unsigned)(q0 + lane);
                            bound += snrm[pI] * nq[u];
                        }
                        nmatch += __popc(bal);
                    }
                }
                __syncwarp();
                // Pre-screen: ||P_IJ||_F <= sum_K ||X_IK||_F ||X_JK||_F.  When that bound is below tau the block is
                // dropped whatever its entries are, so its products -- and the 512-byte operand loads -- are skipped;
                // the outcome is the oracle's (the 1e-9 margin covers the round-off of the norms and of the bound).
                // Most two-hop candidates of a decaying matrix end here.
                bound = warp_sum(bound);
                if (J != I && tau > 0.0 && bound < tau * (1.0 - 1e-9)) nmatch = 0;
                // (2) the block products, EB_PIPE at a time: the operand blocks of row J come from L2 and the loads of a
                // whole group are issued before the first DMMA needs them (one match at a time left every warp waiting
                // a full L2 round trip per block pair; groups cut at the 32-entry chunks of the list held ~4 in flight)
                // Full groups take a path without predicates or zero-filled operands (almost all of them: a surviving
                // candidate has ~64 matches); row I's operands are read through a 32-bit shared-memory address (the
                // generic pointer made the compiler rebuild the shared window base for every block pair).
                int m0 = 0;
                for (; m0 + EB_PIPE <= nmatch; m0 += EB_PIPE)
                    eb_group<BS, EB_PIPE, true>(acc, mlist + m0, EB_PIPE, sA_u32, valJ, g, t);
                if (m0 < nmatch) eb_group<BS, EB_PIPE, false>(acc, mlist + m0, nmatch - m0, sA_u32, valJ, g, t);
                __syncwarp();                              // the list is rewritten for the next candidate
                double nrm2 = 0.0;
#pragma unroll
                for (int m = 0; m < MT; ++m)
#pragma unroll
                    for (int n = 0; n < MT; ++n) {
                        const int r = m * 8 + g, cc = n * 8 + 2 * t;
                        if (r < BS && cc < BS) nrm2 += acc[m][n][0] * acc[m][n][0];
                        if (r < BS && cc + 1 < BS) nrm2 += acc[m][n][1] * acc[m][n][1];
                    }
                nrm2 = warp_sum(nrm2);
                keep = sqrt(nrm2) >= tau || J == I;
            }
            // a kept block takes the next free slot of the row: the upper list is in ARRIVAL order (kernel 2 finds blocks
            // in it with a whole-warp scan, which needs no order; an in-order commit cost 23% of this kernel's warp time
            // in waits behind longer candidates)
            int pos = 0;
            if (keep && lane == 0) pos = atomicAdd(&s_kept, 1);
            pos = __shfl_sync(0xffffffffu, pos, 0);
            if (keep && pos < MB) {
                double *out = tv + ((int64_t)I * MB + pos) * BB;
#pragma unroll
                for (int m = 0; m < MT; ++m)
#pragma unroll
                    for (int n = 0; n < MT; ++n) {
                        const int r = m * 8 + g, cc = n * 8 + 2 * t;
                        if (r < BS && cc + 1 < BS) *(double2 *)(out + r * BS + cc) = make_double2(acc[m][n][0], acc[m][n][1]);
                        else if (r < BS && cc < BS) out[r * BS + cc] = acc[m][n][0];
                    }
                if (lane == 0) ti[(int64_t)I * MB + pos] = J;
            }
            // the mirror block P_JI = P_IJ^T belongs to row J: leave a reference (row, slot) in row J's lower list, so that
            // kernel 2 finds it without searching row I.  The counter counts ALL kept blocks (row lengths stay exact when
            // a list runs over MB); a block that found no slot leaves an invalid reference.
            if (keep && J != I && lane == 0) {
                const int k = atomicAdd(&lcnt[J], 1);
                if (k < MB) lref[(int64_t)J * MB + k] = pos < MB ? (((uint32_t)I << EB_REF_SHIFT) | (uint32_t)pos) : EB_REF_NONE;
            }
        }
        __syncthreads();
        if (use_map) for (int p = tid; p < nI; p += EB_THREADS) spos[sI[p]] = 0;
        const int kept_total = s_kept;
        if (tid == 0) tn[I] = kept_total;      // may exceed MB: kernel 2 reports the overflow
    }
}

// ------------------------------------------------------------------------------------------------------------
// Kernel 2: assemble the full block rows of thr(X X), update, threshold, norms, write-back, finaliser
// ------------------------------------------------------------------------------------------------------------
template <int BS>
__global__ void __launch_bounds__(EB_THREADS, 1)
x2_ellblock_assemble_kernel(double *__restrict__ v0, int32_t *__restrict__ i0, int32_t *__restrict__ n0,
                            double *__restrict__ v1, int32_t *__restrict__ i1, int32_t *__restrict__ n1, int NB, int MB,
                            double tau, int cand_cap, int use_map, int pref_off, Sp2Ctl *__restrict__ ctl,
                            double *__restrict__ partials, const double *__restrict__ tv, const int32_t *__restrict__ ti, const int32_t *__restrict__ tn,
                            const uint32_t *__restrict__ lref, int32_t *__restrict__ lcnt, double *__restrict__ bn0,
                            double *__restrict__ bn1)
{
    constexpr int BB = BS * BS, EPL = (BB + 31) / 32;        // elements of a block per lane
    if (ctl->done) return;
    const int parity = ctl->parity;
    const int branch = ctl->branch_cur;
    const double *__restrict__ xv = parity ? v1 : v0;
    const int32_t *__restrict__ xi = parity ? i1 : i0;
    const int32_t *__restrict__ xn = parity ? n1 : n0;
    double *__restrict__ ov = parity ? v0 : v1;
    int32_t *__restrict__ oi = parity ? i0 : i1;
    int32_t *__restrict__ on = parity ? n0 : n1;
    double *__restrict__ bnO = parity ? bn0 : bn1;                   // Frobenius norms of the blocks of X'

    extern __shared__ __align__(16) uint8_t smem[];
    const int NBW = (NB + 31) >> 5;
    int *sX = (int *)smem;                                           // [MB] block columns of row J of X
    int *cand = sX + MB;                                             // [cand_cap]
    unsigned *bitmap = (unsigned *)(cand + cand_cap);                // [NBW]
    unsigned short *spos = use_map ? (unsigned short *)(bitmap + NBW) : nullptr;   // block column -> 1 + position in row J of X
    uint32_t *pref = (uint32_t *)(smem + pref_off);                  // [cand_cap] where the block of thr(X X) of a candidate is
    __shared__ int s_scan[EB_WARPS], s_keep[EB_WARPS], s_pcnt[EB_WARPS], s_last;
    __shared__ double s_part[EB_WARPS][4];

    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    for (int w = tid; w < NBW; w += EB_THREADS) bitmap[w] = 0u;
    if (use_map) for (int w = tid; w < NB; w += EB_THREADS) spos[w] = 0;
    double w_trp = 0.0, w_e = 0.0, w_x = 0.0, w_trn = 0.0;
    int w_ovf_p = INT32_MAX, w_ovf_u = INT32_MAX, w_max_p = 0, w_max_u = 0;

    for (int J = blockIdx.x; J < NB; J += gridDim.x) {
        const int nX = min(xn[J], MB);
        const int nU = tn[J];                                        // own upper blocks (may exceed MB = overflow)
        const int nL = lcnt[J];                                      // references to the blocks of the rows above (all of them)
        __syncthreads();
        for (int p = tid; p < nX; p += EB_THREADS) {
            const int K = xi[(int64_t)J * MB + p];
            sX[p] = K;
            if (use_map) spos[K] = (unsigned short)(p + 1);
        }
        __syncthreads();
        // The union pattern of row J, in ascending order: the blocks of thr(X X) -- own upper list and the references to
        // blocks of the rows above that kernel 1 left -- and the blocks of X.  (No two-hop enumeration here: a block
        // column that is in neither contributes nothing to the update or to the norms.)  At most 3 MB <= cand_cap entries.
        for (int q = tid; q < min(nU, MB); q += EB_THREADS) {
            const int C = ti[(int64_t)J * MB + q];
            atomicOr(&bitmap[C >> 5], 1u << (C & 31));
        }
        for (int q = tid; q < min(nL, MB); q += EB_THREADS) {
            const uint32_t ref = lref[(int64_t)J * MB + q];
            if (ref != EB_REF_NONE) { const int C = (int)(ref >> EB_REF_SHIFT); atomicOr(&bitmap[C >> 5], 1u << (C & 31)); }
        }
        for (int q = tid; q < nX; q += EB_THREADS) { const int C = sX[q]; atomicOr(&bitmap[C >> 5], 1u << (C & 31)); }
        __syncthreads();
        const int ncand = min(eb_scan_bitmap(bitmap, NBW, cand, cand_cap, s_scan), cand_cap);
        // where the block of thr(X X) of every candidate is: own upper list (row J, slot q) or, transposed, a block of a
        // row above; the positions in the candidate list by binary search in shared memory
        for (int q = tid; q < ncand; q += EB_THREADS) pref[q] = EB_REF_NONE;
        if (tid == 0) lcnt[J] = 0;                                   // every thread has read it (barrier above): for the next product
        __syncthreads();
        for (int q = tid; q < min(nU, MB); q += EB_THREADS) {
            const int c = eb_find(cand, ncand, ti[(int64_t)J * MB + q]);
            if (c >= 0) pref[c] = ((uint32_t)J << EB_REF_SHIFT) | (uint32_t)q;
        }
        for (int q = tid; q < min(nL, MB); q += EB_THREADS) {
            const uint32_t ref = lref[(int64_t)J * MB + q];
            if (ref != EB_REF_NONE) {
                const int c = eb_find(cand, ncand, (int)(ref >> EB_REF_SHIFT));
                if (c >= 0) pref[c] = ref;
            }
        }
        __syncthreads();
        const bool ovf_p = nU + nL > MB;                             // the full row of thr(X X) has nU + nL blocks
        int kept_total = 0;
        const int p_total = nU + nL;
        for (int c0 = 0; c0 < ncand; c0 += EB_WARPS) {
            const int c = c0 + warp;
            bool keep = false, haveP = false;
            double blk_nrm = 0.0;                                    // ||X'_JC||_F of a kept block
            double xnew[EPL];
#pragma unroll
            for (int e = 0; e < EPL; ++e) xnew[e] = 0.0;
            int C = -1;
            if (c < ncand) {
                C = cand[c];
                const uint32_t ref = pref[c];
                const int prow = (int)(ref >> EB_REF_SHIFT);
                const double *P = ref != EB_REF_NONE ? tv + ((int64_t)prow * MB + (ref & ((1u << EB_REF_SHIFT) - 1u))) * BB : nullptr;
                const bool transposed = P && prow != J;
                const int px = use_map ? (int)spos[C] - 1 : eb_find(sX, nX, C);
                const double *X = px >= 0 ? xv + ((int64_t)J * MB + px) * BB : nullptr;
                haveP = P != nullptr;
                double r_e = 0.0, r_x = 0.0, r_trp = 0.0, r_trn = 0.0, nrm2 = 0.0;
#pragma unroll
                for (int e = 0; e < EPL; ++e) {
                    const int el = e * 32 + lane;
                    if (el < BB) {
                        const int r = el / BS, cc = el % BS;
                        const double p = P ? (transposed ? P[cc * BS + r] : P[el]) : 0.0;
                        const double x = X ? X[el] : 0.0;
                        const double d = p - x;
                        r_e += d * d;
                        r_x += x * x;
                        const double xn_ = branch ? (2.0 * x - p) : p;             // Eq. 7 on the union pattern : Eq. 6
                        xnew[e] = xn_;
                        nrm2 += xn_ * xn_;
                        if (C == J && r == cc) { r_trp += p; r_trn += xn_; }
                    }
                }
                nrm2 = warp_sum(nrm2);
                blk_nrm = sqrt(nrm2);
                if (branch) keep = (P || X) && (blk_nrm >= tau || C == J);
                else keep = haveP;                                   // X' = thr(X X) as it stands
                if (P || X) { w_e += r_e; w_x += r_x; w_trp += r_trp; }
                if (keep) w_trn += r_trn;
            }
            if (lane == 0) { s_keep[warp] = keep ? 1 : 0; s_pcnt[warp] = haveP ? 1 : 0; }
            __syncthreads();
            int pos = kept_total, total = 0;
#pragma unroll
            for (int w2 = 0; w2 < EB_WARPS; ++w2) {
                const int k = s_keep[w2];
                if (w2 < warp) pos += k;
                total += k;
            }
            if (keep && pos < MB) {
                double *out = ov + ((int64_t)J * MB + pos) * BB;
#pragma unroll
                for (int e = 0; e < EPL; ++e) {
                    const int el = e * 32 + lane;
                    if (el < BB) out[el] = xnew[e];
                }
                if (lane == 0) { oi[(int64_t)J * MB + pos] = C; bnO[(int64_t)J * MB + pos] = blk_nrm; }
            }
            kept_total += total;
            __syncthreads();
        }
        if (tid == 0) {
            w_max_p = max(w_max_p, ovf_p ? max(p_total, MB + 1) : p_total);
            if (ovf_p) { w_ovf_p = min(w_ovf_p, J); on[J] = 0; }
            else {
                w_max_u = max(w_max_u, kept_total);
                if (kept_total > MB) { w_ovf_u = min(w_ovf_u, J); on[J] = 0; }
                else on[J] = kept_total;
            }
        }
        // slots beyond the count are not written here (every reader goes by nnz); the copy-out zeroes them in D
        if (use_map) { __syncthreads(); for (int p = tid; p < nX; p += EB_THREADS) spos[sX[p]] = 0; }
    }
    // ---------------- per-CTA partials (fixed order), flags, last-CTA finaliser ----------------
    w_trp = warp_sum(w_trp); w_e = warp_sum(w_e); w_x = warp_sum(w_x); w_trn = warp_sum(w_trn);
    if (lane == 0) { s_part[warp][0] = w_trp; s_part[warp][1] = w_e; s_part[warp][2] = w_x; s_part[warp][3] = w_trn; }
    if (tid == 0) {
        if (w_ovf_p != INT32_MAX) atomicMin(&ctl->overflow_row, w_ovf_p);
        if (w_ovf_u != INT32_MAX) atomicMin(&ctl->overflow_upd, w_ovf_u);
        atomicMax(&ctl->nnz_max_p, w_max_p);
        atomicMax(&ctl->nnz_max_upd, w_max_u);
    }
    __syncthreads();
    if (tid < 4) {
        double v = 0.0;
        for (int w2 = 0; w2 < EB_WARPS; ++w2) v += s_part[w2][tid];
        partials[(size_t)blockIdx.x * 4 + tid] = v;
    }
    __threadfence();
    __syncthreads();
    if (tid == 0) {
        __threadfence();
        const uint32_t prev = atomicAdd(&ctl->arrivals, 1u);
        __threadfence();
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
// Gershgorin rows, rescale (Eq. 5, missing diagonal block inserted, ascending block columns), trace, copy-out
// ------------------------------------------------------------------------------------------------------------
// one warp per scalar row: rowlh[2 i] = H_ii - radius, rowlh[2 i + 1] = H_ii + radius (compensated radius)
__global__ void __launch_bounds__(256) gershgorin_rows_ellblock_kernel(const double *__restrict__ hv,
                                                                       const int32_t *__restrict__ hi,
                                                                       const int32_t *__restrict__ hn, int NB, int MB,
                                                                       int bs, double *__restrict__ rowlh)
{
    const int row = (blockIdx.x * blockDim.x + threadIdx.x) >> 5, lane = threadIdx.x & 31;
    if (row >= NB * bs) return;
    const int I = row / bs, r = row % bs;
    const int n = min(hn[I], MB);
    double s = 0.0, c = 0.0, d = 0.0;
    for (int e = lane; e < n * bs; e += 32) {
        const int p = e / bs, cc = e % bs;
        const double v = hv[(((int64_t)I * MB + p) * bs + r) * bs + cc];
        if (hi[(int64_t)I * MB + p] == I && cc == r) d = v;
        else comp_add(s, c, fabs(v));
    }
    const double rad = comp_warp_sum(s, c);
    d = warp_sum(d);                                       // one lane holds it, the others 0
    if (lane == 0) { rowlh[2 * (size_t)row] = d - rad; rowlh[2 * (size_t)row + 1] = d + rad; }
}

// one warp per block row
__global__ void __launch_bounds__(128)
rescale_ellblock_kernel(const double *__restrict__ hv, const int32_t *__restrict__ hi, const int32_t *__restrict__ hn,
                        int NB, int MB, int bs, const double *__restrict__ bounds, double *__restrict__ xv,
                        int32_t *__restrict__ xi, int32_t *__restrict__ xn, double *__restrict__ diag,
                        int *__restrict__ fail_flag, int sort_cap)
{
    extern __shared__ __align__(16) uint8_t smem[];
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31, nwarps = blockDim.x >> 5;
    unsigned long long *sortbuf = (unsigned long long *)(smem + (size_t)warp * sort_cap * 8);
    const double emin = bounds[0], emax = bounds[1];
    const double s = 1.0 / (emax - emin);
    const int I = blockIdx.x * nwarps + warp;
    if (I >= NB) return;
    const int bb = bs * bs;
    const int n = min(hn[I], MB);
    int has = 0;
    for (int p = lane; p < n; p += 32) {
        const int J = hi[(int64_t)I * MB + p];
        has |= (J == I);
        sortbuf[p] = ((unsigned long long)(unsigned)J << 32) | (unsigned)p;
    }
    has = __any_sync(0xffffffffu, has);
    const int total = n + (has ? 0 : 1);
    if (total > MB) {
        if (lane == 0) { atomicMax(&fail_flag[1], INT32_MAX - I); xn[I] = 0; }
        for (int r = lane; r < bs; r += 32) diag[(size_t)I * bs + r] = 0.0;
        return;
    }
    if (!has && lane == 0) sortbuf[n] = ((unsigned long long)(unsigned)I << 32) | 0xffffffffu;
    int n2 = 32;
    while (n2 < total) n2 <<= 1;
    __syncwarp();
    for (int q = total + lane; q < n2; q += 32) sortbuf[q] = ~0ull;
    __syncwarp();
    for (int k = 2; k <= n2; k <<= 1)
        for (int j = k >> 1; j > 0; j >>= 1) {
            for (int tq = lane; tq < (n2 >> 1); tq += 32) {
                const int a = ((tq & ~(j - 1)) << 1) | (tq & (j - 1)), l = a | j;
                const bool up = (a & k) == 0;
                const unsigned long long x = sortbuf[a], y = sortbuf[l];
                if ((x > y) == up) { sortbuf[a] = y; sortbuf[l] = x; }
            }
            __syncwarp();
        }
    for (int q = 0; q < MB; ++q) {
        double *dst = xv + ((int64_t)I * MB + q) * bb;
        int J = 0;
        const double *src = nullptr;
        bool live = false;
        if (q < total) {
            const unsigned long long e = sortbuf[q];
            J = (int)(e >> 32);
            const unsigned p = (unsigned)(e & 0xffffffffu);
            live = true;
            if (p != 0xffffffffu) src = hv + ((int64_t)I * MB + p) * bb;
        }
        for (int el = lane; el < bb; el += 32) {
            double v = 0.0;
            if (live) {
                const int r = el / bs, c = el % bs;
                const double h = src ? src[el] : 0.0;
                v = (J == I && r == c) ? s * (emax - h) : -s * h;
                if (J == I && r == c) diag[(size_t)I * bs + r] = v;
            }
            dst[el] = v;
        }
        if (lane == 0) xi[(int64_t)I * MB + q] = live ? J : 0;
    }
    if (lane == 0) xn[I] = total;
}

__global__ void __launch_bounds__(1024) trace_ellblock_kernel(const double *__restrict__ v, const int32_t *__restrict__ idx,
                                                              const int32_t *__restrict__ nnz, int NB, int MB, int bs,
                                                              double *__restrict__ out)
{
    __shared__ double s_w[32];
    double s = 0.0;
    for (int row = threadIdx.x; row < NB * bs; row += blockDim.x) {
        const int I = row / bs, r = row % bs;
        const int n = min(nnz[I], MB);
        const int p = eb_find(idx + (int64_t)I * MB, n, I);          // rows of an iterate are in ascending order
        if (p >= 0) s += v[(((int64_t)I * MB + p) * bs + r) * bs + r];
    }
    s = warp_sum(s);
    if ((threadIdx.x & 31) == 0) s_w[threadIdx.x >> 5] = s;
    __syncthreads();
    if (threadIdx.x < 32) {
        double r = s_w[threadIdx.x];
        r = warp_sum(r);
        if (threadIdx.x == 0) *out = r;
    }
}

// trace of an ELLBLOCK matrix whose block rows may be in any order (bml_trace on caller data)
__global__ void __launch_bounds__(1024) trace_ellblock_unsorted_kernel(const double *__restrict__ v,
                                                                       const int32_t *__restrict__ idx,
                                                                       const int32_t *__restrict__ nnz, int NB, int MB, int bs,
                                                                       double *__restrict__ out)
{
    __shared__ double s_w[32];
    double s = 0.0;
    for (int row = threadIdx.x; row < NB * bs; row += blockDim.x) {
        const int I = row / bs, r = row % bs;
        const int n = min(nnz[I], MB);
        for (int p = 0; p < n; ++p)
            if (idx[(int64_t)I * MB + p] == I) s += v[(((int64_t)I * MB + p) * bs + r) * bs + r];
    }
    s = warp_sum(s);
    if ((threadIdx.x & 31) == 0) s_w[threadIdx.x >> 5] = s;
    __syncthreads();
    if (threadIdx.x < 32) {
        double r = s_w[threadIdx.x];
        r = warp_sum(r);
        if (threadIdx.x == 0) *out = r;
    }
}

__global__ void __launch_bounds__(256)
copy_out_ellblock_kernel(const double *__restrict__ v0, const int32_t *__restrict__ i0, const int32_t *__restrict__ n0,
                         const double *__restrict__ v1, const int32_t *__restrict__ i1, const int32_t *__restrict__ n1,
                         int64_t NB, int MB, int bb, const Sp2Ctl *__restrict__ ctl, double *__restrict__ dv,
                         int32_t *__restrict__ di, int32_t *__restrict__ dn)
{
    if (ctl->done && ctl->status < 0) return;
    const int parity = ctl->parity;
    const double *__restrict__ sv = parity ? v1 : v0;
    const int32_t *__restrict__ si = parity ? i1 : i0;
    const int32_t *__restrict__ sn = parity ? n1 : n0;
    const int64_t nv = NB * MB * (int64_t)bb, nm = NB * (int64_t)MB;
    const int64_t stride = (int64_t)gridDim.x * blockDim.x, t0 = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    // slots beyond nnz hold stale data in the iterates: D gets (0, zero block) there, as the format's contract says
    for (int64_t e = t0; e < nv; e += stride) {
        const int64_t slot = e / bb;
        dv[e] = (slot % MB) < sn[slot / MB] ? sv[e] : 0.0;
    }
    for (int64_t e = t0; e < nm; e += stride) di[e] = (e % MB) < sn[e / MB] ? si[e] : 0;
    for (int64_t e = t0; e < NB; e += stride) dn[e] = sn[e];
}

// ------------------------------------------------------------------------------------------------------------
// host launchers
// ------------------------------------------------------------------------------------------------------------
#define EB_CHECK() do { if (cudaGetLastError() != cudaSuccess) return BML_ERR_CUDA; } while (0)

static inline size_t eb_up(size_t x) { return (x + 1023) / 1024 * 1024; }
// candidate list capacity: pre-threshold block fill of one block row (both triangles in kernel 2)
static inline int eb_cand_cap(int MB) { int c = 8 * MB; return c < 256 ? 256 : (c > 8192 ? 8192 : c); }

size_t ellblock_sym_bytes(int64_t NB, int MB, int bs)
{
    const size_t nm = (size_t)NB * (size_t)MB;
    return eb_up(nm * (size_t)bs * bs * 8) + eb_up(nm * 4) + eb_up((size_t)NB * 4) + eb_up(nm * 4) + eb_up((size_t)NB * 4) +
           2 * eb_up(nm * 8);
}
size_t ellblock_rowstats_bytes() { return (size_t)EB_MAX_GRID * 4 * sizeof(double); }

bool ellblock_shape_ok(int64_t NB, int MB, int bs)
{
    if (!(bs == 4 || bs == 8 || bs == 16) || NB < 1 || NB > (1 << 19) || MB < 1 || MB >= (1 << EB_REF_SHIFT) - 1) return false;
    const size_t smem1 = (size_t)MB * bs * bs * 8 + (size_t)MB * 4 + (size_t)eb_cand_cap(MB) * 4 + (size_t)((NB + 31) / 32) * 4 +
                         (NB <= 32768 ? (size_t)NB * 2 + 16 : 0) + 16 + (size_t)EB_WARPS * MB * 4 + (size_t)MB * 8;
    return smem1 <= 227 * 1024 - 2048;
}

template <int BS>
static int launch_x2_ellblock_t(double *v0, int32_t *i0, int32_t *n0, double *v1, int32_t *i1, int32_t *n1, int64_t NB, int MB,
                                double tau, Sp2Ctl *ctl, double *partials, void *sym, cudaStream_t st)
{
    const int sms = device_sm_count();
    if (sms <= 0 || !sym) return BML_ERR_CUDA;
    const size_t nm = (size_t)NB * (size_t)MB;
    uint8_t *p = (uint8_t *)sym;
    double *tv = (double *)p; p += eb_up(nm * (size_t)BS * BS * 8);
    int32_t *ti = (int32_t *)p; p += eb_up(nm * 4);
    int32_t *tn = (int32_t *)p; p += eb_up((size_t)NB * 4);
    uint32_t *lref = (uint32_t *)p; p += eb_up(nm * 4);
    int32_t *lcnt = (int32_t *)p; p += eb_up((size_t)NB * 4);
    double *bn0 = (double *)p; p += eb_up(nm * 8);
    double *bn1 = (double *)p;
    const int cap = eb_cand_cap(MB);
    const size_t nbw = (size_t)((NB + 31) / 32) * 4;
    const int use_map = (NB <= 32768 && MB < 65535) ? 1 : 0;
    const size_t match_off = ((size_t)MB * BS * BS * 8 + (size_t)MB * 4 + (size_t)cap * 4 + nbw + (use_map ? (size_t)NB * 2 + 16 : 0) + 15) / 16 * 16;
    size_t smem1 = match_off + (size_t)EB_WARPS * MB * 4 + (size_t)MB * 8;
    // the per-column bound of the folded pre-screen, when 4 NB more bytes fit
    size_t bound_off = 0;
    if (smem1 + (size_t)NB * 4 <= 227 * 1024 - 2048) { bound_off = smem1; smem1 += (size_t)NB * 4; }
    const size_t pref_off = ((size_t)MB * 4 + (size_t)cap * 4 + nbw + (use_map ? (size_t)NB * 2 + 16 : 0) + 15) / 16 * 16;
    const size_t smem2 = pref_off + (size_t)cap * 4;
    static size_t a1[MAX_DEVICES] = {}, a2[MAX_DEVICES] = {};
    if (ensure_smem_attr(x2_ellblock_upper_kernel<BS>, smem1, a1, 48 * 1024)) return BML_ERR_CUDA;
    if (ensure_smem_attr(x2_ellblock_assemble_kernel<BS>, smem2, a2, 48 * 1024)) return BML_ERR_CUDA;
    int64_t grid1 = NB;
    const int64_t per_sm1 = (int64_t)((227 * 1024) / (smem1 + 1024)) > 0 ? (int64_t)((227 * 1024) / (smem1 + 1024)) : 1;
    const int64_t res1 = per_sm1 * EB_THREADS > 2048 ? 2048 / EB_THREADS : per_sm1;
    if (grid1 > sms * res1) grid1 = sms * res1;
    x2_ellblock_upper_kernel<BS><<<(unsigned)grid1, EB_THREADS, smem1, st>>>(v0, i0, n0, v1, i1, n1, (int)NB, MB, tau, cap, use_map,
                                                                          (int)match_off, (int)bound_off, ctl, tv, ti, tn, lref, lcnt, bn0, bn1);
    EB_CHECK();
    int64_t grid2 = NB;
    if (grid2 > sms * 4) grid2 = sms * 4;
    if (grid2 > EB_MAX_GRID) grid2 = EB_MAX_GRID;
    x2_ellblock_assemble_kernel<BS><<<(unsigned)grid2, EB_THREADS, smem2, st>>>(v0, i0, n0, v1, i1, n1, (int)NB, MB, tau, cap, use_map,
                                                                             (int)pref_off, ctl, partials, tv, ti, tn, lref, lcnt, bn0, bn1);
    EB_CHECK();
    return 0;
}

// Frobenius norms of the stored blocks of an iterate, one warp per block (the pre-screen of kernel 1 reads them; kernel
// 2 writes those of every X' itself, so this runs once per solve, on X_0)
__global__ void __launch_bounds__(256) ellblock_norms_kernel(const double *__restrict__ v, const int32_t *__restrict__ nnz,
                                                             int NB, int MB, int bb, double *__restrict__ bn)
{
    const int lane = threadIdx.x & 31;
    const int64_t slot = (int64_t)blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5);
    if (slot >= (int64_t)NB * MB) return;
    if ((int)(slot % MB) >= min(nnz[slot / MB], MB)) return;
    const double *b = v + slot * bb;
    double s = 0.0;
    for (int e = lane; e < bb; e += 32) s = fma(b[e], b[e], s);
    s = warp_sum(s);
    if (lane == 0) bn[slot] = sqrt(s);
}

// start of a solve (or of a single product on a caller's iterate in buffer 0): the lower-list counters must be zero
// (kernel 2 re-zeroes them after every product), and the block norms of the first iterate are needed
int launch_ellblock_sym_init(void *sym, const double *xv, const int32_t *xn, int64_t NB, int MB, int bs, cudaStream_t st)
{
    const size_t nm = (size_t)NB * (size_t)MB;
    uint8_t *p = (uint8_t *)sym + eb_up(nm * (size_t)bs * bs * 8) + eb_up(nm * 4) + eb_up((size_t)NB * 4) + eb_up(nm * 4);
    if (cudaMemsetAsync(p, 0, (size_t)NB * 4, st) != cudaSuccess) return BML_ERR_CUDA;
    double *bn0 = (double *)(p + eb_up((size_t)NB * 4));
    ellblock_norms_kernel<<<(unsigned)((nm + 7) / 8), 256, 0, st>>>(xv, xn, (int)NB, MB, bs * bs, bn0);
    EB_CHECK();
    return 0;
}

int launch_x2_ellblock(double *v0, int32_t *i0, int32_t *n0, double *v1, int32_t *i1, int32_t *n1, int64_t NB, int MB, int bs,
                       double tau, Sp2Ctl *ctl, double *partials, void *sym, cudaStream_t st)
{
    switch (bs) {
        case 4: return launch_x2_ellblock_t<4>(v0, i0, n0, v1, i1, n1, NB, MB, tau, ctl, partials, sym, st);
        case 8: return launch_x2_ellblock_t<8>(v0, i0, n0, v1, i1, n1, NB, MB, tau, ctl, partials, sym, st);
        case 16: return launch_x2_ellblock_t<16>(v0, i0, n0, v1, i1, n1, NB, MB, tau, ctl, partials, sym, st);
        default: return BML_ERR_INVALID;
    }
}

int launch_gershgorin_rows_ellblock(const double *hv, const int32_t *hi, const int32_t *hn, int64_t NB, int MB, int bs,
                                    double *rowlh, cudaStream_t st)
{
    const int64_t rows = NB * bs;
    gershgorin_rows_ellblock_kernel<<<(unsigned)((rows * 32 + 255) / 256), 256, 0, st>>>(hv, hi, hn, (int)NB, MB, bs, rowlh);
    EB_CHECK();
    return 0;
}

int launch_rescale_ellblock(const double *hv, const int32_t *hi, const int32_t *hn, int64_t NB, int MB, int bs,
                            const double *d_bounds, double *xv, int32_t *xi, int32_t *xn, double *diag, int *fail_flag,
                            cudaStream_t st)
{
    int cap = 32;
    while (cap < MB + 1) cap <<= 1;
    const int nwarps = 4;
    const size_t smem = (size_t)nwarps * cap * 8;
    static size_t have[MAX_DEVICES] = {};
    if (ensure_smem_attr(rescale_ellblock_kernel, smem, have, 48 * 1024)) return BML_ERR_CUDA;
    rescale_ellblock_kernel<<<(unsigned)((NB + nwarps - 1) / nwarps), nwarps * 32, smem, st>>>(hv, hi, hn, (int)NB, MB, bs, d_bounds,
                                                                                            xv, xi, xn, diag, fail_flag, cap);
    EB_CHECK();
    return 0;
}

int launch_trace_ellblock(const double *v, const int32_t *idx, const int32_t *nnz, int64_t NB, int MB, int bs, bool sorted,
                          double *d_out, cudaStream_t st)
{
    if (sorted) trace_ellblock_kernel<<<1, 1024, 0, st>>>(v, idx, nnz, (int)NB, MB, bs, d_out);
    else trace_ellblock_unsorted_kernel<<<1, 1024, 0, st>>>(v, idx, nnz, (int)NB, MB, bs, d_out);
    EB_CHECK();
    return 0;
}

int launch_copy_out_ellblock(const double *v0, const int32_t *i0, const int32_t *n0, const double *v1, const int32_t *i1,
                             const int32_t *n1, int64_t NB, int MB, int bs, const Sp2Ctl *ctl, double *dv, int32_t *di,
                             int32_t *dn, cudaStream_t st)
{
    const int sms = device_sm_count();
    if (sms <= 0) return BML_ERR_CUDA;
    copy_out_ellblock_kernel<<<sms * 8, 256, 0, st>>>(v0, i0, n0, v1, i1, n1, NB, MB, bs * bs, ctl, dv, di, dn);
    EB_CHECK();
    return 0;
}

// other translation units
int launch_gershgorin_reduce(const double *rowlh, int N, double *d_bounds, cudaStream_t st);
int launch_init_ctl(Sp2Ctl *ctl, const double *d_bounds, const double *d_tr0, int n_occ, int max_products,
                    double idem_tol, int loop_mode, int branch0, const int *fail_flag, cudaStream_t st);
int launch_sum_vector(const double *v, int N, double *d_out, cudaStream_t st);
int launch_x2_ellpack_info(const Sp2Ctl *ctl, int32_t *d_info, cudaStream_t st);
int finish_solve(Sp2Ctl *d_ctl, bml_sp2_stats_t *stats, cudaStream_t st);

constexpr size_t EB_CTL_BYTES = 4096, EB_SCAL_BYTES = 256;
static_assert(sizeof(Sp2Ctl) <= EB_CTL_BYTES, "control block does not fit its slot");
struct EbScalars {
    double bounds[2];
    double tr0;
    double pad;
    int32_t fail_flag[4];
};

struct EbWs {
    Sp2Ctl *ctl;
    EbScalars *scal;
    double *rowlh, *rowstats;
    void *sym;
    double *v0, *v1;
    int32_t *i0, *i1, *n0, *n1;
    size_t total;
};

static EbWs carve_ellblock(void *ws, int64_t NB, int MB, int bs, bool with_buffers)
{
    EbWs w;
    uint8_t *p = (uint8_t *)ws;
    size_t off = 0;
    w.ctl = (Sp2Ctl *)(p + off); off += EB_CTL_BYTES;
    w.scal = (EbScalars *)(p + off); off += EB_SCAL_BYTES;
    w.rowlh = (double *)(p + off); off = eb_up(off + (size_t)2 * NB * bs * sizeof(double));
    w.rowstats = (double *)(p + off); off = eb_up(off + ellblock_rowstats_bytes());
    w.sym = p + off; off = eb_up(off + ellblock_sym_bytes(NB, MB, bs));
    w.v0 = w.v1 = nullptr; w.i0 = w.i1 = w.n0 = w.n1 = nullptr;
    if (with_buffers) {
        const size_t nm = (size_t)NB * (size_t)MB, nv = nm * (size_t)bs * bs;
        w.v0 = (double *)(p + off); off = eb_up(off + nv * 8);
        w.v1 = (double *)(p + off); off = eb_up(off + nv * 8);
        w.i0 = (int32_t *)(p + off); off = eb_up(off + nm * 4);
        w.i1 = (int32_t *)(p + off); off = eb_up(off + nm * 4);
        w.n0 = (int32_t *)(p + off); off = eb_up(off + (size_t)NB * 4);
        w.n1 = (int32_t *)(p + off); off = eb_up(off + (size_t)NB * 4);
    }
    w.total = off;
    return w;
}

static bool eb_ok(const bml_ellblock_t *A)
{
    return A && A->value && A->index && A->nnz && ellblock_shape_ok(A->NB, A->MB, A->bs);
}

}  // namespace bmlsp2

using namespace bmlsp2;

extern "C" {

size_t bml_gershgorin_ellblock_workspace_bytes(int64_t NB, int32_t bs)
{
    return (NB > 0 && bs > 0) ? (size_t)2 * (size_t)NB * (size_t)bs * sizeof(double) : 0;
}

int bml_gershgorin_ellblock(const bml_ellblock_t *H, double *d_bounds, void *d_workspace, size_t workspace_bytes,
                            void *cuda_stream)
{
    if (!eb_ok(H) || !d_bounds || !d_workspace || workspace_bytes < bml_gershgorin_ellblock_workspace_bytes(H->NB, H->bs))
        return BML_ERR_INVALID;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    int r = launch_gershgorin_rows_ellblock(H->value, H->index, H->nnz, H->NB, H->MB, H->bs, (double *)d_workspace, st);
    if (r) return r;
    return launch_gershgorin_reduce((const double *)d_workspace, (int)(H->NB * H->bs), d_bounds, st);
}

int bml_trace_ellblock(const bml_ellblock_t *A, double *d_trace, void *cuda_stream)
{
    if (!eb_ok(A) || !d_trace) return BML_ERR_INVALID;
    return launch_trace_ellblock(A->value, A->index, A->nnz, A->NB, A->MB, A->bs, false, d_trace, (cudaStream_t)cuda_stream);
}

size_t bml_sp2_ellblock_workspace_bytes(int64_t NB, int32_t MB, int32_t bs)
{
    if (!ellblock_shape_ok(NB, MB, bs)) return 0;
    return carve_ellblock(nullptr, NB, MB, bs, true).total;
}

size_t bml_x2_ellblock_workspace_bytes(int64_t NB, int32_t MB, int32_t bs)
{
    if (!ellblock_shape_ok(NB, MB, bs)) return 0;
    return carve_ellblock(nullptr, NB, MB, bs, false).total;
}

int bml_sp2_ellblock(const bml_ellblock_t *H, const bml_sp2_params_t *p, bml_ellblock_t *D, void *d_workspace,
                     size_t workspace_bytes, bml_sp2_stats_t *stats, void *cuda_stream)
{
    auto fail = [&](int r) { if (stats) { memset(stats, 0, sizeof(*stats)); stats->status = r; stats->overflow_row = -1; } return r; };
    if (!eb_ok(H) || !eb_ok(D) || D->NB != H->NB || D->MB != H->MB || D->bs != H->bs || !p || p->n_occ <= 0 ||
        (int64_t)p->n_occ >= H->NB * H->bs || !(p->idem_tol > 0.0) || !(p->drop_tol >= 0.0) || p->max_products < 1 ||
        p->max_products > BML_SP2_LOG_LEN || p->precision != 0 || (p->flags & ~BML_SP2_FLAG_CHECK_SYMMETRY) != 0 ||
        !d_workspace || ((uintptr_t)d_workspace & 1023) != 0 || D->value == H->value || D->index == H->index ||
        D->nnz == H->nnz)
        return fail(BML_ERR_INVALID);
    const int64_t NB = H->NB;
    const int MB = H->MB, bs = H->bs;
    EbWs w = carve_ellblock(d_workspace, NB, MB, bs, true);
    if (workspace_bytes < w.total) return fail(BML_ERR_INVALID);
    cudaStream_t st = (cudaStream_t)cuda_stream;
    int r;
    if (cudaMemsetAsync(w.scal, 0, EB_SCAL_BYTES, st) != cudaSuccess) return fail(BML_ERR_CUDA);
    if ((r = launch_gershgorin_rows_ellblock(H->value, H->index, H->nnz, NB, MB, bs, w.rowlh, st))) return fail(r);
    if ((r = launch_gershgorin_reduce(w.rowlh, (int)(NB * bs), w.scal->bounds, st))) return fail(r);
    // the Gershgorin row buffer is free again: the N diagonal values of X_0 go there
    if ((r = launch_rescale_ellblock(H->value, H->index, H->nnz, NB, MB, bs, w.scal->bounds, w.v0, w.i0, w.n0, w.rowlh,
                                     w.scal->fail_flag, st)))
        return fail(r);
    if ((r = launch_sum_vector(w.rowlh, (int)(NB * bs), &w.scal->tr0, st))) return fail(r);
    if ((r = launch_init_ctl(w.ctl, w.scal->bounds, &w.scal->tr0, p->n_occ, p->max_products, p->idem_tol, 1, 0,
                             w.scal->fail_flag, st)))
        return fail(r);
    if ((r = launch_ellblock_sym_init(w.sym, w.v0, w.n0, NB, MB, bs, st))) return fail(r);
    if ((r = enqueue_products([&]() { return launch_x2_ellblock(w.v0, w.i0, w.n0, w.v1, w.i1, w.n1, NB, MB, bs, p->drop_tol,
                                                                w.ctl, w.rowstats, w.sym, st); },
                              w.ctl, p->max_products, st, 0, stats == nullptr)))
        return fail(r);
    if ((r = launch_copy_out_ellblock(w.v0, w.i0, w.n0, w.v1, w.i1, w.n1, NB, MB, bs, w.ctl, D->value, D->index, D->nnz, st)))
        return fail(r);
    return finish_solve(w.ctl, stats, st);
}

int bml_x2_ellblock(const bml_ellblock_t *X, bml_ellblock_t *Xnext, int32_t branch, double drop_tol, double *d_sums,
                    int32_t *d_info, void *d_workspace, size_t workspace_bytes, void *cuda_stream)
{
    if (!eb_ok(X) || !eb_ok(Xnext) || X->NB != Xnext->NB || X->MB != Xnext->MB || X->bs != Xnext->bs ||
        X->value == Xnext->value || X->index == Xnext->index || X->nnz == Xnext->nnz || !d_sums || !d_info || !d_workspace ||
        ((uintptr_t)d_workspace & 1023) != 0 || !(drop_tol >= 0.0) ||
        workspace_bytes < bml_x2_ellblock_workspace_bytes(X->NB, X->MB, X->bs))
        return BML_ERR_INVALID;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    EbWs w = carve_ellblock(d_workspace, X->NB, X->MB, X->bs, false);
    int r = launch_init_ctl(w.ctl, nullptr, nullptr, 1, 1, 1.0, 0, branch ? 1 : 0, nullptr, st);
    if (r) return r;
    if ((r = launch_ellblock_sym_init(w.sym, X->value, X->nnz, X->NB, X->MB, X->bs, st))) return r;
    // buffer 0 = X (read only while parity == 0), buffer 1 = Xnext
    r = launch_x2_ellblock(X->value, X->index, X->nnz, Xnext->value, Xnext->index, Xnext->nnz, X->NB, X->MB, X->bs, drop_tol,
                           w.ctl, w.rowstats, w.sym, st);
    if (r) return r;
    if (cudaMemcpyAsync(d_sums, w.ctl->sums, 4 * sizeof(double), cudaMemcpyDeviceToDevice, st) != cudaSuccess)
        return BML_ERR_CUDA;
    return launch_x2_ellpack_info(w.ctl, d_info, st);
}

}  // extern "C"
