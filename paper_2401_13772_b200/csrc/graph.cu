// graph.cu -- the graph-based density-matrix construction (PAPER.md VIII.B, Eq. 15, Listing 11):
// core-halo parts from the Hamiltonian's own graph, gather of the dense sub-matrices (bml_matrix2submatrix), one
// Chebyshev expansion per part (chebyshev.cu), thresholded scatter of the core rows (bml_submatrix2matrix).
#include <string.h>

#include "dense_fp64_core.cuh"
#include "../../include/bml_graph.h"

namespace bmlsp2 {

// chebyshev.cu
size_t cheb_workspace_bytes(int64_t N, int k, int m);
size_t cheb_batch_workspace_bytes(int64_t N, int k, int m, int P);
int cheb_dense_enqueue_batch(int P, const bml_matrix_t *H, const bml_cheb_params_t *p, const bml_matrix_t *D, void *ws,
                             int *n_launches_out, cudaStream_t st);
double *cheb_batch_result(void *ws, int64_t N, int k, int m, int P, int q, int64_t *ld_out);
int *cheb_fail_flag(void *ws, int q);
// reductions.cu
int launch_gershgorin(const bml_matrix_t *H, double *d_bounds, double *rowlh, cudaStream_t st);
int launch_rescale_dense(const bml_matrix_t *H, const double *d_bounds, double *X, int64_t ldx, cudaStream_t st);
int launch_init_ctl(Sp2Ctl *ctl, const double *d_bounds, const double *d_tr0, int n_occ, int max_products,
                    double idem_tol, int loop_mode, int branch0, const int *fail_flag, cudaStream_t st);
// dense_batch.cu
size_t dense_batch_table_bytes();
int dense_batch_fill(void *h_table, int n_jobs, const int32_t *n, double *const *buf0, double *const *buf1,
                     const int64_t *ld, const uint8_t *const *core);
int launch_x2_dense_fp64_batch(const void *d_table, Sp2Ctl *ctl, double *partials, void *sk, cudaStream_t stream);
int launch_batch_core_trace(const void *d_table, double *d_out, cudaStream_t st);
int launch_batch_final_buffers(const void *d_table, const Sp2Ctl *ctl, const double **d_out, int n_jobs, cudaStream_t st);

// part that owns position q of the core-node list: largest k with offsets[k] <= q
__device__ __forceinline__ int part_of(const int32_t *__restrict__ offs, int n_parts, int q)
{
    int lo = 0, hi = n_parts;
    while (hi - lo > 1) {
        const int mid = (lo + hi) >> 1;
        if (offs[mid] <= q) lo = mid; else hi = mid;
    }
    return lo;
}

// Eq. 15 + P:494, first pass: flag[k][o] = 1 for every neighbour o of a core node of part k.  One warp per core node.
// (All writers store the same value, so plain byte stores suffice; the core marks follow in a second launch.)
__global__ void __launch_bounds__(256) graph_mark_halo_kernel(const double *__restrict__ hv, const int32_t *__restrict__ hi,
                                                              const int32_t *__restrict__ hn, int N, int M,
                                                              const int32_t *__restrict__ offs,
                                                              const int32_t *__restrict__ core_nodes, int n_parts,
                                                              double tau, uint8_t *__restrict__ flag)
{
    const int q = (blockIdx.x * blockDim.x + threadIdx.x) >> 5, lane = threadIdx.x & 31;
    if (q >= N) return;
    const int l = core_nodes[q];
    uint8_t *row = flag + (size_t)part_of(offs, n_parts, q) * N;
    const int n = hn[l];
    for (int p = lane; p < n; p += 32) {
        const int o = hi[(size_t)l * M + p];
        if (o != l && fabs(hv[(size_t)l * M + p]) >= tau) row[o] = 1;
    }
}
__global__ void __launch_bounds__(256) graph_mark_core_kernel(int N, const int32_t *__restrict__ offs,
                                                              const int32_t *__restrict__ core_nodes, int n_parts,
                                                              uint8_t *__restrict__ flag)
{
    const int q = blockIdx.x * blockDim.x + threadIdx.x;
    if (q >= N) return;
    flag[(size_t)part_of(offs, n_parts, q) * N + core_nodes[q]] = 2;
}

// Ascending node list of every part (reading G2): one CTA per part compacts its flag row with a block-wide scan.
constexpr int GC_THREADS = 1024;
__global__ void __launch_bounds__(GC_THREADS) graph_compact_kernel(const uint8_t *__restrict__ flag, int N,
                                                                   int32_t *__restrict__ nodes, uint8_t *__restrict__ is_core,
                                                                   int32_t *__restrict__ sizes)
{
    __shared__ int s_warp[GC_THREADS / 32];
    __shared__ int s_base, s_core;
    const int part = blockIdx.x, lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const uint8_t *row = flag + (size_t)part * N;
    if (threadIdx.x == 0) { s_base = 0; s_core = 0; }
    __syncthreads();
    for (int j0 = 0; j0 < N; j0 += GC_THREADS) {
        const int j = j0 + threadIdx.x;
        const int f = j < N ? row[j] : 0;
        const unsigned bal = __ballot_sync(0xffffffffu, f != 0), balc = __ballot_sync(0xffffffffu, f == 2);
        if (lane == 0) s_warp[warp] = __popc(bal);
        __syncthreads();
        int before = 0, total = 0;
        for (int w = 0; w < GC_THREADS / 32; ++w) { const int c = s_warp[w]; if (w < warp) before += c; total += c; }
        const int base = s_base;
        if (f) {
            const int pos = base + before + __popc(bal & ((1u << lane) - 1u));
            nodes[(size_t)part * N + pos] = j;
            is_core[(size_t)part * N + pos] = (uint8_t)(f == 2);
        }
        if (lane == 0 && balc) atomicAdd(&s_core, __popc(balc));
        __syncthreads();
        if (threadIdx.x == 0) s_base = base + total;
        __syncthreads();
    }
    if (threadIdx.x == 0) { sizes[2 * part] = s_base; sizes[2 * part + 1] = s_core; }
}

// bml_matrix2submatrix: h[a, b] = H[nodes[a], nodes[b]].  One warp per row a: zero the row, then place the stored
// entries whose column is in the (ascending) node list, found by binary search.
__global__ void __launch_bounds__(256) graph_gather_kernel(const double *__restrict__ hv, const int32_t *__restrict__ hi,
                                                           const int32_t *__restrict__ hn, int M,
                                                           const int32_t *__restrict__ nodes, int s, double *__restrict__ h,
                                                           int64_t ld)
{
    const int a = (blockIdx.x * blockDim.x + threadIdx.x) >> 5, lane = threadIdx.x & 31;
    if (a >= s) return;
    double *row = h + (int64_t)a * ld;
    for (int b = lane; b < s; b += 32) row[b] = 0.0;
    __syncwarp();
    const int i = nodes[a], n = hn[i];
    for (int p = lane; p < n; p += 32) {
        const int j = hi[(size_t)i * M + p];
        int lo = 0, hi2 = s - 1;
        while (lo < hi2) {
            const int mid = (lo + hi2) >> 1;
            if (nodes[mid] < j) lo = mid + 1; else hi2 = mid;
        }
        if (nodes[lo] == j) row[lo] = hv[(size_t)i * M + p];
    }
}

// bml_submatrix2matrix: core rows of d -> ELLPACK-R rows of D with the drop rule (readings G4, G5).  One warp per row.
// dsel (may be NULL): the matrix is *dsel instead of d (the SP2 local solver's final iterate sits in the ping-pong
// buffer the device-side control block selected).
__global__ void __launch_bounds__(256) graph_scatter_kernel(const double *__restrict__ d, int64_t ld,
                                                            const int32_t *__restrict__ nodes,
                                                            const uint8_t *__restrict__ is_core, int s, double drop_tol,
                                                            double *__restrict__ dv, int32_t *__restrict__ di,
                                                            int32_t *__restrict__ dn, int M, int32_t *__restrict__ overflow,
                                                            const double *const *__restrict__ dsel)
{
    const int a = (blockIdx.x * blockDim.x + threadIdx.x) >> 5, lane = threadIdx.x & 31;
    if (a >= s || !is_core[a]) return;
    if (dsel) d = *dsel;
    const int i = nodes[a];
    const double *row = d + (int64_t)a * ld;
    // count first: a row that does not fit is left untouched
    int count = 0;
    for (int b0 = 0; b0 < s; b0 += 32) {
        const int b = b0 + lane;
        const bool keep = b < s && (fabs(row[b]) >= drop_tol || nodes[b] == i);
        count += __popc(__ballot_sync(0xffffffffu, keep));
    }
    if (count > M) {
        if (lane == 0) atomicMin(overflow, i);
        return;
    }
    int pos = 0;
    for (int b0 = 0; b0 < s; b0 += 32) {
        const int b = b0 + lane;
        const double v = b < s ? row[b] : 0.0;
        const bool keep = b < s && (fabs(v) >= drop_tol || nodes[b] == i);
        const unsigned bal = __ballot_sync(0xffffffffu, keep);
        if (keep) {
            const int q = pos + __popc(bal & ((1u << lane) - 1u));
            dv[(size_t)i * M + q] = v;
            di[(size_t)i * M + q] = nodes[b];
        }
        pos += __popc(bal);
    }
    for (int q = count + lane; q < M; q += 32) { dv[(size_t)i * M + q] = 0.0; di[(size_t)i * M + q] = 0; }
    if (lane == 0) dn[i] = count;
}

// status word of the whole construction: keeps the first (most negative wins) failure of any part
__global__ void graph_collect_kernel(const int *__restrict__ cheb_fail, int *__restrict__ status)
{
    if (*cheb_fail != 0 && *status == 0) *status = *cheb_fail;
}

// ------------------------------------------------------------------------------------------------------------
// host side
// ------------------------------------------------------------------------------------------------------------
#define G_CHECK() do { if (cudaGetLastError() != cudaSuccess) return BML_ERR_CUDA; } while (0)

int launch_graph_core_halo(const bml_matrix_t *H, const int32_t *offs, const int32_t *core_nodes, int n_parts, double tau,
                           int32_t *part_nodes, uint8_t *is_core, int32_t *sizes, uint8_t *flag, cudaStream_t st)
{
    const int N = (int)H->N;
    if (cudaMemsetAsync(flag, 0, (size_t)n_parts * N, st) != cudaSuccess) return BML_ERR_CUDA;
    graph_mark_halo_kernel<<<(unsigned)(((size_t)N * 32 + 255) / 256), 256, 0, st>>>(H->value, H->index, H->nnz, N, H->M,
                                                                                       offs, core_nodes, n_parts, tau, flag);
    G_CHECK();
    graph_mark_core_kernel<<<(unsigned)((N + 255) / 256), 256, 0, st>>>(N, offs, core_nodes, n_parts, flag);
    G_CHECK();
    graph_compact_kernel<<<(unsigned)n_parts, GC_THREADS, 0, st>>>(flag, N, part_nodes, is_core, sizes);
    G_CHECK();
    return 0;
}

int launch_graph_gather(const bml_matrix_t *H, const int32_t *nodes, int s, double *h, int64_t ld, cudaStream_t st)
{
    graph_gather_kernel<<<(unsigned)(((size_t)s * 32 + 255) / 256), 256, 0, st>>>(H->value, H->index, H->nnz, H->M, nodes, s,
                                                                                    h, ld);
    G_CHECK();
    return 0;
}

static int launch_graph_scatter_sel(const double *d, int64_t ld, const int32_t *nodes, const uint8_t *is_core, int s,
                                    double drop_tol, bml_matrix_t *D, int32_t *overflow, cudaStream_t st,
                                    const double *const *dsel)
{
    graph_scatter_kernel<<<(unsigned)(((size_t)s * 32 + 255) / 256), 256, 0, st>>>(d, ld, nodes, is_core, s, drop_tol,
                                                                                     D->value, D->index, D->nnz, D->M,
                                                                                     overflow, dsel);
    G_CHECK();
    return 0;
}

int launch_graph_scatter(const double *d, int64_t ld, const int32_t *nodes, const uint8_t *is_core, int s, double drop_tol,
                         bml_matrix_t *D, int32_t *overflow, cudaStream_t st)
{
    return launch_graph_scatter_sel(d, ld, nodes, is_core, s, drop_tol, D, overflow, st, nullptr);
}

static inline size_t align_up(size_t x, size_t a) { return (x + a - 1) / a * a; }

struct GraphWs {
    int32_t *scal;          // [0] status, [1] overflow row, [2..] sizes (2 per part)
    uint8_t *flag, *is_core;
    int32_t *nodes;
    double *h, *d;
    void *cheb;
    int64_t ldc;
    size_t total;
};

// Parts of EQUAL size are expanded as one batch (their products share grouped launches, which is what fills the GPU when a
// part is too small to) if the batch's matrices fit a fixed memory budget; otherwise parts run back to back.
constexpr size_t GRAPH_BATCH_BUDGET = (size_t)16 << 30;
static bool graph_batch_ok(int n_parts, int size, int k, int m)
{
    const size_t ld = ((size_t)size + 15) / 16 * 16;
    return n_parts >= 2 && (size_t)n_parts * (size_t)(k + m) * (size_t)size * ld * 8 <= GRAPH_BATCH_BUDGET;
}

static GraphWs carve_graph(void *ws, int64_t N, int n_parts, int cap, int k, int m)
{
    GraphWs w;
    uint8_t *p = (uint8_t *)ws;
    size_t off = 0;
    w.scal = (int32_t *)(p + off); off = align_up(off + (size_t)(2 + 2 * BML_GRAPH_MAX_PARTS) * 4, 1024);
    w.flag = p + off; off = align_up(off + (size_t)n_parts * N, 1024);
    w.is_core = p + off; off = align_up(off + (size_t)n_parts * N, 1024);
    w.nodes = (int32_t *)(p + off); off = align_up(off + (size_t)n_parts * N * 4, 1024);
    w.ldc = ((int64_t)cap + 15) / 16 * 16;
    w.h = (double *)(p + off); off = align_up(off + (size_t)cap * w.ldc * 8, 1024);
    w.d = (double *)(p + off); off = align_up(off + (size_t)cap * w.ldc * 8, 1024);
    w.cheb = p + off;
    size_t cheb_bytes = cheb_workspace_bytes(cap, k, m);
    if (graph_batch_ok(n_parts, cap, k, m)) {
        const size_t b = cheb_batch_workspace_bytes(cap, k, m, n_parts);
        cheb_bytes = b > cheb_bytes ? b : cheb_bytes;
    }
    off = align_up(off + cheb_bytes, 1024);
    w.total = off;
    return w;
}

size_t graph_workspace_bytes(int64_t N, int n_parts, int cap, int k, int m)
{
    return carve_graph(nullptr, N, n_parts, cap, k, m).total;
}

int graph_chebyshev_solve(const bml_matrix_t *H, const int32_t *offs, const int32_t *core_nodes, const bml_graph_params_t *p,
                          bml_matrix_t *D, void *ws, bml_graph_stats_t *stats, cudaStream_t st)
{
    const int64_t N = H->N;
    const int P = p->n_parts;
    GraphWs w = carve_graph(ws, N, P, p->part_capacity, p->k, p->m);
    int32_t h_scal[2 + 2 * BML_GRAPH_MAX_PARTS];
    h_scal[0] = 0; h_scal[1] = INT32_MAX;
    if (cudaMemcpyAsync(w.scal, h_scal, 8, cudaMemcpyHostToDevice, st) != cudaSuccess) return BML_ERR_CUDA;
    int r = launch_graph_core_halo(H, offs, core_nodes, P, p->graph_tol, w.nodes, w.is_core, w.scal + 2, w.flag, st);
    if (r) return r;
    // the part sizes decide the launch shapes: the one host round trip before the end
    if (cudaMemcpyAsync(h_scal + 2, w.scal + 2, (size_t)2 * P * 4, cudaMemcpyDeviceToHost, st) != cudaSuccess ||
        cudaStreamSynchronize(st) != cudaSuccess)
        return BML_ERR_CUDA;
    int max_size = 0;
    for (int q = 0; q < P; ++q) max_size = h_scal[2 + 2 * q] > max_size ? h_scal[2 + 2 * q] : max_size;
    if (stats) {
        memset(stats, 0, sizeof(*stats));
        stats->n_parts = P; stats->overflow_row = -1; stats->max_part_size = max_size;
        for (int q = 0; q < P; ++q) { stats->part_size[q] = h_scal[2 + 2 * q]; stats->core_size[q] = h_scal[3 + 2 * q]; }
    }
    if (max_size > p->part_capacity) return BML_ERR_PART_CAPACITY;

    bml_cheb_params_t cp;
    memset(&cp, 0, sizeof(cp));
    cp.mu = p->mu; cp.beta = p->beta; cp.k = p->k; cp.m = p->m;
    int n_products = 0;
    bool equal = true;
    for (int q = 1; q < P; ++q) equal &= (h_scal[2 + 2 * q] == h_scal[2]);
    if (equal && h_scal[2] >= 1 && graph_batch_ok(P, h_scal[2], p->k, p->m) && graph_batch_ok(P, p->part_capacity, p->k, p->m)) {
        // ---- batched: gather each part and map it to its T_1, expand all parts together, scatter from the batch's slots
        const int s = h_scal[2];
        // h^k is gathered into the batch's RESULT slot of its part (S_0, free until Eq. 12 runs): it is only read to
        // get the bounds and T_1, and the last nesting step of Eq. 10 writes d^k over it in place
        bml_matrix_t hd[BML_GRAPH_MAX_PARTS], dd[BML_GRAPH_MAX_PARTS];
        for (int q = 0; q < P; ++q) {
            int64_t ldr = 0;
            double *res = cheb_batch_result(w.cheb, s, p->k, p->m, P, q, &ldr);
            hd[q] = bml_matrix_t{BML_DENSE, 0, s, ldr, res, nullptr, nullptr};
            dd[q] = hd[q];
            if ((r = launch_graph_gather(H, w.nodes + (size_t)q * N, s, res, ldr, st))) return r;
        }
        if ((r = cheb_dense_enqueue_batch(P, hd, &cp, dd, w.cheb, nullptr, st))) return r;
        for (int q = 0; q < P; ++q) {
            graph_collect_kernel<<<1, 1, 0, st>>>(cheb_fail_flag(w.cheb, q), w.scal);
            G_CHECK();
            if ((r = launch_graph_scatter(dd[q].value, dd[q].ld, w.nodes + (size_t)q * N, w.is_core + (size_t)q * N, s,
                                          p->drop_tol, D, w.scal + 1, st)))
                return r;
            n_products += (p->k - 1) + (p->m - 1);
        }
    } else {
        for (int q = 0; q < P; ++q) {
            const int s = h_scal[2 + 2 * q];
            if (s < 1) continue;
            const int32_t *nodes = w.nodes + (size_t)q * N;
            if ((r = launch_graph_gather(H, nodes, s, w.h, w.ldc, st))) return r;
            bml_matrix_t hd = {BML_DENSE, 0, s, w.ldc, w.h, nullptr, nullptr};
            bml_matrix_t dd = {BML_DENSE, 0, s, w.ldc, w.d, nullptr, nullptr};
            if ((r = cheb_dense_enqueue_batch(1, &hd, &cp, &dd, w.cheb, nullptr, st))) return r;
            graph_collect_kernel<<<1, 1, 0, st>>>(cheb_fail_flag(w.cheb, 0), w.scal);
            G_CHECK();
            if ((r = launch_graph_scatter(w.d, w.ldc, nodes, w.is_core + (size_t)q * N, s, p->drop_tol, D, w.scal + 1, st)))
                return r;
            n_products += (p->k - 1) + (p->m - 1);
        }
    }
    if (cudaMemcpyAsync(h_scal, w.scal, 8, cudaMemcpyDeviceToHost, st) != cudaSuccess ||
        cudaStreamSynchronize(st) != cudaSuccess || cudaGetLastError() != cudaSuccess)
        return BML_ERR_CUDA;
    int status = BML_OK;
    if (h_scal[0] != 0) status = h_scal[0];
    else if (h_scal[1] != INT32_MAX) status = BML_ERR_ELL_OVERFLOW;
    if (stats) {
        stats->status = status;
        stats->n_products = n_products;
        stats->overflow_row = h_scal[1] != INT32_MAX ? h_scal[1] : -1;
    }
    return status;
}

// ------------------------------------------------------------------------------------------------------------
// Listing 11 with SP2 as the local solver (reading G3'): ONE SP2 polynomial for all parts -- the Gershgorin bounds of
// the whole H define Eq. 5 for every part, the branch bit comes from the trace summed over the core orbitals of all
// parts, the stop test from the norms summed over all parts.  A product of the whole batch is one launch of
// x2_dense_fp64_batch_kernel (dense_batch.cu); nothing but the part sizes (launch shapes) goes through the host.
// ------------------------------------------------------------------------------------------------------------
constexpr size_t GS_CTL_BYTES = 4096;
static_assert(sizeof(Sp2Ctl) <= GS_CTL_BYTES, "control block does not fit its slot");

struct GraphSp2Ws {
    int32_t *scal;          // [0] unused, [1] overflow row, [2..] sizes (2 per part)
    uint8_t *flag, *is_core;
    int32_t *nodes;
    Sp2Ctl *ctl;
    double *bounds;         // [0..1] e_min, e_max; [2] tr X_0 over the core orbitals
    double *rowlh, *partials;
    void *sk, *table;
    const double **final_buf;
    double *iter;           // the parts' ping-pong iterates, packed
    size_t iter_doubles, total;
};

static size_t gs_sk_bytes() { return (size_t)SK_MAX_GRID * SK_SLOT_DOUBLES * sizeof(double) + 1024; }

static GraphSp2Ws carve_graph_sp2(void *ws, int64_t N, int n_parts, int cap)
{
    GraphSp2Ws w;
    uint8_t *p = (uint8_t *)ws;
    size_t off = 0;
    w.scal = (int32_t *)(p + off); off = align_up(off + (size_t)(2 + 2 * BML_GRAPH_MAX_PARTS) * 4, 1024);
    w.flag = p + off; off = align_up(off + (size_t)n_parts * N, 1024);
    w.is_core = p + off; off = align_up(off + (size_t)n_parts * N, 1024);
    w.nodes = (int32_t *)(p + off); off = align_up(off + (size_t)n_parts * N * 4, 1024);
    w.ctl = (Sp2Ctl *)(p + off); off += GS_CTL_BYTES;
    w.bounds = (double *)(p + off); off += 1024;
    w.rowlh = (double *)(p + off); off = align_up(off + (size_t)2 * N * 8, 1024);
    w.partials = (double *)(p + off); off = align_up(off + (size_t)SK_MAX_GRID * 4 * 8, 1024);
    w.sk = p + off; off = align_up(off + gs_sk_bytes(), 1024);
    w.table = p + off; off = align_up(off + dense_batch_table_bytes(), 1024);
    w.final_buf = (const double **)(p + off); off = align_up(off + (size_t)BML_GRAPH_MAX_PARTS * 8, 1024);
    const size_t ldc = ((size_t)cap + 15) / 16 * 16;
    w.iter = (double *)(p + off);
    w.iter_doubles = (size_t)n_parts * 2 * (align_up((size_t)cap * ldc * 8, 1024) / 8);
    off = align_up(off + w.iter_doubles * 8, 1024);
    w.total = off;
    return w;
}

size_t graph_sp2_workspace_bytes(int64_t N, int n_parts, int cap) { return carve_graph_sp2(nullptr, N, n_parts, cap).total; }

int graph_sp2_solve(const bml_matrix_t *H, const int32_t *offs, const int32_t *core_nodes, const bml_graph_sp2_params_t *p,
                    bml_matrix_t *D, void *ws, bml_graph_sp2_stats_t *stats, cudaStream_t st)
{
    const int64_t N = H->N;
    const int P = p->n_parts;
    GraphSp2Ws w = carve_graph_sp2(ws, N, P, p->part_capacity);
    int32_t h_scal[2 + 2 * BML_GRAPH_MAX_PARTS];
    h_scal[0] = 0; h_scal[1] = INT32_MAX;
    if (cudaMemcpyAsync(w.scal, h_scal, 8, cudaMemcpyHostToDevice, st) != cudaSuccess) return BML_ERR_CUDA;
    int r = launch_graph_core_halo(H, offs, core_nodes, P, p->graph_tol, w.nodes, w.is_core, w.scal + 2, w.flag, st);
    if (r) return r;
    if ((r = launch_gershgorin(H, w.bounds, w.rowlh, st))) return r;           // one Eq. 5 map for every part
    // the part sizes decide the launch shapes: the one host round trip before the end
    if (cudaMemcpyAsync(h_scal + 2, w.scal + 2, (size_t)2 * P * 4, cudaMemcpyDeviceToHost, st) != cudaSuccess ||
        cudaStreamSynchronize(st) != cudaSuccess)
        return BML_ERR_CUDA;
    int max_size = 0;
    for (int q = 0; q < P; ++q) max_size = h_scal[2 + 2 * q] > max_size ? h_scal[2 + 2 * q] : max_size;
    if (stats) {
        memset(stats, 0, sizeof(*stats));
        stats->n_parts = P; stats->overflow_row = -1; stats->max_part_size = max_size;
        for (int q = 0; q < P; ++q) { stats->part_size[q] = h_scal[2 + 2 * q]; stats->core_size[q] = h_scal[3 + 2 * q]; }
    }
    if (max_size > p->part_capacity) return BML_ERR_PART_CAPACITY;

    // ---- gather h^k and rescale it in place to X_0^k (Eq. 5 with the bounds of H); build the job table
    int32_t n[BML_GRAPH_MAX_PARTS], job_of[BML_GRAPH_MAX_PARTS];
    double *b0[BML_GRAPH_MAX_PARTS], *b1[BML_GRAPH_MAX_PARTS];
    int64_t ld[BML_GRAPH_MAX_PARTS];
    const uint8_t *core[BML_GRAPH_MAX_PARTS];
    int nj = 0;
    size_t used = 0;
    for (int q = 0; q < P; ++q) {
        const int s = h_scal[2 + 2 * q];
        if (s < 1) continue;
        const int64_t l = ((int64_t)s + 15) / 16 * 16;
        const size_t one = align_up((size_t)s * l * 8, 1024) / 8;
        if (used + 2 * one > w.iter_doubles) return BML_ERR_INVALID;
        n[nj] = s; ld[nj] = l; b0[nj] = w.iter + used; b1[nj] = w.iter + used + one; core[nj] = w.is_core + (size_t)q * N;
        job_of[nj] = q;
        used += 2 * one;
        if ((r = launch_graph_gather(H, w.nodes + (size_t)q * N, s, b0[nj], l, st))) return r;
        const bml_matrix_t hd = {BML_DENSE, 0, s, l, b0[nj], nullptr, nullptr};
        if ((r = launch_rescale_dense(&hd, w.bounds, b0[nj], l, st))) return r;
        ++nj;
    }
    if (nj < 1) return BML_ERR_INVALID;
    {
        void *h_table = malloc(dense_batch_table_bytes());
        if (!h_table) return BML_ERR_CUDA;
        r = dense_batch_fill(h_table, nj, n, b0, b1, ld, core);
        // pageable source: the copy is staged before cudaMemcpyAsync returns, so the buffer may be freed right away
        if (!r && cudaMemcpyAsync(w.table, h_table, dense_batch_table_bytes(), cudaMemcpyHostToDevice, st) != cudaSuccess)
            r = BML_ERR_CUDA;
        if (!r && cudaStreamSynchronize(st) != cudaSuccess) r = BML_ERR_CUDA;
        free(h_table);
        if (r) return r;
    }
    if ((r = launch_batch_core_trace(w.table, w.bounds + 2, st))) return r;
    if ((r = launch_init_ctl(w.ctl, w.bounds, w.bounds + 2, p->n_occ, p->max_products, p->idem_tol, 1, 0, nullptr, st)))
        return r;
    if (cudaMemsetAsync((uint8_t *)w.sk + (size_t)SK_MAX_GRID * SK_SLOT_DOUBLES * sizeof(double), 0, 1024, st) != cudaSuccess)
        return BML_ERR_CUDA;
    // ---- products: enqueued ahead of the device, launches behind the stop flag exit at once
    if ((r = enqueue_products([&]() { return launch_x2_dense_fp64_batch(w.table, w.ctl, w.partials, w.sk, st); }, w.ctl,
                              p->max_products, st)))
        return r;
    // ---- D rows of the core orbitals from X_{m*}^k
    if ((r = launch_batch_final_buffers(w.table, w.ctl, w.final_buf, nj, st))) return r;
    for (int j = 0; j < nj; ++j) {
        const int q = job_of[j];
        if ((r = launch_graph_scatter_sel(nullptr, ld[j], w.nodes + (size_t)q * N, w.is_core + (size_t)q * N, n[j],
                                          p->drop_tol, D, w.scal + 1, st, w.final_buf + j)))
            return r;
    }
    Sp2Ctl h;
    if (cudaMemcpyAsync(&h, w.ctl, sizeof(Sp2Ctl), cudaMemcpyDeviceToHost, st) != cudaSuccess ||
        cudaMemcpyAsync(h_scal, w.scal, 8, cudaMemcpyDeviceToHost, st) != cudaSuccess ||
        cudaStreamSynchronize(st) != cudaSuccess || cudaGetLastError() != cudaSuccess)
        return BML_ERR_CUDA;
    int status = h.status;
    if (status >= 0 && h_scal[1] != INT32_MAX) status = BML_ERR_ELL_OVERFLOW;
    if (stats) {
        bml_sp2_stats_t &s2 = stats->sp2;
        s2.status = status; s2.m_star = h.m; s2.n_products = h.n_done; s2.overflow_row = -1;
        s2.emin = h.emin; s2.emax = h.emax;
        memcpy(s2.branch, h.branch, sizeof(h.branch));
        memcpy(s2.trace, h.trace, sizeof(h.trace));
        memcpy(s2.idem, h.idem, sizeof(h.idem));
        stats->status = status;
        stats->overflow_row = h_scal[1] != INT32_MAX ? h_scal[1] : -1;
    }
    return status;
}

}  // namespace bmlsp2
