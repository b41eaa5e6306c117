// api.cu -- the C ABI of include/bml_sp2.h: argument checks, workspace carving, launch sequences.
// No step of the method runs on the host; the host only enqueues kernels and reads the control block back once.
#include <string.h>

#include "common.cuh"
#include "symm_ab.cuh"
#include "../../include/bml_graph.h"
#include "../../include/bml_sp2_testing.h"

namespace bmlsp2 {

// dense_fp64.cu
int make_dense_map(CUtensorMap *map, const double *base, int64_t N, int64_t ld);
int dense_fp64_num_tiles(int64_t N);
int dense_fp64_work_item(int64_t N, int n_ctas, int cta, int it, int32_t out[5]);
int dense_mixed_tile_of_cta(int64_t N, int cta, int32_t out[2]);
size_t dense_fp64_sk_bytes(int64_t N);
int dense_fp64_sk_reset(void *sk, int64_t N, cudaStream_t st);
int launch_x2_dense_fp64(const CUtensorMap &map0, const CUtensorMap &map1, double *buf0, double *buf1, int64_t ld,
                         int64_t N, Sp2Ctl *ctl, double *partials, void *sk, cudaStream_t stream);
bool dense_fp64_loop_available(int64_t N);
int launch_sp2_dense_fp64_loop(const CUtensorMap &map0, const CUtensorMap &map1, double *buf0, double *buf1, int64_t ld,
                               int64_t N, Sp2Ctl *ctl, double *partials, int max_products, cudaStream_t stream);
// dense_mixed.cu
int dense_mixed_num_tiles(int64_t N);
size_t dense_mixed_extra_bytes(int64_t N, int64_t ldx);
int sp2_dense_mixed_solve(const bml_matrix_t *H, const bml_sp2_params_t *p, double *X0, double *X1, int64_t ldx,
                          Sp2Ctl *ctl, double *partials, const double *d_bounds, void *extra, cudaStream_t st,
                          bool no_host_wait);
int x2_dense_mixed_once(const bml_matrix_t *X, bml_matrix_t *Xn, int precision, Sp2Ctl *ctl, double *partials,
                        void *extra, cudaStream_t st);
// reductions.cu
int launch_gershgorin(const bml_matrix_t *H, double *d_bounds, double *rowlh, cudaStream_t st);
int launch_trace_dense(const double *A, int64_t ld, int N, double *d_out, cudaStream_t st);
int launch_trace_ellpack(const bml_matrix_t *A, double *d_out, cudaStream_t st);
int launch_rescale_dense(const bml_matrix_t *H, const double *d_bounds, double *X, int64_t ldx, cudaStream_t st);
int launch_check_symmetry(const bml_matrix_t *H, int *d_flag, cudaStream_t st);
int launch_init_ctl(Sp2Ctl *ctl, const double *d_bounds, const double *d_tr0, int n_occ, int max_products,
                    double idem_tol, int loop_mode, int branch0, const int *fail_flag, cudaStream_t st);
int launch_copy_out_dense(const double *buf0, const double *buf1, int64_t ldx, int N, const Sp2Ctl *ctl, double *D,
                          int64_t ldd, cudaStream_t st);
// ellpack.cu
size_t ellpack_rowstats_bytes(int64_t N);
int launch_rescale_ellpack(const bml_matrix_t *H, const double *d_bounds, double *xv, int32_t *xi, int32_t *xn,
                           double *rowstats, double *d_tr0, int *fail_flag, cudaStream_t st);
size_t ellpack_sym_bytes(int64_t N, int M);
int ellpack_sym_reset(void *sym, int64_t N, int M, cudaStream_t st);
int launch_x2_ellpack(const double *v0, const int32_t *i0, const int32_t *n0, double *v1, int32_t *i1, int32_t *n1,
                      int64_t N, int M, double tau, Sp2Ctl *ctl, double *rowstats, void *sym, cudaStream_t st);
int launch_copy_out_ellpack(const double *v0, const int32_t *i0, const int32_t *n0, const double *v1,
                            const int32_t *i1, const int32_t *n1, int64_t N, int M, const Sp2Ctl *ctl, double *dv,
                            int32_t *di, int32_t *dn, cudaStream_t st);
int launch_x2_ellpack_info(const Sp2Ctl *ctl, int32_t *d_info, cudaStream_t st);
// chebyshev.cu
size_t cheb_workspace_bytes(int64_t N, int k, int m);
int cheb_schedule(int k, int32_t *level, int32_t *a, int32_t *b);
int cheb_dense_solve(const bml_matrix_t *H, const bml_cheb_params_t *p, bml_matrix_t *D, void *ws,
                     bml_cheb_stats_t *stats, cudaStream_t st);
// bounds.cu
size_t lanczos_workspace_doubles(int64_t N);
int launch_lanczos_bounds(const bml_matrix_t *H, int steps, uint64_t seed, double *d_bounds, double *work, cudaStream_t st);
// graph.cu
size_t graph_workspace_bytes(int64_t N, int n_parts, int cap, int k, int m);
int graph_chebyshev_solve(const bml_matrix_t *H, const int32_t *offs, const int32_t *core_nodes, const bml_graph_params_t *p,
                          bml_matrix_t *D, void *ws, bml_graph_stats_t *stats, cudaStream_t st);
int launch_graph_core_halo(const bml_matrix_t *H, const int32_t *offs, const int32_t *core_nodes, int n_parts, double tau,
                           int32_t *part_nodes, uint8_t *is_core, int32_t *sizes, uint8_t *flag, cudaStream_t st);
int launch_graph_gather(const bml_matrix_t *H, const int32_t *nodes, int s, double *h, int64_t ld, cudaStream_t st);
int launch_graph_scatter(const double *d, int64_t ld, const int32_t *nodes, const uint8_t *is_core, int s, double drop_tol,
                         bml_matrix_t *D, int32_t *overflow, cudaStream_t st);
void cheb_graph_cache_release();
size_t graph_sp2_workspace_bytes(int64_t N, int n_parts, int cap);
int graph_sp2_solve(const bml_matrix_t *H, const int32_t *offs, const int32_t *core_nodes, const bml_graph_sp2_params_t *p,
                    bml_matrix_t *D, void *ws, bml_graph_sp2_stats_t *stats, cudaStream_t st);
int dense_batch_work_item(int n_jobs, const int32_t *n, int n_ctas, int cta, int it, int32_t out[5]);
// probe.cu
int run_fp64_tensor_probe(int iters, double *flops, double *ms, cudaStream_t st);

PFN_encodeTiled get_encode_tiled()
{
    static PFN_encodeTiled fn = nullptr;
    static bool tried = false;
    if (!tried) {
        tried = true;
        void *p = nullptr;
        cudaDriverEntryPointQueryResult q;
        if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &p, cudaEnableDefault, &q) == cudaSuccess &&
            q == cudaDriverEntryPointSuccess)
            fn = (PFN_encodeTiled)p;
    }
    return fn;
}

static inline size_t align_up(size_t x, size_t a) { return (x + a - 1) / a * a; }
static inline int64_t padded_ld(int64_t N) { return (N + 15) / 16 * 16; }

constexpr size_t CTL_BYTES = 4096;      // Sp2Ctl
constexpr size_t SCAL_BYTES = 256;      // bounds[2], tr0, flags
static_assert(sizeof(Sp2Ctl) <= CTL_BYTES, "control block does not fit its slot");

struct ScalarSlots {
    double bounds[2];
    double tr0;
    double pad;
    int32_t fail_flag[4];
};
static_assert(sizeof(ScalarSlots) <= SCAL_BYTES, "scalar slots");

// per-CTA partial-sum slots: enough for the grid of either dense product kernel
static inline size_t partial_slots(int64_t N)
{
    // the whole-solve kernel of small matrices (N <= 1024) alternates between two sets of per-CTA partial sums
    const int a = dense_fp64_num_tiles(N) * (N <= 1024 ? 2 : 1), b = dense_mixed_num_tiles(N);
    return (size_t)(a > b ? a : b);
}

// per-row scratch shared by the Gershgorin pass (2N doubles) and the optional Lanczos pass (3N + its control block)
static inline size_t row_scratch_doubles(int64_t N)
{
    const size_t a = (size_t)2 * (size_t)N, b = lanczos_workspace_doubles(N);
    return a > b ? a : b;
}
static inline int lanczos_steps(uint32_t flags) { return (int)((flags >> 8) & 0xffu); }

struct DenseWs {
    Sp2Ctl *ctl;
    ScalarSlots *scal;
    double *rowlh, *partials, *X0, *X1;
    void *sk;          // split-tile scratch of the persistent FP64 kernel
    void *extra;
    int64_t ldx;
    size_t total;
};

static DenseWs carve_dense(void *ws, int64_t N, int precision)
{
    DenseWs w;
    uint8_t *p = (uint8_t *)ws;
    size_t off = 0;
    w.ctl = (Sp2Ctl *)(p + off); off += CTL_BYTES;
    w.scal = (ScalarSlots *)(p + off); off += SCAL_BYTES;
    w.rowlh = (double *)(p + off); off = align_up(off + row_scratch_doubles(N) * sizeof(double), 1024);
    w.partials = (double *)(p + off);
    off = align_up(off + partial_slots(N) * 4 * sizeof(double), 1024);
    w.sk = (void *)(p + off); off = align_up(off + dense_fp64_sk_bytes(N), 1024);
    w.ldx = padded_ld(N);
    w.X0 = (double *)(p + off); off = align_up(off + (size_t)N * w.ldx * sizeof(double), 1024);
    w.X1 = (double *)(p + off); off = align_up(off + (size_t)N * w.ldx * sizeof(double), 1024);
    w.extra = (void *)(p + off);
    if (precision != 0) off = align_up(off + dense_mixed_extra_bytes(N, w.ldx), 1024);
    w.total = off;
    return w;
}

struct EllWs {
    Sp2Ctl *ctl;
    ScalarSlots *scal;
    double *rowlh, *rowstats;
    void *sym;          // scratch of the symmetric product (upper parts + lower lists)
    double *v0, *v1;
    int32_t *i0, *i1, *n0, *n1;
    size_t total;
};

static EllWs carve_ell(void *ws, int64_t N, int M, bool with_buffers)
{
    EllWs w;
    uint8_t *p = (uint8_t *)ws;
    size_t off = 0;
    w.ctl = (Sp2Ctl *)(p + off); off += CTL_BYTES;
    w.scal = (ScalarSlots *)(p + off); off += SCAL_BYTES;
    w.rowlh = (double *)(p + off); off = align_up(off + row_scratch_doubles(N) * sizeof(double), 1024);
    w.rowstats = (double *)(p + off); off = align_up(off + ellpack_rowstats_bytes(N), 1024);
    w.sym = (void *)(p + off); off = align_up(off + ellpack_sym_bytes(N, M), 1024);
    w.v0 = w.v1 = nullptr; w.i0 = w.i1 = w.n0 = w.n1 = nullptr;
    if (with_buffers) {
        const size_t nm = (size_t)N * (size_t)M;
        w.v0 = (double *)(p + off); off = align_up(off + nm * 8, 1024);
        w.v1 = (double *)(p + off); off = align_up(off + nm * 8, 1024);
        w.i0 = (int32_t *)(p + off); off = align_up(off + nm * 4, 1024);
        w.i1 = (int32_t *)(p + off); off = align_up(off + nm * 4, 1024);
        w.n0 = (int32_t *)(p + off); off = align_up(off + (size_t)N * 4, 1024);
        w.n1 = (int32_t *)(p + off); off = align_up(off + (size_t)N * 4, 1024);
    }
    w.total = off;
    return w;
}

static bool dense_ok(const bml_matrix_t *A)
{
    return A && A->type == BML_DENSE && A->value && A->N > 0 && A->N <= 0x3fffffff && A->ld >= A->N;
}
static bool ell_ok(const bml_matrix_t *A)
{
    return A && A->type == BML_ELLPACK && A->value && A->index && A->nnz && A->N > 0 && A->N < (1 << 29) - 1 &&
           A->M >= 1 && A->M <= BML_ELL_MAX_M;
}
static bool params_ok(const bml_sp2_params_t *p, int64_t N)
{
    return p && p->n_occ > 0 && (int64_t)p->n_occ < N && p->idem_tol > 0.0 && p->max_products >= 1 &&
           p->max_products <= BML_SP2_LOG_LEN && p->drop_tol >= 0.0 && p->precision >= 0 && p->precision <= 2 &&
           (lanczos_steps(p->flags) == 0 || (lanczos_steps(p->flags) >= 8 && lanczos_steps(p->flags) <= 64));
}

static void fill_stats(bml_sp2_stats_t *stats, const Sp2Ctl &c)
{
    if (!stats) return;
    memset(stats, 0, sizeof(*stats));
    stats->status = c.status;
    stats->m_star = c.m;
    stats->n_products = c.n_done;
    stats->overflow_row = c.fail_row;
    stats->emin = c.emin;
    stats->emax = c.emax;
    memcpy(stats->branch, c.branch, sizeof(c.branch));
    memcpy(stats->trace, c.trace, sizeof(c.trace));
    memcpy(stats->idem, c.idem, sizeof(c.idem));
    memcpy(stats->max_row_nnz, c.max_row_nnz, sizeof(c.max_row_nnz));
}

EnqueueState &enqueue_state()
{
    static thread_local EnqueueState es;
    return es;
}

// stats == NULL: the call is fully asynchronous -- nothing is copied back, the stream is not synchronised and the
// return value only says that everything was enqueued (the verdict of the solve stays in the device control block,
// whose first words bml_sp2_read_status copies out later).
int finish_solve(Sp2Ctl *d_ctl, bml_sp2_stats_t *stats, cudaStream_t st)
{
    if (!stats) return cudaGetLastError() == cudaSuccess ? BML_OK : BML_ERR_CUDA;
    Sp2Ctl h;
    if (cudaMemcpyAsync(&h, d_ctl, sizeof(Sp2Ctl), cudaMemcpyDeviceToHost, st) != cudaSuccess) return BML_ERR_CUDA;
    if (cudaStreamSynchronize(st) != cudaSuccess) return BML_ERR_CUDA;
    if (cudaGetLastError() != cudaSuccess) return BML_ERR_CUDA;
    fill_stats(stats, h);
    return h.status;
}

// CUDA-graph replay of the static head of a small dense FP64 solve (prelude + first batch of product launches).
// Same rules as the Chebyshev replay (chebyshev.cu): N <= 1024, not while capturing, not on the legacy default stream,
// the first solve of a tile size runs plainly (it sets kernel attributes), failures fall back to plain enqueueing.
struct Sp2GraphKey {
    const void *H, *ws;
    int64_t N, ldh;
    double idem_tol;
    int32_t n_occ, max_products;
    uint32_t flags;
    cudaStream_t st;
    int dev;            // device ordinal: a graph exec belongs to the device it was instantiated on
    bool operator==(const Sp2GraphKey &o) const
    {
        return H == o.H && ws == o.ws && N == o.N && ldh == o.ldh && idem_tol == o.idem_tol && n_occ == o.n_occ &&
               max_products == o.max_products && flags == o.flags && st == o.st && dev == o.dev;
    }
};
struct Sp2GraphSlot {
    Sp2GraphKey key;
    cudaGraphExec_t exec = nullptr;
    uint64_t stamp = 0;
};

// The cache is per host thread and holds the caller's H / workspace pointers as KEYS only (they are compared, never
// dereferenced by the host); bml_sp2_release_cached() drops it.
static thread_local Sp2GraphSlot g_sp2_slots[4];
static thread_local uint64_t g_sp2_clock = 0;
static thread_local bool g_sp2_warmed[MAX_DEVICES][2] = {};

void sp2_graph_cache_release()
{
    for (auto &sl : g_sp2_slots) {
        if (sl.exec) cudaGraphExecDestroy(sl.exec);
        sl = Sp2GraphSlot();
    }
}

template <class EnqueueFn>
static int sp2_first_batch_cached(const Sp2GraphKey &key, EnqueueFn &&enqueue)
{
    Sp2GraphSlot (&slots)[4] = g_sp2_slots;
    uint64_t &clock_ = g_sp2_clock;
    cudaStream_t st = key.st;
    cudaStreamCaptureStatus cs = cudaStreamCaptureStatusNone;
    const bool capturing = cudaStreamIsCapturing(st, &cs) == cudaSuccess && cs != cudaStreamCaptureStatusNone;
    const int bti = key.N <= 512 ? 0 : 1;
    if (key.dev < 0) return enqueue();
    bool *warmed = g_sp2_warmed[key.dev];
    if (key.N > 1024 || capturing || st == nullptr || !warmed[bti]) {
        if (key.N <= 1024) warmed[bti] = true;
        return enqueue();
    }
    Sp2GraphSlot *hit = nullptr, *victim = &slots[0];
    for (auto &sl : slots) {
        if (sl.exec && sl.key == key) hit = &sl;
        if (sl.stamp < victim->stamp) victim = &sl;
    }
    if (!hit) {
        cudaGraph_t graph = nullptr;
        if (cudaStreamBeginCapture(st, cudaStreamCaptureModeThreadLocal) != cudaSuccess) {
            cudaGetLastError();
            return enqueue();
        }
        const int r = enqueue();
        const cudaError_t ce = cudaStreamEndCapture(st, &graph);
        cudaGraphExec_t exec = nullptr;
        if (r != 0 || ce != cudaSuccess || !graph || cudaGraphInstantiate(&exec, graph, 0) != cudaSuccess) {
            if (graph) cudaGraphDestroy(graph);
            cudaGetLastError();
            return enqueue();
        }
        cudaGraphDestroy(graph);
        if (victim->exec) cudaGraphExecDestroy(victim->exec);
        victim->key = key; victim->exec = exec;
        hit = victim;
    }
    hit->stamp = ++clock_;
    if (cudaGraphLaunch(hit->exec, st) != cudaSuccess) {
        cudaGetLastError();
        return enqueue();
    }
    return 0;
}

}  // namespace bmlsp2

using namespace bmlsp2;

#define TRY(x) do { int _r = (x); if (_r != 0) { if (stats) { memset(stats, 0, sizeof(*stats)); stats->status = _r; stats->overflow_row = -1; } return _r; } } while (0)

extern "C" {

const char *bml_version(void) { return "0.1.0 (sm_100a)"; }

const char *bml_status_string(int status)
{
    switch (status) {
        case BML_OK: return "converged (S1: e_m < idem_tol)";
        case BML_NOISE_FLOOR: return "stopped on the noise floor (S2); D valid, tolerance not reached";
        case BML_MAX_PRODUCTS: return "max_products reached (S3); not converged";
        case BML_ERR_INVALID: return "invalid argument";
        case BML_ERR_DEGENERATE: return "degenerate spectral bounds (e_max - e_min <= 0)";
        case BML_ERR_ELL_OVERFLOW: return "ELLPACK-R overflow: a row needs more than M slots";
        case BML_ERR_CUDA: return "CUDA error";
        case BML_ERR_NOT_SYMMETRIC: return "H is not symmetric";
        case BML_ERR_ACC_CAPACITY: return "ELLPACK X^2 accumulator capacity exceeded";
        case BML_ERR_PART_CAPACITY: return "graph solver: a core+halo part exceeds part_capacity";
        default: return "unknown status";
    }
}

size_t bml_gershgorin_workspace_bytes(int64_t N) { return N > 0 ? (size_t)2 * (size_t)N * sizeof(double) : 0; }

int bml_gershgorin(const bml_matrix_t *H, double *d_bounds, void *d_workspace, size_t workspace_bytes,
                   void *cuda_stream)
{
    if (!H || !d_bounds || !d_workspace) return BML_ERR_INVALID;
    if (!(H->type == BML_DENSE ? dense_ok(H) : ell_ok(H))) return BML_ERR_INVALID;
    if (workspace_bytes < bml_gershgorin_workspace_bytes(H->N)) return BML_ERR_INVALID;
    return launch_gershgorin(H, d_bounds, (double *)d_workspace, (cudaStream_t)cuda_stream);
}

size_t bml_lanczos_bounds_workspace_bytes(int64_t N)
{
    return N > 0 ? row_scratch_doubles(N) * sizeof(double) : 0;
}

int bml_lanczos_bounds(const bml_matrix_t *H, int32_t steps, uint64_t seed, double *d_bounds, void *d_workspace,
                       size_t workspace_bytes, void *cuda_stream)
{
    if (!H || !d_bounds || !d_workspace || steps < 8 || steps > 64) return BML_ERR_INVALID;
    if (!(H->type == BML_DENSE ? dense_ok(H) : ell_ok(H))) return BML_ERR_INVALID;
    if (workspace_bytes < bml_lanczos_bounds_workspace_bytes(H->N) || ((uintptr_t)d_workspace & 7) != 0)
        return BML_ERR_INVALID;
    int r = launch_gershgorin(H, d_bounds, (double *)d_workspace, (cudaStream_t)cuda_stream);
    if (r) return r;
    return launch_lanczos_bounds(H, steps, seed, d_bounds, (double *)d_workspace, (cudaStream_t)cuda_stream);
}

int bml_trace(const bml_matrix_t *A, double *d_trace, void *cuda_stream)
{
    if (!A || !d_trace) return BML_ERR_INVALID;
    if (A->type == BML_DENSE) {
        if (!dense_ok(A)) return BML_ERR_INVALID;
        return launch_trace_dense(A->value, A->ld, (int)A->N, d_trace, (cudaStream_t)cuda_stream);
    }
    if (!ell_ok(A)) return BML_ERR_INVALID;
    return launch_trace_ellpack(A, d_trace, (cudaStream_t)cuda_stream);
}

size_t bml_sp2_workspace_bytes(const bml_matrix_t *H, const bml_sp2_params_t *p)
{
    if (!H || H->N <= 0) return 0;
    if (H->type == BML_DENSE) return carve_dense(nullptr, H->N, p ? p->precision : 0).total;
    if (H->M < 1) return 0;
    return carve_ell(nullptr, H->N, H->M, true).total;
}

int bml_sp2_dense(const bml_matrix_t *H, const bml_sp2_params_t *p, bml_matrix_t *D, void *d_workspace,
                  size_t workspace_bytes, bml_sp2_stats_t *stats, void *cuda_stream)
{
    if (!dense_ok(H) || !dense_ok(D) || D->N != H->N || !params_ok(p, H->N) || !d_workspace ||
        D->value == H->value || ((uintptr_t)d_workspace & 1023) != 0)
        TRY(BML_ERR_INVALID);
    const int64_t N = H->N;
    DenseWs w = carve_dense(d_workspace, N, p->precision);
    if (workspace_bytes < w.total) TRY(BML_ERR_INVALID);
    cudaStream_t st = (cudaStream_t)cuda_stream;

    // D0 + D1 + control block: everything before the first product
    auto prelude = [&]() -> int {
        int r;
        if (cudaMemsetAsync(w.scal, 0, SCAL_BYTES, st) != cudaSuccess) return BML_ERR_CUDA;
        if ((r = launch_gershgorin(H, w.scal->bounds, w.rowlh, st))) return r;                    // D0
        if (lanczos_steps(p->flags) &&
            (r = launch_lanczos_bounds(H, lanczos_steps(p->flags), 0, w.scal->bounds, w.rowlh, st)))
            return r;
        if ((p->flags & BML_SP2_FLAG_CHECK_SYMMETRY) && (r = launch_check_symmetry(H, w.scal->fail_flag, st))) return r;
        if ((r = launch_rescale_dense(H, w.scal->bounds, w.X0, w.ldx, st))) return r;             // D1
        if ((r = launch_trace_dense(w.X0, w.ldx, (int)N, &w.scal->tr0, st))) return r;
        return launch_init_ctl(w.ctl, w.scal->bounds, &w.scal->tr0, p->n_occ, p->max_products, p->idem_tol, 1, 0,
                               w.scal->fail_flag, st);
    };
    if (p->precision != 0) {
        TRY(prelude());
        TRY(sp2_dense_mixed_solve(H, p, w.X0, w.X1, w.ldx, w.ctl, w.partials, w.scal->bounds, w.extra, st,
                                  stats == nullptr));
    } else {
        CUtensorMap map0, map1;
        TRY(make_dense_map(&map0, w.X0, N, w.ldx));
        TRY(make_dense_map(&map1, w.X1, N, w.ldx));
        auto launch_one = [&]() { return launch_x2_dense_fp64(map0, map1, w.X0, w.X1, w.ldx, N, w.ctl, w.partials, w.sk, st); };
        // D2-D5: products are enqueued ahead of the device; launches after the stop rule fired exit at once.
        // Small matrices: the prelude and the first batch of launches are launch-latency bound and form a static
        // sequence, replayed as a CUDA graph when the stream allows it (sp2_first_batch_cached).
        // Small matrices (N <= 1024): a product is a few microseconds of work, so ALL products run inside one
        // cooperative launch (sp2_dense_fp64_loop_kernel: grid barrier + device-side stop test between products); the
        // prelude and that launch form a static sequence, replayed as a CUDA graph when the stream allows it.
        auto small_solve = [&]() -> int {
            int r = prelude();
            if (r) return r;
            r = launch_sp2_dense_fp64_loop(map0, map1, w.X0, w.X1, w.ldx, N, w.ctl, w.partials, p->max_products, st);
            return r == 1 ? BML_ERR_CUDA : r;
        };
        if (dense_fp64_loop_available(N)) {
            const Sp2GraphKey key = {H->value, d_workspace, N, H->ld, p->idem_tol, p->n_occ, p->max_products, p->flags, st,
                                     current_device()};
            TRY(sp2_first_batch_cached(key, small_solve));
        } else {
            TRY(prelude());
            TRY(dense_fp64_sk_reset(w.sk, N, st));
            TRY(enqueue_products(launch_one, w.ctl, p->max_products, st, 0, stats == nullptr));
        }
    }
    TRY(launch_copy_out_dense(w.X0, w.X1, w.ldx, (int)N, w.ctl, D->value, D->ld, st));        // D6
    return finish_solve(w.ctl, stats, st);
}

void bml_sp2_release_cached(void)
{
    sp2_graph_cache_release();
    cheb_graph_cache_release();
}

int bml_sp2_read_stats(const void *d_workspace, bml_sp2_stats_t *stats, void *cuda_stream)
{
    if (!d_workspace || !stats || ((uintptr_t)d_workspace & 1023) != 0) return BML_ERR_INVALID;
    return finish_solve((Sp2Ctl *)d_workspace, stats, (cudaStream_t)cuda_stream);
}

size_t bml_x2_dense_workspace_bytes(int64_t N, int32_t precision)
{
    if (N <= 0) return 0;
    size_t off = CTL_BYTES;
    off = align_up(off + partial_slots(N) * 4 * sizeof(double), 1024);
    off = align_up(off + dense_fp64_sk_bytes(N), 1024);
    if (precision != 0) off = align_up(off + dense_mixed_extra_bytes(N, padded_ld(N)), 1024);
    return off;
}

int bml_x2_dense(const bml_matrix_t *X, bml_matrix_t *Xnext, int32_t branch, int32_t precision, double *d_sums,
                 void *d_workspace, size_t workspace_bytes, void *cuda_stream)
{
    if (!dense_ok(X) || !dense_ok(Xnext) || X->N != Xnext->N || X->ld != Xnext->ld || (X->ld % 16) != 0 ||
        ((uintptr_t)X->value & 127) != 0 || ((uintptr_t)Xnext->value & 127) != 0 || X->value == Xnext->value ||
        !d_sums || !d_workspace || ((uintptr_t)d_workspace & 1023) != 0 || precision < 0 || precision > 2 ||
        workspace_bytes < bml_x2_dense_workspace_bytes(X->N, precision))
        return BML_ERR_INVALID;
    // the 16-bit planes and the FP64 diagonal in the workspace are sized by bml_x2_dense_workspace_bytes for the pitch
    // padded_ld(N), and the mixed kernel carves them with the iterate's own ld: any wider ld would run past the end
    if (precision != 0 && X->ld != padded_ld(X->N)) return BML_ERR_INVALID;
    const int64_t N = X->N;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    uint8_t *p = (uint8_t *)d_workspace;
    Sp2Ctl *ctl = (Sp2Ctl *)p;
    double *partials = (double *)(p + CTL_BYTES);
    void *sk = p + align_up(CTL_BYTES + partial_slots(N) * 4 * sizeof(double), 1024);
    void *extra = (uint8_t *)sk + align_up(dense_fp64_sk_bytes(N), 1024);
    int r = launch_init_ctl(ctl, nullptr, nullptr, 1, 1, 1.0, 0, branch ? 1 : 0, nullptr, st);
    if (r) return r;
    if (precision != 0) {
        r = x2_dense_mixed_once(X, Xnext, precision, ctl, partials, extra, st);
    } else {
        CUtensorMap map0, map1;
        if ((r = make_dense_map(&map0, X->value, N, X->ld))) return r;
        if ((r = make_dense_map(&map1, Xnext->value, N, X->ld))) return r;
        if ((r = dense_fp64_sk_reset(sk, N, st))) return r;
        r = launch_x2_dense_fp64(map0, map1, X->value, Xnext->value, X->ld, N, ctl, partials, sk, st);
    }
    if (r) return r;
    if (cudaMemcpyAsync(d_sums, ctl->sums, 4 * sizeof(double), cudaMemcpyDeviceToDevice, st) != cudaSuccess)
        return BML_ERR_CUDA;
    return 0;
}

int bml_sp2_ellpack(const bml_matrix_t *H, const bml_sp2_params_t *p, bml_matrix_t *D, void *d_workspace,
                    size_t workspace_bytes, bml_sp2_stats_t *stats, void *cuda_stream)
{
    if (!ell_ok(H) || !ell_ok(D) || D->N != H->N || D->M != H->M || !params_ok(p, H->N) || p->precision != 0 ||
        !d_workspace || D->value == H->value || D->index == H->index || D->nnz == H->nnz ||
        ((uintptr_t)d_workspace & 1023) != 0)
        TRY(BML_ERR_INVALID);
    const int64_t N = H->N;
    const int M = H->M;
    EllWs w = carve_ell(d_workspace, N, M, true);
    if (workspace_bytes < w.total) TRY(BML_ERR_INVALID);
    cudaStream_t st = (cudaStream_t)cuda_stream;

    if (cudaMemsetAsync(w.scal, 0, SCAL_BYTES, st) != cudaSuccess) TRY(BML_ERR_CUDA);
    TRY(launch_gershgorin(H, w.scal->bounds, w.rowlh, st));                                   // S0
    if (lanczos_steps(p->flags)) TRY(launch_lanczos_bounds(H, lanczos_steps(p->flags), 0, w.scal->bounds, w.rowlh, st));
    // the Gershgorin row buffer (2N doubles) is free again: reuse it for the N diagonal values of X_0
    TRY(launch_rescale_ellpack(H, w.scal->bounds, w.v0, w.i0, w.n0, w.rowlh, &w.scal->tr0, w.scal->fail_flag, st));
    TRY(launch_init_ctl(w.ctl, w.scal->bounds, &w.scal->tr0, p->n_occ, p->max_products, p->idem_tol, 1, 0,
                        w.scal->fail_flag, st));
    TRY(ellpack_sym_reset(w.sym, N, M, st));
    TRY(enqueue_products([&]() { return launch_x2_ellpack(w.v0, w.i0, w.n0, w.v1, w.i1, w.n1, N, M, p->drop_tol, w.ctl,
                                                          w.rowstats, w.sym, st); },
                         w.ctl, p->max_products, st, 0, stats == nullptr));                       // S2-S5
    TRY(launch_copy_out_ellpack(w.v0, w.i0, w.n0, w.v1, w.i1, w.n1, N, M, w.ctl, D->value, D->index, D->nnz, st));
    return finish_solve(w.ctl, stats, st);
}

size_t bml_x2_ellpack_workspace_bytes(int64_t N, int32_t M)
{
    if (N <= 0 || M < 1) return 0;
    return carve_ell(nullptr, N, M, false).total;
}

int bml_x2_ellpack(const bml_matrix_t *X, bml_matrix_t *Xnext, int32_t branch, double drop_tol, double *d_sums,
                   int32_t *d_info, void *d_workspace, size_t workspace_bytes, void *cuda_stream)
{
    if (!ell_ok(X) || !ell_ok(Xnext) || X->N != Xnext->N || X->M != Xnext->M || X->value == Xnext->value ||
        X->index == Xnext->index || X->nnz == Xnext->nnz || !d_sums || !d_info || !d_workspace ||
        ((uintptr_t)d_workspace & 1023) != 0 || !(drop_tol >= 0.0) ||
        workspace_bytes < bml_x2_ellpack_workspace_bytes(X->N, X->M))
        return BML_ERR_INVALID;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    EllWs w = carve_ell(d_workspace, X->N, X->M, false);
    int r = launch_init_ctl(w.ctl, nullptr, nullptr, 1, 1, 1.0, 0, branch ? 1 : 0, nullptr, st);
    if (r) return r;
    if ((r = ellpack_sym_reset(w.sym, X->N, X->M, st))) return r;
    r = launch_x2_ellpack(X->value, X->index, X->nnz, Xnext->value, Xnext->index, Xnext->nnz, X->N, X->M, drop_tol,
                          w.ctl, w.rowstats, w.sym, st);
    if (r) return r;
    if (cudaMemcpyAsync(d_sums, w.ctl->sums, 4 * sizeof(double), cudaMemcpyDeviceToDevice, st) != cudaSuccess)
        return BML_ERR_CUDA;
    return launch_x2_ellpack_info(w.ctl, d_info, st);
}

int bml_dense_work_item(int64_t N, int32_t n_ctas, int32_t cta, int32_t it, int32_t *out5)
{
    if (!out5) return BML_ERR_INVALID;
    return dense_fp64_work_item(N, n_ctas, cta, it, out5);
}

int bml_dense_mixed_tile_count(int64_t N) { return N < 1 ? 0 : dense_mixed_num_tiles(N); }

int bml_dense_mixed_tile_of_cta(int64_t N, int32_t cta, int32_t *out2)
{
    if (!out2) return BML_ERR_INVALID;
    return dense_mixed_tile_of_cta(N, cta, out2);
}

// ---------------------------------------------- bml_chebyshev.h ----------------------------------------------
static bool cheb_params_ok(const bml_cheb_params_t *p)
{
    return p && p->k >= 2 && p->k <= BML_CHEB_MAX_K && p->m >= 1 && p->m <= BML_CHEB_MAX_M &&
           p->k * p->m <= BML_CHEB_MAX_TERMS && p->beta > 0.0 && p->mu == p->mu;
}

size_t bml_chebyshev_workspace_bytes(int64_t N, int32_t k, int32_t m)
{
    if (N <= 0 || k < 2 || k > BML_CHEB_MAX_K || m < 1 || m > BML_CHEB_MAX_M) return 0;
    return cheb_workspace_bytes(N, k, m);
}

int bml_chebyshev_dense(const bml_matrix_t *H, const bml_cheb_params_t *p, bml_matrix_t *D, void *d_workspace,
                        size_t workspace_bytes, bml_cheb_stats_t *stats, void *cuda_stream)
{
    int r = BML_OK;
    if (!dense_ok(H) || !dense_ok(D) || D->N != H->N || !cheb_params_ok(p) || !d_workspace ||
        D->value == H->value || ((uintptr_t)d_workspace & 1023) != 0 ||
        workspace_bytes < bml_chebyshev_workspace_bytes(H->N, p->k, p->m))
        r = BML_ERR_INVALID;
    else
        r = cheb_dense_solve(H, p, D, d_workspace, stats, (cudaStream_t)cuda_stream);
    if (r < 0 && stats) { memset(stats, 0, sizeof(*stats)); stats->status = r; }
    return r;
}

size_t bml_symm_ab_workspace_bytes(void) { return symm_ab_sk_bytes(); }

int bml_symm_ab_dense(double *base, int64_t N, int64_t ld, int64_t slot_elems, int32_t n_slots, int32_t n_jobs,
                      const int32_t *a_slot, const int32_t *b_slot, const int32_t *c_slot, const int32_t *out_slot,
                      const double *alpha, const double *beta, const double *gamma, void *d_workspace,
                      size_t workspace_bytes, void *cuda_stream)
{
    if (!base || N < 1 || N > 0x3fffffff || ld < N || (ld % 16) != 0 || ((uintptr_t)base & 127) != 0 ||
        slot_elems < N * ld || (slot_elems % 16) != 0 || n_slots < 1 || n_jobs < 1 || n_jobs > BML_SYMM_MAX_JOBS ||
        !a_slot || !b_slot || !c_slot || !out_slot || !alpha || !beta || !gamma || !d_workspace ||
        ((uintptr_t)d_workspace & 1023) != 0 || workspace_bytes < symm_ab_sk_bytes())
        return BML_ERR_INVALID;
    SymmBatch batch;
    memset(&batch, 0, sizeof(batch));
    batch.n_jobs = n_jobs;
    for (int q = 0; q < n_jobs; ++q) {
        if (a_slot[q] < 0 || a_slot[q] >= n_slots || b_slot[q] < 0 || b_slot[q] >= n_slots || c_slot[q] < -1 ||
            c_slot[q] >= n_slots || out_slot[q] < 0 || out_slot[q] >= n_slots)
            return BML_ERR_INVALID;
        for (int q2 = 0; q2 < n_jobs; ++q2)      // an output must not be an operand of the same launch
            if (out_slot[q] == a_slot[q2] || out_slot[q] == b_slot[q2] || (q2 != q && out_slot[q] == out_slot[q2]) ||
                (q2 != q && out_slot[q] == c_slot[q2]))
                return BML_ERR_INVALID;
        SymmJob &jb = batch.job[q];
        jb.a = a_slot[q]; jb.b = b_slot[q];
        jb.C = c_slot[q] < 0 ? nullptr : base + (int64_t)c_slot[q] * slot_elems;
        jb.Out = base + (int64_t)out_slot[q] * slot_elems;
        jb.ldc = ld; jb.ldo = ld;
        jb.alpha = alpha[q]; jb.beta = beta[q]; jb.gamma = gamma[q];
    }
    cudaStream_t st = (cudaStream_t)cuda_stream;
    CUtensorMap map;
    int r = make_slab_map(&map, base, N, ld, slot_elems, n_slots);
    if (r) return r;
    if ((r = symm_ab_sk_reset(d_workspace, st))) return r;
    return launch_symm_ab(map, batch, N, d_workspace, 1u, st);
}

int bml_cheb_schedule(int32_t k, int32_t *level, int32_t *a, int32_t *b) { return cheb_schedule(k, level, a, b); }

int bml_symm_work_item(int64_t N, int32_t n_jobs, int32_t n_ctas, int32_t cta, int32_t it, int32_t *out6)
{
    if (!out6) return BML_ERR_INVALID;
    return symm_ab_work_item(N, n_jobs, n_ctas, cta, it, out6);
}

// ------------------------------------------------ bml_graph.h ------------------------------------------------
// ELLPACK-R descriptor whose row capacity may exceed the SP2 kernels' BML_ELL_MAX_M (rows of a graph-built D are as
// long as a core+halo part unless drop_tol cuts them)
static bool ell_ok_wide(const bml_matrix_t *A)
{
    return A && A->type == BML_ELLPACK && A->value && A->index && A->nnz && A->N > 0 && A->N < (1 << 29) - 1 &&
           A->M >= 1 && A->M <= (1 << 20);
}
static bool graph_params_ok(const bml_graph_params_t *p, int64_t N)
{
    return p && p->n_parts >= 1 && p->n_parts <= BML_GRAPH_MAX_PARTS && p->part_capacity >= 1 &&
           (int64_t)p->part_capacity <= N && p->k >= 2 && p->k <= BML_CHEB_MAX_K && p->m >= 1 && p->m <= BML_CHEB_MAX_M &&
           p->k * p->m <= BML_CHEB_MAX_TERMS && p->beta > 0.0 && p->mu == p->mu && p->graph_tol >= 0.0 &&
           p->drop_tol >= 0.0;
}

size_t bml_graph_workspace_bytes(int64_t N, int32_t n_parts, int32_t part_capacity, int32_t k, int32_t m)
{
    if (N <= 0 || n_parts < 1 || n_parts > BML_GRAPH_MAX_PARTS || part_capacity < 1 || part_capacity > N || k < 2 ||
        k > BML_CHEB_MAX_K || m < 1 || m > BML_CHEB_MAX_M)
        return 0;
    return graph_workspace_bytes(N, n_parts, part_capacity, k, m);
}

int bml_graph_chebyshev_ellpack(const bml_matrix_t *H, const int32_t *d_core_offsets, const int32_t *d_core_nodes,
                                const bml_graph_params_t *p, bml_matrix_t *D, void *d_workspace, size_t workspace_bytes,
                                bml_graph_stats_t *stats, void *cuda_stream)
{
    int r;
    if (!ell_ok_wide(H) || !ell_ok_wide(D) || D->N != H->N || !graph_params_ok(p, H->N) || !d_core_offsets ||
        !d_core_nodes || !d_workspace || D->value == H->value || D->index == H->index || D->nnz == H->nnz ||
        ((uintptr_t)d_workspace & 1023) != 0 ||
        workspace_bytes < bml_graph_workspace_bytes(H->N, p->n_parts, p->part_capacity, p->k, p->m)) {
        r = BML_ERR_INVALID;
        if (stats) memset(stats, 0, sizeof(*stats));
    } else {
        r = graph_chebyshev_solve(H, d_core_offsets, d_core_nodes, p, D, d_workspace, stats, (cudaStream_t)cuda_stream);
    }
    if (stats) stats->status = r;
    return r;
}

size_t bml_graph_sp2_workspace_bytes(int64_t N, int32_t n_parts, int32_t part_capacity)
{
    if (N <= 0 || n_parts < 1 || n_parts > BML_GRAPH_MAX_PARTS || part_capacity < 1 || part_capacity > N) return 0;
    return graph_sp2_workspace_bytes(N, n_parts, part_capacity);
}

int bml_graph_sp2_ellpack(const bml_matrix_t *H, const int32_t *d_core_offsets, const int32_t *d_core_nodes,
                          const bml_graph_sp2_params_t *p, bml_matrix_t *D, void *d_workspace, size_t workspace_bytes,
                          bml_graph_sp2_stats_t *stats, void *cuda_stream)
{
    int r;
    if (!ell_ok_wide(H) || !ell_ok_wide(D) || D->N != H->N || !p || p->n_parts < 1 || p->n_parts > BML_GRAPH_MAX_PARTS ||
        p->part_capacity < 1 || (int64_t)p->part_capacity > H->N || p->n_occ <= 0 || (int64_t)p->n_occ >= H->N ||
        !(p->idem_tol > 0.0) || !(p->graph_tol >= 0.0) || !(p->drop_tol >= 0.0) || p->max_products < 1 ||
        p->max_products > BML_SP2_LOG_LEN || !d_core_offsets || !d_core_nodes || !d_workspace || D->value == H->value ||
        D->index == H->index || D->nnz == H->nnz || ((uintptr_t)d_workspace & 1023) != 0 ||
        workspace_bytes < bml_graph_sp2_workspace_bytes(H->N, p->n_parts, p->part_capacity)) {
        r = BML_ERR_INVALID;
        if (stats) memset(stats, 0, sizeof(*stats));
    } else {
        r = graph_sp2_solve(H, d_core_offsets, d_core_nodes, p, D, d_workspace, stats, (cudaStream_t)cuda_stream);
    }
    if (stats) { stats->status = r; stats->sp2.status = r; }
    return r;
}

int bml_dense_batch_work_item(int32_t n_jobs, const int32_t *n, int32_t n_ctas, int32_t cta, int32_t it, int32_t *out5)
{
    if (!n || !out5) return BML_ERR_INVALID;
    return dense_batch_work_item(n_jobs, n, n_ctas, cta, it, out5);
}

int bml_graph_core_halo(const bml_matrix_t *H, const int32_t *d_core_offsets, const int32_t *d_core_nodes, int32_t n_parts,
                        double graph_tol, int32_t *d_part_nodes, uint8_t *d_is_core, int32_t *d_part_sizes,
                        void *d_workspace, size_t workspace_bytes, void *cuda_stream)
{
    if (!ell_ok_wide(H) || !d_core_offsets || !d_core_nodes || n_parts < 1 || n_parts > BML_GRAPH_MAX_PARTS ||
        !(graph_tol >= 0.0) || !d_part_nodes || !d_is_core || !d_part_sizes || !d_workspace ||
        workspace_bytes < (size_t)n_parts * (size_t)H->N)
        return BML_ERR_INVALID;
    return launch_graph_core_halo(H, d_core_offsets, d_core_nodes, n_parts, graph_tol, d_part_nodes, d_is_core,
                                  d_part_sizes, (uint8_t *)d_workspace, (cudaStream_t)cuda_stream);
}

int bml_matrix2submatrix_ellpack(const bml_matrix_t *H, const int32_t *d_nodes, int32_t s, double *d_h, int64_t ld,
                                 void *cuda_stream)
{
    if (!ell_ok_wide(H) || !d_nodes || s < 1 || (int64_t)s > H->N || !d_h || ld < s) return BML_ERR_INVALID;
    return launch_graph_gather(H, d_nodes, s, d_h, ld, (cudaStream_t)cuda_stream);
}

int bml_submatrix2matrix_ellpack(const double *d_d, int64_t ld, const int32_t *d_nodes, const uint8_t *d_is_core, int32_t s,
                                 double drop_tol, bml_matrix_t *D, int32_t *d_overflow_row, void *cuda_stream)
{
    if (!ell_ok_wide(D) || !d_d || !d_nodes || !d_is_core || s < 1 || (int64_t)s > D->N || ld < s || !(drop_tol >= 0.0) ||
        !d_overflow_row)
        return BML_ERR_INVALID;
    return launch_graph_scatter(d_d, ld, d_nodes, d_is_core, s, drop_tol, D, d_overflow_row, (cudaStream_t)cuda_stream);
}

int bml_probe_fp64_tensor_peak(int32_t iters, double *flops_out, double *ms_out, void *cuda_stream)
{
    if (iters < 1 || !flops_out || !ms_out) return BML_ERR_INVALID;
    return run_fp64_tensor_probe(iters, flops_out, ms_out, (cudaStream_t)cuda_stream);
}

}  // extern "C"
