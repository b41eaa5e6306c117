// chebyshev.cu -- the Chebyshev / Paterson-Stockmeyer Fermi-operator path (PAPER.md IV.B):
// device-side coefficients (c_n of Eq. 8, d_{i,j} of Eq. 10), the map H -> H~ = T_1, the partial sums S_j (Eq. 12) and
// the launch sequence.  The matrix products themselves are the grouped kernel of symm_ab.cu.
#include <string.h>

#include "symm_ab.cuh"

namespace bmlsp2 {

// reductions.cu
int launch_gershgorin(const bml_matrix_t *H, double *d_bounds, double *rowlh, cudaStream_t st);
int launch_trace_dense(const double *A, int64_t ld, int N, double *d_out, cudaStream_t st);
int launch_check_symmetry(const bml_matrix_t *H, int *d_flag, cudaStream_t st);

// Device-resident record of one expansion; copied to the host once, at the end of the call.
struct ChebCtl {
    double bounds[2];      // Gershgorin e_min, e_max
    double trace;          // tr D
    int32_t fail;          // 0, or BML_ERR_DEGENERATE
    int32_t not_symmetric; // set by the symmetry check
    int32_t pad[2];
    double c[BML_CHEB_MAX_TERMS];
    double d[BML_CHEB_MAX_TERMS];      // d_{i,j} at d[j * k + i]
};
constexpr size_t CHEB_CTL_BYTES = (sizeof(ChebCtl) + 1023) / 1024 * 1024;
constexpr size_t CHEB_CTL_STRIDE = CHEB_CTL_BYTES;

// f_mu(eps) = 1 / (1 + exp(beta (eps - mu))), written so that exp never overflows (reading C2)
__device__ __forceinline__ double fermi_fn(double eps, double mu, double beta)
{
    const double z = beta * (eps - mu);
    if (z >= 0.0) { const double e = exp(-z); return e / (1.0 + e); }
    return 1.0 / (1.0 + exp(z));
}

// ------------------------------------------------------------------------------------------------------------
// c_n (Eq. 8) by Chebyshev-Gauss quadrature on N_q = 2 (L + 1) nodes (reading C3), then d_{i,j} (Eq. 10) by dividing
// the series by T_k with Eq. 11 (reading C4).  One CTA; scalar work: O(L N_q) table look-ups, then m division steps of
// 2k parallel chains of <= m / 2 subtractions.
// ------------------------------------------------------------------------------------------------------------
constexpr int CC_THREADS = 1024;
__global__ void __launch_bounds__(CC_THREADS, 1) cheb_coeff_kernel(ChebCtl *ctl, double mu, double beta, int k, int m)
{
    // dynamic shared memory, cheb_coeff_smem_bytes(k m): node values, the two division buffers and the cosine table
    // (every lane of a warp reads a different entry of it)
    extern __shared__ double s_dyn[];
    const int terms = k * m, Nq = 2 * terms;
    double *s_f = s_dyn;                   // [N_q]      f at the nodes
    double *s_p = s_f + Nq;                // [terms]    dividend of the current division step
    double *s_q = s_p + terms;             // [terms]    its quotient
    double *tab = s_q + terms;             // [4 N_q]    cos(pi j / (2 N_q))
    const double emin = ctl->bounds[0], emax = ctl->bounds[1];
    if (threadIdx.x == 0) ctl->fail = (emax - emin > 0.0) ? 0 : BML_ERR_DEGENERATE;
    // exact angles: every cosine needed is cos(pi j / (2 N_q)) with an integer j reduced mod 4 N_q
    for (int j = threadIdx.x; j < 4 * Nq; j += CC_THREADS) tab[j] = cospi((double)j / (double)(2 * Nq));
    __syncthreads();
    // f at the nodes, folded: cos(n pi (N_q - q - 1/2) / N_q) = (-1)^n cos(n pi (q + 1/2) / N_q), so the sum over the
    // N_q nodes is a sum over the first N_q / 2 of f_q +- f_{N_q-1-q} (N_q is even).  This O(L N_q) loop runs on ONE SM
    // and is issue-bound (4 schedulers): the fold halves it.  s_f[q] = f_q + f_mirror, s_f[N_q/2 + q] = f_q - f_mirror.
    const int Nh = Nq / 2;
    for (int q = threadIdx.x; q < Nh; q += CC_THREADS) {
        const double x = tab[2 * q + 1];                                // cos(pi (q + 1/2) / N_q); the mirror node is -x
        const double fa = fermi_fn(0.5 * (emax - emin) * x + 0.5 * (emax + emin), mu, beta);
        const double fb = fermi_fn(-0.5 * (emax - emin) * x + 0.5 * (emax + emin), mu, beta);
        s_f[q] = fa + fb;
        s_f[Nh + q] = fa - fb;
    }
    __syncthreads();
    // one warp per coefficient, the N_q / 2 nodes dealt out to its lanes: table index j = n (2 q + 1) mod 4 N_q,
    // advanced by 64 n
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    for (int n = warp; n < terms; n += CC_THREADS / 32) {
        const unsigned period = (unsigned)(4 * Nq);
        unsigned j = ((unsigned)n * (2u * (unsigned)lane + 1u)) % period;
        const unsigned step = (64u * (unsigned)n) % period;
        const double *fs = s_f + ((n & 1) ? Nh : 0);
        double s = 0.0;
        for (int q = lane; q < Nh; q += 32) {
            s = fma(fs[q], tab[j], s);
            j += step;
            if (j >= period) j -= period;
        }
        s = warp_sum(s);
        const double cn = (n == 0 ? 1.0 : 2.0) / (double)Nq * s;
        if (lane == 0) { ctl->c[n] = cn; s_p[n] = cn; }
    }
    __syncthreads();
    // p = T_k q + r, deg r < k: for n > k, T_n = 2 T_k T_{n-k} - T_{|n-2k|}; T_k = T_k T_0 (Eq. 11), highest n first.
    // Going down from the highest n, p_n is final once p_{n+2k} has been subtracted from it, so the 2k residue classes
    // of n mod 2k are independent chains (one thread each); the reflected targets |n - 2k| = 2k - n, k < n < 2k, come
    // after the chains.  Every p_i sees the same subtractions in the same order as in the one-thread loop.
    // Only the first two warps take part (2k <= 64 chains), synchronised by a named barrier of 64 threads: a barrier of
    // the whole 1024-thread CTA per phase was most of this kernel's time.  The quotient is built in a second buffer.
    const int tid = threadIdx.x;
    if (tid >= 64) return;
    auto bar64 = []() { asm volatile("bar.sync 1, 64;" ::: "memory"); };
    double *pp = s_p, *qq = s_q;
    int len = terms;
    for (int j = 0; j < m; ++j) {
        const int qlen = len - k;
        if (tid < 2 * k && tid < len) {
            int n = tid + (len - 1 - tid) / (2 * k) * (2 * k);           // largest index of this class below len
            double above = pp[n];
            for (n -= 2 * k; n >= 0; n -= 2 * k) {
                above = pp[n] - above;
                pp[n] = above;
            }
        }
        bar64();
        if (tid > 0 && tid < k && 2 * k - tid < len) pp[tid] -= pp[2 * k - tid];
        bar64();
        if (tid < k) ctl->d[j * k + tid] = pp[tid];
        for (int i = tid; i < qlen; i += 64) qq[i] = (i == 0) ? pp[k] : 2.0 * pp[i + k];
        bar64();
        double *t = pp; pp = qq; qq = t;
        len = qlen;
    }
}

// ------------------------------------------------------------------------------------------------------------
// T_1 = H~ = (2 H - (e_max + e_min) I) / (e_max - e_min)   (reading C1).  One pass: N^2 x 8 B read + written.
// ------------------------------------------------------------------------------------------------------------
__global__ void cheb_map_kernel(const double *__restrict__ H, int64_t ldh, double *__restrict__ T1, int64_t ld, int N,
                                const ChebCtl *__restrict__ ctl)
{
    const double emin = ctl->bounds[0], emax = ctl->bounds[1];
    const double shift = emax + emin, width = emax - emin;
    const int c = blockIdx.x * blockDim.x + threadIdx.x;
    if (c >= N) return;
    for (int r = blockIdx.y; r < N; r += gridDim.y) {
        const double h = H[(int64_t)r * ldh + c];
        T1[(int64_t)r * ld + c] = (2.0 * h - (r == c ? shift : 0.0)) / width;
    }
}

// ------------------------------------------------------------------------------------------------------------
// S_j = sum_{i<k} d_{i,j} T_i, j = 0 .. m-1 (Eq. 12), all m sums in ONE pass over T_1 .. T_{k-1} (T_0 = I adds
// d_{0,j} on the diagonal): every T_i element is read once and feeds m accumulators held in registers, where the paper
// computes the S_j as m separate sums on concurrent streams.  HBM-bound: (k - 1 + m) N^2 x 8 B.
// slab: slot s holds the matrix at slab + s * slot_elems; T_i in slot i - 1, S_j in slot k + j.
// ------------------------------------------------------------------------------------------------------------
static size_t cheb_coeff_smem_bytes(int terms) { return (size_t)(2 + 1 + 1 + 8) * (size_t)terms * sizeof(double); }

static int launch_cheb_coeff(ChebCtl *ctl, double mu, double beta, int k, int m, cudaStream_t st)
{
    static size_t have[MAX_DEVICES] = {};
    if (ensure_smem_attr(cheb_coeff_kernel, cheb_coeff_smem_bytes(BML_CHEB_MAX_TERMS), have)) return BML_ERR_CUDA;
    cheb_coeff_kernel<<<1, CC_THREADS, cheb_coeff_smem_bytes(k * m), st>>>(ctl, mu, beta, k, m);
    return cudaGetLastError() == cudaSuccess ? 0 : BML_ERR_CUDA;
}

template <int MJ, int CW>
__global__ void __launch_bounds__(256, (MJ * CW <= 16) ? 4 : 2)
cheb_sums_kernel(double *__restrict__ slab, int64_t slot_elems, int64_t ld, int N, int k, int m,
                 const ChebCtl *__restrict__ ctl)
{
    // s_d[i * MJ + j] = d_{i,j} (0 for j >= m): the MJ coefficients of one T_i are contiguous -> 128-bit broadcast loads
    __shared__ __align__(16) double s_d[BML_CHEB_MAX_K * MJ];
    for (int idx = threadIdx.x; idx < k * MJ; idx += blockDim.x) {
        const int i = idx / MJ, j = idx - i * MJ;
        s_d[idx] = j < m ? ctl->d[j * k + i] : 0.0;
    }
    __syncthreads();
    // CW adjacent columns per thread.  CW = 2 (few sums: registers to spare) makes every access 16 bytes -- ld is even
    // and rows are 128-byte aligned; a pair that straddles N reads a pad column and stores only its first element.
    // CW = 1 (16 or 32 sums) keeps the accumulators at MJ registers pairs so that 4 CTAs fit an SM: the kernel is
    // latency-bound and needs the warps more than the wider accesses.
    const int c = (blockIdx.x * blockDim.x + threadIdx.x) * CW;
    if (c >= N) return;
    const bool two = (CW == 2) && (c + 1 < N);
    for (int r = blockIdx.y; r < N; r += gridDim.y) {
        const int64_t off = (int64_t)r * ld + c;
        double acc[CW][MJ];
#pragma unroll
        for (int j = 0; j < MJ; ++j) {
#pragma unroll
            for (int q = 0; q < CW; ++q) acc[q][j] = (r == c + q) ? s_d[j] : 0.0;
        }
#pragma unroll 8
        for (int i = 1; i < k; ++i) {
            const double *src = slab + (int64_t)(i - 1) * slot_elems + off;
            double t[CW];
            if (CW == 2) { const double2 v = __ldg((const double2 *)src); t[0] = v.x; t[CW - 1] = v.y; }
            else t[0] = __ldg(src);
#pragma unroll
            for (int j = 0; j < MJ; ++j) {
                const double dij = s_d[i * MJ + j];
#pragma unroll
                for (int q = 0; q < CW; ++q) acc[q][j] = fma(dij, t[q], acc[q][j]);
            }
        }
#pragma unroll
        for (int j = 0; j < MJ; ++j) {
            if (j < m) {
                double *dst = slab + (int64_t)(k + j) * slot_elems + off;
                if (two) *(double2 *)dst = make_double2(acc[0][j], acc[CW - 1][j]);
                else *dst = acc[0][j];
            }
        }
    }
}

template <int MJ, int CW>
static int launch_sums_t(double *slab, int64_t slot_elems, int64_t ld, int N, int k, int m, const ChebCtl *ctl,
                         cudaStream_t st)
{
    // a few CTAs per SM in total, each walking several rows: the staging of d_{i,j} is paid once per CTA
    const unsigned gx = (unsigned)((N + 256 * CW - 1) / (256 * CW));
    unsigned gy = (16u * 148u + gx - 1) / gx;
    if (gy > (unsigned)N) gy = (unsigned)N;
    const dim3 grid(gx, gy);
    cheb_sums_kernel<MJ, CW><<<grid, 256, 0, st>>>(slab, slot_elems, ld, N, k, m, ctl);
    return cudaGetLastError() == cudaSuccess ? 0 : BML_ERR_CUDA;
}

// ------------------------------------------------------------------------------------------------------------
// host side
// ------------------------------------------------------------------------------------------------------------
// doubling schedule of reading C5: T_i = 2 T_a T_b - T_{a-b}, a = ceil(i / 2), b = floor(i / 2); level = ceil(log2 i)
int cheb_schedule(int k, int32_t *level, int32_t *a, int32_t *b)
{
    if (k < 2 || k > BML_CHEB_MAX_K) return BML_ERR_INVALID;
    int levels = 0;
    for (int i = 2; i <= k; ++i) {
        int lv = 0;
        while ((1 << lv) < i) ++lv;
        if (level) level[i - 2] = lv;
        if (a) a[i - 2] = (i + 1) / 2;
        if (b) b[i - 2] = i / 2;
        if (lv > levels) levels = lv;
    }
    return levels;
}

static inline size_t align_up(size_t x, size_t a) { return (x + a - 1) / a * a; }

struct ChebWs {
    uint8_t *ctl0;          // P control blocks, CHEB_CTL_STRIDE bytes apart
    double *rowlh;
    void *sk;
    double *slab;           // P x (k + m) slots: problem q owns slots q (k + m) .. ; T_i at +i - 1, S_j at +k + j
    int64_t ld, slot_elems;
    size_t total;
    ChebCtl *ctl(int q) const { return (ChebCtl *)(ctl0 + (size_t)q * CHEB_CTL_STRIDE); }
};

static ChebWs carve_cheb(void *ws, int64_t N, int k, int m, int P)
{
    ChebWs w;
    uint8_t *p = (uint8_t *)ws;
    size_t off = 0;
    w.ctl0 = p + off; off = align_up(off + (size_t)P * CHEB_CTL_STRIDE, 1024);
    w.rowlh = (double *)(p + off); off = align_up(off + (size_t)2 * N * sizeof(double), 1024);
    w.sk = (void *)(p + off); off = align_up(off + symm_ab_sk_bytes(), 1024);
    w.ld = (N + 15) / 16 * 16;
    w.slot_elems = (int64_t)align_up((size_t)N * w.ld, 128);
    w.slab = (double *)(p + off); off = align_up(off + (size_t)P * (k + m) * w.slot_elems * sizeof(double), 1024);
    w.total = off;
    return w;
}

size_t cheb_workspace_bytes(int64_t N, int k, int m) { return carve_cheb(nullptr, N, k, m, 1).total; }
size_t cheb_batch_workspace_bytes(int64_t N, int k, int m, int P) { return carve_cheb(nullptr, N, k, m, P).total; }

// Enqueue P independent expansions of the same size N (steps C0-C6 each), no host synchronisation.  The products of
// the P problems share launches: a doubling level or a nesting step of ALL problems goes out in grouped launches of up
// to BML_SYMM_MAX_JOBS products (this is what fills the GPU when one problem is too small to).
// D[q] may point into the workspace (cheb_batch_result): the last nesting step then works in place.
// The device-side verdict of problem q (0 or BML_ERR_DEGENERATE) is left in *cheb_fail_flag(ws, q).
int cheb_dense_enqueue_batch(int P, const bml_matrix_t *H, const bml_cheb_params_t *p, const bml_matrix_t *D, void *ws,
                             int *n_launches_out, cudaStream_t st)
{
    const int64_t N = H[0].N;
    const int k = p->k, m = p->m, SL = k + m;
    ChebWs w = carve_cheb(ws, N, k, m, P);
    auto slot = [&](int q, int s) { return w.slab + (int64_t)(q * SL + s) * w.slot_elems; };
#define CK(x) do { int _r = (x); if (_r != 0) return _r; } while (0)
    for (int q = 0; q < P; ++q) {
        if (cudaMemsetAsync(w.ctl(q), 0, 64, st) != cudaSuccess) return BML_ERR_CUDA;
        CK(launch_gershgorin(&H[q], w.ctl(q)->bounds, w.rowlh, st));
        if (p->flags & BML_SP2_FLAG_CHECK_SYMMETRY) CK(launch_check_symmetry(&H[q], &w.ctl(q)->not_symmetric, st));
        CK(launch_cheb_coeff(w.ctl(q), p->mu, p->beta, k, m, st));
        const dim3 grid((unsigned)((N + 255) / 256), (unsigned)(N < 2048 ? N : 2048));
        cheb_map_kernel<<<grid, 256, 0, st>>>(H[q].value, H[q].ld, slot(q, 0), w.ld, (int)N, w.ctl(q));
        if (cudaGetLastError() != cudaSuccess) return BML_ERR_CUDA;
    }

    CUtensorMap map;
    CK(make_slab_map(&map, w.slab, N, w.ld, w.slot_elems, P * SL));
    CK(symm_ab_sk_reset(w.sk, st));
    unsigned int epoch = 0;
    int n_launches = 0;
    SymmBatch batch;
    memset(&batch, 0, sizeof(batch));
    auto flush = [&]() -> int {
        if (batch.n_jobs == 0) return 0;
        const int r = launch_symm_ab(map, batch, N, w.sk, ++epoch, st);
        ++n_launches;
        memset(&batch, 0, sizeof(batch));
        return r;
    };
    auto add = [&](const SymmJob &jb) -> int {
        batch.job[batch.n_jobs++] = jb;
        return batch.n_jobs == BML_SYMM_MAX_JOBS ? flush() : 0;
    };

    // T_2 .. T_k of every problem, level by level (Eq. 13-14)
    int32_t level[BML_CHEB_MAX_K], ta[BML_CHEB_MAX_K], tb[BML_CHEB_MAX_K];
    const int levels = cheb_schedule(k, level, ta, tb);
    for (int lv = 1; lv <= levels; ++lv) {
        for (int q = 0; q < P; ++q)
            for (int i = 2; i <= k; ++i) {
                if (level[i - 2] != lv) continue;
                SymmJob jb;
                memset(&jb, 0, sizeof(jb));
                jb.a = q * SL + ta[i - 2] - 1; jb.b = q * SL + tb[i - 2] - 1;
                jb.Out = slot(q, i - 1); jb.ldo = w.ld; jb.ldc = w.ld;
                jb.alpha = 2.0;
                if (ta[i - 2] == tb[i - 2]) { jb.C = nullptr; jb.beta = 0.0; jb.gamma = -1.0; }     // - T_0
                else { jb.C = slot(q, 0); jb.beta = -1.0; jb.gamma = 0.0; }                         // - T_1
                CK(add(jb));
            }
        CK(flush());                    // the next level reads this one
    }

    // S_0 .. S_{m-1} (Eq. 12)
    for (int q = 0; q < P; ++q) {
        double *base = slot(q, 0);
        if (m <= 4) CK((launch_sums_t<4, 2>(base, w.slot_elems, w.ld, (int)N, k, m, w.ctl(q), st)));
        else if (m <= 8) CK((launch_sums_t<8, 2>(base, w.slot_elems, w.ld, (int)N, k, m, w.ctl(q), st)));
        else if (m <= 16) CK((launch_sums_t<16, 1>(base, w.slot_elems, w.ld, (int)N, k, m, w.ctl(q), st)));
        else CK((launch_sums_t<32, 1>(base, w.slot_elems, w.ld, (int)N, k, m, w.ctl(q), st)));
    }

    // Eq. 10, innermost bracket first: R_{m-1} = S_{m-1}; R_j = T_k R_{j+1} + S_j, written over S_j; R_0 -> D
    for (int j = m - 2; j >= 0; --j) {
        for (int q = 0; q < P; ++q) {
            SymmJob jb;
            memset(&jb, 0, sizeof(jb));
            jb.a = q * SL + k - 1; jb.b = q * SL + k + j + 1;
            jb.C = slot(q, k + j); jb.ldc = w.ld;
            jb.Out = (j == 0) ? D[q].value : slot(q, k + j);
            jb.ldo = (j == 0) ? D[q].ld : w.ld;
            jb.alpha = 1.0; jb.beta = 1.0; jb.gamma = 0.0;
            CK(add(jb));
        }
        CK(flush());
    }
    for (int q = 0; q < P; ++q) {
        if (m == 1 && D[q].value != slot(q, k) &&
            cudaMemcpy2DAsync(D[q].value, (size_t)D[q].ld * 8, slot(q, k), (size_t)w.ld * 8, (size_t)N * 8, (size_t)N,
                              cudaMemcpyDeviceToDevice, st) != cudaSuccess)
            return BML_ERR_CUDA;
        CK(launch_trace_dense(D[q].value, D[q].ld, (int)N, &w.ctl(q)->trace, st));
    }
#undef CK
    if (n_launches_out) *n_launches_out = n_launches;
    return 0;
}

// where problem q of a batch leaves its result when D[q] is not supplied by the caller: its S_0 slot (leading dim ld)
double *cheb_batch_result(void *ws, int64_t N, int k, int m, int P, int q, int64_t *ld_out)
{
    ChebWs w = carve_cheb(ws, N, k, m, P);
    if (ld_out) *ld_out = w.ld;
    return w.slab + (int64_t)(q * (k + m) + k) * w.slot_elems;
}

// Enqueue one expansion: the batch of one.
int cheb_dense_enqueue(const bml_matrix_t *H, const bml_cheb_params_t *p, bml_matrix_t *D, void *ws, int *n_launches_out,
                       cudaStream_t st)
{
    return cheb_dense_enqueue_batch(1, H, p, D, ws, n_launches_out, st);
}

int *cheb_fail_flag(void *ws, int q) { return &((ChebCtl *)((uint8_t *)ws + (size_t)q * CHEB_CTL_STRIDE))->fail; }

// ------------------------------------------------------------------------------------------------------------
// CUDA-graph replay of one expansion.  The launch sequence of an expansion is static -- no host decision, no
// data-dependent launch shape -- so it is captured once per (pointers, shapes, parameters) and replayed: for small
// matrices the ~25 launches are launch-latency bound.  A handful of instantiated graphs is kept per
// host thread; anything that fails to capture or instantiate falls back to plain enqueueing (never to another
// implementation).
// ------------------------------------------------------------------------------------------------------------
struct ChebGraphKey {
    const void *H, *D, *ws;
    int64_t N, ldh, ldd;
    double mu, beta;
    int32_t k, m;
    uint32_t flags;
    cudaStream_t st;
    int dev;            // device ordinal the graph was instantiated on
    bool operator==(const ChebGraphKey &o) const
    {
        return H == o.H && D == o.D && ws == o.ws && N == o.N && ldh == o.ldh && ldd == o.ldd && mu == o.mu &&
               beta == o.beta && k == o.k && m == o.m && flags == o.flags && st == o.st && dev == o.dev;
    }
};
struct ChebGraphSlot {
    ChebGraphKey key;
    cudaGraphExec_t exec = nullptr;
    int n_launches = 0;
    uint64_t stamp = 0;
};
constexpr int CHEB_GRAPH_SLOTS = 4;
constexpr int64_t CHEB_GRAPH_MAX_N = 2048;      // above this the launches are long: nothing to gain

// per host thread; the caller's pointers are keys only.  bml_sp2_release_cached() drops it.
static thread_local ChebGraphSlot g_cheb_slots[CHEB_GRAPH_SLOTS];
static thread_local uint64_t g_cheb_clock = 0;
static thread_local bool g_cheb_warmed[MAX_DEVICES][3] = {};

void cheb_graph_cache_release()
{
    for (auto &sl : g_cheb_slots) {
        if (sl.exec) cudaGraphExecDestroy(sl.exec);
        sl = ChebGraphSlot();
    }
}

static int cheb_enqueue_cached(const bml_matrix_t *H, const bml_cheb_params_t *p, bml_matrix_t *D, void *ws,
                               int *n_launches_out, cudaStream_t st)
{
    ChebGraphSlot (&slots)[CHEB_GRAPH_SLOTS] = g_cheb_slots;
    uint64_t &clock_ = g_cheb_clock;
    const int dev = current_device();
    if (dev < 0) return BML_ERR_CUDA;
    bool *warmed = g_cheb_warmed[dev];
    cudaStreamCaptureStatus cs = cudaStreamCaptureStatusNone;
    const bool capturing = cudaStreamIsCapturing(st, &cs) == cudaSuccess && cs != cudaStreamCaptureStatusNone;
    const int bti = H->N <= 512 ? 0 : (H->N <= 1024 ? 1 : 2);
    if (H->N > CHEB_GRAPH_MAX_N || capturing || st == nullptr || !warmed[bti]) {
        // the first expansion of a tile size runs plainly: it sets the kernels' shared-memory attributes, which must
        // not happen inside a capture; the legacy default stream cannot be captured
        warmed[bti] = true;
        return cheb_dense_enqueue(H, p, D, ws, n_launches_out, st);
    }
    const ChebGraphKey key = {H->value, D->value, ws, H->N, H->ld, D->ld, p->mu, p->beta, p->k, p->m, p->flags, st, dev};
    ChebGraphSlot *hit = nullptr, *victim = &slots[0];
    for (auto &sl : slots) {
        if (sl.exec && sl.key == key) hit = &sl;
        if (sl.stamp < victim->stamp) victim = &sl;
    }
    if (!hit) {
        cudaGraph_t graph = nullptr;
        int nl = 0;
        if (cudaStreamBeginCapture(st, cudaStreamCaptureModeThreadLocal) != cudaSuccess) {
            cudaGetLastError();
            return cheb_dense_enqueue(H, p, D, ws, n_launches_out, st);
        }
        const int r = cheb_dense_enqueue(H, p, D, ws, &nl, st);
        const cudaError_t ce = cudaStreamEndCapture(st, &graph);
        cudaGraphExec_t exec = nullptr;
        if (r != 0 || ce != cudaSuccess || !graph || cudaGraphInstantiate(&exec, graph, 0) != cudaSuccess) {
            if (graph) cudaGraphDestroy(graph);
            cudaGetLastError();
            return cheb_dense_enqueue(H, p, D, ws, n_launches_out, st);
        }
        cudaGraphDestroy(graph);
        if (victim->exec) cudaGraphExecDestroy(victim->exec);
        victim->key = key; victim->exec = exec; victim->n_launches = nl;
        hit = victim;
    }
    hit->stamp = ++clock_;
    if (n_launches_out) *n_launches_out = hit->n_launches;
    if (cudaGraphLaunch(hit->exec, st) != cudaSuccess) {
        cudaGetLastError();
        return cheb_dense_enqueue(H, p, D, ws, n_launches_out, st);
    }
    return 0;
}

int cheb_dense_solve(const bml_matrix_t *H, const bml_cheb_params_t *p, bml_matrix_t *D, void *ws, bml_cheb_stats_t *stats,
                     cudaStream_t st)
{
    const int k = p->k, m = p->m;
    ChebWs w = carve_cheb(ws, H->N, k, m, 1);
    int n_launches = 0;
    const int r = cheb_enqueue_cached(H, p, D, ws, &n_launches, st);
    if (r) return r;
    // the one host round trip of the call
    ChebCtl h;
    if (cudaMemcpyAsync(&h, w.ctl(0), sizeof(h), cudaMemcpyDeviceToHost, st) != cudaSuccess) return BML_ERR_CUDA;
    if (cudaStreamSynchronize(st) != cudaSuccess) return BML_ERR_CUDA;
    if (cudaGetLastError() != cudaSuccess) return BML_ERR_CUDA;
    int status = BML_OK;
    if (h.fail) status = h.fail;
    else if (h.not_symmetric) status = BML_ERR_NOT_SYMMETRIC;
    if (stats) {
        memset(stats, 0, sizeof(*stats));
        stats->status = status;
        stats->n_products = (k - 1) + (m - 1);
        stats->n_launches = n_launches;
        stats->L = k * m - 1;
        stats->emin = h.bounds[0]; stats->emax = h.bounds[1];
        stats->trace = h.trace;
        memcpy(stats->c, h.c, sizeof(double) * (size_t)(k * m));
        memcpy(stats->d, h.d, sizeof(double) * (size_t)(k * m));
    }
    return status;
}

}  // namespace bmlsp2
