// dense_mixed.cu -- mixed-precision dense X^2 (BASELINE.json configs[3]; not in the paper, readings item 17).
//
// X (FP64 master) is kept next to its three-way BF16 split  X = Xh + Xm + Xl  (Xh = bf16(X), Xm = bf16(X - Xh),
// Xl = bf16(X - Xh - Xm): 3 x 8 mantissa bits).  One product tile P_IJ = sum_K X_IK X_JK^T is evaluated on the 5th-gen
// tensor cores as the six cross terms of weight <= 2
//        Xh Xl^T + Xl Xh^T + Xm Xm^T + Xh Xm^T + Xm Xh^T + Xh Xh^T
// with tcgen05.mma.kind::f16 (BF16 x BF16 products are exact in FP32), FP32 accumulation in TMEM over a K-chunk of
// M_KC columns only; every chunk is read back with tcgen05.ld and added to FP64 accumulators held in registers by the
// eight epilogue warps (two TMEM accumulator buffers: the next chunk's MMAs run while the previous chunk is promoted).
// The FP64 epilogue is the one of the FP64 kernel (Eq. 6 / Eq. 7, tr P, ||P - X||^2, ||X||^2, tr X', mirrored write,
// last-CTA finaliser) and additionally writes the BF16 planes of X' for the next product.
//
// Roles (384 threads): warp 0 = TMA producer (one lane), warp 1 = MMA issuer (one lane), warp 2 = TMEM allocator,
// warps 4..11 = epilogue (thread <-> one accumulator row, 64 columns).  Shared memory: M_STAGES x { A planes h,m,l ;
// B planes h,m,l } of 128 rows x 32 bf16 (64-byte rows, SWIZZLE_64B, K-major UMMA canonical layout).
#include <cuda_bf16.h>

#include "common.cuh"

namespace bmlsp2 {

constexpr int M_BM = 128;
constexpr int M_BN = 128;
constexpr int M_BK = 32;                       // bf16 elements per k-slab = 64 bytes = one SWIZZLE_64B row
constexpr int M_STAGES = 4;
constexpr int M_KC_SLABS = 4;                  // K-chunk promoted to FP64 = 4 slabs = 128 columns
constexpr int M_PLANE_TILE = M_BM * M_BK * 2;  // 8 KB
constexpr int M_STAGE_BYTES = 6 * M_PLANE_TILE;
constexpr int M_EPI_WARPS = 8;
constexpr int M_CTRL_WARPS = 4;
constexpr int M_THREADS = (M_CTRL_WARPS + M_EPI_WARPS) * 32;
constexpr int M_REGS_CTRL = 56;
constexpr int M_REGS_EPI = 224;                // 128 x 56 + 256 x 224 = 64512
constexpr int M_TMEM_COLS = 256;               // two 128-column FP32 accumulator buffers
constexpr size_t M_SMEM_BYTES = (size_t)M_STAGES * M_STAGE_BYTES + 1024 /*align*/ + 1024 /*barriers, scratch*/;

// tcgen05 instruction descriptor (kind::f16): D = F32, A = B = BF16, both K-major, N = 128, M = 128
constexpr uint32_t M_IDESC = (1u << 4) | (1u << 7) | (1u << 10) | ((uint32_t)(M_BN >> 3) << 17) | ((uint32_t)(M_BM >> 4) << 24);

// shared-memory matrix descriptor: K-major, SWIZZLE_64B, 8-row groups 512 bytes apart, sm_100 descriptor version 1
__device__ __forceinline__ uint64_t umma_desc(uint32_t saddr)
{
    return (uint64_t)((saddr >> 4) & 0x3FFFu) | ((uint64_t)(512u >> 4) << 32) | (1ull << 46) | (4ull << 61);
}

__device__ __forceinline__ void umma_bf16(uint32_t tmem_d, uint64_t adesc, uint64_t bdesc, uint32_t accumulate)
{
    asm volatile(
        "{\n\t.reg .pred p;\n\t"
        "setp.ne.b32 p, %4, 0;\n\t"
        "tcgen05.mma.cta_group::1.kind::f16 [%0], %1, %2, %3, p;\n\t}"
        ::"r"(tmem_d), "l"(adesc), "l"(bdesc), "r"(M_IDESC), "r"(accumulate)
        : "memory");
}
__device__ __forceinline__ void umma_commit(uint64_t *bar)
{
    asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%0];" ::"r"(smem_u32(bar))
                 : "memory");
}
__device__ __forceinline__ void tc_fence_before() { asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory"); }
__device__ __forceinline__ void tc_fence_after() { asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory"); }

// 32 lanes x 32 consecutive FP32 columns of TMEM -> 32 registers per thread (thread = its own lane)
__device__ __forceinline__ void tmem_ld32(uint32_t taddr, uint32_t (&v)[32])
{
    asm volatile(
        "tcgen05.ld.sync.aligned.32x32b.x32.b32 "
        "{%0, %1, %2, %3, %4, %5, %6, %7, %8, %9, %10, %11, %12, %13, %14, %15, "
        "%16, %17, %18, %19, %20, %21, %22, %23, %24, %25, %26, %27, %28, %29, %30, %31}, [%32];"
        : "=r"(v[0]), "=r"(v[1]), "=r"(v[2]), "=r"(v[3]), "=r"(v[4]), "=r"(v[5]), "=r"(v[6]), "=r"(v[7]), "=r"(v[8]),
          "=r"(v[9]), "=r"(v[10]), "=r"(v[11]), "=r"(v[12]), "=r"(v[13]), "=r"(v[14]), "=r"(v[15]), "=r"(v[16]),
          "=r"(v[17]), "=r"(v[18]), "=r"(v[19]), "=r"(v[20]), "=r"(v[21]), "=r"(v[22]), "=r"(v[23]), "=r"(v[24]),
          "=r"(v[25]), "=r"(v[26]), "=r"(v[27]), "=r"(v[28]), "=r"(v[29]), "=r"(v[30]), "=r"(v[31])
        : "r"(taddr)
        : "memory");
}
__device__ __forceinline__ void tmem_ld_wait() { asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory"); }

// X = h + m + l in BF16 (round to nearest at every level)
__device__ __forceinline__ void split3(double x, __nv_bfloat16 &h, __nv_bfloat16 &m, __nv_bfloat16 &l)
{
    h = __double2bfloat16(x);
    const double r1 = x - (double)__bfloat162float(h);
    m = __double2bfloat16(r1);
    const double r2 = r1 - (double)__bfloat162float(m);
    l = __double2bfloat16(r2);
}

// planes[p][r][c], p = 0 (h), 1 (m), 2 (l); leading dimension ldp elements
__global__ void __launch_bounds__(256)
split_planes_kernel(const double *__restrict__ X, int64_t ld, int N, __nv_bfloat16 *__restrict__ planes, int64_t ldp)
{
    const int64_t plane = (int64_t)N * ldp;
    const int64_t total = (int64_t)N * N;
    for (int64_t e = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; e < total; e += (int64_t)gridDim.x * blockDim.x) {
        const int64_t r = e / N, c = e - r * N;
        __nv_bfloat16 h, m, l;
        split3(X[r * ld + c], h, m, l);
        planes[r * ldp + c] = h;
        planes[plane + r * ldp + c] = m;
        planes[2 * plane + r * ldp + c] = l;
    }
}

__global__ void __launch_bounds__(M_THREADS, 1)
x2_dense_mixed_kernel(const __grid_constant__ CUtensorMap map0, const __grid_constant__ CUtensorMap map1,
                      double *__restrict__ buf0, double *__restrict__ buf1, __nv_bfloat16 *__restrict__ pl0,
                      __nv_bfloat16 *__restrict__ pl1, int64_t ld, int N, Sp2Ctl *__restrict__ ctl,
                      double *__restrict__ partials)
{
    if (ctl->done) return;
    const int parity = ctl->parity;
    const int branch = ctl->branch_cur;
    const CUtensorMap *map = parity ? &map1 : &map0;
    const double *__restrict__ X = parity ? buf1 : buf0;
    double *__restrict__ Xn = parity ? buf0 : buf1;
    __nv_bfloat16 *__restrict__ Pn = parity ? pl0 : pl1;

    extern __shared__ uint8_t smem_raw[];
    uint8_t *smem = smem_raw + ((1024u - (smem_u32(smem_raw) & 1023u)) & 1023u);
    uint64_t *full_bar = (uint64_t *)(smem + (size_t)M_STAGES * M_STAGE_BYTES);
    uint64_t *empty_bar = full_bar + M_STAGES;
    uint64_t *tfull_bar = empty_bar + M_STAGES;       // [2] accumulator buffer ready for the epilogue
    uint64_t *tempty_bar = tfull_bar + 2;             // [2] accumulator buffer drained
    double (*s_red)[4] = (double (*)[4])(tempty_bar + 2);   // [M_EPI_WARPS][4]
    uint32_t *s_tmem = (uint32_t *)(s_red + M_EPI_WARPS);
    int *s_last = (int *)(s_tmem + 1);

    const int warp_all = threadIdx.x >> 5, lane = threadIdx.x & 31;
    int I, J;
    const bool valid = tile_sb_decode((int)blockIdx.x, (N + M_BM - 1) / M_BM, I, J);    // CTA-uniform
    const bool diag = (I == J);
    const int nslabs = (N + M_BK - 1) / M_BK;
    const int nchunks = (nslabs + M_KC_SLABS - 1) / M_KC_SLABS;

    if (threadIdx.x == 0) {
        for (int s = 0; s < M_STAGES; ++s) { mbar_init(&full_bar[s], 1); mbar_init(&empty_bar[s], 1); }
        for (int b = 0; b < 2; ++b) { mbar_init(&tfull_bar[b], 1); mbar_init(&tempty_bar[b], M_EPI_WARPS); }
        mbar_fence_init();
        fence_proxy_async();
    }
    if (threadIdx.x < M_EPI_WARPS * 4) ((double *)s_red)[threadIdx.x] = 0.0;     // empty slots contribute zero
    if (valid && warp_all == 2) {
        asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(smem_u32(s_tmem)),
                     "n"(M_TMEM_COLS)
                     : "memory");
        asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
    }
    tc_fence_before();
    __syncthreads();
    tc_fence_after();
    const uint32_t tmem_base = *(volatile uint32_t *)s_tmem;

    if (!valid) {
        // slot below the diagonal / outside the tile grid: nothing to compute
    } else if (warp_all < M_CTRL_WARPS) {
        asm volatile("setmaxnreg.dec.sync.aligned.u32 %0;" ::"n"(M_REGS_CTRL));
        if (warp_all == 0 && lane == 0) {
            // ===================== TMA producer =====================
            tma_prefetch_desc(map);
            const uint32_t tx = (diag ? 3u : 6u) * M_PLANE_TILE;
            for (int slab = 0; slab < nslabs; ++slab) {
                const int s = slab % M_STAGES;
                const uint32_t ph = (uint32_t)(slab / M_STAGES) & 1u;
                mbar_wait(&empty_bar[s], ph ^ 1u);
                mbar_expect_tx(&full_bar[s], tx);
                uint8_t *dst = smem + (size_t)s * M_STAGE_BYTES;
#pragma unroll
                for (int p = 0; p < 3; ++p)
                    tma_load_2d(dst + p * M_PLANE_TILE, map, slab * M_BK, p * N + I * M_BM, &full_bar[s]);
                if (!diag) {
#pragma unroll
                    for (int p = 0; p < 3; ++p)
                        tma_load_2d(dst + (3 + p) * M_PLANE_TILE, map, slab * M_BK, p * N + J * M_BN, &full_bar[s]);
                }
            }
        } else if (warp_all == 1 && lane == 0) {
            // ===================== MMA issuer =====================
            // cross terms, smallest first: (A plane, B plane)
            const int ta[6] = {0, 2, 1, 0, 1, 0};
            const int tb[6] = {2, 0, 1, 1, 0, 0};
            for (int slab = 0; slab < nslabs; ++slab) {
                const int s = slab % M_STAGES;
                const uint32_t ph = (uint32_t)(slab / M_STAGES) & 1u;
                const int chunk = slab / M_KC_SLABS, within = slab % M_KC_SLABS;
                const int buf = chunk & 1;
                if (within == 0) {
                    mbar_wait(&tempty_bar[buf], (((uint32_t)chunk >> 1) & 1u) ^ 1u);
                    tc_fence_after();
                }
                mbar_wait(&full_bar[s], ph);
                tc_fence_after();
                const uint32_t a_base = smem_u32(smem + (size_t)s * M_STAGE_BYTES);
                const uint32_t b_base = diag ? a_base : a_base + 3 * M_PLANE_TILE;
                const uint32_t d_tmem = tmem_base + (uint32_t)buf * M_BN;
#pragma unroll
                for (int t = 0; t < 6; ++t) {
                    const uint64_t ad = umma_desc(a_base + ta[t] * M_PLANE_TILE);
                    const uint64_t bd = umma_desc(b_base + tb[t] * M_PLANE_TILE);
#pragma unroll
                    for (int ks = 0; ks < M_BK / 16; ++ks)     // UMMA_K = 16 bf16 = 32 bytes = 2 descriptor units
                        umma_bf16(d_tmem, ad + 2 * ks, bd + 2 * ks, (within | t | ks) != 0 ? 1u : 0u);
                }
                umma_commit(&empty_bar[s]);                   // frees the smem stage when these MMAs have read it
                if (within == M_KC_SLABS - 1 || slab == nslabs - 1) umma_commit(&tfull_bar[buf]);
            }
        }
    } else {
        // ===================== epilogue warps: promote every K-chunk to FP64, then the fused SP2 epilogue ============
        asm volatile("setmaxnreg.inc.sync.aligned.u32 %0;" ::"n"(M_REGS_EPI));
        const int e = warp_all - M_CTRL_WARPS;          // 0..7; TMEM lane quarter = warp_all % 4 = e % 4
        const int q = e & 3, half = e >> 2;
        double acc[64];
#pragma unroll
        for (int i = 0; i < 64; ++i) acc[i] = 0.0;
        const uint32_t t_lane = tmem_base + ((uint32_t)(q * 32) << 16) + (uint32_t)(half * 64);
        for (int chunk = 0; chunk < nchunks; ++chunk) {
            const int buf = chunk & 1;
            mbar_wait(&tfull_bar[buf], ((uint32_t)chunk >> 1) & 1u);
            tc_fence_after();
#pragma unroll
            for (int hh = 0; hh < 2; ++hh) {
                uint32_t v[32];
                tmem_ld32(t_lane + (uint32_t)(buf * M_BN + hh * 32), v);
                tmem_ld_wait();
#pragma unroll
                for (int i = 0; i < 32; ++i) acc[hh * 32 + i] += (double)__uint_as_float(v[i]);
            }
            tc_fence_before();
            __syncwarp();
            if (lane == 0) mbar_arrive(&tempty_bar[buf]);
        }

        // fused epilogue (D4): this thread owns row r, columns c0 .. c0 + 63 of the tile
        double s_trp = 0.0, s_e = 0.0, s_x = 0.0, s_trn = 0.0;
        const int r = I * M_BM + q * 32 + lane;
        const int c0 = J * M_BN + half * 64;
        const int64_t plane = (int64_t)N * ld;
        if (r < N) {
#pragma unroll
            for (int i = 0; i < 64; ++i) {
                const int c = c0 + i;
                if (c < N && (!diag || r <= c)) {
                    const double p = acc[i];
                    const double x = X[(int64_t)r * ld + c];
                    const double d = p - x;
                    const double xn = branch ? (2.0 * x - p) : p;     // Eq. 7 : Eq. 6
                    __nv_bfloat16 h, m, l;
                    split3(xn, h, m, l);
                    const int64_t o = (int64_t)r * ld + c;
                    Xn[o] = xn;
                    Pn[o] = h; Pn[plane + o] = m; Pn[2 * plane + o] = l;
                    if (r == c) {
                        s_trp += p; s_trn += xn; s_e += d * d; s_x += x * x;
                    } else {
                        const int64_t ot = (int64_t)c * ld + r;       // mirror
                        Xn[ot] = xn;
                        Pn[ot] = h; Pn[plane + ot] = m; Pn[2 * plane + ot] = l;
                        s_e += 2.0 * (d * d); s_x += 2.0 * (x * x);
                    }
                }
            }
        }
        s_trp = warp_sum(s_trp); s_e = warp_sum(s_e); s_x = warp_sum(s_x); s_trn = warp_sum(s_trn);
        if (lane == 0) { s_red[e][0] = s_trp; s_red[e][1] = s_e; s_red[e][2] = s_x; s_red[e][3] = s_trn; }
    }
    tc_fence_before();
    __syncthreads();
    if (valid && warp_all == 2) {
        tc_fence_after();
        asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(tmem_base), "n"(M_TMEM_COLS) : "memory");
    }

    // ===================== per-tile partials, last-CTA finaliser (D5) =====================
    if (threadIdx.x < 4) {
        double v = 0.0;
#pragma unroll
        for (int w = 0; w < M_EPI_WARPS; ++w) v += s_red[w][threadIdx.x];
        partials[(size_t)blockIdx.x * 4 + threadIdx.x] = v;
        __threadfence();
    }
    __syncthreads();
    if (threadIdx.x == 0) {
        const uint32_t prev = atomicAdd(&ctl->arrivals, 1u);
        *s_last = (prev + 1u == gridDim.x);
    }
    __syncthreads();
    if (*s_last && warp_all == 0) {
        __threadfence();
        double s[4] = {0.0, 0.0, 0.0, 0.0};
        const volatile double *vp = partials;
        for (int tI = lane; tI < (int)gridDim.x; tI += 32) {
#pragma unroll
            for (int k = 0; k < 4; ++k) s[k] += vp[(size_t)tI * 4 + k];
        }
#pragma unroll
        for (int k = 0; k < 4; ++k) s[k] = warp_sum(s[k]);
        if (lane == 0) sp2_finalise(ctl, s);
    }
}

// ------------------------------------------------------------------------------------------------------------
// host side
// ------------------------------------------------------------------------------------------------------------
int dense_fp64_num_tiles(int64_t N);

// the three BF16 planes of one iterate, stacked: rows p * N + r, leading dimension ldp (= the FP64 iterate's ld)
static int make_plane_map(CUtensorMap *map, const __nv_bfloat16 *base, int64_t N, int64_t ldp)
{
    PFN_encodeTiled enc = get_encode_tiled();
    if (!enc) return BML_ERR_CUDA;
    const cuuint64_t dims[2] = {(cuuint64_t)N, (cuuint64_t)(3 * N)};
    const cuuint64_t strides[1] = {(cuuint64_t)ldp * sizeof(__nv_bfloat16)};
    const cuuint32_t box[2] = {(cuuint32_t)M_BK, (cuuint32_t)M_BM};
    const cuuint32_t estr[2] = {1, 1};
    CUresult r = enc(map, CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, 2, (void *)base, dims, strides, box, estr,
                     CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_64B, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
                     CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    return r == CUDA_SUCCESS ? 0 : BML_ERR_CUDA;
}

static inline size_t plane_set_bytes(int64_t N, int64_t ldx)
{
    return ((size_t)3 * (size_t)N * (size_t)ldx * sizeof(__nv_bfloat16) + 1023) / 1024 * 1024;
}

size_t dense_mixed_extra_bytes(int64_t N, int64_t ldx) { return 2 * plane_set_bytes(N, ldx); }

static int launch_split(const double *X, int64_t ld, int64_t N, __nv_bfloat16 *planes, cudaStream_t st)
{
    int64_t blocks = (N * N + 255) / 256;
    if (blocks > 148 * 16) blocks = 148 * 16;
    split_planes_kernel<<<(unsigned)blocks, 256, 0, st>>>(X, ld, (int)N, planes, ld);
    return cudaGetLastError() == cudaSuccess ? 0 : BML_ERR_CUDA;
}

static int launch_x2_mixed(const CUtensorMap &m0, const CUtensorMap &m1, double *b0, double *b1, __nv_bfloat16 *p0,
                           __nv_bfloat16 *p1, int64_t ld, int64_t N, Sp2Ctl *ctl, double *partials, cudaStream_t st)
{
    static bool attr_set = false;
    if (!attr_set) {
        if (cudaFuncSetAttribute(x2_dense_mixed_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)M_SMEM_BYTES) !=
            cudaSuccess)
            return BML_ERR_CUDA;
        attr_set = true;
    }
    x2_dense_mixed_kernel<<<dense_fp64_num_tiles(N), M_THREADS, M_SMEM_BYTES, st>>>(m0, m1, b0, b1, p0, p1, ld, (int)N,
                                                                                    ctl, partials);
    return cudaGetLastError() == cudaSuccess ? 0 : BML_ERR_CUDA;
}

// X0 (already rescaled, in buffer 0) -> planes of buffer 0, then max_products fused products
int sp2_dense_mixed_solve(const bml_matrix_t *H, const bml_sp2_params_t *p, double *X0, double *X1, int64_t ldx,
                          Sp2Ctl *ctl, double *partials, const double *, void *extra, cudaStream_t st)
{
    const int64_t N = H->N;
    __nv_bfloat16 *p0 = (__nv_bfloat16 *)extra;
    __nv_bfloat16 *p1 = (__nv_bfloat16 *)((uint8_t *)extra + plane_set_bytes(N, ldx));
    CUtensorMap m0, m1;
    int r;
    if ((r = make_plane_map(&m0, p0, N, ldx))) return r;
    if ((r = make_plane_map(&m1, p1, N, ldx))) return r;
    if ((r = launch_split(X0, ldx, N, p0, st))) return r;
    return enqueue_products([&]() { return launch_x2_mixed(m0, m1, X0, X1, p0, p1, ldx, N, ctl, partials, st); }, ctl,
                            p->max_products, st);
}

int x2_dense_mixed_once(const bml_matrix_t *X, bml_matrix_t *Xn, Sp2Ctl *ctl, double *partials, void *extra,
                        cudaStream_t st)
{
    const int64_t N = X->N, ld = X->ld;
    __nv_bfloat16 *p0 = (__nv_bfloat16 *)extra;
    __nv_bfloat16 *p1 = (__nv_bfloat16 *)((uint8_t *)extra + plane_set_bytes(N, ld));
    CUtensorMap m0, m1;
    int r;
    if ((r = make_plane_map(&m0, p0, N, ld))) return r;
    if ((r = make_plane_map(&m1, p1, N, ld))) return r;
    if ((r = launch_split(X->value, ld, N, p0, st))) return r;
    return launch_x2_mixed(m0, m1, X->value, Xn->value, p0, p1, ld, N, ctl, partials, st);
}

}  // namespace bmlsp2
