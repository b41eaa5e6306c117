// probe.cu -- measurement helper (not part of the method): the FP64 tensor-pipe issue peak.
// Every warp keeps 16 independent 8x8 FP64 accumulator fragments in registers and issues `iters` rounds of 16
// back-to-back mma.sync m8n8k4 f64 (SASS DMMA.8x8x4) with register-resident operands: no memory traffic at all, so
// flops / time is the tensor pipe's issue peak at the clocks of the run.
#include "common.cuh"

namespace bmlsp2 {

constexpr int PROBE_ACC = 16;

__global__ void __launch_bounds__(256) fp64_tensor_probe_kernel(int iters, double *sink)
{
    double c[PROBE_ACC][2];
#pragma unroll
    for (int q = 0; q < PROBE_ACC; ++q) { c[q][0] = 0.0; c[q][1] = 0.0; }
    const double a = 1.0 + 1e-9 * (double)threadIdx.x, b = 1.0 - 1e-9 * (double)(threadIdx.x & 7);
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int q = 0; q < PROBE_ACC; ++q) dmma884(c[q][0], c[q][1], a, b);
    }
    double s = 0.0;
#pragma unroll
    for (int q = 0; q < PROBE_ACC; ++q) s += c[q][0] + c[q][1];
    if (s == -1.0) sink[0] = s;   // never true: keeps the chain alive
}

int run_fp64_tensor_probe(int iters, double *flops, double *ms, cudaStream_t st)
{
    int dev = 0, sms = 0;
    if (cudaGetDevice(&dev) != cudaSuccess) return BML_ERR_CUDA;
    if (cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess) return BML_ERR_CUDA;
    double *sink = nullptr;
    if (cudaMalloc(&sink, sizeof(double)) != cudaSuccess) return BML_ERR_CUDA;   // helper only: 8 bytes, freed below
    cudaEvent_t e0, e1;
    cudaEventCreate(&e0); cudaEventCreate(&e1);
    const int grid = sms * 2, block = 256;    // 16 warps per SM, 4 per scheduler
    fp64_tensor_probe_kernel<<<grid, block, 0, st>>>(iters / 8 + 1, sink);      // warm-up
    cudaEventRecord(e0, st);
    fp64_tensor_probe_kernel<<<grid, block, 0, st>>>(iters, sink);
    cudaEventRecord(e1, st);
    int rc = 0;
    if (cudaStreamSynchronize(st) != cudaSuccess || cudaGetLastError() != cudaSuccess) rc = BML_ERR_CUDA;
    float t = 0.f;
    cudaEventElapsedTime(&t, e0, e1);
    cudaEventDestroy(e0); cudaEventDestroy(e1);
    cudaFree(sink);
    *ms = (double)t;
    // one m8n8k4 = 8*8*4 FMAs = 512 flops
    *flops = (double)grid * (block / 32) * (double)iters * PROBE_ACC * 512.0;
    return rc;
}

}  // namespace bmlsp2
