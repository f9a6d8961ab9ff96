// Self test that backs the fp64 peak used by bench.py's roofline_alu: a kernel of independent DFMA
// chains, timed with CUDA events.  Not part of the hot path.
#include "gp_internal.h"

namespace gp {

// 8 independent chains of dependent DFMAs per thread: enough instruction-level parallelism, together with the
// resident warps, to keep the fp64 pipe issuing every cycle it can.
__global__ void __launch_bounds__(256)
k_dfma_rate(int iters, double seed, double* __restrict__ sink) {
    double a[8];
#pragma unroll
    for (int q = 0; q < 8; ++q) a[q] = seed + q + threadIdx.x * 1e-3;
    const double m = 1.0 - 1e-9, c = 1e-9;
    for (int i = 0; i < iters; ++i) {
#pragma unroll
        for (int u = 0; u < 8; ++u) {
#pragma unroll
            for (int q = 0; q < 8; ++q) a[q] = fma(a[q], m, c);
        }
    }
    double s = 0.0;
#pragma unroll
    for (int q = 0; q < 8; ++q) s += a[q];
    if (s == 12345.678) sink[0] = s;      // never true; keeps the chains alive
}

int fp64_rate_selftest(double* thread_inst_per_s, double* ms_out) {
    int dev = 0, sms = 0;
    GP_CUDA(cudaGetDevice(&dev));
    GP_CUDA(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev));
    double* sink = nullptr;
    GP_CUDA(cudaMalloc(&sink, sizeof(double)));
    cudaEvent_t e0, e1;
    GP_CUDA(cudaEventCreate(&e0));
    GP_CUDA(cudaEventCreate(&e1));
    const int blocks = sms * 8, threads = 256, iters = 4096;
    k_dfma_rate<<<blocks, threads>>>(64, 1.0, sink);            // warm-up
    float best = 1e30f;
    for (int rep = 0; rep < 5; ++rep) {
        cudaEventRecord(e0);
        k_dfma_rate<<<blocks, threads>>>(iters, 1.0 + rep, sink);
        cudaEventRecord(e1);
        cudaError_t e = cudaEventSynchronize(e1);
        if (e != cudaSuccess) { cudaFree(sink); GP_CUDA(e); }
        float ms = 0.f;
        cudaEventElapsedTime(&ms, e0, e1);
        if (ms < best) best = ms;
    }
    cudaEventDestroy(e0);
    cudaEventDestroy(e1);
    cudaFree(sink);
    const double inst = (double)blocks * threads * 64.0 * iters;   // 8 chains x 8 unrolled DFMAs per iteration
    *thread_inst_per_s = inst / (best * 1e-3);
    if (ms_out) *ms_out = best;
    return GP_OK;
}

}  // namespace gp
