// probe.cu — FP64 throughput probes for the roofline denominators (MEASURED_PEAKS.json has no FP64
// entry).  kind 0: register-resident DFMA chains (8 independent chains per thread); kind 1: mma.sync
// m8n8k4 f64 chains (8 independent accumulator tiles per warp).  Not on the hot path.
#include "amp_internal.cuh"

namespace amp {

__global__ void __launch_bounds__(256) k_probe_dfma(int iters, double* sink) {
    double a0 = threadIdx.x * 1e-9, a1 = a0 + 1, a2 = a0 + 2, a3 = a0 + 3, a4 = a0 + 4, a5 = a0 + 5, a6 = a0 + 6, a7 = a0 + 7;
    const double b = 1.0 + 1e-12, c = 1e-13;
    for (int i = 0; i < iters; ++i) {
#pragma unroll
        for (int u = 0; u < 8; ++u) {
            a0 = fma(a0, b, c); a1 = fma(a1, b, c); a2 = fma(a2, b, c); a3 = fma(a3, b, c);
            a4 = fma(a4, b, c); a5 = fma(a5, b, c); a6 = fma(a6, b, c); a7 = fma(a7, b, c);
        }
    }
    const double s = a0 + a1 + a2 + a3 + a4 + a5 + a6 + a7;
    if (s == 123.456) sink[0] = s;
}

__device__ __forceinline__ void dmma884(double& d0, double& d1, double a, double b) {
    asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};\n" : "+d"(d0), "+d"(d1) : "d"(a), "d"(b));
}

__global__ void __launch_bounds__(256) k_probe_dmma(int iters, double* sink) {
    double acc[8][2];
#pragma unroll
    for (int t = 0; t < 8; ++t) acc[t][0] = acc[t][1] = 0.0;
    const double a = 1.0 + threadIdx.x * 1e-9, b = 1e-9;
    for (int i = 0; i < iters; ++i) {
#pragma unroll
        for (int u = 0; u < 4; ++u)
#pragma unroll
            for (int t = 0; t < 8; ++t) dmma884(acc[t][0], acc[t][1], a, b);
    }
    double s = 0;
#pragma unroll
    for (int t = 0; t < 8; ++t) s += acc[t][0] + acc[t][1];
    if (s == 123.456) sink[0] = s;
}

cudaError_t probe_fp64(int kind, int iters, double* flops, cudaStream_t s) {
    double* sink = nullptr;
    cudaError_t e = cudaMalloc(&sink, 8);
    if (e != cudaSuccess) return e;
    cudaEvent_t t0, t1;
    cudaEventCreate(&t0);
    cudaEventCreate(&t1);
    const int grid = 148 * 8, block = 256;
    double best = 0;
    for (int rep = 0; rep < 4; ++rep) {   // rep 0 is warm-up
        cudaEventRecord(t0, s);
        if (kind == 0) k_probe_dfma<<<grid, block, 0, s>>>(iters, sink);
        else k_probe_dmma<<<grid, block, 0, s>>>(iters, sink);
        cudaEventRecord(t1, s);
        e = cudaEventSynchronize(t1);
        if (e != cudaSuccess) break;
        float ms = 0;
        cudaEventElapsedTime(&ms, t0, t1);
        // flops: DFMA: 64 fma/thread/iter; DMMA: 32 mma/warp/iter x 8*8*4 fma
        const double fl = (kind == 0) ? 2.0 * 64.0 * iters * (double)grid * block : 2.0 * 32.0 * 256.0 * iters * (double)grid * (block / 32);
        const double f = fl / (ms * 1e-3);
        if (rep && f > best) best = f;
    }
    cudaEventDestroy(t0);
    cudaEventDestroy(t1);
    cudaFree(sink);
    if (e == cudaSuccess) e = cudaGetLastError();
    *flops = best;
    return e;
}

}  // namespace amp
