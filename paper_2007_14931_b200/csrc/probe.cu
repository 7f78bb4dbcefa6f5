// probe.cu — FP64 throughput probes for the roofline denominators (MEASURED_PEAKS.json has no FP64
// entry).  kind 0: register-resident DFMA chains (8 independent chains per thread); kind 1: mma.sync
// m8n8k4 f64 chains (8 independent accumulator tiles per warp).  Not on the hot path.
// probe_hbm_read: the streaming kernels' own access pattern with the arithmetic taken out — the ceiling k_stream's
// achieved GB/s is to be read against, next to the copy figure of MEASURED_PEAKS.json.
#include "stream_core.cuh"

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
    const int grid = sm_count() * 8, block = 256;
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

// k_stream's tile pipeline (stream.cu) without the model: a persistent grid of 2 CTAs per SM, one elected thread
// streaming 512-event blocks of NCOL_ALL + 1 columns (184 B per event, the normalisation cache) into shared memory as two
// TMA bulk regions with one mbarrier each, a region refilled as soon as every thread has taken its two events
// of each column into registers.  One DADD per loaded double keeps the loads alive.
__global__ void __launch_bounds__(THREADS, 2) k_probe_read(const double* __restrict__ buf, long long ntiles, double* sink) {
    extern __shared__ __align__(128) unsigned char smem_raw[];
    double* stage = reinterpret_cast<double*>(smem_raw);   // [NCOL_ALL + 1][TILE]
    __shared__ uint64_t full[2];
    const int ncolw = NCOL_ALL + 1;
    if (threadIdx.x == 0) {
        mbar_init(&full[0], 1);
        mbar_init(&full[1], 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();
    if (threadIdx.x == 0 && (long long)blockIdx.x < ntiles) {
        issue_cols(buf, ncolw, blockIdx.x, stage, &full[0], 0, NCOL_K, true);
        issue_cols(buf, ncolw, blockIdx.x, stage, &full[1], NCOL_K, NCOL_ALL, false);
    }
    double acc = 0.0;
    uint32_t parity = 0;
    for (long long tile = blockIdx.x; tile < ntiles; tile += gridDim.x, parity ^= 1) {
        const bool has_next = tile + gridDim.x < ntiles;
        mbar_wait(&full[0], parity);
#pragma unroll
        for (int c = 0; c < NCOL_K; ++c) { const Ev v = load_col(stage, c); acc += v.v[0] + v.v[E - 1]; }
        { const Ev v = load_col(stage, NCOL_ALL); acc += v.v[0] + v.v[E - 1]; }
        __syncthreads();
        if (threadIdx.x == 0 && has_next) issue_cols(buf, ncolw, tile + gridDim.x, stage, &full[0], 0, NCOL_K, true);
        mbar_wait(&full[1], parity);
#pragma unroll
        for (int c = NCOL_K; c < NCOL_ALL; ++c) { const Ev v = load_col(stage, c); acc += v.v[0] + v.v[E - 1]; }
        __syncthreads();
        if (threadIdx.x == 0 && has_next) issue_cols(buf, ncolw, tile + gridDim.x, stage, &full[1], NCOL_K, NCOL_ALL, false);
    }
    if (acc == 123.456) sink[0] = acc;
}

cudaError_t probe_hbm_read(long long bytes, double* gbs, cudaStream_t s) {
    *gbs = 0.0;
    const size_t tile_bytes = (size_t)(NCOL_ALL + 1) * TILE * sizeof(double);
    const long long ntiles = bytes / (long long)tile_bytes;
    if (ntiles < 1) return cudaErrorInvalidValue;
    double* buf = nullptr;
    cudaError_t e = cudaMalloc(&buf, (size_t)ntiles * tile_bytes + 8);
    if (e != cudaSuccess) return e;
    double* sink = buf + (size_t)ntiles * tile_bytes / sizeof(double);
    e = cudaMemsetAsync(buf, 0, (size_t)ntiles * tile_bytes + 8, s);
    if (e == cudaSuccess) e = cudaFuncSetAttribute(k_probe_read, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)tile_bytes);
    const int sms = sm_count();
    cudaEvent_t t0, t1;
    cudaEventCreate(&t0);
    cudaEventCreate(&t1);
    const int grid = (int)(ntiles < 2LL * sms ? ntiles : 2LL * sms);
    double best = 0;
    for (int rep = 0; rep < 6 && e == cudaSuccess; ++rep) {   // rep 0 is warm-up
        cudaEventRecord(t0, s);
        k_probe_read<<<grid, THREADS, tile_bytes, s>>>(buf, ntiles, sink);
        cudaEventRecord(t1, s);
        e = cudaEventSynchronize(t1);
        if (e != cudaSuccess) break;
        float ms = 0;
        cudaEventElapsedTime(&ms, t0, t1);
        const double g = (double)ntiles * tile_bytes / (ms * 1e-3) / 1e9;
        if (rep && g > best) best = g;
    }
    cudaEventDestroy(t0);
    cudaEventDestroy(t1);
    cudaFree(buf);
    if (e == cudaSuccess) e = cudaGetLastError();
    *gbs = best;
    return e;
}

}  // namespace amp
