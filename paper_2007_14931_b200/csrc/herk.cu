// herk.cu — step a4: the Hermitian normalisation matrix  M_kl = sum_j w_j sum_xi conj(B_k,xi(j)) B_l,xi(j)  over the
// phase-space Monte Carlo sample, built once per lineshape state by a ZHERK-style kernel on the FP64
// tensor cores, so that the normalisation integral of any parameter point is the quadratic form I(p) = c(p)^H M c(p).
//
// Realified: with b' = (Re B_0, Im B_0, Re B_1, Im B_1, ...) the real Gram matrix G' = sum_j w_j b'(j) b'(j)^T holds
//   Re M_kl = G'[2k][2l] + G'[2k+1][2l+1],   Im M_kl = G'[2k][2l+1] - G'[2k+1][2l].
// G' is cut in 8 x 8 tiles; one mma.sync.m8n8k4.f64 adds four events to a tile (the contraction index is the event),
// both operands are fragments of the same shared-memory basis tile that batch.cu uses.  Only tiles (I <= J) that some
// parameter point needs are computed (for a gradient batch: base x base, base x variant, variant x same variant).
// Each CTA keeps its tiles in registers over all its events and writes one partial per tile; k_herk_reduce adds the
// CTA partials in a fixed order (deterministic), k_gram_expand mirrors the triangle, k_quadform evaluates c^H M c.
#include "tile_basis.cuh"

namespace amp {

constexpr int HERK_MAXT = 24;   // tiles per warp (8 warps -> up to 192 tiles)

__global__ void __launch_bounds__(BT_THREADS, 1) k_herk(const __grid_constant__ HerkArgs h) {
    extern __shared__ __align__(16) double smem[];
    const BatchArgs& a = h.b;
    const int KP = a.nent * 2;   // realified rows, multiple of 8
    const TileSmem t = carve_tile_smem(smem, KP, a.ncolu);
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int nang = a.have_z ? BT_NANG : 6;
    const int t0 = h.tile_start[warp], nt = h.tile_start[warp + 1] - t0;

    double acc[HERK_MAXT][2];
#pragma unroll
    for (int i = 0; i < HERK_MAXT; ++i) acc[i][0] = acc[i][1] = 0.0;

    const long long ntiles = (a.n + BT_EVENTS - 1) / BT_EVENTS;
    if (tid == 0) {
        bmbar_init(t.full, 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();
    if (tid == 0 && (long long)blockIdx.x < ntiles) issue_stage(a, blockIdx.x, t.scol, t.sang, t.sw, t.full, nang, true);
    uint32_t parity = 0;
    for (long long tile = blockIdx.x; tile < ntiles; tile += gridDim.x, parity ^= 1) {
        bmbar_wait(t.full, parity);
        build_basis_tile(a, t, tile, KP, true);
        __syncthreads();   // basis tile complete, staging consumed: stream the next tile in during the DMMA phase
        if (tid == 0 && tile + gridDim.x < ntiles) issue_stage(a, tile + gridDim.x, t.scol, t.sang, t.sw, t.full, nang, true);
#pragma unroll 1
        for (int xi = 0; xi < 2; ++xi) {
#pragma unroll 1
            for (int ks = 0; ks < BT_EVENTS / 4; ++ks) {
                // fragment element of this lane: basis row (tile row lane/4), event 4 ks + lane%4
                const double* fb = t.Bs + (size_t)xi * KP * BT_STRIDE + (size_t)(lane >> 2) * BT_STRIDE + 4 * ks + (lane & 3);
                const double wv = t.ws[4 * ks + (lane & 3)];
                int lastI = -1;
                double afr = 0.0;
#pragma unroll
                for (int i = 0; i < HERK_MAXT; ++i) {
                    if (i < nt) {
                        const int2 c = h.tiles[t0 + i];   // (row tile I, column tile J), sorted by I within a warp
                        if (c.x != lastI) { afr = fb[(size_t)8 * c.x * BT_STRIDE] * wv; lastI = c.x; }
                        const double bfr = fb[(size_t)8 * c.y * BT_STRIDE];
                        dmma884(acc[i], afr, bfr);
                    }
                }
            }
        }
        __syncthreads();
    }
#pragma unroll
    for (int i = 0; i < HERK_MAXT; ++i)
        if (i < nt) {
            double* o = h.partial + ((size_t)blockIdx.x * h.ntile + t0 + i) * 64 + 2 * lane;   // C fragment: row lane/4, columns 2 (lane%4) + {0,1}
            o[0] = acc[i][0];
            o[1] = acc[i][1];
        }
}

// G'[tile][64] = sum over CTAs of partial[cta][tile][64], CTA order fixed
__global__ void __launch_bounds__(64) k_herk_reduce(const double* __restrict__ partial, int ncta, int ntile, double* __restrict__ gt) {
    const int tile = blockIdx.x, e = threadIdx.x;
    double s = 0.0;
    for (int c = 0; c < ncta; ++c) s += partial[((size_t)c * ntile + tile) * 64 + e];
    gt[(size_t)tile * 64 + e] = s;
}

// dense symmetric G'[KP][KP] from the computed upper-triangle tiles (zero elsewhere)
__global__ void __launch_bounds__(64) k_gram_expand(const double* __restrict__ gt, const int2* __restrict__ tiles, int KP, double* __restrict__ G) {
    const int2 c = tiles[blockIdx.x];
    const int r = threadIdx.x >> 3, q = threadIdx.x & 7;
    const double v = gt[(size_t)blockIdx.x * 64 + threadIdx.x];
    G[(size_t)(8 * c.x + r) * KP + 8 * c.y + q] = v;
    if (c.x != c.y) G[(size_t)(8 * c.y + q) * KP + 8 * c.x + r] = v;
}

// out[p] = sum_{e,f} Re( conj(C[p][e]) M_ef C[p][f] ), one block per point, fixed summation order
__global__ void __launch_bounds__(256) k_quadform(const double* __restrict__ G, int KP, const double2* __restrict__ C, int nent,
                                                  double* __restrict__ out) {
    const int p = blockIdx.x;
    const double2* c = C + (size_t)p * nent;
    double s = 0.0;
    for (int idx = threadIdx.x; idx < nent * nent; idx += 256) {
        const int e = idx / nent, f = idx % nent;
        const double2 ce = c[e], cf = c[f];
        if ((ce.x == 0.0 && ce.y == 0.0) || (cf.x == 0.0 && cf.y == 0.0)) continue;
        const double* g = G + (size_t)(2 * e) * KP + 2 * f;
        const double mre = g[0] + g[KP + 1], mim = g[1] - g[KP];
        // Re( conj(ce) (mre + i mim) cf )
        const double tr = mre * cf.x - mim * cf.y, ti = mre * cf.y + mim * cf.x;
        s += ce.x * tr + ce.y * ti;
    }
    __shared__ double sm[8];
#pragma unroll
    for (int o = 16; o; o >>= 1) s += __shfl_xor_sync(0xffffffffu, s, o);
    if ((threadIdx.x & 31) == 0) sm[threadIdx.x >> 5] = s;
    __syncthreads();
    if (threadIdx.x == 0) {
        double tsum = 0.0;
        for (int wv = 0; wv < 8; ++wv) tsum += sm[wv];
        out[p] = tsum;
    }
}

int herk_max_tiles() { return HERK_MAXT * 8; }

cudaError_t launch_herk(const HerkArgs& h, int grid, cudaStream_t s) {
    static bool attr_done = false;
    cudaError_t e = cudaSuccess;
    if (!attr_done) { e = cudaFuncSetAttribute(k_herk, cudaFuncAttributeMaxDynamicSharedMemorySize, 224 * 1024); attr_done = true; }
    if (e != cudaSuccess) return e;
    k_herk<<<grid, BT_THREADS, tile_smem_bytes(h.b.nent, h.b.ncolu), s>>>(h);
    return cudaGetLastError();
}

cudaError_t launch_herk_finish(const double* partial, int ncta, int ntile, const int2* tiles, int KP, double* gt, double* G, cudaStream_t s) {
    cudaError_t e = cudaMemsetAsync(G, 0, sizeof(double) * (size_t)KP * KP, s);
    if (e != cudaSuccess) return e;
    k_herk_reduce<<<ntile, 64, 0, s>>>(partial, ncta, ntile, gt);
    k_gram_expand<<<ntile, 64, 0, s>>>(gt, tiles, KP, G);
    return cudaGetLastError();
}

cudaError_t launch_quadform(const double* G, int KP, const double2* C, int nent, int P, double* out, cudaStream_t s) {
    k_quadform<<<P, 256, 0, s>>>(G, KP, C, nent, out);
    return cudaGetLastError();
}

}  // namespace amp
