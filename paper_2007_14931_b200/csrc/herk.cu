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

// CTAs per SM: a CTA alternates between building a basis tile (plain ALUs) and multiplying it (tensor pipe) with a barrier in
// between, so two resident CTAs keep the tensor pipe fed while the other one builds (the tile's shared memory is ~80 KB)
constexpr int HERK_MINB = 2;
constexpr int HERK_MAXRUN = 12;   // runs per warp; a run = one row tile I with two column tiles J0, J1 (3 fragment loads, 2 DMMA)

__device__ __forceinline__ double lds_f64(uint32_t addr) {
    double v;
    asm volatile("ld.shared.f64 %0, [%1];" : "=d"(v) : "r"(addr));
    return v;
}

// The basis tile is built with every event scaled by sqrt(w_j), so G' = sum_j (sqrt(w) b')(sqrt(w) b')^T needs no
// per-fragment weight and both MMA operands are plain fragment loads of the same tile.
template <int NRUN>
__global__ void __launch_bounds__(BT_THREADS, (NRUN <= 4 ? HERK_MINB : 1)) k_herk(const __grid_constant__ HerkArgs h) {
    extern __shared__ __align__(16) double smem[];
    const BatchArgs& a = h.b;
    const int KP = a.nent * 2;   // realified rows, multiple of 8
    const TileSmem t = carve_tile_smem(smem, KP, a.ncolu);
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int nang = a.have_z ? BT_NANG : 6;

    double acc[NRUN][2][2];
    uint32_t offA[NRUN], offB[NRUN][2];   // byte offsets of the fragments' row tiles inside one helicity plane
    int outidx[NRUN][2];                  // tile index in the partial buffer, -1: padding
#pragma unroll
    for (int r = 0; r < NRUN; ++r) {
        const int4 run = h.runs[warp * NRUN + r];   // (I, J0, J1, flags: bit0 J0 real, bit1 J1 real) ; outs in runs_out
        const int2 ro = h.runs_out[warp * NRUN + r];
        offA[r] = (uint32_t)(8 * run.x * BT_STRIDE * sizeof(double));
        offB[r][0] = (uint32_t)(8 * run.y * BT_STRIDE * sizeof(double));
        offB[r][1] = (uint32_t)(8 * run.z * BT_STRIDE * sizeof(double));
        outidx[r][0] = ro.x; outidx[r][1] = ro.y;
        acc[r][0][0] = acc[r][0][1] = acc[r][1][0] = acc[r][1][1] = 0.0;
    }

    const long long ntiles = (a.n + BT_EVENTS - 1) / BT_EVENTS;
    if (tid == 0) {
        bmbar_init(t.full, 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    stage_tile_entries(a, t);
    __syncthreads();
    if (tid == 0 && (long long)blockIdx.x < ntiles) issue_stage(a, blockIdx.x, t.scol, t.sang, t.sw, t.full, nang, true);
    uint32_t parity = 0;
    const uint32_t bs32 = bsmem_u32(t.Bs) + (uint32_t)(((lane >> 2) * BT_STRIDE + (lane & 3)) * sizeof(double));
    for (long long tile = blockIdx.x; tile < ntiles; tile += gridDim.x, parity ^= 1) {
        bmbar_wait(t.full, parity);
        build_basis_tile(a, t, tile, KP, true, true);
        __syncthreads();   // basis tile complete, staging consumed: stream the next tile in during the DMMA phase
        if (tid == 0 && tile + gridDim.x < ntiles) issue_stage(a, tile + gridDim.x, t.scol, t.sang, t.sw, t.full, nang, true);
#pragma unroll 1
        for (int xi = 0; xi < 2; ++xi) {
#pragma unroll 4   // fragment loads of the next steps issue under the DMMAs of this one (4.2 -> 3.9 ms for K = 27 at 10M events)
            for (int ks = 0; ks < BT_EVENTS / 4; ++ks) {
                // fragment element of this lane: basis row (tile row lane/4), event 4 ks + lane%4
                const uint32_t fb = bs32 + (uint32_t)((xi * KP * BT_STRIDE + 4 * ks) * sizeof(double));
#pragma unroll
                for (int r = 0; r < NRUN; ++r) {
                    const double af = lds_f64(fb + offA[r]);
                    const double b0 = lds_f64(fb + offB[r][0]), b1 = lds_f64(fb + offB[r][1]);
                    dmma884(acc[r][0], af, b0);
                    dmma884(acc[r][1], af, b1);
                }
            }
        }
        __syncthreads();
    }
#pragma unroll
    for (int r = 0; r < NRUN; ++r)
#pragma unroll
        for (int c = 0; c < 2; ++c)
            if (outidx[r][c] >= 0) {
                double* o = h.partial + ((size_t)blockIdx.x * h.ntile + outidx[r][c]) * 64 + 2 * lane;   // C fragment: row lane/4, columns 2 (lane%4) + {0,1}
                o[0] = acc[r][c][0];
                o[1] = acc[r][c][1];
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

int herk_max_runs() { return HERK_MAXRUN; }

// persistent grid: as many CTAs per SM as the basis tile's shared memory allows, at most HERK_MINB
int herk_grid(long long n, int nent, int ncolu) {
    const long long ntiles = (n + BT_EVENTS - 1) / BT_EVENTS;
    long long per_sm = (long long)((224 * 1024) / (tile_smem_bytes(nent, ncolu) + 1024));
    if (per_sm > HERK_MINB) per_sm = HERK_MINB;
    if (per_sm < 1) per_sm = 1;
    const long long cap = (long long)sm_count() * per_sm;
    return (int)(ntiles < 1 ? 1 : (ntiles > cap ? cap : ntiles));
}
int herk_grid_max() { return sm_count() * HERK_MINB; }

template <int NRUN>
static cudaError_t launch_herk_n(const HerkArgs& h, int grid, cudaStream_t s) {
    static DeviceOnce attr_done;
    cudaError_t e = cudaSuccess;
    if (attr_done.first()) { e = cudaFuncSetAttribute(k_herk<NRUN>, cudaFuncAttributeMaxDynamicSharedMemorySize, 224 * 1024); }
    if (e != cudaSuccess) return e;
    k_herk<NRUN><<<grid, BT_THREADS, tile_smem_bytes(h.b.nent, h.b.ncolu), s>>>(h);
    return cudaGetLastError();
}

// h.nrun = runs per warp (the host pads every warp's list to this length)
cudaError_t launch_herk(const HerkArgs& h, int grid, cudaStream_t s) {
    switch (h.nrun) {
        case 1: case 2: return launch_herk_n<2>(h, grid, s);
        case 3: case 4: return launch_herk_n<4>(h, grid, s);
        case 5: case 6: return launch_herk_n<6>(h, grid, s);
        case 7: case 8: return launch_herk_n<8>(h, grid, s);
        case 9: case 10: return launch_herk_n<10>(h, grid, s);
        case 11: case 12: return launch_herk_n<12>(h, grid, s);
    }
    return cudaErrorInvalidValue;
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
