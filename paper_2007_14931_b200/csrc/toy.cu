// toy.cu — accept-reject toy generator ("a distribution according to the fit model is generated
// through MC techniques").  DESIGN.md "Toy generator" states the method; in short, for candidate number i:
//   twelve words of Philox4x32-10 (counter (i lo, i hi, j, 0), key = seed, j = 0..2) -> five 53-bit uniforms ->
//   x = (m_lo + (m_hi - m_lo) U0, (2 U1 - 1) c_max, (2 U2 - 1) c_max, (2 U3 - 1) pi),  accepted iff  U4 f_max < p_B q S(x).
// The model density S comes from the same kinematics and streaming kernels as the likelihood (api.cu runs them on the candidate
// block); this file holds the three steps around them: draw the candidates, count the accepted ones per block, and compact
// them IN CANDIDATE ORDER (block counts -> exclusive scan -> scatter), so that the toy does not depend on scheduling.
// Every product / sum of the candidate map is a single rounded FP64 operation (__dmul_rn / __dadd_rn: no FMA contraction):
// the candidate stream is bit-reproducible by any implementation of the recipe.
#include "amp_internal.cuh"

namespace amp {

namespace {

constexpr int TOY_THREADS = 256;
constexpr int TOY_SLABS = 4;                             // a block owns TOY_SLABS consecutive slabs of TOY_THREADS candidates
constexpr int TOY_BLOCK = TOY_THREADS * TOY_SLABS;

__device__ __forceinline__ uint4 philox4x32_10(uint4 c, uint2 k) {
    constexpr unsigned M0 = 0xD2511F53u, M1 = 0xCD9E8D57u, W0 = 0x9E3779B9u, W1 = 0xBB67AE85u;
#pragma unroll
    for (int r = 0; r < 10; ++r) {
        const unsigned hi0 = __umulhi(M0, c.x), lo0 = M0 * c.x;
        const unsigned hi1 = __umulhi(M1, c.z), lo1 = M1 * c.z;
        c = make_uint4(hi1 ^ c.y ^ k.x, lo1, hi0 ^ c.w ^ k.y, lo0);
        k.x += W0;
        k.y += W1;
    }
    return c;
}

__device__ __forceinline__ double uniform53(unsigned a, unsigned b) {
    return __dmul_rn(__dadd_rn(__dmul_rn((double)(a >> 5), 67108864.0), (double)(b >> 6)), 1.0 / 9007199254740992.0);
}

__global__ void __launch_bounds__(TOY_THREADS) k_toy_candidates(const ToyArgs t) {
    const uint2 key = make_uint2((unsigned)(t.seed & 0xffffffffull), (unsigned)(t.seed >> 32));
    for (long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x; i < t.n; i += (long long)gridDim.x * blockDim.x) {
        const unsigned long long c = t.first + (unsigned long long)i;
        const unsigned lo = (unsigned)(c & 0xffffffffull), hi = (unsigned)(c >> 32);
        const uint4 w0 = philox4x32_10(make_uint4(lo, hi, 0u, 0u), key);
        const uint4 w1 = philox4x32_10(make_uint4(lo, hi, 1u, 0u), key);
        const uint4 w2 = philox4x32_10(make_uint4(lo, hi, 2u, 0u), key);
        const double U0 = uniform53(w0.x, w0.y), U1 = uniform53(w0.z, w0.w), U2 = uniform53(w1.x, w1.y), U3 = uniform53(w1.z, w1.w);
        t.x[i] = __dadd_rn(t.m_lo, __dmul_rn(t.m_span, U0));
        t.x[t.n + i] = __dmul_rn(__dadd_rn(__dmul_rn(2.0, U1), -1.0), t.cos_max);
        t.x[2 * t.n + i] = __dmul_rn(__dadd_rn(__dmul_rn(2.0, U2), -1.0), t.cos_max);
        t.x[3 * t.n + i] = __dmul_rn(__dadd_rn(__dmul_rn(2.0, U3), -1.0), 3.14159265358979323846);
        t.u[i] = uniform53(w2.x, w2.y);
    }
}

// f = p_B q S of candidate i (S from the streaming kernel, p_B and q from the kinematics cache) and the decision
__device__ __forceinline__ bool toy_accept(const ToyArgs& t, long long i, double* f_out) {
    if (i >= t.n) { *f_out = 0.0; return false; }
    const double q = t.cache[cache_idx(t.ncolw, C_Q, i)], pB = t.cache[cache_idx(t.ncolw, C_PB, i)];
    const double f = pB * q * t.S[i];
    *f_out = f;
    return __dmul_rn(t.u[i], t.f_max) < f;
}

__global__ void __launch_bounds__(TOY_THREADS) k_toy_count(const ToyArgs t) {
    const long long base = (long long)blockIdx.x * TOY_BLOCK;
    int total = 0;
    double fm = 0.0;
    bool bad = false;
    for (int sl = 0; sl < TOY_SLABS; ++sl) {
        double f;
        const bool acc = toy_accept(t, base + sl * TOY_THREADS + threadIdx.x, &f);
        bad |= !(f >= 0.0) || !isfinite(f);
        fm = fmax(fm, f);
        total += __syncthreads_count(acc);
    }
    if (threadIdx.x == 0) t.count[blockIdx.x] = total;
#pragma unroll
    for (int o = 16; o; o >>= 1) fm = fmax(fm, __shfl_xor_sync(0xffffffffu, fm, o));
    if ((threadIdx.x & 31) == 0 && fm > 0.0) atomicMax(t.f_seen, (unsigned long long)__double_as_longlong(fm));   // f >= 0: bit order = value order
    if (bad) atomicOr(t.flag, 2);
}

// exclusive scan of the block counts (in place) by one CTA; count[nb] receives the total.  nb <= 4 * 1024.
__global__ void __launch_bounds__(1024) k_toy_scan(int* __restrict__ count, int nb) {
    __shared__ int warp_tot[32];
    const int t = threadIdx.x, lane = t & 31, wp = t >> 5;
    int v[4], own = 0;
#pragma unroll
    for (int j = 0; j < 4; ++j) { const int k = 4 * t + j; v[j] = k < nb ? count[k] : 0; own += v[j]; }
    int incl = own;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) { const int y = __shfl_up_sync(0xffffffffu, incl, o); if (lane >= o) incl += y; }
    if (lane == 31) warp_tot[wp] = incl;
    __syncthreads();
    if (wp == 0) {
        int w = warp_tot[lane], wi = w;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) { const int y = __shfl_up_sync(0xffffffffu, wi, o); if (lane >= o) wi += y; }
        warp_tot[lane] = wi - w;
        if (lane == 31) count[nb] = wi;
    }
    __syncthreads();
    int run = warp_tot[wp] + incl - own;
#pragma unroll
    for (int j = 0; j < 4; ++j) { const int k = 4 * t + j; if (k < nb) count[k] = run; run += v[j]; }
}

__global__ void __launch_bounds__(TOY_THREADS) k_toy_scatter(const ToyArgs t) {
    __shared__ int wcount[TOY_THREADS / 32];
    const long long base = (long long)blockIdx.x * TOY_BLOCK;
    const int lane = threadIdx.x & 31, wp = threadIdx.x >> 5;
    long long run = t.out_base + t.count[blockIdx.x];
    for (int sl = 0; sl < TOY_SLABS; ++sl) {
        const long long i = base + sl * TOY_THREADS + threadIdx.x;
        double f;
        const bool acc = toy_accept(t, i, &f);
        const unsigned b = __ballot_sync(0xffffffffu, acc);
        if (lane == 0) wcount[wp] = __popc(b);
        __syncthreads();
        int before = 0, slab = 0;
#pragma unroll
        for (int w = 0; w < TOY_THREADS / 32; ++w) { const int c = wcount[w]; before += w < wp ? c : 0; slab += c; }
        const long long dst = run + before + __popc(b & ((1u << lane) - 1u));
        if (acc && dst < t.capacity) {
#pragma unroll
            for (int c = 0; c < 4; ++c) t.x_out[c * t.capacity + dst] = t.x[c * t.n + i];
            if (t.index_out) t.index_out[dst] = (long long)(t.first + (unsigned long long)i);
        }
        run += slab;
        __syncthreads();
    }
}

}  // namespace

int toy_blocks(long long n) { return (int)((n + TOY_BLOCK - 1) / TOY_BLOCK); }

cudaError_t launch_toy_candidates(const ToyArgs& t, cudaStream_t s) {
    const long long blocks = (t.n + TOY_THREADS - 1) / TOY_THREADS;
    k_toy_candidates<<<(int)(blocks < sm_count() * 8 ? (blocks < 1 ? 1 : blocks) : sm_count() * 8), TOY_THREADS, 0, s>>>(t);
    return cudaGetLastError();
}

cudaError_t launch_toy_select(const ToyArgs& t, cudaStream_t s) {
    const int nb = toy_blocks(t.n);
    if (nb < 1 || nb > 4096) return cudaErrorInvalidValue;
    k_toy_count<<<nb, TOY_THREADS, 0, s>>>(t);
    k_toy_scan<<<1, 1024, 0, s>>>(t.count, nb);
    k_toy_scatter<<<nb, TOY_THREADS, 0, s>>>(t);
    return cudaGetLastError();
}

}  // namespace amp
