// stream_core.cuh — pieces shared by the streaming kernels (stream.cu: one parameter point; delta.cu: gradient batches):
// the two-events-per-thread register layout, the TMA bulk-copy tile pipeline, the per-spin coherent sums with
// lineshapes evaluated in registers, the model-shape specialisation and the fixed-order block reductions.
#pragma once
#include "amp_internal.cuh"

namespace amp {

// E consecutive events per thread: each cache column is read with one 16-byte (E = 2) load per thread
// (a warp covers 512 contiguous bytes), the group / resonance constants and couplings are fetched once
// for E events, and the E independent dependency chains give the FP64 pipe instruction-level parallelism.
#ifndef AMP_STREAM_E
#define AMP_STREAM_E 2
#endif
#ifndef AMP_STREAM_MINB
#define AMP_STREAM_MINB 2
#endif
constexpr int E = AMP_STREAM_E;

#ifndef AMP_STREAM_THREADS
#define AMP_STREAM_THREADS 256
#endif
constexpr int THREADS = AMP_STREAM_THREADS;
constexpr int NWARPS = THREADS / 32;
constexpr int TILE = THREADS * E;          // events per pipeline stage

struct Ev {   // per-thread event registers
    double v[E];
};
// The E events of this thread from column c of a staged tile (shared memory, [column][TILE] doubles):
// consecutive threads read consecutive 16-byte words — conflict-free.
__device__ __forceinline__ Ev load_col(const double* __restrict__ stage, int c) {
    Ev r;
    const double* p = stage + c * TILE + threadIdx.x * E;
    if (E == 2) {
        const double2 t = *reinterpret_cast<const double2*>(p);
        r.v[0] = t.x; r.v[E - 1] = t.y;
    } else {
#pragma unroll
        for (int e = 0; e < E; ++e) r.v[e] = p[e];
    }
    return r;
}

// ---- TMA bulk-copy pipeline (cp.async.bulk + mbarrier): one elected thread streams whole cache columns of the
// next tile into shared memory while all warps compute on the current one, so no register holds data in flight.
__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(uint64_t* bar, int count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count));
}
__device__ __forceinline__ void mbar_expect_tx(uint64_t* bar, uint32_t bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint64_t* bar, uint32_t parity) {
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "WAIT_%=:\n"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
        "@p bra DONE_%=;\n"
        "bra WAIT_%=;\n"
        "DONE_%=:\n"
        "}\n" ::"r"(smem_u32(bar)), "r"(parity) : "memory");
}
__device__ __forceinline__ void bulk_g2s(void* dst, const void* src, uint32_t bytes, uint64_t* bar) {
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(smem_u32(dst)), "l"(src),
                 "r"(bytes), "r"(smem_u32(bar))
                 : "memory");
}
// Columns [c0, c1) of block `tile` of a tiled cache (and, if with_w, its weight column) -> the same places of the stage.
// The columns of a block are contiguous, so a region is ONE bulk copy (40 KB for the K* chain, 48 KB for the Z chain).
static_assert(TILE == CACHE_TILE, "a streaming tile is one cache block");
__device__ __forceinline__ void issue_cols(const double* cache, int ncolw, long long tile, double* stage, uint64_t* bar, int c0, int c1, bool with_w) {
    const double* blk = cache + (size_t)tile * ncolw * TILE;
    const uint32_t bytes = (uint32_t)(c1 - c0) * TILE * sizeof(double), wbytes = TILE * sizeof(double);
    mbar_expect_tx(bar, bytes + (with_w ? wbytes : 0));
    bulk_g2s(stage + c0 * TILE, blk + c0 * TILE, bytes, bar);
    if (with_w) bulk_g2s(stage + (ncolw - 1) * TILE, blk + (ncolw - 1) * TILE, wbytes, bar);
}
// MODE_FUSED walks one tile space: the data tiles first, then the normalisation tiles (second dataset of StreamArgs).
template <int MODE>
__device__ __forceinline__ void issue_tile(const StreamArgs& a, long long ntd, long long tile, double* stage, uint64_t* bar, int c0, int c1,
                                           bool region_has_w) {
    if (MODE == MODE_FUSED && tile >= ntd)
        issue_cols(a.cache2, a.ncolw, tile - ntd, stage, bar, c0, c1, region_has_w);
    else
        issue_cols(a.cache, a.ncolw, tile, stage, bar, c0, c1, region_has_w && MODE != MODE_DATA && MODE != MODE_FUSED && MODE != MODE_DATA_M);
}

// fixed-order block sum: xor-shuffle tree, then the 8 warp values in warp order; result valid in thread 0
__device__ __forceinline__ double block_sum(double v, double* sm) {
#pragma unroll
    for (int o = 16; o; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    __syncthreads();   // sm may still be read from a previous use
    if ((threadIdx.x & 31) == 0) sm[threadIdx.x >> 5] = v;
    __syncthreads();
    double t = 0.0;
    if (threadIdx.x == 0)
        for (int wv = 0; wv < NWARPS; ++wv) t += sm[wv];
    return t;
}
// sum of the per-CTA partials in the order k_finalize uses (thread t adds b = t, t + 256, ...; fixed tree): every thread calls it
__device__ __forceinline__ double partial_sum(const double* p, int n, double* sm) {
    double v = 0.0;
    for (int b = threadIdx.x; b < n; b += THREADS) v += __ldcg(p + b);
    return block_sum(v, sm);
}

// One resonance: lineshape (from its pool column or in registers) times its couplings, added to U_l.
template <int J>
__device__ __forceinline__ void add_resonance(const StreamArgs& a, const ResEntry& en, long long i0, const Ev& m2, const double (&F)[E],
                                              const double (&G)[E], double2 (&Um)[E], double2 (&U0)[E], double2 (&Up)[E]) {
    double2 bw[E];
    if (en.column >= 0) {
#pragma unroll
        for (int e = 0; e < E; ++e) bw[e] = a.cols[(size_t)en.column * a.npad + i0 + e];
    } else {
#pragma unroll
        for (int e = 0; e < E; ++e) bw[e] = bw_unscaled(en, m2.v[e], F[e], G[e]);   // couplings carry kN
    }
#pragma unroll
    for (int e = 0; e < E; ++e) {
        U0[e] = cfma(en.c0, bw[e], U0[e]);
        if (J) { Um[e] = cfma(en.cm, bw[e], Um[e]); Up[e] = cfma(en.cp, bw[e], Up[e]); }
    }
}

// Partial sums U_l = sum_{R of spin J} c_{R,l} BW_R.  CNT >= 0: the model has exactly CNT resonances of this
// spin, all with one radius, stored at ent[OFF..OFF+CNT): the loop unrolls and every constant becomes an
// immediate constant-bank operand (no index arithmetic, no constant loads).  CNT < 0: generic model, runtime
// loops over the barrier groups [g0, g1).
// SAVE: also store the group factors (F, G) of the thread's E events at fg[g * TILE + e] (delta.cu re-evaluates
// Breit-Wigners of perturbed points from them).
template <int J, int LRv, int LBv, int CNT, int OFF, int SPIN, bool SAVE = false>
__device__ __forceinline__ void spin_sum(const StreamArgs& a, long long i0, const Ev& m2, const Ev& invm, const Ev& pR, const Ev& pB,
                                         double2 (&Um)[E], double2 (&U0)[E], double2 (&Up)[E], double2* fg = nullptr) {
    double F[E], G[E];
    if (CNT >= 0) {
#pragma unroll
        for (int e = 0; e < E; ++e) group_factors<LRv, LBv>(a.r2_spin[SPIN], invm.v[e], pR.v[e], pB.v[e], &F[e], &G[e]);
        if (SAVE) {
#pragma unroll
            for (int e = 0; e < E; ++e) fg[a.gstart[SPIN] * TILE + e] = make_double2(F[e], G[e]);
        }
#pragma unroll
        for (int t = 0; t < CNT; ++t) add_resonance<J>(a, a.ent[OFF + t], i0, m2, F, G, Um, U0, Up);
    } else {
        for (int g = a.gstart[SPIN]; g < a.gstart[SPIN + 1]; ++g) {
            const BarrierGroup grp = a.grp[g];
#pragma unroll
            for (int e = 0; e < E; ++e) group_factors<LRv, LBv>(grp.r2, invm.v[e], pR.v[e], pB.v[e], &F[e], &G[e]);
            if (SAVE) {
#pragma unroll
                for (int e = 0; e < E; ++e) fg[g * TILE + e] = make_double2(F[e], G[e]);
            }
            for (int t = grp.first; t < grp.first + grp.count; ++t) add_resonance<J>(a, a.ent[t], i0, m2, F, G, Um, U0, Up);
        }
    }
}

// Model shape: number of resonances of K* spin 0..4 and of Z's; Generic = runtime loops.
template <int A0, int A1, int A2, int A3, int A4, int AZ, int AL = 0>
struct Shape {
    static constexpr int n0 = A0, n1 = A1, n2 = A2, n3 = A3, n4 = A4, nz = A4 < 0 ? -1 : AZ;
    static constexpr int nl = A4 < 0 ? -1 : AL;   // LASS terms (Eq. 7): 0 = none compiled in, -1 = runtime count
    static constexpr int o1 = A0, o2 = A0 + A1, o3 = o2 + A2, o4 = o3 + A3, oz = o4 + A4;
};
using Generic = Shape<-1, -1, -1, -1, -1, -1>;

}  // namespace amp
