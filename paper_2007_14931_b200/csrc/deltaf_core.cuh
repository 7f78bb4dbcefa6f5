// deltaf_core.cuh — what the two gradient-batch kernels of the paper's resonance lists share (deltaf.cu: data events, and the
// normalisation events when it runs alone; deltan.cu: normalisation events): the value layout of a model shape, the class-wise
// forward pass, and the per-warp shared-memory tile that sums values over a warp's 32 events.  See deltaf.cu for the method.
#pragma once
#define AMP_STREAM_E 2
#define AMP_STREAM_THREADS 256
#define AMP_STREAM_MINB 1
#include <type_traits>

#include "stream_core.cuh"

namespace amp {

namespace {

constexpr int UNIT = THREADS;   // events per pipeline unit (half a cache block)
constexpr int UPB = CACHE_TILE / UNIT;       // units per cache block
static_assert(UPB * UNIT == CACHE_TILE, "whole units per cache block");

__device__ __forceinline__ void mbar_arrive(uint64_t* bar) {
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(smem_u32(bar)) : "memory");
}

template <class SH>
struct DLay {
    static constexpr int NENT = SH::oz + SH::nz;                        // Breit-Wigner entries, spin-class order
    static constexpr int NSLOT = SH::n0 + 3 * (NENT - SH::n0);          // single-slot coupling positions
    static constexpr int NPOS = NSLOT + SH::nz;                         // + one tied-pair position per Z
    static constexpr int NVAL = 4 * (NPOS + NENT);                      // value slots: 4 per coupling position, then 4 per entry (lineshape points)
    static constexpr int NCH = (NVAL / 4 + 1) / 2;                      // chunks of eight values (two quads)
    __host__ __device__ static constexpr int base(int t) { return t < SH::n0 ? t : SH::n0 + 3 * (t - SH::n0); }
};
static_assert(DLay<Shape<3, 3, 2, 1, 1, 2>>::NPOS <= DELTAF_MAX_POS && DLay<Shape<3, 3, 2, 1, 1, 2>>::NENT <= DELTAF_MAX_ENT, "tables of DeltaFArgs");

// lineshapes of one spin class: U_l += c BW (couplings carry kN); the class's barrier factors are kept for the values pass
template <int J, int LRv, int LBv, int CNT, int OFF, int SPIN>
__device__ __forceinline__ void class_forward(const StreamArgs& a, double m2, double invm, double pR, double pB, double& F, double& G,
                                              double2& Um, double2& U0, double2& Up) {
    group_factors<LRv, LBv>(a.r2_spin[SPIN], invm, pR, pB, &F, &G);
#pragma unroll
    for (int t = 0; t < CNT; ++t) {
        const ResEntry& en = a.ent[OFF + t];
        const double2 bw = bw_unscaled(en, m2, F, G);
        U0 = cfma(en.c0, bw, U0);
        if (J) { Um = cfma(en.cm, bw, Um); Up = cfma(en.cp, bw, Up); }
    }
}

// conj(bw) x
__device__ __forceinline__ double2 conj_mul(double2 bw, double2 x) {
    return make_double2(fma(bw.x, x.x, bw.y * x.y), fma(bw.x, x.y, -bw.y * x.x));
}

// The values of one event-row (32 events of a warp, one per lane) are summed over the events through a per-warp shared-memory
// tile, eight values (two quads) at a time: lane e stores its value v at [v][e] (row stride 256 B: conflict-free), and lane l
// reads the eight events 8 g .. 8 g + 7 of value v = l % 8 as four 16-byte loads and folds them into its accumulator of the
// chunk (a register; NORM: sum, DATA: product of r ~ 1).  So that a quarter-warp's 16-byte loads hit eight different banks
// although every row starts at bank 0, lanes with v >= 4 take the next event group (g = (l / 8 + v / 4) % 4) and every lane
// walks its four slots rotated by v.  Per value this is one store, half a load and one FP64 operation (the exchange tree of
// selects and shuffles it replaces took ~8 instructions per value); the order of the sums is fixed, so the result is
// reproducible.  q (quads pushed so far) only ever changes by constants in straight-line code: every test on it is resolved at
// compile time.
constexpr int TILE_ROW_BYTES = 32 * 8;
constexpr int TILE_BYTES = 8 * TILE_ROW_BYTES;   // per warp
template <bool NORM, int NCH>
struct Tile {
    uint32_t wr;              // shared-space address of [0][lane]
    uint32_t rd[4];           // ... of the four 16-byte slots this lane reads
    double x[8];              // the eight values of the chunk whose loads are under way
    int q;
    double* acc;              // [NCH] the lane's chunk accumulators (registers of the kernel, shared by the two phases)
    __device__ __forceinline__ void init(uint32_t tile, int lane) {
        const int v = lane & 7, g = ((lane >> 3) + (v >> 2)) & 3;
        wr = tile + lane * 8;
#pragma unroll
        for (int i = 0; i < 4; ++i) rd[i] = tile + v * TILE_ROW_BYTES + g * 64 + ((i + v) & 3) * 16;
    }
    __device__ __forceinline__ void reset_event() { q = 0; }
    __device__ __forceinline__ void push4(double y0, double y1, double y2, double y3) {
        const uint32_t w = wr + (q & 1) * 4 * TILE_ROW_BYTES;
        asm volatile("st.shared.f64 [%0], %1;" ::"r"(w), "d"(y0) : "memory");
        asm volatile("st.shared.f64 [%0+256], %1;" ::"r"(w), "d"(y1) : "memory");
        asm volatile("st.shared.f64 [%0+512], %1;" ::"r"(w), "d"(y2) : "memory");
        asm volatile("st.shared.f64 [%0+768], %1;" ::"r"(w), "d"(y3) : "memory");
        if (q & 1) load();             // the chunk is complete: its loads are issued now and used one quad later
        else if (q > 0) fold(q / 2 - 1);
        ++q;
    }
    // the three sums of a coupling position on the normalisation side (the fourth value of the quad is zero)
    __device__ __forceinline__ void push3(double y0, double y1, double y2) { push4(y0, y1, y2, 0.0); }
    // a quad that is not in use: neutral values
    __device__ __forceinline__ void push_identity() { const double id = NORM ? 0.0 : 1.0; push4(id, id, id, id); }
    // A warp's shared-memory accesses are performed in program order, so the stores of the next quad (rows 0-3 again) cannot
    // overtake these loads; the four loads are one statement so that they get four register pairs and issue back to back.
    __device__ __forceinline__ void load() {
        __syncwarp();
        asm volatile(
            "ld.shared.v2.f64 {%0, %1}, [%8];\n\t"
            "ld.shared.v2.f64 {%2, %3}, [%9];\n\t"
            "ld.shared.v2.f64 {%4, %5}, [%10];\n\t"
            "ld.shared.v2.f64 {%6, %7}, [%11];"
            : "=d"(x[0]), "=d"(x[1]), "=d"(x[2]), "=d"(x[3]), "=d"(x[4]), "=d"(x[5]), "=d"(x[6]), "=d"(x[7])
            : "r"(rd[0]), "r"(rd[1]), "r"(rd[2]), "r"(rd[3])
            : "memory");
        __syncwarp();
    }
    __device__ __forceinline__ void fold(int c) {
#pragma unroll
        for (int cc = 0; cc < NCH; ++cc)
            if (cc == c) {
                if (NORM) acc[cc] += ((x[0] + x[1]) + (x[2] + x[3])) + ((x[4] + x[5]) + (x[6] + x[7]));
                else acc[cc] *= ((x[0] * x[1]) * (x[2] * x[3])) * ((x[4] * x[5]) * (x[6] * x[7]));   // r in [0.5, 1.5]: renormalised every 16 units
            }
    }
    __device__ __forceinline__ void pad_block() {   // complete the last chunk with neutral values and take in the loads still under way
        if (q & 1) push_identity();
        fold(q / 2 - 1);
    }
};

}  // namespace

}  // namespace amp
