// tile_basis.cuh — shared by the two FP64 tensor-core kernels (batch.cu: points x events GEMM; herk.cu: Gram matrix):
// a tile of 64 events is staged by TMA bulk copies (lineshape columns, angular cache columns, weights) and turned
// into the basis tile B[xi][realified entry][event] in shared memory.
#pragma once
#include "amp_internal.cuh"

namespace amp {

constexpr int BT_EVENTS = 64;            // events per tile
constexpr int BT_STRIDE = 68;            // row stride in doubles: = 4 (mod 16) -> conflict-free B-fragment reads
constexpr int BT_THREADS = 256;

__device__ __forceinline__ void dmma884(double (&d)[2], double a, double b) {
    asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};\n" : "+d"(d[0]), "+d"(d[1]) : "d"(a), "d"(b));
}

// TMA bulk copy + mbarrier helpers (same PTX as in stream.cu)
__device__ __forceinline__ uint32_t bsmem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void bmbar_init(uint64_t* bar, int count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bsmem_u32(bar)), "r"(count));
}
__device__ __forceinline__ void bmbar_expect_tx(uint64_t* bar, uint32_t bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bsmem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void bmbar_wait(uint64_t* bar, uint32_t parity) {
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "BWAIT_%=:\n"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
        "@p bra BDONE_%=;\n"
        "bra BWAIT_%=;\n"
        "BDONE_%=:\n"
        "}\n" ::"r"(bsmem_u32(bar)), "r"(parity) : "memory");
}
__device__ __forceinline__ void bbulk_g2s(void* dst, const void* src, uint32_t bytes, uint64_t* bar) {
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(bsmem_u32(dst)), "l"(src),
                 "r"(bytes), "r"(bsmem_u32(bar))
                 : "memory");
}

constexpr int BT_NANG = 14;   // staged cache columns: the angular ones (C_CK .. C_SPHI, C_CZ .. C_SA)
__device__ __forceinline__ int ang_col(int j) { return j < 6 ? C_CK + j : C_CZ + (j - 6); }

// raw inputs of one tile -> staging area: the distinct lineshape columns (64 x 16 B each), the angular cache
// columns and the weights (64 x 8 B each); issued by one thread, lands while the previous tile is multiplied
__device__ __forceinline__ void issue_stage(const BatchArgs& a, long long tile, double2* scol, double* sang, double* sw, uint64_t* bar, int nang,
                                            bool with_w) {
    const long long i0 = tile * BT_EVENTS;
    bmbar_expect_tx(bar, (uint32_t)(a.ncolu * BT_EVENTS * 16 + (nang + (with_w ? 1 : 0)) * BT_EVENTS * 8));
#pragma unroll 1
    for (int c = 0; c < a.ncolu; ++c) bbulk_g2s(scol + (size_t)c * BT_EVENTS, a.cols + (size_t)a.colu[c] * a.npad + i0, BT_EVENTS * 16, bar);
#pragma unroll 1
    for (int j = 0; j < nang; ++j) bbulk_g2s(sang + (size_t)j * BT_EVENTS, a.cache + cache_idx(a.ncolw, ang_col(j), i0), BT_EVENTS * 8, bar);
    if (with_w) bbulk_g2s(sw, a.cache + cache_idx(a.ncolw, a.ncolw - 1, i0), BT_EVENTS * 8, bar);   // (64 divides the 512-event cache block)
}

// angular factor g_xi (xi = +1, -1) of one basis entry at one event; `code` is warp-uniform
struct Angles {
    double cK, sK, cpsi, spsi, cphi, sphi;
    double cZ, sZ, ct, st, cpt, spt, ca, sa;
};
__device__ __forceinline__ void angular_factor(const Angles& g, int code, double2* gp, double2* gm) {
    const double RSQRT2 = 0.70710678118654752440;
    const int kind = code >> 8, J = (code >> 4) & 15, lam = (code & 15) - 1;
    if (kind_is_z(kind)) {
        // d^J_{0 l'}(theta_Z) e^{i l' phi~} d^1_{l' xi}(theta~) e^{i xi alpha}   (Eq. 10); J = 0, 1, 2
        double zf;
        if (J == 1) zf = lam == 0 ? g.cZ : (lam > 0 ? RSQRT2 * g.sZ : -RSQRT2 * g.sZ);
        else if (J == 0) zf = lam == 0 ? 1.0 : 0.0;
        else zf = lam == 0 ? fma(1.5, g.cZ * g.cZ, -0.5) : (lam > 0 ? 1.2247448713915890491 : -1.2247448713915890491) * g.sZ * g.cZ;
        const double dp = lam == 0 ? RSQRT2 * g.st : (lam > 0 ? 0.5 * (1.0 + g.ct) : 0.5 * (1.0 - g.ct));    // d^1_{l',+1}
        const double dm = lam == 0 ? -RSQRT2 * g.st : (lam > 0 ? 0.5 * (1.0 - g.ct) : 0.5 * (1.0 + g.ct));   // d^1_{l',-1}
        const double2 eph = lam == 0 ? make_double2(1.0, 0.0) : make_double2(g.cpt, lam > 0 ? g.spt : -g.spt);
        *gp = cscale(zf * dp, cmul(eph, make_double2(g.ca, g.sa)));
        *gm = cscale(zf * dm, cmul(eph, make_double2(g.ca, -g.sa)));
        return;
    }
    // d^J_{l 0}(theta_K*) e^{i l phi} d^1_{l xi}(theta_psi)   (Eq. 4); the constant term is J = 0
    const double c = g.cK, s = g.sK, c2 = c * c;
    double dj;
    if (lam == 0) {
        switch (J) {
            case 0: dj = 1.0; break;
            case 1: dj = c; break;
            case 2: dj = fma(1.5, c2, -0.5); break;
            case 3: dj = c * fma(2.5, c2, -1.5); break;
            default: dj = fma(fma(4.375, c2, -3.75), c2, 0.375); break;
        }
        const double h0 = RSQRT2 * g.spsi;
        *gp = make_double2(dj * h0, 0.0);
        *gm = make_double2(-dj * h0, 0.0);
        return;
    }
    switch (J) {
        case 1: dj = -RSQRT2 * s; break;
        case 2: dj = -1.2247448713915890491 * s * c; break;
        case 3: dj = -0.43301270189221932338 * s * fma(5.0, c2, -1.0); break;
        default: dj = -0.55901699437494742410 * s * c * fma(7.0, c2, -3.0); break;
    }
    if (lam < 0) dj = -dj;                                                 // d^J_{-1,0} = -d^J_{+1,0}
    const double hp = 0.5 * (1.0 + g.cpsi), hm = 0.5 * (1.0 - g.cpsi);
    const double2 eph = make_double2(g.cphi, lam > 0 ? g.sphi : -g.sphi);
    *gp = cscale(dj * (lam > 0 ? hp : hm), eph);
    *gm = cscale(dj * (lam > 0 ? hm : hp), eph);
}


// shared-memory carve-up common to both kernels
struct TileSmem {
    double* Bs;      // [2][KP][BT_STRIDE] basis tile, xi = +1 then -1
    double* ws;      // [BT_EVENTS] weights of the tile being multiplied (0 for padding events)
    double* sw;      // staging: weights
    double* sang;    // staging: [BT_NANG][BT_EVENTS] angular cache columns
    double2* scol;   // staging: [ncolu][BT_EVENTS] lineshape columns
    uint64_t* full;  // mbarrier of the staging area
};
__device__ __forceinline__ TileSmem carve_tile_smem(double* smem, int KP, int ncolu) {
    TileSmem t;
    t.Bs = smem;
    t.ws = smem + (size_t)2 * KP * BT_STRIDE;
    t.sw = t.ws + BT_EVENTS;
    t.sang = t.sw + BT_EVENTS;
    t.scol = reinterpret_cast<double2*>(t.sang + BT_NANG * BT_EVENTS);
    t.full = reinterpret_cast<uint64_t*>(t.scol + (size_t)ncolu * BT_EVENTS);
    return t;
}
static inline size_t tile_smem_bytes(int nent, int ncolu) {
    return ((size_t)2 * nent * 2 * BT_STRIDE + 2 * BT_EVENTS + BT_NANG * BT_EVENTS + (size_t)ncolu * BT_EVENTS * 2) * sizeof(double) + 16;
}

// Basis tile from the staged inputs: thread (part, ev) fills entries part, part+4, ... of event ev for both helicities.
// Call with all BT_THREADS threads after the staging barrier completed; follow with __syncthreads().
// scale_sqrt_w: multiply the event's basis by sqrt(w) (Gram kernel) — then ws holds 1 for live events.
__device__ __forceinline__ void build_basis_tile(const BatchArgs& a, const TileSmem& t, long long tile, int KP, bool with_w,
                                                 bool scale_sqrt_w = false) {
    const int tid = threadIdx.x;
    const int ev = tid & (BT_EVENTS - 1), part = tid / BT_EVENTS;
    const long long i = tile * BT_EVENTS + ev;          // < npad (npad is a multiple of 512)
    const double* sang = t.sang;
    Angles g;
    g.cK = sang[0 * BT_EVENTS + ev]; g.sK = sang[1 * BT_EVENTS + ev]; g.cpsi = sang[2 * BT_EVENTS + ev]; g.spsi = sang[3 * BT_EVENTS + ev];
    g.cphi = sang[4 * BT_EVENTS + ev]; g.sphi = sang[5 * BT_EVENTS + ev];
    if (a.have_z) {
        g.cZ = sang[6 * BT_EVENTS + ev]; g.sZ = sang[7 * BT_EVENTS + ev]; g.ct = sang[8 * BT_EVENTS + ev]; g.st = sang[9 * BT_EVENTS + ev];
        g.cpt = sang[10 * BT_EVENTS + ev]; g.spt = sang[11 * BT_EVENTS + ev]; g.ca = sang[12 * BT_EVENTS + ev]; g.sa = sang[13 * BT_EVENTS + ev];
    }
    const double sc = scale_sqrt_w ? ((i < a.n) ? sqrt(t.sw[ev]) : 0.0) : 1.0;
    for (int e = part; e < a.nent; e += BT_THREADS / BT_EVENTS) {
        const int2 en = a.entries[e];                   // (staged column, code); column -1: empty entry, -2: lineshape == 1
        double2 bp = make_double2(0, 0), bm = bp;
        if (en.x != -1) {
            const double2 bw = en.x >= 0 ? t.scol[(size_t)en.x * BT_EVENTS + ev] : make_double2(1.0, 0.0);
            double2 gp, gm;
            angular_factor(g, en.y, &gp, &gm);
            bp = cmul(bw, gp);
            bm = cmul(bw, gm);
            if (scale_sqrt_w) { bp = cscale(sc, bp); bm = cscale(sc, bm); }
        }
        double* r0 = t.Bs + (size_t)(2 * e) * BT_STRIDE + ev;
        r0[0] = bp.x; r0[BT_STRIDE] = bp.y;
        r0[(size_t)KP * BT_STRIDE] = bm.x; r0[(size_t)KP * BT_STRIDE + BT_STRIDE] = bm.y;
    }
    if (part == 0) t.ws[ev] = (i < a.n) ? (with_w ? t.sw[ev] : 1.0) : 0.0;
}

}  // namespace amp
