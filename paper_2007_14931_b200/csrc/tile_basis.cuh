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

constexpr int BT_NSCAL = 15;  // rows of the scaling table: d^J_{00} (J = 0 .. 4), d^J_{+1,0} (J = 1 .. 4), then per Z spin 0, 1, 2: lambda' = 0, |lambda'| = 1
constexpr int BT_NBASE = 6;   // rows of the base table: K* lambda = -1, 0, +1, then Z lambda' = -1, 0, +1
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

// shared-memory carve-up common to both kernels
struct TileSmem {
    double* Bs;      // [2][KP][BT_STRIDE] basis tile, xi = +1 then -1
    double* ws;      // [BT_EVENTS] weights of the tile being multiplied (0 for padding events)
    double* sw;      // staging: weights
    double* sang;    // staging: [BT_NANG][BT_EVENTS] angular cache columns
    double2* scol;   // staging: [ncolu][BT_EVENTS] lineshape columns
    uint64_t* full;  // mbarrier of the staging area
    double* tabS;    // [BT_NSCAL][BT_EVENTS] the real angular scalings of the tile's events (build_basis_tile)
    double2* tabB;   // [2 BT_NBASE][BT_EVENTS] their complex angular bases, xi = +1 then -1 per helicity row
    int2* sent;      // [nent] (staged column, scaling row | base row << 8) per entry, decoded once per CTA
};
__device__ __forceinline__ TileSmem carve_tile_smem(double* smem, int KP, int ncolu) {
    TileSmem t;
    t.Bs = smem;
    t.ws = smem + (size_t)2 * KP * BT_STRIDE;
    t.sw = t.ws + BT_EVENTS;
    t.sang = t.sw + BT_EVENTS;
    t.scol = reinterpret_cast<double2*>(t.sang + BT_NANG * BT_EVENTS);
    t.full = reinterpret_cast<uint64_t*>(t.scol + (size_t)ncolu * BT_EVENTS);
    t.tabB = reinterpret_cast<double2*>(t.full + 2);
    t.tabS = reinterpret_cast<double*>(t.tabB + 2 * BT_NBASE * BT_EVENTS);
    t.sent = reinterpret_cast<int2*>(t.tabS + BT_NSCAL * BT_EVENTS);
    return t;
}
static inline size_t tile_smem_bytes(int nent, int ncolu) {
    return ((size_t)2 * nent * 2 * BT_STRIDE + 2 * BT_EVENTS + BT_NANG * BT_EVENTS + (size_t)ncolu * BT_EVENTS * 2) * sizeof(double) + 16 +
           ((size_t)4 * BT_NBASE + BT_NSCAL) * BT_EVENTS * sizeof(double) + (size_t)nent * sizeof(int2);
}

// Once per CTA (before the first tile; all threads, followed by a barrier before the first build): the entries as the build reads
// them.  An entry's angular factor g_xi (xi = +1, -1; `code` = kind << 8 | J << 4 | lambda + 1) is scaling x base_xi:
//   K* (Eq. 4):  d^J_{lambda 0}(theta_K*)  x  e^{i lambda phi} d^1_{lambda xi}(theta_psi)        (the constant term is J = 0)
//   Z (Eq. 10):  d^J_{0 lambda'}(theta_Z)  x  e^{i lambda' phi~} d^1_{lambda' xi}(theta~) e^{i xi alpha}
// the scaling real and a function of (chain, J, |lambda|), the base complex and a function of (chain, lambda); the signs
// d^J_{-1,0} = -d^J_{+1,0} and d^J_{0,-1} = -d^J_{0,+1} go into the lambda = -1 bases.
__device__ __forceinline__ void stage_tile_entries(const BatchArgs& a, const TileSmem& t) {
    for (int e = threadIdx.x; e < a.nent; e += BT_THREADS) {
        const int2 en = a.entries[e];
        const int kind = en.y >> 8, J = (en.y >> 4) & 15, lam = (en.y & 15) - 1;
        const bool isz = kind_is_z(kind);
        const int srow = isz ? 9 + 2 * J + (lam != 0) : (lam != 0 ? 4 + J : J);
        const int brow = (isz ? 3 : 0) + lam + 1;
        t.sent[e] = make_int2(en.x, srow | (brow << 8));
    }
}

// Basis tile from the staged inputs, in two steps with a barrier between them.  (1) The four threads of an event fill its rows of
// the two angular tables: K* scalings, K* bases, Z scalings, Z bases (the bases carry sqrt(w) for the Gram kernel).  (2) Thread
// (part, ev) fills entries part, part + 4, ... of event ev for both helicities: B = BW x (scaling x base_xi) — three table loads,
// one column load, twelve FP64 operations and four stores per entry; no switch on the entry's kind in the loop.
// Call with all BT_THREADS threads after the staging barrier completed; follow with __syncthreads().
// scale_sqrt_w: multiply the event's basis by sqrt(w) (Gram kernel) — then ws holds 1 for live events.
__device__ __forceinline__ void build_basis_tile(const BatchArgs& a, const TileSmem& t, long long tile, int KP, bool with_w,
                                                 bool scale_sqrt_w = false) {
    const double RSQRT2 = 0.70710678118654752440;
    const int tid = threadIdx.x;
    const int ev = tid & (BT_EVENTS - 1), part = tid / BT_EVENTS;
    const long long i = tile * BT_EVENTS + ev;          // < npad (npad is a multiple of 512)
    const double* sang = t.sang;
    const double sc = scale_sqrt_w ? ((i < a.n) ? sqrt(t.sw[ev]) : 0.0) : 1.0;
    double* S = t.tabS + ev;
    double2* Bt = t.tabB + ev;
    if (part == 0) {            // d^J_{00}(theta_K*), d^J_{+1,0}(theta_K*)
        const double c = sang[0 * BT_EVENTS + ev], sn = sang[1 * BT_EVENTS + ev], c2 = c * c;
        S[0 * BT_EVENTS] = 1.0;
        S[1 * BT_EVENTS] = c;
        S[2 * BT_EVENTS] = fma(1.5, c2, -0.5);
        S[3 * BT_EVENTS] = c * fma(2.5, c2, -1.5);
        S[4 * BT_EVENTS] = fma(fma(4.375, c2, -3.75), c2, 0.375);
        S[5 * BT_EVENTS] = -RSQRT2 * sn;
        S[6 * BT_EVENTS] = -1.2247448713915890491 * sn * c;
        S[7 * BT_EVENTS] = -0.43301270189221932338 * sn * fma(5.0, c2, -1.0);
        S[8 * BT_EVENTS] = -0.55901699437494742410 * sn * c * fma(7.0, c2, -3.0);
        t.ws[ev] = (i < a.n) ? (with_w ? t.sw[ev] : 1.0) : 0.0;
    } else if (part == 1) {     // e^{i lambda phi} d^1_{lambda xi}(theta_psi); d^J_{-1,0} = -d^J_{+1,0} goes into the lambda = -1 row
        const double cpsi = sang[2 * BT_EVENTS + ev], spsi = sang[3 * BT_EVENTS + ev], cphi = sang[4 * BT_EVENTS + ev], sphi = sang[5 * BT_EVENTS + ev];
        const double hp = sc * 0.5 * (1.0 + cpsi), hm = sc * 0.5 * (1.0 - cpsi), h0 = sc * RSQRT2 * spsi;
        Bt[0 * BT_EVENTS] = make_double2(-hm * cphi, hm * sphi);     // lambda = -1, xi = +1: -d^1_{-1,+1} e^{-i phi}
        Bt[1 * BT_EVENTS] = make_double2(-hp * cphi, hp * sphi);     //              xi = -1
        Bt[2 * BT_EVENTS] = make_double2(h0, 0.0);                   // lambda = 0
        Bt[3 * BT_EVENTS] = make_double2(-h0, 0.0);
        Bt[4 * BT_EVENTS] = make_double2(hp * cphi, hp * sphi);      // lambda = +1
        Bt[5 * BT_EVENTS] = make_double2(hm * cphi, hm * sphi);
    } else if (part == 2) {     // d^J_{0 lambda'}(theta_Z): J = 0, 1, 2; lambda' = 0, |lambda'| = 1 (the sign of lambda' < 0 in the base)
        if (a.have_z) {
            const double cZ = sang[6 * BT_EVENTS + ev], sZ = sang[7 * BT_EVENTS + ev];
            S[9 * BT_EVENTS] = 1.0;
            S[10 * BT_EVENTS] = 0.0;
            S[11 * BT_EVENTS] = cZ;
            S[12 * BT_EVENTS] = RSQRT2 * sZ;
            S[13 * BT_EVENTS] = fma(1.5, cZ * cZ, -0.5);
            S[14 * BT_EVENTS] = 1.2247448713915890491 * sZ * cZ;
        }
    } else {                    // e^{i lambda' phi~} d^1_{lambda' xi}(theta~) e^{i xi alpha}   (Eq. 10)
        if (a.have_z) {
            const double ct = sang[8 * BT_EVENTS + ev], st = sang[9 * BT_EVENTS + ev], cpt = sang[10 * BT_EVENTS + ev], spt = sang[11 * BT_EVENTS + ev];
            const double ca = sang[12 * BT_EVENTS + ev], sa = sang[13 * BT_EVENTS + ev];
            const double gp = sc * 0.5 * (1.0 + ct), gm = sc * 0.5 * (1.0 - ct), g0 = sc * RSQRT2 * st;
            const double2 ap = make_double2(ca, sa), am = make_double2(ca, -sa);
            const double2 ep = cmul(make_double2(cpt, spt), ap), em = cmul(make_double2(cpt, spt), am);       // e^{+i phi~} e^{+-i alpha}
            const double2 fp = cmul(make_double2(cpt, -spt), ap), fm = cmul(make_double2(cpt, -spt), am);     // e^{-i phi~} e^{+-i alpha}
            Bt[6 * BT_EVENTS] = cscale(-gm, fp);                     // lambda' = -1: d^1_{-1,+1} = gm, sign of d^J_{0,-1} folded in
            Bt[7 * BT_EVENTS] = cscale(-gp, fm);
            Bt[8 * BT_EVENTS] = cscale(g0, ap);                      // lambda' = 0: d^1_{0,+1} = g0, d^1_{0,-1} = -g0
            Bt[9 * BT_EVENTS] = cscale(-g0, am);
            Bt[10 * BT_EVENTS] = cscale(gp, ep);                     // lambda' = +1
            Bt[11 * BT_EVENTS] = cscale(gm, em);
        }
    }
    __syncthreads();
#pragma unroll 2
    for (int e = part; e < a.nent; e += BT_THREADS / BT_EVENTS) {
        const int2 en = t.sent[e];                      // (staged column, table rows); column -1: empty entry, -2: lineshape == 1
        double2 bp = make_double2(0, 0), bm = bp;
        if (en.x != -1) {
            const double2 bw = en.x >= 0 ? t.scol[(size_t)en.x * BT_EVENTS + ev] : make_double2(1.0, 0.0);
            const double sv = S[(en.y & 255) * BT_EVENTS];
            const double2 gp = cscale(sv, Bt[2 * (en.y >> 8) * BT_EVENTS]), gm = cscale(sv, Bt[(2 * (en.y >> 8) + 1) * BT_EVENTS]);
            bp = cmul(bw, gp);
            bm = cmul(bw, gm);
        }
        double* r0 = t.Bs + (size_t)(2 * e) * BT_STRIDE + ev;
        r0[0] = bp.x; r0[BT_STRIDE] = bp.y;
        r0[(size_t)KP * BT_STRIDE] = bm.x; r0[(size_t)KP * BT_STRIDE + BT_STRIDE] = bm.y;
    }
}

}  // namespace amp
