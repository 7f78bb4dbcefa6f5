// batch.cu — step a3 for P > 1 parameter points: the amplitude combine as the dense complex contraction it is,
//   A_xi(p, i) = sum_e C(p, e) B_{e,xi}(i),      S(p, i) = |A_+|^2 + |A_-|^2,
// on the FP64 tensor cores (mma.sync.m8n8k4.f64 — DMMA; tcgen05 has no f64 kind), fused with the -log L /
// normalisation reduction (a5).  Eqs. 4, 5, 10, 12.
//
// Realified GEMM, rows = parameter points, columns = events, contraction index = (basis entry, re/im):
//   Re A(p) = sum_e  c_re(p,e) b_re(e) - c_im(p,e) b_im(e)      (m-tile "RE" of a point octet)
//   Im A(p) = sum_e  c_im(p,e) b_re(e) + c_re(p,e) b_im(e)      (m-tile "IM" of the same octet)
// so the real and imaginary parts of one (point, event) pair land in the same thread and |A|^2 needs no shuffle.
// A warp owns 16 points (two octets = four m-tiles) and keeps their coefficient fragments in registers for the
// whole kernel; the basis tile B (events x entries, both muon helicities) is formed on the fly from the
// lineshape columns and the kinematics cache into shared memory and read as B fragments by all eight warps.
//
// Extended basis: a point that moves a resonance's mass or width uses another lineshape column for that
// resonance's slots.  Those (column, slot) pairs are appended as extra basis entries after the K base entries;
// the coefficient matrix is block-sparse there, and only the (k-tile, octet) blocks that are non-zero are
// multiplied (the per-warp item list), so a MINUIT-style gradient batch costs ~10 % more than the base GEMM.
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
    for (int j = 0; j < nang; ++j) bbulk_g2s(sang + (size_t)j * BT_EVENTS, a.cache + (size_t)ang_col(j) * a.npad + i0, BT_EVENTS * 8, bar);
    if (with_w) bbulk_g2s(sw, a.weight + i0, BT_EVENTS * 8, bar);
}

// angular factor g_xi (xi = +1, -1) of one basis entry at one event; `code` is warp-uniform
struct Angles {
    double cK, sK, cpsi, spsi, cphi, sphi;
    double cZ, sZ, ct, st, cpt, spt, ca, sa;
};
__device__ __forceinline__ void angular_factor(const Angles& g, int code, double2* gp, double2* gm) {
    const double RSQRT2 = 0.70710678118654752440;
    const int kind = code >> 8, J = (code >> 4) & 15, lam = (code & 15) - 1;
    if (kind == AMP_Z) {
        // d^1_{0 l'}(theta_Z) e^{i l' phi~} d^1_{l' xi}(theta~) e^{i xi alpha}   (Eq. 10)
        const double zf = lam == 0 ? g.cZ : (lam > 0 ? RSQRT2 * g.sZ : -RSQRT2 * g.sZ);
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

template <int NKT, int MODE>
__global__ void __launch_bounds__(BT_THREADS, 1) k_batch(const __grid_constant__ BatchArgs a) {
    extern __shared__ __align__(16) double smem[];
    const int KP = a.nent * 2;                                 // realified rows (multiple of 4)
    double* Bs = smem;                                         // [2][KP][BT_STRIDE]
    double* ws = smem + (size_t)2 * KP * BT_STRIDE;            // [BT_EVENTS] weights of the tile being multiplied
    double* sw = ws + BT_EVENTS;                               // staging: weights, angular columns, lineshape columns
    double* sang = sw + BT_EVENTS;                             // [BT_NANG][BT_EVENTS]
    double2* scol = reinterpret_cast<double2*>(sang + BT_NANG * BT_EVENTS);   // [ncolu][BT_EVENTS]
    uint64_t* full = reinterpret_cast<uint64_t*>(scol + (size_t)a.ncolu * BT_EVENTS);
    const int nang = a.have_z ? BT_NANG : 6;
    const bool with_w = MODE == MODE_NORM;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;

    // coefficient fragments of this warp's 16 points: [octet][re/im][k-tile]
    double Afr[2][2][NKT];
#pragma unroll
    for (int o = 0; o < 2; ++o)
#pragma unroll
        for (int ri = 0; ri < 2; ++ri)
#pragma unroll
            for (int kt = 0; kt < NKT; ++kt) Afr[o][ri][kt] = a.Adense[((((size_t)(2 * warp + o) * 2 + ri) * NKT) + kt) * 32 + lane];
    const int it0 = a.item_start[warp], it1 = a.item_start[warp + 1];
    const int prow = lane >> 2;                                // point row within an octet
    // row -> parameter point (the host spreads the points that own extended-basis blocks evenly over the warps)
    const int pt0 = a.point_of_row[16 * warp + prow], pt1 = a.point_of_row[16 * warp + 8 + prow];
    const bool live0 = pt0 >= 0, live1 = pt1 >= 0;
    const bool warp_live = __any_sync(0xffffffffu, live0 || live1);

    double sum[2] = {0.0, 0.0}, prod[2] = {1.0, 1.0};
    bool bad = false;
    const long long ntiles = (a.n + BT_EVENTS - 1) / BT_EVENTS;
    if (tid == 0) {
        bmbar_init(full, 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();
    if (tid == 0 && (long long)blockIdx.x < ntiles) issue_stage(a, blockIdx.x, scol, sang, sw, full, nang, with_w);
    uint32_t parity = 0;
    for (long long tile = blockIdx.x; tile < ntiles; tile += gridDim.x, parity ^= 1) {
        // ---- basis tile from the staged inputs: thread (part, ev) fills entries part, part+4, ... of event ev, both helicities
        bmbar_wait(full, parity);
        {
            const int ev = tid & (BT_EVENTS - 1), part = tid / BT_EVENTS;
            const long long i = tile * BT_EVENTS + ev;          // < npad (npad is a multiple of 512)
            Angles g;
            g.cK = sang[0 * BT_EVENTS + ev]; g.sK = sang[1 * BT_EVENTS + ev]; g.cpsi = sang[2 * BT_EVENTS + ev]; g.spsi = sang[3 * BT_EVENTS + ev];
            g.cphi = sang[4 * BT_EVENTS + ev]; g.sphi = sang[5 * BT_EVENTS + ev];
            if (a.have_z) {
                g.cZ = sang[6 * BT_EVENTS + ev]; g.sZ = sang[7 * BT_EVENTS + ev]; g.ct = sang[8 * BT_EVENTS + ev]; g.st = sang[9 * BT_EVENTS + ev];
                g.cpt = sang[10 * BT_EVENTS + ev]; g.spt = sang[11 * BT_EVENTS + ev]; g.ca = sang[12 * BT_EVENTS + ev]; g.sa = sang[13 * BT_EVENTS + ev];
            }
            for (int e = part; e < a.nent; e += BT_THREADS / BT_EVENTS) {
                const int2 en = a.entries[e];                   // (staged column, code); column -1: empty entry, -2: lineshape == 1
                double2 bp = make_double2(0, 0), bm = bp;
                if (en.x != -1) {
                    const double2 bw = en.x >= 0 ? scol[(size_t)en.x * BT_EVENTS + ev] : make_double2(1.0, 0.0);
                    double2 gp, gm;
                    angular_factor(g, en.y, &gp, &gm);
                    bp = cmul(bw, gp);
                    bm = cmul(bw, gm);
                }
                double* r0 = Bs + (size_t)(2 * e) * BT_STRIDE + ev;
                r0[0] = bp.x; r0[BT_STRIDE] = bp.y;
                r0[(size_t)KP * BT_STRIDE] = bm.x; r0[(size_t)KP * BT_STRIDE + BT_STRIDE] = bm.y;
            }
            if (part == 0) ws[ev] = (i < a.n) ? (with_w ? sw[ev] : 1.0) : 0.0;
        }
        __syncthreads();   // basis tile complete, staging area consumed: stream the next tile into it during the DMMA phase
        if (tid == 0 && tile + gridDim.x < ntiles) issue_stage(a, tile + gridDim.x, scol, sang, sw, full, nang, with_w);
        // ---- DMMA: this warp's 16 points x 64 events x both helicities
#pragma unroll 1
        for (int nt = 0; nt < (warp_live ? BT_EVENTS / 8 : 0); ++nt) {
            // both helicities side by side: eight independent accumulator chains per warp keep the DMMA pipe fed
            double acc[2][2][2][2];   // [xi][octet][re/im][event pair]
#pragma unroll
            for (int xi = 0; xi < 2; ++xi)
#pragma unroll
                for (int o = 0; o < 2; ++o)
#pragma unroll
                    for (int ri = 0; ri < 2; ++ri) acc[xi][o][ri][0] = acc[xi][o][ri][1] = 0.0;
            const double* bbase = Bs + (size_t)(lane & 3) * BT_STRIDE + 8 * nt + (lane >> 2);
            const size_t xoff = (size_t)KP * BT_STRIDE;
#pragma unroll
            for (int kt = 0; kt < NKT; ++kt) {
                const double bP = bbase[(size_t)4 * kt * BT_STRIDE], bM = bbase[xoff + (size_t)4 * kt * BT_STRIDE];
                dmma884(acc[0][0][0], Afr[0][0][kt], bP);
                dmma884(acc[1][0][0], Afr[0][0][kt], bM);
                dmma884(acc[0][0][1], Afr[0][1][kt], bP);
                dmma884(acc[1][0][1], Afr[0][1][kt], bM);
                dmma884(acc[0][1][0], Afr[1][0][kt], bP);
                dmma884(acc[1][1][0], Afr[1][0][kt], bM);
                dmma884(acc[0][1][1], Afr[1][1][kt], bP);
                dmma884(acc[1][1][1], Afr[1][1][kt], bM);
            }
            for (int it = it0; it < it1; ++it) {           // non-zero blocks of the extended (variant) basis
                const int2 item = a.items[it];               // (first realified row of the k-tile, octet 0/1 of this warp)
                const double bP = bbase[(size_t)item.x * BT_STRIDE], bM = bbase[xoff + (size_t)item.x * BT_STRIDE];
                const double are = a.itemA[((size_t)it * 2) * 32 + lane], aim = a.itemA[((size_t)it * 2 + 1) * 32 + lane];
                if (item.y == 0) {
                    dmma884(acc[0][0][0], are, bP); dmma884(acc[1][0][0], are, bM);
                    dmma884(acc[0][0][1], aim, bP); dmma884(acc[1][0][1], aim, bM);
                } else {
                    dmma884(acc[0][1][0], are, bP); dmma884(acc[1][1][0], are, bM);
                    dmma884(acc[0][1][1], aim, bP); dmma884(acc[1][1][1], aim, bM);
                }
            }
            double S[2][2];
#pragma unroll
            for (int o = 0; o < 2; ++o)
#pragma unroll
                for (int j = 0; j < 2; ++j)
                    S[o][j] = fma(acc[0][o][0][j], acc[0][o][0][j], fma(acc[0][o][1][j], acc[0][o][1][j],
                              fma(acc[1][o][0][j], acc[1][o][0][j], acc[1][o][1][j] * acc[1][o][1][j])));
            const double w0 = ws[8 * nt + 2 * (lane & 3)], w1 = ws[8 * nt + 2 * (lane & 3) + 1];
            if (MODE == MODE_NORM) {
#pragma unroll
                for (int o = 0; o < 2; ++o) {
                    bad |= !isfinite(S[o][0]) || !isfinite(S[o][1]);
                    sum[o] = fma(w0, S[o][0], fma(w1, S[o][1], sum[o]));
                }
            } else {
                // sum of logs: multiply four S values (two events x two n-tiles), one log per product
#pragma unroll
                for (int o = 0; o < 2; ++o) {
                    const bool live = o ? live1 : live0;
                    const double s0 = (live && w0 > 0.0) ? S[o][0] : 1.0, s1 = (live && w1 > 0.0) ? S[o][1] : 1.0;
                    bad |= !(s0 > 0.0) || !(s1 > 0.0) || !isfinite(s0) || !isfinite(s1);
                    prod[o] *= s0 * s1;
                    if (nt & 1) { sum[o] += log(prod[o]); prod[o] = 1.0; }
                }
            }
        }
        __syncthreads();
    }
    if (bad) atomicOr(a.flag, 2);
    // the four lanes of a row hold different events of the same point: fixed xor tree, then one partial per (point, CTA)
#pragma unroll
    for (int o = 0; o < 2; ++o) {
        double v = sum[o];
        v += __shfl_xor_sync(0xffffffffu, v, 1);
        v += __shfl_xor_sync(0xffffffffu, v, 2);
        const int p = o ? pt1 : pt0;
        if ((lane & 3) == 0 && p >= 0) a.partial[(size_t)p * a.partial_stride + blockIdx.x] = v;
    }
}

size_t batch_smem(int nent, int ncolu) {
    return ((size_t)2 * nent * 2 * BT_STRIDE + 2 * BT_EVENTS + BT_NANG * BT_EVENTS + (size_t)ncolu * BT_EVENTS * 2) * sizeof(double) + 16;
}
bool batch_fits(int nent, int ncolu) { return ncolu <= BATCH_MAX_COLS && batch_smem(nent, ncolu) <= (size_t)224 * 1024; }

int batch_grid(long long n) {
    const long long ntiles = (n + BT_EVENTS - 1) / BT_EVENTS;
    return (int)(ntiles < 1 ? 1 : (ntiles > 148 ? 148 : ntiles));   // persistent: one CTA per SM
}

cudaError_t launch_batch(const BatchArgs& a, int grid, cudaStream_t s) {
    const size_t smem = batch_smem(a.nent, a.ncolu);
    cudaError_t e = cudaSuccess;
#define AMP_LAUNCH(NKT, M)                                                                                           \
    {                                                                                                                \
        static bool attr_done = false;                                                                               \
        if (!attr_done) { e = cudaFuncSetAttribute(k_batch<NKT, M>, cudaFuncAttributeMaxDynamicSharedMemorySize, 224 * 1024); attr_done = true; } \
        if (e == cudaSuccess) k_batch<NKT, M><<<grid, BT_THREADS, smem, s>>>(a);                                     \
    }
    if (a.nkt != BATCH_NKT) return cudaErrorInvalidValue;
    if (a.mode == MODE_NORM) AMP_LAUNCH(BATCH_NKT, MODE_NORM) else AMP_LAUNCH(BATCH_NKT, MODE_DATA)
#undef AMP_LAUNCH
    return e != cudaSuccess ? e : cudaGetLastError();
}

}  // namespace amp
