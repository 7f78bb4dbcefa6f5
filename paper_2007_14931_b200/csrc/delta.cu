// delta.cu — steps a2 + a3 + a4 + a5 for a GRADIENT BATCH: P parameter points of which points 1..P-1 differ from
// point 0 in a few resonances only (MINUIT's finite-difference pattern, BASELINE.json configs[4]: the central value
// plus theta_k +- h_k for ~60 parameters; "> 60 free parameters").
//
// With B_k,xi the basis terms of Eqs. 4 and 10, a point that changes resonance R only gives
//   A_xi(p) = A_xi(0) + sum_{l in R} [ c_{R,l}(p) BW_R(p) - c_{R,l}(0) BW_R(0) ] g_{R,l,xi}          (Eq. 12 is linear in c BW)
// i.e. one to three complex multiply-adds per muon helicity instead of the 27 of the dense contraction, and the
// perturbed Breit-Wigner (Eqs. 2-3) costs ~12 FP64 instructions because the barrier factors of its spin group are
// those of point 0.  One fused persistent launch walks the data tiles (sum_i log S_i(p)) and then the normalisation
// tiles (sum_j w_j S_j(p)) for ALL points; no lineshape column, no normalisation matrix, no second pass.
//
// Thread = one event.  Per tile: (1) point 0 exactly as the streaming kernel does it, but the Breit-Wigners and the
// group factors (F, G) of the event are kept in a thread-private shared-memory record; (2) the points, 32 at a time:
// every lane evaluates S(p) of its own event for the 32 points of a block in order, and a recursive-halving
// exchange (one shuffle + one add/multiply per point and lane) leaves lane l with the total of point 32 b + l over
// the warp's 32 events.  Data side: S = f 2^e is split with integer ops, mantissas are multiplied and exponents
// added, so the sum of logs needs ONE log per (point, warp) at the very end instead of one per (point, event).
// Everything is fixed-order: bit-reproducible.  Bound: plain FP64 ALUs.
#include "amp_internal.cuh"

namespace amp {

namespace {

constexpr int DT = DELTA_TILE;       // events per tile = threads per CTA
constexpr int DNCOL = NCOL_ALL + 1;  // staged columns per tile: the cache + the weight
constexpr int DBLK = DELTA_MAX_SORTED / 32;

__device__ __forceinline__ uint32_t d_smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void d_mbar_init(uint64_t* bar, int count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(d_smem_u32(bar)), "r"(count));
}
__device__ __forceinline__ void d_mbar_expect_tx(uint64_t* bar, uint32_t bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(d_smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void d_mbar_wait(uint64_t* bar, uint32_t parity) {
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "DWAIT_%=:\n"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
        "@p bra DDONE_%=;\n"
        "bra DWAIT_%=;\n"
        "DDONE_%=:\n"
        "}\n" ::"r"(d_smem_u32(bar)), "r"(parity) : "memory");
}
__device__ __forceinline__ void d_bulk_g2s(void* dst, const void* src, uint32_t bytes, uint64_t* bar) {
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(d_smem_u32(dst)), "l"(src),
                 "r"(bytes), "r"(d_smem_u32(bar))
                 : "memory");
}

// all columns of one 256-event tile (unified tile space: data tiles first, then normalisation tiles) -> stage
__device__ __forceinline__ void issue_tile(const StreamArgs& a, long long ntd, long long tile, int ncache, double* stage, uint64_t* bar) {
    const bool is_norm = tile >= ntd;
    const double* cache = is_norm ? a.cache2 : a.cache;
    const long long npad = is_norm ? a.npad2 : a.npad, lt = is_norm ? tile - ntd : tile;
    const uint32_t col_bytes = DT * sizeof(double);
    d_mbar_expect_tx(bar, col_bytes * (ncache + (is_norm ? 1 : 0)));
#pragma unroll 1
    for (int c = 0; c < ncache; ++c) d_bulk_g2s(stage + c * DT, cache + (size_t)c * npad + lt * DT, col_bytes, bar);
    if (is_norm) d_bulk_g2s(stage + NCOL_ALL * DT, a.weight2 + lt * DT, col_bytes, bar);
}

// S = f 2^e with f in [0.5, 1) for normal positive S (integer ops on the exponent field)
__device__ __forceinline__ void split_exp(double S, double* f, int* e) {
    if (S < 1e-290) { S *= 1.3407807929942597e154; *e = -512; } else *e = 0;   // 2^512: keeps subnormals out of the bit trick
    const int hi = __double2hiint(S), lo = __double2loint(S);
    *e += ((hi >> 20) & 0x7ff) - 1022;
    *f = __hiloint2double((hi & 0x800fffff) | 0x3fe00000, lo);
}

struct EvK {   // what the point loop needs of one event (registers)
    double2 Ap, Am;                 // A_xi(0)
    double m2, mZ2;
    double cK, sK;
    double h0, a1, a2, a3, a4;      // d^1_{0,+}(theta_psi); hp cos phi, hp sin phi, hm cos phi, hm sin phi
};

// d^J_{00}, d^J_{+1,0} (Eq. 4), J warp-uniform
__device__ __forceinline__ void dJ(int J, double c, double s, double* d0, double* d1) {
    const double c2 = c * c;
    switch (J) {
        case 0: *d0 = 1.0; *d1 = 0.0; break;
        case 1: *d0 = c; *d1 = -0.70710678118654752440 * s; break;
        case 2: *d0 = fma(1.5, c2, -0.5); *d1 = -1.2247448713915890491 * s * c; break;
        case 3: *d0 = c * fma(2.5, c2, -1.5); *d1 = -0.43301270189221932338 * s * fma(5.0, c2, -1.0); break;
        default: *d0 = fma(fma(4.375, c2, -3.75), c2, 0.375); *d1 = -0.55901699437494742410 * s * c * fma(7.0, c2, -3.0); break;
    }
}

// Point 0 of one event: Eqs. 2-5, 10, 12 with the resonances grouped by spin (as stream.cu), E = 1, runtime group loops.
// Stores BW_R(0) of every entry and (F, G) of every barrier group in the thread's shared-memory record.
template <int J, int LR, int LB>
__device__ __forceinline__ void spin_group(const StreamArgs& a, int sp, double m2, double invm, double pR, double pB, double2* bw_rec, double2* fg_rec,
                                           double2& Um, double2& U0, double2& Up) {
    for (int g = a.gstart[sp]; g < a.gstart[sp + 1]; ++g) {
        double F, G;
        group_factors<LR, LB>(a.grp[g].r2, invm, pR, pB, &F, &G);
        fg_rec[g * DT] = make_double2(F, G);
        for (int t = a.grp[g].first; t < a.grp[g].first + a.grp[g].count; ++t) {
            const double2 bw = bw_from_factors(a.ent[t], m2, F, G);
            bw_rec[t * DT] = bw;
            U0 = cfma(a.ent[t].c0, bw, U0);
            if (J) { Um = cfma(a.ent[t].cm, bw, Um); Up = cfma(a.ent[t].cp, bw, Up); }
        }
    }
}

// fixed-order block sum (xor-shuffle tree, then the 8 warp values in warp order); valid in thread 0
__device__ __forceinline__ double block_sum(double v, double* sm) {
#pragma unroll
    for (int o = 16; o; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    __syncthreads();
    if ((threadIdx.x & 31) == 0) sm[threadIdx.x >> 5] = v;
    __syncthreads();
    double t = 0.0;
    if (threadIdx.x == 0)
        for (int wv = 0; wv < 8; ++wv) t += sm[wv];
    return t;
}

// S(p) of this thread's event for the point whose items start at items[it]; advances it past the point.
__device__ __forceinline__ double point_density(const DeltaItem* __restrict__ items, int& it, const EvK& k, const double2* bw_rec,
                                                const double2* fg_rec, const double* zst /* this event's slot in the staged tile */) {
    const double RSQRT2 = 0.70710678118654752440;
    double2 Ap = k.Ap, Am = k.Am;
    int flags;
    do {
        const DeltaItem* d = items + it++;
        flags = d->flags;
        if ((flags & 0xe) == 0) continue;                      // empty point (padding, or identical to point 0)
        const bool isz = d->J == 256;
        const double2 bw0 = bw_rec[d->ent * DT];
        double2 gam[3];                                        // c(p) BW(p) - c(0) BW(0) per helicity
        if (flags & 1) {
            const double2 fg = fg_rec[d->grp * DT];
            const double2 bw1 = bw_from_consts(d->kN, d->kG, d->M2, isz ? k.mZ2 : k.m2, fg.x, fg.y);
#pragma unroll
            for (int l = 0; l < 3; ++l)
                if (flags & (2 << l)) {
                    const double2 t = cmul(d->c0[l], bw0);
                    gam[l] = cfma(d->g[l], bw1, make_double2(-t.x, -t.y));
                }
        } else {
#pragma unroll
            for (int l = 0; l < 3; ++l)
                if (flags & (2 << l)) gam[l] = cmul(d->g[l], bw0);
        }
        if (!isz) {
            // Eq. 4: d^J_{l0}(theta_K*) e^{i l phi} d^1_{l xi}(theta_psi); d^J_{-1,0} = -d^J_{+1,0}
            double d0, d1;
            dJ(d->J, k.cK, k.sK, &d0, &d1);
            if (flags & 4) { const double t = d0 * k.h0; Ap.x = fma(t, gam[1].x, Ap.x); Ap.y = fma(t, gam[1].y, Ap.y); Am.x = fma(-t, gam[1].x, Am.x); Am.y = fma(-t, gam[1].y, Am.y); }
            if (flags & 8) {   // lambda = +1: e^{+i phi} (hp, hm)
                const double2 t = cscale(d1, gam[2]);
                Ap = cfma(t, make_double2(k.a1, k.a2), Ap);
                Am = cfma(t, make_double2(k.a3, k.a4), Am);
            }
            if (flags & 2) {   // lambda = -1: e^{-i phi} (hm, hp), sign of d^J_{-1,0}
                const double2 t = cscale(-d1, gam[0]);
                Ap = cfma(t, make_double2(k.a3, -k.a4), Ap);
                Am = cfma(t, make_double2(k.a1, -k.a2), Am);
            }
        } else {
            // Eq. 10: d^1_{0 l'}(theta_Z) e^{i l' phi~} d^1_{l' xi}(theta~) e^{i xi alpha}; angles from the staged tile
            const double cZ = zst[C_CZ * DT], sZ = zst[C_SZ * DT], ct = zst[C_CT * DT], st = zst[C_ST * DT];
            const double cpt = zst[C_CPT * DT], spt = zst[C_SPT * DT], ca = zst[C_CA * DT], sa = zst[C_SA * DT];
            const double z1 = RSQRT2 * sZ, gp = 0.5 * (1.0 + ct), gm = 0.5 * (1.0 - ct), g0 = RSQRT2 * st;
            double2 Zp = make_double2(0, 0), Zm = Zp;
            if (flags & 4) { const double2 T0 = cscale(cZ, gam[1]); Zp = cscale(g0, T0); Zm = cscale(-g0, T0); }
            if (flags & 8) {
                const double2 Tp = cscale(z1, cmul(make_double2(cpt, spt), gam[2]));
                Zp.x = fma(gp, Tp.x, Zp.x); Zp.y = fma(gp, Tp.y, Zp.y); Zm.x = fma(gm, Tp.x, Zm.x); Zm.y = fma(gm, Tp.y, Zm.y);
            }
            if (flags & 2) {
                const double2 Tm = cscale(-z1, cmul(make_double2(cpt, -spt), gam[0]));
                Zp.x = fma(gm, Tm.x, Zp.x); Zp.y = fma(gm, Tm.y, Zp.y); Zm.x = fma(gp, Tm.x, Zm.x); Zm.y = fma(gp, Tm.y, Zm.y);
            }
            Ap = cfma(make_double2(ca, sa), Zp, Ap);
            Am = cfma(make_double2(ca, -sa), Zm, Am);
        }
    } while (!(flags & 16));
    return fma(Ap.x, Ap.x, fma(Ap.y, Ap.y, fma(Am.x, Am.x, Am.y * Am.y)));
}

// Recursive halving over the 32 lanes: `a` belongs to the earlier half of the points, `b` to the later half; lanes with
// bit `level` clear keep the earlier half.  After levels 0..4 lane l holds the total of point l of the block.
template <bool NORM>
__device__ __forceinline__ void halve(int level, int lane, double a, int ea, double b, int eb, double* v, int* e) {
    const bool up = (lane >> level) & 1;
    const double send = up ? a : b, keep = up ? b : a;
    const double recv = __shfl_xor_sync(0xffffffffu, send, 1 << level);
    if (NORM) {
        *v = keep + recv;
    } else {
        const int es = up ? ea : eb, ek = up ? eb : ea;
        *v = keep * recv;
        *e = ek + __shfl_xor_sync(0xffffffffu, es, 1 << level);
    }
}

// one point of this thread's event as a tree leaf: NORM: w S; DATA: (mantissa, exponent) of S
template <bool NORM>
__device__ __forceinline__ void leaf(const DeltaItem* __restrict__ items, int& it, const EvK& k, const double2* bw_rec, const double2* fg_rec,
                                     const double* zst, double w, bool live, bool& bad, double* v, int* e) {
    const double S = point_density(items, it, k, bw_rec, fg_rec, zst);
    if (NORM) {
        bad |= live && !isfinite(S);
        *v = w * S;
        *e = 0;
    } else {
        const bool ok = S > 0.0 && isfinite(S);
        bad |= live && !ok;
        split_exp((live && ok) ? S : 1.0, v, e);
    }
}

// The 32 points of one block for this thread's event; on return lane l holds the warp total of point 32 blk + l
// (NORM: sum of w S; DATA: product of mantissas in *v, sum of exponents in *e).
template <bool NORM>
__device__ __forceinline__ void eval_block(const DeltaItem* __restrict__ items, int& it, const EvK& k, const double2* bw_rec, const double2* fg_rec,
                                           const double* zst, double w, bool live, bool& bad, int lane, double* v, int* e) {
    double s2 = 0, s3 = 0, s4 = 0;
    int e2 = 0, e3 = 0, e4 = 0;
#pragma unroll 1
    for (int g = 0; g < 8; ++g) {
        double v0, v1, u0, u1, x;
        int f0, f1, q0, q1, ex;
        leaf<NORM>(items, it, k, bw_rec, fg_rec, zst, w, live, bad, &v0, &f0);
        leaf<NORM>(items, it, k, bw_rec, fg_rec, zst, w, live, bad, &v1, &f1);
        halve<NORM>(0, lane, v0, f0, v1, f1, &u0, &q0);
        leaf<NORM>(items, it, k, bw_rec, fg_rec, zst, w, live, bad, &v0, &f0);
        leaf<NORM>(items, it, k, bw_rec, fg_rec, zst, w, live, bad, &v1, &f1);
        halve<NORM>(0, lane, v0, f0, v1, f1, &u1, &q1);
        halve<NORM>(1, lane, u0, q0, u1, q1, &x, &ex);
        // binary-counter carries through levels 2, 3, 4 (g is uniform)
        if ((g & 1) == 0) { s2 = x; e2 = ex; continue; }
        halve<NORM>(2, lane, s2, e2, x, ex, &x, &ex);
        if ((g & 2) == 0) { s3 = x; e3 = ex; continue; }
        halve<NORM>(3, lane, s3, e3, x, ex, &x, &ex);
        if ((g & 4) == 0) { s4 = x; e4 = ex; continue; }
        halve<NORM>(4, lane, s4, e4, x, ex, v, e);
    }
}

}  // namespace

__global__ void __launch_bounds__(DT, 1) k_delta(const __grid_constant__ DeltaArgs d) {
    const StreamArgs& a = d.a;
    const double RSQRT2 = 0.70710678118654752440;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const bool have_z = a.gstart[6] > a.gstart[5];
    const int ncache = have_z ? NCOL_ALL : NCOL_K;
    int nent = 0;
    for (int sp = 0; sp < 6; ++sp) nent += a.shape[sp];
    const int ngrp = a.gstart[6];
    const int nblk = d.nsorted / 32;

    extern __shared__ __align__(128) unsigned char smem_raw[];
    double* stage = reinterpret_cast<double*>(smem_raw);                       // [2][DNCOL][DT]
    double2* bw_base = reinterpret_cast<double2*>(stage + 2 * DNCOL * DT);      // [nent][DT]
    double2* fg_base = bw_base + (size_t)nent * DT;                             // [ngrp][DT]
    double* accN = reinterpret_cast<double*>(fg_base + (size_t)ngrp * DT);      // [DBLK][8 warps][32] sum w S
    double* accF = accN + DBLK * DT;                                            // [DBLK][8][32] mantissa products (data)
    int* accE = reinterpret_cast<int*>(accF + DBLK * DT);                       // [DBLK][8][32] exponent sums (data)
    uint64_t* full = reinterpret_cast<uint64_t*>(accE + DBLK * DT);             // [2]
    __shared__ double sm[8];
    __shared__ bool s_last;
    for (int b = 0; b < DBLK; ++b) { accN[b * DT + tid] = 0.0; accF[b * DT + tid] = 1.0; accE[b * DT + tid] = 0; }
    if (tid == 0) {
        d_mbar_init(&full[0], 1);
        d_mbar_init(&full[1], 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();
    const long long ntd = d.want_nll ? (a.n + DT - 1) / DT : 0;
    const long long ntiles = ntd + (a.n2 + DT - 1) / DT;
    if (tid == 0 && (long long)blockIdx.x < ntiles) issue_tile(a, ntd, blockIdx.x, ncache, stage, &full[0]);

    double2* bw_rec = bw_base + tid;
    double2* fg_rec = fg_base + tid;
    double acc0N = 0.0, acc0F = 1.0;   // point 0: sum w S ; mantissa product and exponent sum of S
    int acc0E = 0;
    bool bad = false;
    uint32_t par0 = 0, par1 = 0;
    int buf = 0;
    for (long long tile = blockIdx.x; tile < ntiles; tile += gridDim.x, buf ^= 1) {
        // the other buffer was last read before the __syncthreads that closed the previous iteration: refill it now
        if (tid == 0 && tile + gridDim.x < ntiles) issue_tile(a, ntd, tile + gridDim.x, ncache, stage + (buf ^ 1) * DNCOL * DT, &full[buf ^ 1]);
        const bool is_norm = tile >= ntd;
        const long long lt = is_norm ? tile - ntd : tile;
        const bool live = lt * DT + tid < (is_norm ? a.n2 : a.n);
        if (buf == 0) { d_mbar_wait(&full[0], par0); par0 ^= 1; } else { d_mbar_wait(&full[1], par1); par1 ^= 1; }
        const double* st = stage + buf * DNCOL * DT + tid;

        // ---- point 0 (as stream.cu, one event per thread)
        EvK k;
        k.m2 = st[C_M2 * DT];
        k.cK = st[C_CK * DT]; k.sK = st[C_SK * DT];
        double2 V0 = a.cconst, Vp = make_double2(0, 0), Vm = Vp;
        {
            const double invm = st[C_INVM * DT], q = st[C_Q * DT], pB = st[C_PB * DT];
            const double c = k.cK, s = k.sK;
#define AMP_DSPIN(J, LB)                                                                         \
            if (a.gstart[J + 1] > a.gstart[J]) {                                                   \
                double2 Um = make_double2(0, 0), U0 = Um, Up = Um;                                 \
                spin_group<J, J, LB>(a, J, k.m2, invm, q, pB, bw_rec, fg_rec, Um, U0, Up);         \
                double d0, d1;                                                                     \
                dJ(J, c, s, &d0, &d1);                                                             \
                V0 = cadd(V0, cscale(d0, U0));                                                     \
                if (J) { Vp = cadd(Vp, cscale(d1, Up)); Vm = cadd(Vm, cscale(-d1, Um)); }          \
            }
            AMP_DSPIN(0, 1)
            AMP_DSPIN(1, 0)
            AMP_DSPIN(2, 1)
            AMP_DSPIN(3, 2)
            AMP_DSPIN(4, 3)
#undef AMP_DSPIN
        }
        {
            const double cpsi = st[C_CPSI * DT], spsi = st[C_SPSI * DT], cphi = st[C_CPHI * DT], sphi = st[C_SPHI * DT];
            const double hp = 0.5 * (1.0 + cpsi), hm = 0.5 * (1.0 - cpsi);
            k.h0 = RSQRT2 * spsi;
            k.a1 = hp * cphi; k.a2 = hp * sphi; k.a3 = hm * cphi; k.a4 = hm * sphi;
            // A_xi = sum_l e^{i l phi} d^1_{l xi}(theta_psi) V_l
            k.Ap = make_double2(k.h0 * V0.x, k.h0 * V0.y);
            k.Am = make_double2(-k.Ap.x, -k.Ap.y);
            k.Ap = cfma(Vp, make_double2(k.a1, k.a2), k.Ap);
            k.Am = cfma(Vp, make_double2(k.a3, k.a4), k.Am);
            k.Ap = cfma(Vm, make_double2(k.a3, -k.a4), k.Ap);
            k.Am = cfma(Vm, make_double2(k.a1, -k.a2), k.Am);
        }
        k.mZ2 = 0.0;
        if (have_z) {
            k.mZ2 = st[C_MZ2 * DT];
            const double invmZ = st[C_INVMZ * DT], qZ = st[C_QZ * DT], pBZ = st[C_PBZ * DT];
            double2 Um = make_double2(0, 0), U0 = Um, Up = Um;
            spin_group<1, 0, 1>(a, 5, k.mZ2, invmZ, qZ, pBZ, bw_rec, fg_rec, Um, U0, Up);   // 1+ Z: L_R = 0, L_B = 1
            const double cZ = st[C_CZ * DT], sZ = st[C_SZ * DT], ct = st[C_CT * DT], stt = st[C_ST * DT];
            const double cpt = st[C_CPT * DT], spt = st[C_SPT * DT], ca = st[C_CA * DT], sa = st[C_SA * DT];
            const double z1 = RSQRT2 * sZ;
            const double2 T0 = cscale(cZ, U0);
            const double2 Tp = cscale(z1, cmul(make_double2(cpt, spt), Up));
            const double2 Tm = cscale(-z1, cmul(make_double2(cpt, -spt), Um));
            const double gp = 0.5 * (1.0 + ct), gm = 0.5 * (1.0 - ct), g0 = RSQRT2 * stt;
            const double2 Zp = make_double2(g0 * T0.x + gp * Tp.x + gm * Tm.x, g0 * T0.y + gp * Tp.y + gm * Tm.y);
            const double2 Zm = make_double2(-g0 * T0.x + gm * Tp.x + gp * Tm.x, -g0 * T0.y + gm * Tp.y + gp * Tm.y);
            k.Ap = cfma(make_double2(ca, sa), Zp, k.Ap);
            k.Am = cfma(make_double2(ca, -sa), Zm, k.Am);
        }
        const double S0 = fma(k.Ap.x, k.Ap.x, fma(k.Ap.y, k.Ap.y, fma(k.Am.x, k.Am.x, k.Am.y * k.Am.y)));
        const double w = is_norm ? st[NCOL_ALL * DT] : 0.0;
        if (is_norm) {
            bad |= live && !isfinite(S0);
            acc0N = fma(w, S0, acc0N);      // padding events carry w = 0
        } else {
            const bool ok = S0 > 0.0 && isfinite(S0);
            bad |= live && !ok;
            double f; int e1, e2;
            split_exp((live && ok) ? S0 : 1.0, &f, &e1);
            split_exp(acc0F * f, &acc0F, &e2);   // running product of mantissas, renormalised to [0.5, 1)
            acc0E += e1 + e2;
        }
        // ---- the points, 32 per block; the warp totals go to the per-warp accumulators
        int it = 0;
        for (int b = 0; b < nblk; ++b) {
            double v; int e;
            const int slot = b * DT + warp * 32 + lane;
            if (is_norm) {
                eval_block<true>(d.items, it, k, bw_rec, fg_rec, st, w, live, bad, lane, &v, &e);
                accN[slot] += v;
            } else {
                eval_block<false>(d.items, it, k, bw_rec, fg_rec, st, w, live, bad, lane, &v, &e);
                double f; int e2;
                split_exp(accF[slot] * v, &f, &e2);
                accF[slot] = f;
                accE[slot] += e + e2;
            }
        }
        __syncthreads();   // every thread is done with this buffer
    }
    if (bad) atomicOr(a.flag, 2);

    // ---- per-CTA partials: partial[(seg * rows + row) * stride + cta], seg 0 = sum log S (data), 1 = sum w S (norm);
    //      row 0 = point 0, row 1 + s = sorted point s
    const double LN2 = 0.69314718055994530942;
    const int rows = 1 + d.nsorted;
    {
        const double t0 = block_sum(log(acc0F) + (double)acc0E * LN2, sm);
        const double t1 = block_sum(acc0N, sm);
        if (tid == 0) { d.partial[(size_t)0 * d.stride + blockIdx.x] = t0; d.partial[(size_t)rows * d.stride + blockIdx.x] = t1; }
    }
    for (int idx = tid; idx < d.nsorted; idx += DT) {
        const int b = idx >> 5, l = idx & 31;
        double sN = 0.0, sL = 0.0;
        for (int wv = 0; wv < 8; ++wv) {   // the 8 warp totals in warp order
            const int slot = b * DT + wv * 32 + l;
            sN += accN[slot];
            sL += log(accF[slot]) + (double)accE[slot] * LN2;
        }
        d.partial[(size_t)(1 + idx) * d.stride + blockIdx.x] = sL;
        d.partial[(size_t)(rows + 1 + idx) * d.stride + blockIdx.x] = sN;
    }
    // ---- the last CTA to finish adds the partials of every row in CTA order and forms NLL(p), I(p)
    __threadfence();
    __syncthreads();
    if (tid == 0) s_last = atomicAdd(a.ticket, 1u) == gridDim.x - 1;
    __syncthreads();
    if (!s_last) return;
    __threadfence();
    double* tot = accN;   // [2 rows] (accN/accF are dead; 2 * 129 doubles fit)
    for (int r = tid; r < 2 * rows; r += DT) {
        const double* p = d.partial + (size_t)r * d.stride;
        double s = 0.0;
        for (unsigned c = 0; c < gridDim.x; ++c) s += __ldcg(p + c);
        tot[r] = s;
    }
    __syncthreads();
    for (int r = tid; r < rows; r += DT) {
        const int p = r == 0 ? 0 : d.point_of_sorted[r - 1];
        if (p < 0) continue;
        const double I = tot[rows + r] / a.wsum;
        d.result[d.P + p] = I;
        double v = -(tot[r] + a.sum_log_eff) + (double)a.n * log(I);
        if (!isfinite(v) || !(I > 0.0)) v = INFINITY;
        d.result[p] = d.want_nll ? v : 0.0;
    }
    if (tid == 0) {
        d.result[2 * d.P] = (double)atomicExch(a.flag, 0);
        *a.ticket = 0u;
    }
}

namespace {

size_t delta_smem(int nent, int ngrp) {
    return (size_t)2 * DNCOL * DT * sizeof(double) + (size_t)(nent + ngrp) * DT * sizeof(double2) + (size_t)DBLK * DT * (2 * sizeof(double) + sizeof(int)) +
           2 * sizeof(uint64_t);
}

}  // namespace

bool delta_fits(int nent, int ngrp) { return delta_smem(nent, ngrp) <= (size_t)224 * 1024; }

int delta_grid(long long n_data, long long n_norm) {
    const long long ntiles = (n_data + DT - 1) / DT + (n_norm + DT - 1) / DT;
    return (int)(ntiles < 1 ? 1 : (ntiles > 148 ? 148 : ntiles));   // persistent: one CTA per SM
}

cudaError_t launch_delta(const DeltaArgs& d, int grid, cudaStream_t s) {
    static bool attr_done = false;
    cudaError_t e = cudaSuccess;
    if (!attr_done) { e = cudaFuncSetAttribute(k_delta, cudaFuncAttributeMaxDynamicSharedMemorySize, 224 * 1024); attr_done = true; }
    if (e != cudaSuccess) return e;
    int nent = 0;
    for (int sp = 0; sp < 6; ++sp) nent += d.a.shape[sp];
    k_delta<<<grid, DT, delta_smem(nent, d.a.gstart[6]), s>>>(d);
    return cudaGetLastError();
}

}  // namespace amp
