// deltan.cu — the NORMALISATION events of a gradient batch of the paper's resonance lists (deltaf.cu has the method and the
// data events; PAPER.md:53 for the Monte Carlo integral, PAPER.md:191 for the batch).  On this side nothing depends on the point:
//   sum_j w_j S_j(p) = sum_j w_j S0_j + a sum_j L'_k.x + b sum_j L'_k.y + c2 sum_j n'_k        (coupling point on position k)
//   sum_j w_j S_j(p) = sum_j w_j S0_j + sum_j x_j(p)                                           (lineshape point)
// with L'_k = 2 w conj(BW_R) d^J_{lambda 0} W_lambda and n'_k = w |BW_R|^2 (d^J_{lambda 0})^2 sum_xi (d^1_{lambda xi})^2, so every
// sum can be a REGISTER of the thread that owns the event, as in gradf.cu (whose leaves the sums of L' are): no exchange between
// lanes, independent FMAs, one reduction per CTA.  All of them do not fit one thread (2 NSLOT + ~2 NENT + 4 NENT doubles next to
// the forward pass's working set), so the sample is walked TWICE, each pass with the forward pass of point 0:
//   PASS 0   sum w S0 and the 2 NSLOT sums of L' (four FMAs per slot and event)                           — gradf.cu's loop
//   PASS 1   the sums of n' (one or two per entry, a Z's tied pair a third) and the four lineshape sums x of every entry that has
//            lineshape points; its last CTA adds the per-CTA partials of both passes in CTA order and scatters the totals into
//            k_deltaf's value rows (DeltaFArgs::norm_tot), which the data-side launch that follows on the same stream picks up.
// Measured on configs[4] (10M normalisation events): 0.44 + 0.91 ms, against 1.7 ms for the same events inside k_deltaf (two CTAs of
// 128 registers per SM, every sum through the shared-memory tile); one pass with everything in registers spills to L2 (1.74 ms),
// the lineshape sums in thread-private shared-memory columns instead of (spilling) registers: 0.96 ms.
//
// Pipeline: gradf.cu's (256-event units, TMA bulk copies with full / empty mbarriers, producer duty rotating over the warps, one
// CTA of 256 threads per SM); four stages in pass 0, two in pass 1 (which leaves the L1 room for its 0.4 KB of spills per thread).
// Fixed order everywhere: bit-reproducible.  Bound: plain FP64 ALUs.
#include "deltaf_core.cuh"

namespace amp {

namespace {


constexpr int RED_DOUBLES = 2048;   // the flush buffer (the partial rows of every warp), then the totals of the finish

// acc += conj(bw) x
__device__ __forceinline__ void conj_fma(double2 bw, double2 x, double2& acc) {
    acc.x = fma(bw.x, x.x, fma(bw.y, x.y, acc.x));
    acc.y = fma(bw.x, x.y, fma(-bw.y, x.x, acc.y));
}

// lineshapes of one spin class, kept: U_l += c BW (couplings carry kN), rec[t] = BW / kN, F / G the class's barrier factors
template <int J, int LRv, int LBv, int CNT, int OFF, int SPIN>
__device__ __forceinline__ void class_forward_keep(const StreamArgs& a, double m2, double invm, double pR, double pB, double2* rec, double& F,
                                                   double& G, double2& Um, double2& U0, double2& Up) {
    group_factors<LRv, LBv>(a.r2_spin[SPIN], invm, pR, pB, &F, &G);
#pragma unroll
    for (int t = 0; t < CNT; ++t) {
        const ResEntry& en = a.ent[OFF + t];
        const double2 bw = bw_unscaled(en, m2, F, G);
        rec[OFF + t] = bw;
        U0 = cfma(en.c0, bw, U0);
        if (J) { Um = cfma(en.cm, bw, Um); Up = cfma(en.cp, bw, Up); }
    }
}

}  // namespace

template <class SH, int PASS>
__global__ void __launch_bounds__(THREADS, 1) k_deltan(const __grid_constant__ DeltaFArgs d) {
    using L = DLay<SH>;
    constexpr int NENT = L::NENT, NSLOT = L::NSLOT;
    constexpr int NROW = 1 + 2 * NSLOT + 8 * NENT;   // partial rows: sum w S0; the leaves (x, y per slot); eight values per entry
    constexpr bool have_z = SH::nz > 0;
    constexpr int NSTAGE_N = PASS == 0 ? 4 : 2;
    const StreamArgs& a = d.a;
    const double RSQRT2 = 0.70710678118654752440;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int ncolw = a.ncolw;

    extern __shared__ __align__(128) unsigned char smem_raw[];
    double* stage0 = reinterpret_cast<double*>(smem_raw);                                        // [NSTAGE_N][ncolw][UNIT]
    double* red = stage0 + (size_t)NSTAGE_N * ncolw * UNIT;                                      // flush: [NWARPS][NRED]; finish: NROW totals
    uint64_t* full = reinterpret_cast<uint64_t*>(red + RED_DOUBLES);
    __shared__ double sm[NWARPS];
    __shared__ bool s_last;
    uint64_t* empty = full + NSTAGE_N;
    if (tid == 0) {
        for (int s = 0; s < NSTAGE_N; ++s) { mbar_init(&full[s], 1); mbar_init(&empty[s], NWARPS); }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();
    const long long nunits = UPB * ((a.n2 + CACHE_TILE - 1) / CACHE_TILE);
    auto issue = [&](long long unit, int s) {   // one warp: one 2 KB copy per cache column
        const double* src = a.cache2 + (size_t)(unit / UPB) * ncolw * CACHE_TILE + (size_t)(unit % UPB) * UNIT;
        if (lane == 0) mbar_expect_tx(&full[s], (uint32_t)ncolw * UNIT * sizeof(double));
        __syncwarp();
        if (lane < ncolw) bulk_g2s(stage0 + ((size_t)s * ncolw + lane) * UNIT, src + (size_t)lane * CACHE_TILE, UNIT * sizeof(double), &full[s]);
    };
    if (warp == 0)
        for (int s = 0; s < NSTAGE_N; ++s)
            if (blockIdx.x + (long long)s * gridDim.x < nunits) issue(blockIdx.x + (long long)s * gridDim.x, s);

    double2 acc[PASS == 0 ? NSLOT : 1];     // sums of L' per coupling slot (entry order; lambda = -1, 0, +1 within an entry of spin >= 1)
    double nacc[PASS == 1 ? NENT : 1][3];   // sums of n' per entry: lambda = 0; lambda = +-1; a Z's tied pair
    double lacc[PASS == 1 ? NENT : 1][4];   // the four lineshape sums per entry (the ones of entries without lineshape points stay zero)
#pragma unroll
    for (int q = 0; q < (PASS == 0 ? NSLOT : 1); ++q) acc[q] = make_double2(0.0, 0.0);
#pragma unroll
    for (int t = 0; t < (PASS == 1 ? NENT : 1); ++t) {
        nacc[t][0] = nacc[t][1] = nacc[t][2] = 0.0;
        lacc[t][0] = lacc[t][1] = lacc[t][2] = lacc[t][3] = 0.0;
    }
    double accW = 0.0;
    bool bad = false;

    long long k = 0;
    for (long long unit = blockIdx.x; unit < nunits; unit += gridDim.x, ++k) {
        const int s = (int)(k % NSTAGE_N);
        const uint32_t parity = (uint32_t)((k / NSTAGE_N) & 1);
        const bool live = unit * UNIT + tid < a.n2;
        mbar_wait(&full[s], parity);
        const double* st = stage0 + (size_t)s * ncolw * UNIT + tid;
        // ---- point 0: K* chain (Eq. 4)
        const double m2 = st[C_M2 * UNIT], invm = st[C_INVM * UNIT], q = st[C_Q * UNIT], pB = st[C_PB * UNIT];
        const double cK = st[C_CK * UNIT], sK = st[C_SK * UNIT], cK2 = cK * cK;
        // d^J_{00} = P_J(cK), d^J_{+1,0} = -sK P_J'(cK) / sqrt(J(J+1))
        const double d10 = cK, d11 = -RSQRT2 * sK;
        const double d20 = fma(1.5, cK2, -0.5), d21 = -1.2247448713915890491 * sK * cK;
        const double d30 = cK * fma(2.5, cK2, -1.5), d31 = -0.43301270189221932338 * sK * fma(5.0, cK2, -1.0);
        const double d40 = fma(fma(4.375, cK2, -3.75), cK2, 0.375), d41 = -0.55901699437494742410 * sK * cK * fma(7.0, cK2, -3.0);
        double2 V0 = make_double2(0, 0), Vp = V0, Vm = V0;
        double2 rec[NENT];      // BW_R / kN of this event
        double Fc[6], Gc[6];    // barrier factors of the spin classes (5: the Z's)
#define AMP_FSPIN(J, LB, CNT, OFF, D0, D1)                                                            \
        if (CNT > 0) {                                                                                 \
            double2 Um = make_double2(0, 0), U0 = Um, Up = Um;                                         \
            class_forward_keep<J, J, LB, CNT, OFF, J>(a, m2, invm, q, pB, rec, Fc[J], Gc[J], Um, U0, Up); \
            V0 = cadd(V0, cscale(D0, U0));                                                             \
            if (J) { Vp = cadd(Vp, cscale(D1, Up)); Vm = cadd(Vm, cscale(-(D1), Um)); }                \
        }
        AMP_FSPIN(0, 1, SH::n0, 0, 1.0, 0.0)
        AMP_FSPIN(1, 0, SH::n1, SH::o1, d10, d11)
        AMP_FSPIN(2, 1, SH::n2, SH::o2, d20, d21)
        AMP_FSPIN(3, 2, SH::n3, SH::o3, d30, d31)
        AMP_FSPIN(4, 3, SH::n4, SH::o4, d40, d41)
#undef AMP_FSPIN
        // A_xi = sum_l g_{l,xi} V_l with g_{0,+-} = +-h0, g_{+1,+} = a1 + i a2, g_{+1,-} = a3 + i a4, g_{-1,+} = a3 - i a4, g_{-1,-} = a1 - i a2
        const double cpsi = st[C_CPSI * UNIT], spsi = st[C_SPSI * UNIT], cphi = st[C_CPHI * UNIT], sphi = st[C_SPHI * UNIT];
        const double hp = 0.5 * (1.0 + cpsi), hm = 0.5 * (1.0 - cpsi), h0 = RSQRT2 * spsi;
        const double a1 = hp * cphi, a2 = hp * sphi, a3 = hm * cphi, a4 = hm * sphi;
        double2 Ap = make_double2(h0 * V0.x, h0 * V0.y);
        double2 Am = make_double2(-Ap.x, -Ap.y);
        Ap = cfma(Vp, make_double2(a1, a2), Ap);
        Am = cfma(Vp, make_double2(a3, a4), Am);
        Ap = cfma(Vm, make_double2(a3, -a4), Ap);
        Am = cfma(Vm, make_double2(a1, -a2), Am);
        // ---- point 0: Z chain (Eq. 10), 1+ only in the specialised shapes
        double mZ2 = 0, zc0 = 0, zcp = 0, gp = 0, gm = 0, g0 = 0, cpt = 0, spt = 0, ca = 0, sa = 0;
        if (have_z) {
            mZ2 = st[C_MZ2 * UNIT];
            const double invmZ = st[C_INVMZ * UNIT], qZ = st[C_QZ * UNIT], pBZ = st[C_PBZ * UNIT];
            zc0 = st[C_CZ * UNIT];                       // d^1_{00}(theta_Z)
            zcp = RSQRT2 * st[C_SZ * UNIT];              // d^1_{0,+1}(theta_Z) = -d^1_{0,-1}
            const double ct = st[C_CT * UNIT], stt = st[C_ST * UNIT];
            cpt = st[C_CPT * UNIT]; spt = st[C_SPT * UNIT]; ca = st[C_CA * UNIT]; sa = st[C_SA * UNIT];
            double2 Um = make_double2(0, 0), U0 = Um, Up = Um;
            class_forward_keep<1, 0, 1, SH::nz, SH::oz, 5>(a, mZ2, invmZ, qZ, pBZ, rec, Fc[5], Gc[5], Um, U0, Up);
            const double2 T0 = cscale(zc0, U0);
            const double2 Tp = cmul(make_double2(cpt, spt), cscale(zcp, Up));      // e^{+i phi~}
            const double2 Tm = cmul(make_double2(cpt, -spt), cscale(-zcp, Um));    // e^{-i phi~}
            gp = 0.5 * (1.0 + ct); gm = 0.5 * (1.0 - ct); g0 = RSQRT2 * stt;
            const double2 Zp = make_double2(g0 * T0.x + gp * Tp.x + gm * Tm.x, g0 * T0.y + gp * Tp.y + gm * Tm.y);
            const double2 Zm = make_double2(-g0 * T0.x + gm * Tp.x + gp * Tm.x, -g0 * T0.y + gm * Tp.y + gp * Tm.y);
            Ap = cfma(make_double2(ca, sa), Zp, Ap);      // e^{+i alpha}
            Am = cfma(make_double2(ca, -sa), Zm, Am);     // e^{-i alpha}
        }
        const double wgt = st[(ncolw - 1) * UNIT];       // padding events carry w = 0
        __syncwarp();
        if (lane == 0) mbar_arrive(&empty[s]);   // this warp has read everything it needs from the stage
        // refill the stage of the PREVIOUS unit with the unit NSTAGE_N - 1 steps ahead; the warps take turns as producer (gradf.cu)
        if (k > 0 && warp == (int)(k & (NWARPS - 1)) && unit + (long long)(NSTAGE_N - 1) * gridDim.x < nunits) {
            const int ps = (int)((k - 1) % NSTAGE_N);
            mbar_wait(&empty[ps], (uint32_t)(((k - 1) / NSTAGE_N) & 1));
            issue(unit + (long long)(NSTAGE_N - 1) * gridDim.x, ps);
        }
        const double S0 = fma(Ap.x, Ap.x, fma(Ap.y, Ap.y, fma(Am.x, Am.x, Am.y * Am.y)));
        bad |= live && !isfinite(S0);
        if (PASS == 0) accW = fma(wgt, S0, accW);
        // weights as in deltaf.cu: the linear terms carry uw = 2 w, the quadratic ones un = w
        const double un = wgt, uw = un + un;
        const double2 uAp = cscale(uw, Ap), uAm = cscale(uw, Am);
        // W_l = uw sum_xi conj(g_{l,xi}) A_xi;  conj(x + i y) A = (x A.x + y A.y, x A.y - y A.x)
        const double2 W0 = make_double2(h0 * (uAp.x - uAm.x), h0 * (uAp.y - uAm.y));
        const double2 Wp = make_double2(fma(a1, uAp.x, fma(a2, uAp.y, fma(a3, uAm.x, a4 * uAm.y))),
                                        fma(a1, uAp.y, fma(-a2, uAp.x, fma(a3, uAm.y, -a4 * uAm.x))));
        // lambda = -1: g_+ = -a3 + i a4, g_- = -a1 + i a2 (the sign of d^J_{-1,0} folded in, so X_{J,-1} = d^J_{+1,0} Wm)
        const double2 Wm = make_double2(fma(-a3, uAp.x, fma(a4, uAp.y, fma(-a1, uAm.x, a2 * uAm.y))),
                                        fma(-a3, uAp.y, fma(-a4, uAp.x, fma(-a1, uAm.y, -a2 * uAm.x))));
        // sum_xi |g_{l,xi}|^2 times un: lambda = 0: 2 h0^2; lambda = +-1: hp^2 + hm^2
        const double N0 = 2.0 * h0 * h0 * un, N1 = fma(hp, hp, hm * hm) * un;

        // lineshape points of one entry (deltaf.cu): Delta = rho BW(p)/kN(p) - BW(0)/kN(0), x = Re(conj(Delta) Q) + |Delta|^2 nR
        auto lineshape_quad = [&](const int t, const double2 bw0, const double mm2, const double F, const double G, const double2 Q,
                                  const double nR) {
#pragma unroll
            for (int j = 0; j < 4; ++j) {
                const double MG = d.mw[t][j][1] * G, dre = d.mw[t][j][2] - mm2;
                const double sc = d.mw[t][j][0] * F * fast_rcp(fma(dre, dre, MG * MG));
                const double Dx = fma(sc, dre, -bw0.x), Dy = fma(sc, MG, -bw0.y);
                lacc[PASS == 1 ? t : 0][j] += fma(Dx, Q.x, fma(Dy, Q.y, fma(Dx, Dx, Dy * Dy) * nR));
            }
        };
        // one K* spin class: pass 0: the leaves; pass 1: per entry n_{lambda=0}, n_{lambda=+-1} and, if it has lineshape points, their four sums
        auto kstar_class = [&](auto Jc, auto CNTc, auto OFFc, const double d0, const double d1) {
            constexpr int J = decltype(Jc)::value, CNT = decltype(CNTc)::value, OFF = decltype(OFFc)::value;
            if (CNT == 0) return;
            const double2 X0 = cscale(d0, W0), Xp = cscale(d1, Wp), Xm = cscale(d1, Wm);
            const double n0v = d0 * d0 * N0, nm = d1 * d1 * N1;
#pragma unroll
            for (int t = 0; t < CNT; ++t) {
                const double2 bw = rec[OFF + t];
                const int b = L::base(OFF + t);
                const double bw2 = fma(bw.x, bw.x, bw.y * bw.y);
                if (PASS == 0) {
                    if (J == 0) {
                        conj_fma(bw, X0, acc[b]);
                    } else {
                        conj_fma(bw, Xm, acc[b]);
                        conj_fma(bw, X0, acc[b + 1]);
                        conj_fma(bw, Xp, acc[b + 2]);
                    }
                    continue;
                }
                nacc[PASS == 1 ? OFF + t : 0][0] = fma(bw2, n0v, nacc[PASS == 1 ? OFF + t : 0][0]);
                if (J) nacc[PASS == 1 ? OFF + t : 0][1] = fma(bw2, nm, nacc[PASS == 1 ? OFF + t : 0][1]);
                if (!((d.ent_active >> (OFF + t)) & 1u)) continue;
                const ResEntry& en = a.ent[OFF + t];
                // Q = sum_l conj(c_l) X_l;  G_xi = sum_l c_l d^J_{l0} g_{l,xi} (the sign of d^J_{-1,0} with the lambda = -1 term)
                double2 Q = conj_mul(en.c0, X0);
                double2 Gp = make_double2(d0 * h0 * en.c0.x, d0 * h0 * en.c0.y), Gm = make_double2(-Gp.x, -Gp.y);
                if (J) {
                    const double2 qp = conj_mul(en.cp, Xp), qm = conj_mul(en.cm, Xm);
                    Q = make_double2(Q.x + qp.x + qm.x, Q.y + qp.y + qm.y);
                    const double2 cp = cscale(d1, en.cp), cm = cscale(-d1, en.cm);
                    Gp = cfma(cp, make_double2(a1, a2), Gp);
                    Gm = cfma(cp, make_double2(a3, a4), Gm);
                    Gp = cfma(cm, make_double2(a3, -a4), Gp);
                    Gm = cfma(cm, make_double2(a1, -a2), Gm);
                }
                const double nR = fma(Gp.x, Gp.x, fma(Gp.y, Gp.y, fma(Gm.x, Gm.x, Gm.y * Gm.y))) * un;
                lineshape_quad(OFF + t, bw, m2, Fc[J], Gc[J], Q, nR);
            }
        };
        {
            using std::integral_constant;
            kstar_class(integral_constant<int, 0>{}, integral_constant<int, SH::n0>{}, integral_constant<int, 0>{}, 1.0, 0.0);
            kstar_class(integral_constant<int, 1>{}, integral_constant<int, SH::n1>{}, integral_constant<int, SH::o1>{}, d10, d11);
            kstar_class(integral_constant<int, 2>{}, integral_constant<int, SH::n2>{}, integral_constant<int, SH::o2>{}, d20, d21);
            kstar_class(integral_constant<int, 3>{}, integral_constant<int, SH::n3>{}, integral_constant<int, SH::o3>{}, d30, d31);
            kstar_class(integral_constant<int, 4>{}, integral_constant<int, SH::n4>{}, integral_constant<int, SH::o4>{}, d40, d41);
        }
        if (have_z) {
            // Z chain: B_{l',xi} = BW_Z d^1_{0 l'}(theta_Z) e^{i l' phi~} d^1_{l' xi}(theta~) e^{i xi alpha}
            const double2 Bp = make_double2(fma(ca, uAp.x, sa * uAp.y), fma(ca, uAp.y, -sa * uAp.x));    // conj(e^{+i alpha}) uw A+
            const double2 Bm = make_double2(fma(ca, uAm.x, -sa * uAm.y), fma(ca, uAm.y, sa * uAm.x));    // conj(e^{-i alpha}) uw A-
            const double2 Y0 = make_double2(zc0 * g0 * (Bp.x - Bm.x), zc0 * g0 * (Bp.y - Bm.y));
            const double2 Rp = make_double2(fma(gp, Bp.x, gm * Bm.x), fma(gp, Bp.y, gm * Bm.y));         // l' = +1: d^1_{1,+} = gp, d^1_{1,-} = gm
            const double2 Rm = make_double2(fma(gm, Bp.x, gp * Bm.x), fma(gm, Bp.y, gp * Bm.y));         // l' = -1
            // conj(e^{+-i phi~}) R, times d^1_{0,+-1}(theta_Z) = +-zcp
            const double2 Yp = make_double2(zcp * fma(cpt, Rp.x, spt * Rp.y), zcp * fma(cpt, Rp.y, -spt * Rp.x));
            const double2 Ym = make_double2(-zcp * fma(cpt, Rm.x, -spt * Rm.y), -zcp * fma(cpt, Rm.y, spt * Rm.x));
            // sum_xi |d^1_{0 l'} d^1_{l' xi}|^2 un, and for the tied pair (l' = -1 and +1 moving together) the cross term (deltaf.cu)
            const double NZ0 = zc0 * zc0 * 2.0 * g0 * g0 * un;
            const double NZ1 = zcp * zcp * fma(gp, gp, gm * gm) * un;
            const double NZc = -4.0 * zcp * zcp * gp * gm * fma(cpt, cpt, -spt * spt) * un;
#pragma unroll
            for (int z = 0; z < SH::nz; ++z) {
                const double2 bw = rec[SH::oz + z];
                const int b = L::base(SH::oz + z);
                const double bw2 = fma(bw.x, bw.x, bw.y * bw.y);
                if (PASS == 0) {
                    conj_fma(bw, Ym, acc[b]);
                    conj_fma(bw, Y0, acc[b + 1]);
                    conj_fma(bw, Yp, acc[b + 2]);
                    continue;
                }
                {
                    double* na = nacc[PASS == 1 ? SH::oz + z : 0];
                    na[0] = fma(bw2, NZ0, na[0]);
                    na[1] = fma(bw2, NZ1, na[1]);
                    na[2] = fma(bw2, NZ1 + NZ1 + NZc, na[2]);
                }
                if (!((d.ent_active >> (SH::oz + z)) & 1u)) continue;
                const ResEntry& en = a.ent[SH::oz + z];
                const double2 q0 = conj_mul(en.c0, Y0), qp = conj_mul(en.cp, Yp), qm = conj_mul(en.cm, Ym);
                const double2 Q = make_double2(q0.x + qp.x + qm.x, q0.y + qp.y + qm.y);
                // G_xi / e^{i xi alpha} = sum_l' c_l' d^1_{0 l'} e^{i l' phi~} d^1_{l' xi}(theta~): the forward combination with c in place of U
                const double2 T0 = cscale(zc0, en.c0);
                const double2 Tp = cmul(make_double2(cpt, spt), cscale(zcp, en.cp));
                const double2 Tm = cmul(make_double2(cpt, -spt), cscale(-zcp, en.cm));
                const double2 Zp = make_double2(g0 * T0.x + gp * Tp.x + gm * Tm.x, g0 * T0.y + gp * Tp.y + gm * Tm.y);
                const double2 Zm = make_double2(-g0 * T0.x + gm * Tp.x + gp * Tm.x, -g0 * T0.y + gm * Tp.y + gp * Tm.y);
                const double nR = fma(Zp.x, Zp.x, fma(Zp.y, Zp.y, fma(Zm.x, Zm.x, Zm.y * Zm.y))) * un;
                lineshape_quad(SH::oz + z, bw, mZ2, Fc[5], Gc[5], Q, nR);
            }
        }
    }
    if (bad) atomicOr(a.flag, 2);

    // ---- per-CTA partials: row 0 = sum w S0; rows 1 + 2 q, 2 + 2 q = the leaf of slot q; rows 1 + 2 NSLOT + 8 t + r = value r of entry t
    constexpr int NRED = 2 * NSLOT + 8 * NENT;
    static_assert(NWARPS * NRED <= RED_DOUBLES && NROW <= RED_DOUBLES, "the flush buffer");
    __syncthreads();
    if (PASS == 0) {
#pragma unroll
        for (int qq = 0; qq < (PASS == 0 ? NSLOT : 1); ++qq) {   // summed over the warp by a fixed xor tree
            double x = acc[qq].x, y = acc[qq].y;
#pragma unroll
            for (int o = 16; o; o >>= 1) { x += __shfl_xor_sync(0xffffffffu, x, o); y += __shfl_xor_sync(0xffffffffu, y, o); }
            if (lane == 0) { red[warp * NRED + 2 * qq] = x; red[warp * NRED + 2 * qq + 1] = y; }
        }
    } else {
#pragma unroll
        for (int t = 0; t < (PASS == 1 ? NENT : 1); ++t)
#pragma unroll
            for (int r = 0; r < 8; ++r) {
                double v = r < 3 ? nacc[t][r] : (r == 3 ? 0.0 : lacc[t][r - 4]);
#pragma unroll
                for (int o = 16; o; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
                if (lane == 0) red[warp * NRED + 2 * NSLOT + 8 * t + r] = v;
            }
    }
    __syncthreads();
    for (int idx = tid + (PASS == 0 ? 0 : 2 * NSLOT); idx < (PASS == 0 ? 2 * NSLOT : NRED); idx += THREADS) {   // over the warps in warp order
        double s = 0.0;
        for (int wv = 0; wv < NWARPS; ++wv) s += red[wv * NRED + idx];
        d.npartial[(size_t)(1 + idx) * d.stride + blockIdx.x] = s;
    }
    __syncthreads();
    if (PASS == 0) {
        const double t1 = block_sum(accW, sm);
        if (tid == 0) d.npartial[blockIdx.x] = t1;
        return;
    }
    // ---- the last CTA to finish adds the partials of every row in CTA order and scatters the totals into k_deltaf's value rows
    __threadfence();
    __syncthreads();
    if (tid == 0) s_last = atomicAdd(a.ticket, 1u) == gridDim.x - 1;
    __syncthreads();
    if (!s_last) return;
    __threadfence();
    double* tot = red;
    for (int r = tid; r < NROW; r += THREADS) {
        const double* p = d.npartial + (size_t)r * d.stride;
        double s = 0.0;
        for (unsigned c = 0; c < gridDim.x; ++c) s += __ldcg(p + c);
        tot[r] = s;
    }
    __syncthreads();
    double* out = d.norm_tot + 1;
    const double* leaf = tot + 1;               // (x, y) of slot q at leaf[2 q], leaf[2 q + 1]
    const double* tv = tot + 1 + 2 * NSLOT;     // value r of entry t at tv[8 t + r]: n_{lambda=0}, n_{lambda=+-1}, n of a Z's tied pair, -, then the four lineshape values
    for (int t = tid; t < NENT; t += THREADS) {
        const int b = L::base(t);
        if (t < SH::n0) {
            double* o = out + 4 * d.quad_of_pos[b];
            o[0] = leaf[2 * b]; o[1] = leaf[2 * b + 1]; o[2] = tv[8 * t]; o[3] = 0.0;
        } else {
            for (int j = 0; j < 3; ++j) {
                double* o = out + 4 * d.quad_of_pos[b + j];
                o[0] = leaf[2 * (b + j)]; o[1] = leaf[2 * (b + j) + 1]; o[2] = tv[8 * t + (j == 1 ? 0 : 1)]; o[3] = 0.0;
            }
            if (t >= SH::oz) {   // a Z: the tied pair moves lambda' = -1 and +1 together
                double* o = out + 4 * d.quad_of_pos[NSLOT + (t - SH::oz)];
                o[0] = leaf[2 * b] + leaf[2 * (b + 2)]; o[1] = leaf[2 * b + 1] + leaf[2 * (b + 2) + 1]; o[2] = tv[8 * t + 2]; o[3] = 0.0;
            }
        }
        double* o = out + 4 * d.quad_of_ent[t];
        for (int j = 0; j < 4; ++j) o[j] = tv[8 * t + 4 + j];
    }
    if (tid == 0) {
        d.norm_tot[0] = tot[0];
        *a.ticket = 0u;     // (the domain flag stays for the data-side launch, which reports and clears it)
    }
}

namespace {

template <class SH>
size_t deltan_smem(int ncolw, int nstage) {
    return (size_t)nstage * ncolw * UNIT * sizeof(double) + (size_t)RED_DOUBLES * sizeof(double) + 2 * nstage * sizeof(uint64_t);
}

template <class SH>
cudaError_t launch_deltan_shape(const DeltaFArgs& d, int grid, int pass, cudaStream_t s) {
    static DeviceOnce attr_done;
    cudaError_t e = cudaSuccess;
    if (attr_done.first()) {
        e = cudaFuncSetAttribute(k_deltan<SH, 0>, cudaFuncAttributeMaxDynamicSharedMemorySize, 224 * 1024);
        if (e == cudaSuccess) e = cudaFuncSetAttribute(k_deltan<SH, 1>, cudaFuncAttributeMaxDynamicSharedMemorySize, 224 * 1024);
    }
    if (e != cudaSuccess) return e;
    if (pass == 0) k_deltan<SH, 0><<<grid, THREADS, deltan_smem<SH>(d.a.ncolw, 4), s>>>(d);
    else k_deltan<SH, 1><<<grid, THREADS, deltan_smem<SH>(d.a.ncolw, 2), s>>>(d);
    return cudaGetLastError();
}

}  // namespace

int deltan_grid(long long n_norm) {
    const long long nunits = UPB * ((n_norm + CACHE_TILE - 1) / CACHE_TILE);
    return (int)(nunits < 1 ? 1 : (nunits > sm_count() ? sm_count() : nunits));   // persistent: one CTA per SM
}

// the shapes of deltaf.cu (deltaf_layout decides); pass 0, then pass 1 with the same grid on the same stream
cudaError_t launch_deltan(const DeltaFArgs& d, int grid, int pass, cudaStream_t s) {
    switch (d.a.shape[5]) {
        case 0: return launch_deltan_shape<Shape<3, 3, 2, 1, 1, 0>>(d, grid, pass, s);
        case 1: return launch_deltan_shape<Shape<3, 3, 2, 1, 1, 1>>(d, grid, pass, s);
        default: return launch_deltan_shape<Shape<3, 3, 2, 1, 1, 2>>(d, grid, pass, s);
    }
}

}  // namespace amp
