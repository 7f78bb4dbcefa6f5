// deltaf.cu — steps a2 + a3 + a4 + a5 for a GRADIENT BATCH of the paper's resonance lists: the shape-specialised form of delta.cu
// ("> 60 free parameters": MINUIT's finite-difference step is the central point plus theta_k +- h_k; BASELINE.json
// configs[4]).  Every point other than point 0 changes ONE thing:
//   a coupling H_k by delta (or the two tied helicities of a 1+ Z, Eq. 11, by the same delta), or
//   the mass / width of one resonance R.
// Eq. 12 is linear in (coupling x lineshape), so with A_xi = A_xi(0), S0 = sum_xi |A_xi|^2 and B_k,xi the basis
// terms of Eqs. 4 and 10
//   S(p) = S0 + 2 Re(conj(delta) L_k) + |delta|^2 n_k,        L_k = sum_xi conj(B_k,xi) A_xi,   n_k = sum_xi |B_k,xi|^2
//   S(p) = S0 + 2 Re(conj(Delta) Q_R) + |Delta|^2 n_R,        Delta = BW_R(p) - BW_R(0) (per event),
//                                                             Q_R = sum_l conj(c_R,l) L_(R,l) / conj(BW_R),  n_R = sum_xi |sum_l c_R,l g_(R,l),xi|^2
// exactly (no truncation).  L_k factors as in the analytic gradient (gradf.cu): three complex W_lambda per event and chain, one
// real scaling per spin, one complex multiply per slot; n_k = |BW_R|^2 (d^J_{lambda 0})^2 sum_xi (d^1_{lambda xi})^2.
//   data events:           log S(p) = log S0 + log r,  r = 1 + [2 Re(conj(delta) L_k) + |delta|^2 n_k] / S0 — three FMAs per point; the
//                          r of a point are multiplied up (no logarithm and no exponent bookkeeping per event: r is near 1)
//   normalisation events:  a coupling point needs NO per-point work: sum_j w_j S_j(p) = sum w S0 + 2 Re(conj(delta) sum_j w_j L_k) +
//                          |delta|^2 sum_j w_j n_k, three sums per SLOT; lineshape points accumulate w (S(p) - S0).
// NLL(p) - NLL(0) is thus formed from small quantities directly, not as a difference of two 1e6-sized sums.
//
// The set of values per event is STATIC for a model shape — four per coupling position (entry order; J = 0: lambda = 0; J >= 1:
// lambda = -1, 0, +1; per Z one more position for the tied pair) and four per entry for its lineshape points — so the code is
// straight-line: no program decode, no slot records, no per-point branches.  The host fills the coefficient tables of the
// positions in use (DeltaFArgs, kernel parameter space: operands come from the constant bank) and maps points to value slots.
// Values are summed over a warp's 32 events through a per-warp shared-memory tile (struct Tile below: one store, half a 16-byte
// load and one add or multiply per value and lane), which leaves lane l with the total of value 8 c + l % 8 of chunk c over a
// quarter of the events in a register; per-CTA partials, last-CTA finish: bit-reproducible.
// A change so large that r leaves [0.5, 1.5] trips the guard (flag 1024): the host repeats the call with delta.cu's exact form.
//
// Pipeline: as gradf.cu (256-event units, a ring of TMA-fed stages with full / empty mbarriers, producer duty rotates over the
// warps), but TWO CTAs of 256 threads per SM at 128 registers with two stages each: the values pass is long dependent chains, and
// sixteen warps hide them better than eight (measured on configs[4]: 2.53 ms against 2.76 ms for one CTA at 255 registers with
// four stages; four CTAs of 128 threads or one of 512: 2.41 / 2.44 against 2.29 ms).  To fit, the lineshapes of point 0 are not kept across the forward pass (they are
// re-evaluated class by class from the saved barrier factors) and the Z-chain angles are read again from the stage, which a
// warp releases only after its values pass.  Bound: plain FP64 ALUs.
#include "deltaf_core.cuh"

namespace amp {

namespace {

constexpr int NSTAGE = 2;       // stages per CTA
constexpr int DELTAF_MINB = 2;               // CTAs per SM

}  // namespace

// The unrolled body of one phase is ~50 KB of code, more than the SM's 32 KB instruction cache, and sixteen warps drifting apart in
// it made instruction fetch the bound (I-cache hit rate 77 %, GPC instruction-cache requests at 86 % of peak).  A CTA's warps
// therefore meet at a named barrier at the start of every unit, so that each CTA is ONE stream through the code (hit rate > 92 %).
// With the exchange tree of the first version meeting again at every spin class paid (2.57 -> 2.28 ms); with the shared-memory
// tile it no longer does (2.29 against 2.20 ms for the unit-only barrier), and finer meeting points never did.
__device__ __forceinline__ void align_warps() { asm volatile("bar.sync 1, %0;" ::"n"(THREADS) : "memory"); }

template <class SH>
__global__ void __launch_bounds__(THREADS, DELTAF_MINB) k_deltaf(const __grid_constant__ DeltaFArgs d) {
    using L = DLay<SH>;
    constexpr int NENT = L::NENT, NSLOT = L::NSLOT, NPOS = L::NPOS, NVAL = L::NVAL, NCH = L::NCH, NVP = 8 * NCH;
    constexpr bool have_z = SH::nz > 0;
    const StreamArgs& a = d.a;
    const double RSQRT2 = 0.70710678118654752440, LN2 = 0.69314718055994530942;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int ncolw = a.ncolw;                      // cache columns per block, the weight last

    extern __shared__ __align__(128) unsigned char smem_raw[];
    double* stage0 = reinterpret_cast<double*>(smem_raw);                                        // [NSTAGE][ncolw][UNIT]
    double* red = stage0 + (size_t)NSTAGE * ncolw * UNIT;                                        // [NWARPS] value tiles of 2 KB; flush: [NWARPS][NVP]; finish: 2 + 2 NVAL totals
    uint64_t* full = reinterpret_cast<uint64_t*>(red + NWARPS * (TILE_BYTES / 8));
    __shared__ double sm[NWARPS];
    __shared__ bool s_last;
    uint64_t* empty = full + NSTAGE;   // a stage is free again once every warp has read its event's columns
    if (tid == 0) {
        for (int s = 0; s < NSTAGE; ++s) { mbar_init(&full[s], 1); mbar_init(&empty[s], NWARPS); }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();
    // units: the halves of the data blocks, then the halves of the normalisation blocks
    const long long nud = d.want_nll ? UPB * ((a.n + CACHE_TILE - 1) / CACHE_TILE) : 0, nunits = nud + UPB * ((a.n2 + CACHE_TILE - 1) / CACHE_TILE);
    auto issue = [&](long long unit, int s) {   // one warp: one 2 KB copy per cache column
        const bool nrm = unit >= nud;
        const long long lu = nrm ? unit - nud : unit;
        const double* src = (nrm ? a.cache2 : a.cache) + (size_t)(lu / UPB) * ncolw * CACHE_TILE + (size_t)(lu % UPB) * UNIT;
        if (lane == 0) mbar_expect_tx(&full[s], (uint32_t)ncolw * UNIT * sizeof(double));
        __syncwarp();
        if (lane < ncolw) bulk_g2s(stage0 + ((size_t)s * ncolw + lane) * UNIT, src + (size_t)lane * CACHE_TILE, UNIT * sizeof(double), &full[s]);
    };
    if (warp == 0)
        for (int s = 0; s < NSTAGE; ++s)
            if (blockIdx.x + (long long)s * gridDim.x < nunits) issue(blockIdx.x + (long long)s * gridDim.x, s);

    double accv[NCH];       // the lane's chunk accumulators: products of r (data units, with exponents accx), then sums (normalisation units)
    int accx[NCH];
    Tile<false, NCH> td;    // data side: products of r
    Tile<true, NCH> tn;     // normalisation side: sums
    td.init(smem_u32(red) + warp * TILE_BYTES, lane);
    tn.init(smem_u32(red) + warp * TILE_BYTES, lane);
    td.acc = tn.acc = accv;
#pragma unroll
    for (int c = 0; c < NCH; ++c) { accv[c] = 1.0; accx[c] = 0; }
    double acc0F = 1.0, acc0W = 0.0;   // point 0: sum log S as mantissa product / exponent sum; sum w S
    int acc0E = 0;
    int bad = 0;                       // 1: a density that is not finite and positive; 2: the guard on r tripped
    bool in_norm = false;

    // per-CTA partial rows [row0, row0 + NVAL) of the lanes' block accumulators: summed over the warps in warp order
    auto flush = [&](int row0, bool data) {
        __syncthreads();   // (every warp is done with its value tile: the flush buffer lies over the tiles)
#pragma unroll
        for (int c = 0; c < NCH; ++c) {
            // lane l holds value 8 c + l % 8 over a quarter of the warp's events: the four quarters in a fixed order
            double t = data ? log(accv[c]) + (double)accx[c] * LN2 : accv[c];
            t += __shfl_xor_sync(0xffffffffu, t, 8);
            t += __shfl_xor_sync(0xffffffffu, t, 16);
            if (lane < 8) red[warp * NVP + 8 * c + lane] = t;
        }
#pragma unroll
        for (int c = 0; c < NCH; ++c) { accv[c] = 0.0; accx[c] = 0; }   // (after the data flush: the sums of the normalisation units start)
        __syncthreads();
        for (int idx = tid; idx < NVAL; idx += THREADS) {
            double s = 0.0;
            for (int wv = 0; wv < NWARPS; ++wv) s += red[wv * NVP + idx];
            d.partial[(size_t)(row0 + idx) * d.stride + blockIdx.x] = s;
        }
        __syncthreads();
    };

    long long k = 0;
    for (long long unit = blockIdx.x; unit < nunits; unit += gridDim.x, ++k) {
        const int s = (int)(k % NSTAGE);
        const uint32_t parity = (uint32_t)((k / NSTAGE) & 1);
        const bool is_norm = unit >= nud;
        if (is_norm && !in_norm) {   // this CTA's data units are complete
            const double t0 = block_sum(log(acc0F) + (double)acc0E * LN2, sm);
            if (tid == 0) d.partial[(size_t)0 * d.stride + blockIdx.x] = t0;
            flush(2, true);
            in_norm = true;
        }
        const long long lu = is_norm ? unit - nud : unit;
        const bool live = lu * UNIT + tid < (is_norm ? a.n2 : a.n);
        // Refill the stage of the PREVIOUS unit (every warp releases it at the end of its values pass) with the unit NSTAGE - 1 steps
        // ahead, at the START of this unit so that the copy has the whole unit to land; the warps take turns as producer (gradf.cu).
        if (k > 0 && warp == (int)(k & (NWARPS - 1)) && unit + (long long)(NSTAGE - 1) * gridDim.x < nunits) {
            const int ps = (int)((k - 1) % NSTAGE);
            mbar_wait(&empty[ps], (uint32_t)(((k - 1) / NSTAGE) & 1));
            issue(unit + (long long)(NSTAGE - 1) * gridDim.x, ps);
        }
        mbar_wait(&full[s], parity);
        align_warps();
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
#define AMP_FSPIN(J, LB, CNT, OFF, D0, D1)                                                  \
        if (CNT > 0) {                                                                       \
            double2 Um = make_double2(0, 0), U0 = Um, Up = Um;                               \
            double Fc, Gc;                                                                   \
            class_forward<J, J, LB, CNT, OFF, J>(a, m2, invm, q, pB, Fc, Gc, Um, U0, Up);    \
            V0 = cadd(V0, cscale(D0, U0));                                                   \
            if (J) { Vp = cadd(Vp, cscale(D1, Up)); Vm = cadd(Vm, cscale(-(D1), Um)); }      \
        }
        AMP_FSPIN(0, 1, SH::n0, 0, 1.0, 0.0)
        AMP_FSPIN(1, 0, SH::n1, SH::o1, d10, d11)
        AMP_FSPIN(2, 1, SH::n2, SH::o2, d20, d21)
        AMP_FSPIN(3, 2, SH::n3, SH::o3, d30, d31)
        AMP_FSPIN(4, 3, SH::n4, SH::o4, d40, d41)
#undef AMP_FSPIN
        // A_xi = sum_l g_{l,xi} V_l with g_{0,+-} = +-h0, g_{+1,+} = a1 + i a2, g_{+1,-} = a3 + i a4, g_{-1,+} = a3 - i a4, g_{-1,-} = a1 - i a2
        // (the sign of d^J_{-1,0} = -d^J_{+1,0} is in Vm)
        const double cpsi = st[C_CPSI * UNIT], spsi = st[C_SPSI * UNIT], cphi = st[C_CPHI * UNIT], sphi = st[C_SPHI * UNIT];
        const double hp = 0.5 * (1.0 + cpsi), hm = 0.5 * (1.0 - cpsi), h0 = RSQRT2 * spsi;
        const double a1 = hp * cphi, a2 = hp * sphi, a3 = hm * cphi, a4 = hm * sphi;
        double2 Ap = make_double2(h0 * V0.x, h0 * V0.y);
        double2 Am = make_double2(-Ap.x, -Ap.y);
        Ap = cfma(Vp, make_double2(a1, a2), Ap);
        Am = cfma(Vp, make_double2(a3, a4), Am);
        Ap = cfma(Vm, make_double2(a3, -a4), Ap);
        Am = cfma(Vm, make_double2(a1, -a2), Am);
        // ---- point 0: Z chain (Eq. 10), 1+ only in the specialised shapes; its angles are read again from the stage by the values pass
        if (have_z) {
            const double mZ2 = st[C_MZ2 * UNIT], invmZ = st[C_INVMZ * UNIT], qZ = st[C_QZ * UNIT], pBZ = st[C_PBZ * UNIT];
            const double zc0 = st[C_CZ * UNIT], zcp = RSQRT2 * st[C_SZ * UNIT];   // d^1_{00}(theta_Z); d^1_{0,+1}(theta_Z) = -d^1_{0,-1}
            const double ct = st[C_CT * UNIT], stt = st[C_ST * UNIT];
            const double cpt = st[C_CPT * UNIT], spt = st[C_SPT * UNIT], ca = st[C_CA * UNIT], sa = st[C_SA * UNIT];
            double2 Um = make_double2(0, 0), U0 = Um, Up = Um;
            double Fc, Gc;
            class_forward<1, 0, 1, SH::nz, SH::oz, 5>(a, mZ2, invmZ, qZ, pBZ, Fc, Gc, Um, U0, Up);
            const double2 T0 = cscale(zc0, U0);
            const double2 Tp = cmul(make_double2(cpt, spt), cscale(zcp, Up));      // e^{+i phi~}
            const double2 Tm = cmul(make_double2(cpt, -spt), cscale(-zcp, Um));    // e^{-i phi~}
            const double gp = 0.5 * (1.0 + ct), gm = 0.5 * (1.0 - ct), g0 = RSQRT2 * stt;
            const double2 Zp = make_double2(g0 * T0.x + gp * Tp.x + gm * Tm.x, g0 * T0.y + gp * Tp.y + gm * Tm.y);
            const double2 Zm = make_double2(-g0 * T0.x + gm * Tp.x + gp * Tm.x, -g0 * T0.y + gm * Tp.y + gp * Tm.y);
            Ap = cfma(make_double2(ca, sa), Zp, Ap);      // e^{+i alpha}
            Am = cfma(make_double2(ca, -sa), Zm, Am);     // e^{-i alpha}
        }
        const double wgt = st[(ncolw - 1) * UNIT];
        const double S0 = fma(Ap.x, Ap.x, fma(Ap.y, Ap.y, fma(Am.x, Am.x, Am.y * Am.y)));
        // weights: the linear terms carry uw = 2 w (normalisation) or 2 / S0 (data), the quadratic ones un = uw / 2
        double un;
        if (is_norm) {
            bad |= (live && !isfinite(S0)) ? 1 : 0;
            acc0W = fma(wgt, S0, acc0W);        // padding events carry w = 0
            un = wgt;
        } else {
            const bool ok = S0 > 0.0 && isfinite(S0);
            bad |= (live && !ok) ? 1 : 0;
            double f; int x1, x2;
            split_exp((live && ok) ? S0 : 1.0, &f, &x1);
            split_exp(acc0F * f, &acc0F, &x2);
            acc0E += x1 + x2;
            un = (live && ok) ? fast_rcp(S0) : 0.0;   // padding and bad events: every r = 1
        }
        const double uw = un + un;
        const double2 uAp = cscale(uw, Ap), uAm = cscale(uw, Am);

        // ---- the values of this event, class by class: [coupling positions of the class's entries][tied pairs (Z)][lineshape quads]
        // coupling position: L = conj(bw) X, n = |bw|^2 nf.  Data: r_j = 1 + a_j L.x + b_j L.y + c2_j n, guarded through
        // cmax (|a_j|, |b_j| <= cmax[0], c2_j <= cmax[1]): |r - 1| <= cmax[0] (|L.x| + |L.y|) + cmax[1] n.  Normalisation: the three sums of the slot.
        auto position = [&](auto& tree, const bool norm, const int pos, const double2 Lk, const double nk) {
            if (!((d.pos_active >> pos) & 1u)) { tree.push_identity(); return; }
            if (norm) { tree.push3(Lk.x, Lk.y, nk); return; }
            if (fma(d.cmax[pos][0], fabs(Lk.x) + fabs(Lk.y), d.cmax[pos][1] * nk) > 0.5) bad |= 2;
            double r[4];
#pragma unroll
            for (int j = 0; j < 4; ++j) r[j] = fma(d.cq[pos][j][0], Lk.x, fma(d.cq[pos][j][1], Lk.y, fma(d.cq[pos][j][2], nk, 1.0)));
            tree.push4(r[0], r[1], r[2], r[3]);
        };
        // lineshape points of one entry: Delta = rho BW(p)/kN(p) - BW(0)/kN(0) with the class's barrier factors of this event,
        // x = Re(conj(Delta) Q) + |Delta|^2 nR (weights inside Q and nR); data: r = 1 + x, normalisation: x
        auto lineshape_points = [&](auto& tree, const bool norm, const int t, const double2 bw0, const double mm2, const double F, const double G,
                                    const double2 Q, const double nR) {
            double y[4];
#pragma unroll
            for (int j = 0; j < 4; ++j) {
                const double MG = d.mw[t][j][1] * G, dre = d.mw[t][j][2] - mm2;
                const double sc = d.mw[t][j][0] * F * fast_rcp(fma(dre, dre, MG * MG));
                const double Dx = fma(sc, dre, -bw0.x), Dy = fma(sc, MG, -bw0.y);
                const double x = fma(Dx, Q.x, fma(Dy, Q.y, fma(Dx, Dx, Dy * Dy) * nR));
                if (!norm && !(fabs(x) <= 0.5)) bad |= 2;
                y[j] = norm ? x : 1.0 + x;
            }
            tree.push4(y[0], y[1], y[2], y[3]);
        };
        // one K* spin class: X_{J,l} = d^J_{l0} W_l (lambda = -1 carries d^J_{+1,0}: see Wm), nf = (d^J_{l0})^2 N_l
        auto kstar_class = [&](auto& tree, const bool norm, auto Jc, auto CNTc, auto OFFc, const double2 W0,
                               const double2 Wp, const double2 Wm, const double N0, const double N1) {
            constexpr int J = decltype(Jc)::value, CNT = decltype(CNTc)::value, OFF = decltype(OFFc)::value;
            if (CNT == 0) return;
            // the class's d functions and barrier factors again (cheaper than keeping them in registers across the other classes:
            // the kernel runs two CTAs per SM at 128 registers)
            double d0, d1;
            {
                const double c = st[C_CK * UNIT], sn = st[C_SK * UNIT], c2 = c * c;
                if (J == 0) { d0 = 1.0; d1 = 0.0; }
                else if (J == 1) { d0 = c; d1 = -RSQRT2 * sn; }
                else if (J == 2) { d0 = fma(1.5, c2, -0.5); d1 = -1.2247448713915890491 * sn * c; }
                else if (J == 3) { d0 = c * fma(2.5, c2, -1.5); d1 = -0.43301270189221932338 * sn * fma(5.0, c2, -1.0); }
                else { d0 = fma(fma(4.375, c2, -3.75), c2, 0.375); d1 = -0.55901699437494742410 * sn * c * fma(7.0, c2, -3.0); }
            }
            double Fc, Gc;
            group_factors<J, (J == 0 ? 1 : J - 1)>(a.r2_spin[J], st[C_INVM * UNIT], st[C_Q * UNIT], st[C_PB * UNIT], &Fc, &Gc);
            const double cps = st[C_CPSI * UNIT], h0 = RSQRT2 * st[C_SPSI * UNIT];
            const double hp = 0.5 * (1.0 + cps), hm = 0.5 * (1.0 - cps);
            const double a1 = hp * st[C_CPHI * UNIT], a2 = hp * st[C_SPHI * UNIT], a3 = hm * st[C_CPHI * UNIT], a4 = hm * st[C_SPHI * UNIT];
            const double2 X0 = cscale(d0, W0), Xp = cscale(d1, Wp), Xm = cscale(d1, Wm);
            const double n0v = d0 * d0 * N0, nm = d1 * d1 * N1;
            double2 bwc[CNT > 0 ? CNT : 1];
#pragma unroll
            for (int t = 0; t < CNT; ++t) {
                const double2 bw = bw_unscaled(a.ent[OFF + t], m2, Fc, Gc);
                bwc[t] = bw;
                const double bw2 = fma(bw.x, bw.x, bw.y * bw.y);
                const int b = L::base(OFF + t);
                if (J == 0) {
                    position(tree, norm, b, conj_mul(bw, X0), bw2 * n0v);
                } else {
                    position(tree, norm, b, conj_mul(bw, Xm), bw2 * nm);
                    position(tree, norm, b + 1, conj_mul(bw, X0), bw2 * n0v);
                    position(tree, norm, b + 2, conj_mul(bw, Xp), bw2 * nm);
                }
            }
#pragma unroll
            for (int t = 0; t < CNT; ++t) {
                if (!((d.ent_active >> (OFF + t)) & 1u)) { tree.push_identity(); continue; }
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
                lineshape_points(tree, norm, OFF + t, bwc[t], m2, Fc, Gc, Q, nR);
            }
        };
        auto all_values = [&](auto& tree, const bool norm) {
            tree.reset_event();
            using std::integral_constant;
            {
                // W_l = uw sum_xi conj(g_{l,xi}) A_xi;  conj(x + i y) A = (x A.x + y A.y, x A.y - y A.x)
                const double2 W0 = make_double2(h0 * (uAp.x - uAm.x), h0 * (uAp.y - uAm.y));
                const double2 Wp = make_double2(fma(a1, uAp.x, fma(a2, uAp.y, fma(a3, uAm.x, a4 * uAm.y))),
                                                fma(a1, uAp.y, fma(-a2, uAp.x, fma(a3, uAm.y, -a4 * uAm.x))));
                // lambda = -1: g_+ = -a3 + i a4, g_- = -a1 + i a2 (the sign of d^J_{-1,0} folded in, so X_{J,-1} = d^J_{+1,0} Wm)
                const double2 Wm = make_double2(fma(-a3, uAp.x, fma(a4, uAp.y, fma(-a1, uAm.x, a2 * uAm.y))),
                                                fma(-a3, uAp.y, fma(-a4, uAp.x, fma(-a1, uAm.y, -a2 * uAm.x))));
                // sum_xi |g_{l,xi}|^2 times un: lambda = 0: 2 h0^2; lambda = +-1: hp^2 + hm^2
                const double N0 = 2.0 * h0 * h0 * un, N1 = fma(hp, hp, hm * hm) * un;
                kstar_class(tree, norm, integral_constant<int, 0>{}, integral_constant<int, SH::n0>{}, integral_constant<int, 0>{}, W0, Wp, Wm, N0, N1);
                kstar_class(tree, norm, integral_constant<int, 1>{}, integral_constant<int, SH::n1>{}, integral_constant<int, SH::o1>{}, W0, Wp, Wm, N0, N1);
                kstar_class(tree, norm, integral_constant<int, 2>{}, integral_constant<int, SH::n2>{}, integral_constant<int, SH::o2>{}, W0, Wp, Wm, N0, N1);
                kstar_class(tree, norm, integral_constant<int, 3>{}, integral_constant<int, SH::n3>{}, integral_constant<int, SH::o3>{}, W0, Wp, Wm, N0, N1);
                kstar_class(tree, norm, integral_constant<int, 4>{}, integral_constant<int, SH::n4>{}, integral_constant<int, SH::o4>{}, W0, Wp, Wm, N0, N1);
            }
            if (have_z) {
                // the Z chain's angles again from the stage (not kept in registers across the K* classes)
                const double mZ2 = st[C_MZ2 * UNIT];
                const double zc0 = st[C_CZ * UNIT], zcp = RSQRT2 * st[C_SZ * UNIT];
                const double ct = st[C_CT * UNIT], stt = st[C_ST * UNIT];
                const double cpt = st[C_CPT * UNIT], spt = st[C_SPT * UNIT], ca = st[C_CA * UNIT], sa = st[C_SA * UNIT];
                const double gp = 0.5 * (1.0 + ct), gm = 0.5 * (1.0 - ct), g0 = RSQRT2 * stt;
                const double2 Bp = make_double2(fma(ca, uAp.x, sa * uAp.y), fma(ca, uAp.y, -sa * uAp.x));    // conj(e^{+i alpha}) uw A+
                const double2 Bm = make_double2(fma(ca, uAm.x, -sa * uAm.y), fma(ca, uAm.y, sa * uAm.x));    // conj(e^{-i alpha}) uw A-
                const double2 Y0 = make_double2(zc0 * g0 * (Bp.x - Bm.x), zc0 * g0 * (Bp.y - Bm.y));
                const double2 Rp = make_double2(fma(gp, Bp.x, gm * Bm.x), fma(gp, Bp.y, gm * Bm.y));         // l' = +1: d^1_{1,+} = gp, d^1_{1,-} = gm
                const double2 Rm = make_double2(fma(gm, Bp.x, gp * Bm.x), fma(gm, Bp.y, gp * Bm.y));         // l' = -1
                // conj(e^{+-i phi~}) R, times d^1_{0,+-1}(theta_Z) = +-zcp
                const double2 Yp = make_double2(zcp * fma(cpt, Rp.x, spt * Rp.y), zcp * fma(cpt, Rp.y, -spt * Rp.x));
                const double2 Ym = make_double2(-zcp * fma(cpt, Rm.x, -spt * Rm.y), -zcp * fma(cpt, Rm.y, spt * Rm.x));
                // sum_xi |d^1_{0 l'} d^1_{l' xi}|^2 un, and for the tied pair (l' = -1 and +1 moving together) the cross term
                //   2 Re sum_xi conj(B_-1,xi) B_+1,xi / |BW|^2 = -zcp^2 (2 gp gm) 2 cos(2 phi~)
                const double NZ0 = zc0 * zc0 * 2.0 * g0 * g0 * un;
                const double NZ1 = zcp * zcp * fma(gp, gp, gm * gm) * un;
                const double NZc = -4.0 * zcp * zcp * gp * gm * fma(cpt, cpt, -spt * spt) * un;
                double Fz, Gz;
                group_factors<0, 1>(a.r2_spin[5], st[C_INVMZ * UNIT], st[C_QZ * UNIT], st[C_PBZ * UNIT], &Fz, &Gz);
                double2 bwz[SH::nz > 0 ? SH::nz : 1];
#pragma unroll
                for (int z = 0; z < SH::nz; ++z) {
                    const double2 bw = bw_unscaled(a.ent[SH::oz + z], mZ2, Fz, Gz);
                    bwz[z] = bw;
                    const double bw2 = fma(bw.x, bw.x, bw.y * bw.y);
                    const int b = L::base(SH::oz + z);
                    const double2 Lm = conj_mul(bw, Ym), Lp = conj_mul(bw, Yp);
                    position(tree, norm, b, Lm, bw2 * NZ1);
                    position(tree, norm, b + 1, conj_mul(bw, Y0), bw2 * NZ0);
                    position(tree, norm, b + 2, Lp, bw2 * NZ1);
                    // tied pair: both helicities +-1 move by the same delta
                    position(tree, norm, NSLOT + z, make_double2(Lm.x + Lp.x, Lm.y + Lp.y), bw2 * (NZ1 + NZ1 + NZc));
                }
    #pragma unroll
                for (int z = 0; z < SH::nz; ++z) {
                    if (!((d.ent_active >> (SH::oz + z)) & 1u)) { tree.push_identity(); continue; }
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
                    lineshape_points(tree, norm, SH::oz + z, bwz[z], mZ2, Fz, Gz, Q, nR);
                }
            }
            tree.pad_block();
        };
        if (is_norm) {
            all_values(tn, true);
        } else {
            all_values(td, false);
            if ((k & 15) == 15) {   // the products of r in [0.5, 1.5] (eight per unit and chunk) back to [0.5, 1)
#pragma unroll
                for (int c = 0; c < NCH; ++c) { int e; split_exp(accv[c], &accv[c], &e); accx[c] += e; }
            }
        }
        __syncwarp();
        if (lane == 0) mbar_arrive(&empty[s]);   // this warp has read everything it needs from the stage
    }
    if (bad & 1) atomicOr(a.flag, 2);
    if (bad & 2) atomicOr(a.flag, 1024);

    // ---- per-CTA partials: rows 0, 1 = sum log S0, sum w S0; rows 2 + v = data-side value slot v (sum of log r); rows 2 + NVAL + v = normalisation side
    if (!in_norm) {   // this CTA saw data units only (or none)
        const double t0 = block_sum(log(acc0F) + (double)acc0E * LN2, sm);
        if (tid == 0) d.partial[(size_t)0 * d.stride + blockIdx.x] = t0;
        flush(2, true);
    }
    flush(2 + NVAL, false);
    {
        const double t1 = block_sum(acc0W, sm);
        if (tid == 0) d.partial[(size_t)1 * d.stride + blockIdx.x] = t1;
    }
    // ---- the last CTA to finish adds the partials of every row in CTA order and forms NLL(p), I(p)
    __threadfence();
    __syncthreads();
    if (tid == 0) s_last = atomicAdd(a.ticket, 1u) == gridDim.x - 1;
    __syncthreads();
    if (!s_last) return;
    __threadfence();
    double* tot = red;   // 2 + 2 NVAL totals (the tiles are larger)
    constexpr int ROWS = 2 + 2 * NVAL;
    for (int r = tid; r < ROWS; r += THREADS) {
        const double* p = d.partial + (size_t)r * d.stride;
        double s = 0.0;
        for (unsigned c = 0; c < gridDim.x; ++c) s += __ldcg(p + c);
        tot[r] = s;
    }
    __syncthreads();
    if (d.norm_tot) {   // the normalisation events were walked by k_deltan (this launch saw none): its totals in their place
        for (int r = tid; r < 1 + NVAL; r += THREADS) tot[r == 0 ? 1 : 1 + NVAL + r] = __ldcg(d.norm_tot + r);
        __syncthreads();
    }
    for (int p = tid; p < d.P; p += THREADS) {
        const int v = p == 0 ? -1 : d.val_of_point[p];      // value slot of the point; -1: equal to point 0
        double slog = tot[0], swS = tot[1];
        if (v >= 0) {
            slog += tot[2 + v];
            const int pos = d.pos_of_point[p], j = v & 3;
            if (pos >= 0) {       // coupling point: from the three sums of its position (the first three values of its quad)
                const double* row = tot + 2 + NVAL + (v & ~3);
                swS += fma(d.cq[pos][j][0], row[0], fma(d.cq[pos][j][1], row[1], d.cq[pos][j][2] * row[2]));
            } else {
                swS += tot[2 + NVAL + v];
            }
        }
        const double I = swS / a.wsum;
        d.result[d.P + p] = I;
        d.result[2 * d.P + 1 + p] = slog;
        d.result[3 * d.P + 1 + p] = swS;
        double nll = -(slog + a.sum_log_eff) + (double)a.n * log(I);
        if (!isfinite(nll) || !(I > 0.0)) nll = INFINITY;
        d.result[p] = d.want_nll ? nll : 0.0;
    }
    // the result block may live in mapped host memory: every writer's values are in place system-wide before the stamp goes out
    __threadfence_system();
    __syncthreads();
    if (tid == 0) {
        d.result[2 * d.P] = (double)atomicExch(a.flag, 0);   // domain flag of this launch, cleared for the next one
        *a.ticket = 0u;
        __threadfence_system();
        *reinterpret_cast<volatile double*>(d.result + 4 * d.P + 1) = d.seq;
    }
}

namespace {

template <class SH>
size_t deltaf_smem(int ncolw) {
    return (size_t)NSTAGE * ncolw * UNIT * sizeof(double) + (size_t)NWARPS * TILE_BYTES + 2 * NSTAGE * sizeof(uint64_t);
}

template <class SH>
cudaError_t launch_deltaf_shape(const DeltaFArgs& d, int grid, cudaStream_t s) {
    static_assert(NWARPS * TILE_BYTES / 8 >= 2 + 2 * DLay<SH>::NVAL && TILE_BYTES / 8 >= 8 * DLay<SH>::NCH, "the flush and the finish reuse the value tiles");
    static DeviceOnce attr_done;
    cudaError_t e = cudaSuccess;
    if (attr_done.first()) { e = cudaFuncSetAttribute(k_deltaf<SH>, cudaFuncAttributeMaxDynamicSharedMemorySize, 224 * 1024); }
    if (e != cudaSuccess) return e;
    k_deltaf<SH><<<grid, THREADS, deltaf_smem<SH>(d.a.ncolw), s>>>(d);
    return cudaGetLastError();
}

}  // namespace

int deltaf_grid(long long n_data, long long n_norm) {
    const long long nunits = UPB * ((n_data + CACHE_TILE - 1) / CACHE_TILE) + UPB * ((n_norm + CACHE_TILE - 1) / CACHE_TILE);
    const long long cap = (long long)sm_count() * DELTAF_MINB;
    return (int)(nunits < 1 ? 1 : (nunits > cap ? cap : nunits));   // persistent: one CTA per SM
}

// the shapes this kernel is compiled for: the paper's ten K* (3, 3, 2, 1, 1 per spin, one radius per spin) with zero to two 1+ Z's,
// no constant or LASS term.  Fills the layout numbers the host needs to build the tables of DeltaFArgs.
bool deltaf_layout(const StreamArgs& a, DeltaFLayout* lay) {
    const int* n = a.shape;
    if (!a.shape_fixed || a.nlass > 0 || a.bkg || a.cconst.x != 0.0 || a.cconst.y != 0.0) return false;
    if (n[6] + n[7] + n[8] + n[9] != 0) return false;
    if (!(n[0] == 3 && n[1] == 3 && n[2] == 2 && n[3] == 1 && n[4] == 1 && n[5] >= 0 && n[5] <= 2)) return false;
    if (a.ncolw != (n[5] > 0 ? NCOL_ALL : NCOL_K) + 1) return false;
    const int ne = 10 + n[5];
    lay->nent = ne;
    lay->nslot = 3 + 3 * (ne - 3);
    lay->npos = lay->nslot + n[5];
    // the kernel's value order, a quad (four values) at a time: per spin class the coupling positions of its entries (a Z: its three
    // helicities, then the tied pair), then the lineshape quads of its entries
    int quad = 0, t = 0;
    for (int cls = 0; cls < 6; ++cls) {
        const int t0 = t;
        for (int e = 0; e < n[cls]; ++e, ++t) {
            const int b = t < n[0] ? t : n[0] + 3 * (t - n[0]);
            for (int j = 0; j < (cls == 0 ? 1 : 3); ++j) lay->quad_of_pos[b + j] = quad++;
            if (cls == 5) lay->quad_of_pos[lay->nslot + e] = quad++;
        }
        for (int e = t0; e < t; ++e) lay->quad_of_ent[e] = quad++;
    }
    lay->nquad = quad;
    return true;
}

cudaError_t launch_deltaf(const DeltaFArgs& d, int grid, cudaStream_t s) {
    switch (d.a.shape[5]) {
        case 0: return launch_deltaf_shape<Shape<3, 3, 2, 1, 1, 0>>(d, grid, s);
        case 1: return launch_deltaf_shape<Shape<3, 3, 2, 1, 1, 1>>(d, grid, s);
        default: return launch_deltaf_shape<Shape<3, 3, 2, 1, 1, 2>>(d, grid, s);
    }
}

}  // namespace amp
