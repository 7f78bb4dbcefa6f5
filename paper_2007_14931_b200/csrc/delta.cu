// delta.cu — steps a2 + a3 + a4 + a5 for a GRADIENT BATCH: P parameter points of which points 1..P-1 differ from
// point 0 in a few resonances only (MINUIT's finite-difference pattern, BASELINE.json configs[4]: the central value
// plus theta_k +- h_k for ~60 parameters; "> 60 free parameters").
//
// Eq. 12 is linear in (coupling x lineshape), so with g_k,xi the angular factors of Eqs. 4 and 10
// a point that changes resonance R only gives
//   A_xi(p) = A_xi(0) + sum_{l in R} [ c_{R,l}(p) BW_R(p) - c_{R,l}(0) BW_R(0) ] g_{R,l,xi}
// — one complex multiply-add per muon helicity instead of the 27 of the dense contraction, and a perturbed
// Breit-Wigner (Eqs. 2-3) costs ~12 FP64 instructions because the barrier factors (F, G) of its spin group are those
// of point 0.  The host compiles the batch into contributions `coef * SLOT` (amp_internal.cuh, DeltaContrib); the
// kernel is the streaming kernel (stream.cu: TMA-fed 512-event tiles, two events per thread, point 0 with lineshapes
// in registers) followed, per tile, by the point loop.  One fused persistent launch walks the data tiles
// (sum_i log S_i(p)) and then the normalisation tiles (sum_j w_j S_j(p)) for ALL points: no lineshape column, no
// normalisation matrix, no second pass.
//
// Point loop: every lane evaluates S(p) of its two events for the 32 points of a block in order; a recursive-halving
// exchange (one shuffle + one add or multiply per point and lane) leaves lane l with the total of point 32 b + l over
// the warp's 64 events.  Data side: S = f 2^e is split with integer ops, mantissas are multiplied and exponents
// added, so the sum of logs takes ONE log per (point, warp) at the very end instead of one per (point, event).
// Everything is fixed-order: bit-reproducible.  Bound: plain FP64 ALUs.
// One event per thread x 512 threads (16 warps per SM, 128 registers): the point loop is chains of short dependent FP64
// sequences and the extra warps hide their latency.  Measured on configs[4] (with the four-point blocks): 5.55 ms, against
// 5.74 ms for two events per thread x 256 threads (8 warps, 229 registers), which pays the warp-uniform per-point overhead once
// for two events but stalls more.
#define AMP_STREAM_E 1
#define AMP_STREAM_THREADS 512
#include "stream_core.cuh"
#include "delta_core.cuh"

namespace amp {

namespace {

constexpr int DBLK = DELTA_MAX_SORTED / 32;

struct SlotVal {   // the current slot of one event
    double2 Sp, Sm;                 // xi = +1, -1
    double2 bw0;                    // BW(0) of the slot's resonance (kind-1 contributions subtract it)
    // A point with ONE contribution coef x SLOT has S = |A(0) + coef SLOT|^2 = S(0) + Re(coef T2) + |coef|^2 n with
    //   T2 = 2 sum_xi conj(A_xi(0)) SLOT_xi,  n = sum_xi |SLOT_xi|^2:
    // three FMAs per point instead of twelve once T2 and n are known per (event, slot) — a slot serves 2-4 points.
    double2 T2;
    double n;
};
// below this fraction of S(0) the expansion's cancellation would cost more than three digits: the guard trips (flag 1024) and the
// host repeats the call with the amplitudes summed term by term (k_delta<Generic, false>)
constexpr double DELTA_CANCEL = 1e-3;

// BW of entry `ent` at point 0 for one event, from the saved group factors
__device__ __forceinline__ double2 bw_point0(const StreamArgs& a, int ent, int grp, bool isz, const EvK& k, const double2* fg) {
    const double2 f = fg[grp * TILE];
    return bw_from_consts(a.ent[ent].kN, a.ent[ent].kG, a.ent[ent].M2, isz ? k.mZ2 : k.m2, f.x, f.y);
}

// Evaluate the slot record at `rec` (shared memory) for the thread's E events.  A slot belongs to ONE resonance (its terms are
// helicities of that resonance): entry, barrier group, spin and chain are decoded once, the Breit-Wigner of point 0 and the
// d functions are computed once, and only the helicity-dependent factors run per term (at most three).
template <bool FAST>
__device__ __forceinline__ void eval_slot(const StreamArgs& a, const double* rec, const EvK (&k)[E], const double2* fg, const double* zst,
                                          SlotVal (&sv)[E]) {
    const double RSQRT2 = 0.70710678118654752440;
    const int2 h = *reinterpret_cast<const int2*>(rec);
    const int th0 = *reinterpret_cast<const int*>(rec + 1);
    const int ent = th0 & 255, grp = (th0 >> 8) & 15, J = (th0 >> 12) & 7;
    const bool isz = (th0 >> 17) & 1, unit = (th0 >> 18) & 1;
#pragma unroll
    for (int e = 0; e < E; ++e) {
        double2 Sp = make_double2(0.0, 0.0), Sm = Sp;
        if (!isz) {
            double d0, d1;
            dJ(J, k[e].cK, k[e].sK, &d0, &d1);
            const double t0 = d0 * k[e].h0;
#pragma unroll
            for (int t = 0; t < 3; ++t) {
                if (t < h.x) {
                    const int lam = ((*reinterpret_cast<const int*>(rec + 1 + 3 * t) >> 15) & 3) - 1;
                    double2 gp, gm;
                    if (lam == 0) { gp = make_double2(t0, 0.0); gm = make_double2(-t0, 0.0); }
                    else if (lam > 0) { gp = make_double2(d1 * k[e].a1, d1 * k[e].a2); gm = make_double2(d1 * k[e].a3, d1 * k[e].a4); }
                    else { gp = make_double2(-d1 * k[e].a3, d1 * k[e].a4); gm = make_double2(-d1 * k[e].a1, d1 * k[e].a2); }
                    if (!unit) {
                        const double2 wgt = make_double2(rec[2 + 3 * t], rec[3 + 3 * t]);
                        gp = cmul(wgt, gp);
                        gm = cmul(wgt, gm);
                    }
                    Sp = cadd(Sp, gp);
                    Sm = cadd(Sm, gm);
                }
            }
        } else {
            // d^1_{0 l'}(theta_Z) e^{i l' phi~} d^1_{l' xi}(theta~) e^{i xi alpha} (the plans of this kernel hold 1+ Zs only)
            const double* z = zst + e;
            const double cZ = z[C_CZ * TILE], sZ = z[C_SZ * TILE], ct = z[C_CT * TILE], st = z[C_ST * TILE];
            const double cpt = z[C_CPT * TILE], spt = z[C_SPT * TILE], ca = z[C_CA * TILE], sa = z[C_SA * TILE];
            const double z1 = RSQRT2 * sZ, g0 = RSQRT2 * st, gpp = 0.5 * (1.0 + ct), gmm = 0.5 * (1.0 - ct);
            // T = sum_l' w_l' d^1_{0 l'} e^{i l' phi~} (.)  accumulated per xi before the alpha phase
            double2 Zp = make_double2(0.0, 0.0), Zm = Zp;
#pragma unroll
            for (int t = 0; t < 3; ++t) {
                if (t < h.x) {
                    const int lam = ((*reinterpret_cast<const int*>(rec + 1 + 3 * t) >> 15) & 3) - 1;
                    double2 f = lam == 0 ? make_double2(cZ, 0.0) : (lam > 0 ? make_double2(z1 * cpt, z1 * spt) : make_double2(-z1 * cpt, z1 * spt));
                    if (!unit) f = cmul(make_double2(rec[2 + 3 * t], rec[3 + 3 * t]), f);
                    const double dp = lam == 0 ? g0 : (lam > 0 ? gpp : gmm), dm = lam == 0 ? -g0 : (lam > 0 ? gmm : gpp);
                    Zp = make_double2(fma(dp, f.x, Zp.x), fma(dp, f.y, Zp.y));
                    Zm = make_double2(fma(dm, f.x, Zm.x), fma(dm, f.y, Zm.y));
                }
            }
            Sp = cmul(make_double2(ca, sa), Zp);
            Sm = cmul(make_double2(ca, -sa), Zm);
        }
        if (ent != 255) {
            const double2 bw = bw_point0(a, ent, grp, isz, k[e], fg + e);
            Sp = cmul(bw, Sp);
            Sm = cmul(bw, Sm);
        }
        sv[e].Sp = Sp;
        sv[e].Sm = Sm;
    }
    if (h.y >= 0) {
#pragma unroll
        for (int e = 0; e < E; ++e) sv[e].bw0 = bw_point0(a, h.y & 255, (h.y >> 8) & 15, (h.y >> 12) & 1, k[e], fg + e);
    }
    if (!FAST) return;
#pragma unroll
    for (int e = 0; e < E; ++e) {
        const double2 Ap = k[e].Ap, Am = k[e].Am, Sp = sv[e].Sp, Sm = sv[e].Sm;
        const double tr = fma(Ap.x, Sp.x, fma(Ap.y, Sp.y, fma(Am.x, Sm.x, Am.y * Sm.y)));
        const double ti = fma(Ap.x, Sp.y, fma(-Ap.y, Sp.x, fma(Am.x, Sm.y, -Am.y * Sm.x)));
        sv[e].T2 = make_double2(tr + tr, ti + ti);
        sv[e].n = fma(Sp.x, Sp.x, fma(Sp.y, Sp.y, fma(Sm.x, Sm.x, Sm.y * Sm.y)));
    }
}


// NORM: sum_e w_e S_e; DATA: mantissa product / exponent sum of the S_e (the tail of a leaf)
template <bool NORM>
__device__ __forceinline__ void leaf_value(const double (&S)[E], const double (&w)[E], const bool (&live)[E], int& bad, double* v, int* ex) {
    if (NORM) {
        double t = 0.0;
#pragma unroll
        for (int e = 0; e < E; ++e) t = fma(w[e], S[e], t);
        *v = t;
        *ex = 0;
    } else {
        double f = 1.0;
        int x = 0;
#pragma unroll
        for (int e = 0; e < E; ++e) {
            const bool ok = S[e] > 0.0 && isfinite(S[e]);
            bad |= live[e] && !ok;
            double fe; int xe;
            split_exp((live[e] && ok) ? S[e] : 1.0, &fe, &xe);
            f *= fe; x += xe;
        }
        *v = f;
        *ex = x;
    }
}

// coef * SLOT of one contribution added to (Bp, Bm) -> (Ap, Am), for the thread's E events
__device__ __forceinline__ void apply_contrib(int hdr, double ca, double2 bc, const EvK (&k)[E], const double2* fg, const SlotVal (&sv)[E],
                                              const double2 (&Bp)[E], const double2 (&Bm)[E], double2 (&Ap)[E], double2 (&Am)[E]) {
    const int kind = hdr & 3;
#pragma unroll
    for (int e = 0; e < E; ++e) {
        double2 coef = make_double2(ca, bc.x);
        if (kind) {
            const double2 f = fg[((hdr >> 8) & 15) * TILE + e];
            coef = bw_from_consts(ca, bc.x, bc.y, (hdr & 32) ? k[e].mZ2 : k[e].m2, f.x, f.y);
            if (kind == 1) { coef.x -= sv[e].bw0.x; coef.y -= sv[e].bw0.y; }
        }
        Ap[e] = cfma(coef, sv[e].Sp, Bp[e]);
        Am[e] = cfma(coef, sv[e].Sm, Bm[e]);
    }
}

// One point for the thread's E events as a leaf of the reduction tree.  NORM: *v = sum_e w_e S_e; DATA: *v = product of
// the mantissas of S_e, *ex = sum of their exponents.  `it` walks the contribution list; `sv` caches the current slot.
// The first contribution is applied straight onto A(0) (no copy of the four complex amplitudes per point).
template <bool NORM, bool FAST>
__device__ __forceinline__ void leaf(const StreamArgs& a, const DeltaContrib* prog, const double* slots, int& it, const EvK (&k)[E],
                                     const double2* fg, const double* zst, SlotVal (&sv)[E], const double (&w)[E], const bool (&live)[E],
                                     int& bad, double* v, int* ex) {
    double2 A0p[E], A0m[E];
#pragma unroll
    for (int e = 0; e < E; ++e) { A0p[e] = k[e].Ap; A0m[e] = k[e].Am; }
    int4 h4 = *reinterpret_cast<const int4*>(prog + it);                      // hdr, slot, a (two words)
    double2 bc = *reinterpret_cast<const double2*>(&prog[it].b);              // b, c
    ++it;
    int hdr = h4.x;
    double S[E];
    if ((hdr & 20) == 4) {
        // the common gradient point: ONE contribution.  Its own copy of the tail keeps the amplitudes of the general
        // path out of the merge (no register moves per point).
        if (hdr & 8) eval_slot<FAST>(a, slots + h4.y, k, fg, zst, sv);
        double2 Ap[E], Am[E];
        apply_contrib(hdr, __hiloint2double(h4.w, h4.z), bc, k, fg, sv, A0p, A0m, Ap, Am);
#pragma unroll
        for (int e = 0; e < E; ++e) S[e] = fma(Ap[e].x, Ap[e].x, fma(Ap[e].y, Ap[e].y, fma(Am[e].x, Am[e].x, Am[e].y * Am[e].y)));
    } else {
        double2 Ap[E], Am[E];
#pragma unroll
        for (int e = 0; e < E; ++e) { Ap[e] = A0p[e]; Am[e] = A0m[e]; }
        if (!(hdr & 16)) {                                                    // (an empty point has S(p) = S(0))
            for (;;) {
                if (hdr & 8) eval_slot<FAST>(a, slots + h4.y, k, fg, zst, sv);
                apply_contrib(hdr, __hiloint2double(h4.w, h4.z), bc, k, fg, sv, Ap, Am, Ap, Am);
                if (hdr & 4) break;
                h4 = *reinterpret_cast<const int4*>(prog + it);
                bc = *reinterpret_cast<const double2*>(&prog[it].b);
                ++it;
                hdr = h4.x;
            }
        }
#pragma unroll
        for (int e = 0; e < E; ++e) S[e] = fma(Ap[e].x, Ap[e].x, fma(Ap[e].y, Ap[e].y, fma(Am[e].x, Am[e].x, Am[e].y * Am[e].y)));
    }
    leaf_value<NORM>(S, w, live, bad, v, ex);   // (NORM: a non-finite S makes the point's total non-finite: flagged at the end)
}

// NP = 2 or 4 consecutive single-contribution points of the same kind on the same slot (theta_k +- h; modulus and phase of
// one coupling; mass and width of one resonance) as ONE straight-line block: NP points x E events independent dependency
// chains, which is what keeps the FP64 pipe busy with two warps per scheduler.
template <bool NORM, int KIND, int NP, bool FAST>
__device__ __forceinline__ void leaf_multi(const int4 (&h4)[NP], const double2 (&bc)[NP], const EvK (&k)[E], const double2* fg,
                                           const SlotVal (&sv)[E], const double (&w)[E], const bool (&live)[E], int& bad, double (&v)[NP],
                                           int (&ex)[NP]) {
    double S[NP][E];
    bool trip = false;   // (one predicate for the NP x E comparisons, folded into `bad` once)
#pragma unroll
    for (int j = 0; j < NP; ++j) {
        const double ca = __hiloint2double(h4[j].w, h4[j].z);
#pragma unroll
        for (int e = 0; e < E; ++e) {
            double2 coef = make_double2(ca, bc[j].x);
            if (KIND) {
                const double2 f = fg[((h4[j].x >> 8) & 15) * TILE + e];
                coef = bw_from_consts(ca, bc[j].x, bc[j].y, (h4[j].x & 32) ? k[e].mZ2 : k[e].m2, f.x, f.y);
                if (KIND == 1) { coef.x -= sv[e].bw0.x; coef.y -= sv[e].bw0.y; }
            }
            double Sv;
            if (FAST) {
                // S(0) + Re(coef T2) + |coef|^2 n; kind 0 carries |coef|^2 in the contribution's third constant.  A change that
                // nearly cancels A(0) would lose digits here: it trips the guard and the host repeats the call with FAST = false
                const double c2 = KIND ? fma(coef.x, coef.x, coef.y * coef.y) : bc[j].y;
                Sv = fma(c2, sv[e].n, fma(coef.x, sv[e].T2.x, fma(-coef.y, sv[e].T2.y, k[e].S0)));
                trip |= Sv < k[e].Sguard;
            } else {
                const double2 Ap = cfma(coef, sv[e].Sp, k[e].Ap), Am = cfma(coef, sv[e].Sm, k[e].Am);
                Sv = fma(Ap.x, Ap.x, Ap.y * Ap.y) + fma(Am.x, Am.x, Am.y * Am.y);
            }
            S[j][e] = Sv;
        }
    }
    if (FAST && trip) bad |= 2;
#pragma unroll
    for (int j = 0; j < NP; ++j) leaf_value<NORM>(S[j], w, live, bad, &v[j], &ex[j]);
}

// The 32 points of one block; on return lane l holds the warp total of point 32 blk + l (NORM: sum of w S; DATA:
// product of mantissas in *v — at least 2^-64 — and sum of exponents in *ex).  Binary-counter carries: q is uniform.
template <bool NORM, bool FAST>
__device__ __forceinline__ void eval_block(const StreamArgs& a, const DeltaContrib* prog, const double* slots, int& it, const EvK (&k)[E],
                                           const double2* fg, const double* zst, SlotVal (&sv)[E], const double (&w)[E],
                                           const bool (&live)[E], int& bad, int lane, double* v, int* ex) {
    double s2 = 0, s3 = 0, s4 = 0;
    int e2 = 0, e3 = 0, e4 = 0;
    // two points: as one block if both are single-contribution, non-empty, of one kind and on one slot, else one by one
    auto two_points = [&](double* y, int* ye) {
        int4 h4[2];
        double2 bc[2];
#pragma unroll
        for (int j = 0; j < 2; ++j) {
            h4[j] = *reinterpret_cast<const int4*>(prog + it + j);
            bc[j] = *reinterpret_cast<const double2*>(&prog[it + j].b);
        }
        if ((h4[0].x & 20) == 4 && (h4[1].x & 28) == 4 && ((h4[0].x ^ h4[1].x) & 3) == 0) {
            it += 2;
            if (h4[0].x & 8) eval_slot<FAST>(a, slots + h4[0].y, k, fg, zst, sv);
            double v2[2]; int x2[2];
            const int kind = h4[0].x & 3;
            if (kind == 0) leaf_multi<NORM, 0, 2, FAST>(h4, bc, k, fg, sv, w, live, bad, v2, x2);
            else if (kind == 1) leaf_multi<NORM, 1, 2, FAST>(h4, bc, k, fg, sv, w, live, bad, v2, x2);
            else leaf_multi<NORM, 2, 2, FAST>(h4, bc, k, fg, sv, w, live, bad, v2, x2);
            y[0] = v2[0]; ye[0] = x2[0]; y[1] = v2[1]; ye[1] = x2[1];
        } else {
            leaf<NORM, FAST>(a, prog, slots, it, k, fg, zst, sv, w, live, bad, &y[0], &ye[0]);
            leaf<NORM, FAST>(a, prog, slots, it, k, fg, zst, sv, w, live, bad, &y[1], &ye[1]);
        }
    };
    // (not unrolled: the body is large, and two or four copies of it measured slower)
#pragma unroll 1
    for (int q = 0; q < 32; q += 4) {
        double y[4]; int ye[4];
        {
            int4 h4[4];
            double2 bc[4];
#pragma unroll
            for (int j = 0; j < 4; ++j) {
                h4[j] = *reinterpret_cast<const int4*>(prog + it + j);
                bc[j] = *reinterpret_cast<const double2*>(&prog[it + j].b);
            }
            // four single-contribution points of kind 0 or 1 on one slot (the gradient pattern, marked by the host): one straight-line block
            const int kind = h4[0].x & 3;
            const bool quad = (h4[0].x & 64) != 0;
            if (quad) {
                it += 4;
                if (h4[0].x & 8) eval_slot<FAST>(a, slots + h4[0].y, k, fg, zst, sv);
                if (NORM && FAST && kind == 0) {
                    // normalisation side of four coupling points on one slot: their coefficients do not depend on the event, so
                    //   sum_j w_j S_j(p) = sum w S(0) + Re(coef(p) sum_j w_j T2_j) + |coef(p)|^2 sum_j w_j n_j
                    // and the three sums of the SLOT take the places of the four points here; the last CTA forms the points
                    // from them (quad_points_from_slot_sums).  The cancellation guard stays with the data events.
                    double t0 = 0.0, t1 = 0.0, t2 = 0.0;
#pragma unroll
                    for (int e = 0; e < E; ++e) {
                        t0 = fma(w[e], sv[e].T2.x, t0);
                        t1 = fma(w[e], sv[e].T2.y, t1);
                        t2 = fma(w[e], sv[e].n, t2);
                    }
                    y[0] = t0; y[1] = t1; y[2] = t2; y[3] = 0.0;
                    ye[0] = ye[1] = ye[2] = ye[3] = 0;
                }
                else if (kind == 0) leaf_multi<NORM, 0, 4, FAST>(h4, bc, k, fg, sv, w, live, bad, y, ye);
                else leaf_multi<NORM, 1, 4, FAST>(h4, bc, k, fg, sv, w, live, bad, y, ye);
            } else {
                two_points(&y[0], &ye[0]);
                two_points(&y[2], &ye[2]);
            }
        }
        double x, u; int xe, ue;
        halve<NORM>(0, lane, y[0], ye[0], y[1], ye[1], &u, &ue);
        halve<NORM>(0, lane, y[2], ye[2], y[3], ye[3], &x, &xe);
        halve<NORM>(1, lane, u, ue, x, xe, &x, &xe);
        if (!(q & 4)) { s2 = x; e2 = xe; continue; }
        halve<NORM>(2, lane, s2, e2, x, xe, &x, &xe);
        if (!(q & 8)) { s3 = x; e3 = xe; continue; }
        halve<NORM>(3, lane, s3, e3, x, xe, &x, &xe);
        if (!(q & 16)) { s4 = x; e4 = xe; continue; }
        halve<NORM>(4, lane, s4, e4, x, xe, v, ex);
    }
}

}  // namespace

template <class SH, bool FAST>
__global__ void __launch_bounds__(THREADS, 1) k_delta(const __grid_constant__ DeltaArgs d) {
    const StreamArgs& a = d.a;
    const double RSQRT2 = 0.70710678118654752440;
    const int tid = threadIdx.x, lane = tid & 31;
    const bool have_z = SH::nz > 0 || (SH::nz < 0 && a.gstart[NSPIN] > a.gstart[5]);
    const int ncache = have_z ? NCOL_ALL : NCOL_K;
    const int ngrp = a.gstart[NSPIN];
    const int nblk = d.nsorted / 32;

    // shared memory: staged tile (two regions, as k_stream) | group factors | per-lane point accumulators | the program
    extern __shared__ __align__(128) unsigned char smem_raw[];
    double* stage = reinterpret_cast<double*>(smem_raw);                          // [ncache + 1][TILE]
    double2* fg_base = reinterpret_cast<double2*>(stage + (size_t)(ncache + 1) * TILE);   // [ngrp][TILE]
    double* accN = reinterpret_cast<double*>(fg_base + (size_t)ngrp * TILE);      // [DBLK][THREADS] sum w S
    double* accF = accN + DBLK * THREADS;                                         // [DBLK][THREADS] mantissa products (data)
    int* accE = reinterpret_cast<int*>(accF + DBLK * THREADS);                    // [DBLK][THREADS] exponent sums (data)
    DeltaContrib* prog = reinterpret_cast<DeltaContrib*>(accE + DBLK * THREADS);  // [DELTA_MAX_CONTRIB]
    double* slots = reinterpret_cast<double*>(prog + DELTA_MAX_CONTRIB);          // [DELTA_MAX_SLOTWORDS]
    uint64_t* full = reinterpret_cast<uint64_t*>(slots + DELTA_MAX_SLOTWORDS);    // [2]
    __shared__ double sm[NWARPS];
    __shared__ bool s_last;
    for (int b = 0; b < DBLK; ++b) { accN[b * THREADS + tid] = 0.0; accF[b * THREADS + tid] = 1.0; accE[b * THREADS + tid] = 0; }
    for (int i = tid; i < d.ncontrib * 4; i += THREADS) reinterpret_cast<double*>(prog)[i] = reinterpret_cast<const double*>(d.contrib)[i];
    for (int i = tid; i < d.nslotwords; i += THREADS) slots[i] = d.slots[i];
    if (tid == 0) {
        mbar_init(&full[0], 1);
        mbar_init(&full[1], 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();
    const long long ntd = d.want_nll ? (a.n + TILE - 1) / TILE : 0;              // data tiles first, then normalisation tiles
    const long long ntiles = ntd + (a.n2 + TILE - 1) / TILE;
    auto issue = [&](long long tile, int region) {
        const bool nrm = tile >= ntd;
        const double* cache = nrm ? a.cache2 : a.cache;
        const long long lt = nrm ? tile - ntd : tile;
        if (region == 0) issue_cols(cache, a.ncolw, lt, stage, &full[0], 0, NCOL_K, nrm);
        else issue_cols(cache, a.ncolw, lt, stage, &full[1], NCOL_K, NCOL_ALL, false);
    };
    if (tid == 0 && (long long)blockIdx.x < ntiles) {
        issue(blockIdx.x, 0);
        if (have_z) issue(blockIdx.x, 1);
    }
    double2* fg = fg_base + tid * E;
    const double* zst = stage + tid * E;
    double acc0N = 0.0, acc0F = 1.0;   // point 0: sum w S ; mantissa product and exponent sum of S
    int acc0E = 0;
    int bad = 0;   // 1: a density that is not finite and positive; 2: the expansion guard tripped (FAST)
    uint32_t parity = 0;
    for (long long tile = blockIdx.x; tile < ntiles; tile += gridDim.x, parity ^= 1) {
        const bool has_next = tile + gridDim.x < ntiles;
        const bool is_norm = tile >= ntd;
        const long long lt = is_norm ? tile - ntd : tile;
        const long long i0 = lt * TILE + tid * E;
        const long long nlive = is_norm ? a.n2 : a.n;
        // ---- point 0: the K* chain (as k_stream)
        mbar_wait(&full[0], parity);
        const Ev m2 = load_col(stage, C_M2), invm = load_col(stage, C_INVM);
        const Ev q = load_col(stage, C_Q), pB = load_col(stage, C_PB);
        const Ev cK = load_col(stage, C_CK), sK = load_col(stage, C_SK);
        const Ev cpsi = load_col(stage, C_CPSI), spsi = load_col(stage, C_SPSI);
        const Ev cphi = load_col(stage, C_CPHI), sphi = load_col(stage, C_SPHI);
        Ev wv;
        if (is_norm) wv = load_col(stage, ncache);
        __syncthreads();   // K* region consumed by every thread: stream the next tile into it during the point loop
        if (tid == 0 && has_next) issue(tile + gridDim.x, 0);

        double2 V0[E], Vp[E], Vm[E];
#pragma unroll
        for (int e = 0; e < E; ++e) { V0[e] = a.cconst; Vp[e] = make_double2(0, 0); Vm[e] = make_double2(0, 0); }
#define AMP_SPIN(J, LB, CNT, OFF, D0, D1)                                                              \
        if (CNT != 0 && (CNT > 0 || a.gstart[J + 1] > a.gstart[J])) {                                  \
            double2 Um[E], U0[E], Up[E];                                                               \
            _Pragma("unroll") for (int e = 0; e < E; ++e) Um[e] = U0[e] = Up[e] = make_double2(0, 0);  \
            spin_sum<J, J, LB, CNT, OFF, J, true>(a, i0, m2, invm, q, pB, Um, U0, Up, fg);             \
            _Pragma("unroll") for (int e = 0; e < E; ++e) {                                            \
                const double c = cK.v[e], s = sK.v[e], c2 = c * c;                                     \
                (void)s; (void)c2;                                                                     \
                const double d0 = (D0), d1 = (D1);                                                     \
                V0[e] = cadd(V0[e], cscale(d0, U0[e]));                                                \
                if (J) { Vp[e] = cadd(Vp[e], cscale(d1, Up[e])); Vm[e] = cadd(Vm[e], cscale(-d1, Um[e])); } \
            }                                                                                          \
        }
        AMP_SPIN(0, 1, SH::n0, 0, 1.0, 0.0)
        AMP_SPIN(1, 0, SH::n1, SH::o1, c, -RSQRT2 * s)
        AMP_SPIN(2, 1, SH::n2, SH::o2, fma(1.5, c2, -0.5), -1.2247448713915890491 * s * c)
        AMP_SPIN(3, 2, SH::n3, SH::o3, c * fma(2.5, c2, -1.5), -0.43301270189221932338 * s * fma(5.0, c2, -1.0))
        AMP_SPIN(4, 3, SH::n4, SH::o4, fma(fma(4.375, c2, -3.75), c2, 0.375), -0.55901699437494742410 * s * c * fma(7.0, c2, -3.0))
#undef AMP_SPIN
        EvK k[E];
#pragma unroll
        for (int e = 0; e < E; ++e) {
            const double hp = 0.5 * (1.0 + cpsi.v[e]), hm = 0.5 * (1.0 - cpsi.v[e]);
            k[e].m2 = m2.v[e]; k[e].mZ2 = 0.0;
            k[e].cK = cK.v[e]; k[e].sK = sK.v[e];
            k[e].h0 = RSQRT2 * spsi.v[e];
            k[e].a1 = hp * cphi.v[e]; k[e].a2 = hp * sphi.v[e]; k[e].a3 = hm * cphi.v[e]; k[e].a4 = hm * sphi.v[e];
            // A_xi = sum_l e^{i l phi} d^1_{l xi}(theta_psi) V_l
            k[e].Ap = make_double2(k[e].h0 * V0[e].x, k[e].h0 * V0[e].y);
            k[e].Am = make_double2(-k[e].Ap.x, -k[e].Ap.y);
            k[e].Ap = cfma(Vp[e], make_double2(k[e].a1, k[e].a2), k[e].Ap);
            k[e].Am = cfma(Vp[e], make_double2(k[e].a3, k[e].a4), k[e].Am);
            k[e].Ap = cfma(Vm[e], make_double2(k[e].a3, -k[e].a4), k[e].Ap);
            k[e].Am = cfma(Vm[e], make_double2(k[e].a1, -k[e].a2), k[e].Am);
        }
        // ---- point 0: the Z chain; its staged columns stay in place for the point loop (Z slots read the angles)
        if (have_z) {
            mbar_wait(&full[1], parity);
            const Ev mZ2 = load_col(stage, C_MZ2), invmZ = load_col(stage, C_INVMZ);
            const Ev qZ = load_col(stage, C_QZ), pBZ = load_col(stage, C_PBZ);
            const Ev cZ = load_col(stage, C_CZ), sZ = load_col(stage, C_SZ);
            const Ev ct = load_col(stage, C_CT), st = load_col(stage, C_ST);
            const Ev cpt = load_col(stage, C_CPT), spt = load_col(stage, C_SPT);
            const Ev ca = load_col(stage, C_CA), sa = load_col(stage, C_SA);
            double2 Um[E], U0[E], Up[E];
#pragma unroll
            for (int e = 0; e < E; ++e) Um[e] = U0[e] = Up[e] = make_double2(0, 0);
            spin_sum<1, 0, 1, SH::nz, SH::oz, 5, true>(a, i0, mZ2, invmZ, qZ, pBZ, Um, U0, Up, fg);   // 1+ Z: L_R = 0, L_B = 1
#pragma unroll
            for (int e = 0; e < E; ++e) {
                const double z1 = RSQRT2 * sZ.v[e];
                const double2 T0 = cscale(cZ.v[e], U0[e]);
                const double2 Tp = cscale(z1, cmul(make_double2(cpt.v[e], spt.v[e]), Up[e]));
                const double2 Tm = cscale(-z1, cmul(make_double2(cpt.v[e], -spt.v[e]), Um[e]));
                const double gp = 0.5 * (1.0 + ct.v[e]), gm = 0.5 * (1.0 - ct.v[e]), g0 = RSQRT2 * st.v[e];
                const double2 Zp = make_double2(g0 * T0.x + gp * Tp.x + gm * Tm.x, g0 * T0.y + gp * Tp.y + gm * Tm.y);
                const double2 Zm = make_double2(-g0 * T0.x + gm * Tp.x + gp * Tm.x, -g0 * T0.y + gm * Tp.y + gp * Tm.y);
                k[e].Ap = cfma(make_double2(ca.v[e], sa.v[e]), Zp, k[e].Ap);
                k[e].Am = cfma(make_double2(ca.v[e], -sa.v[e]), Zm, k[e].Am);
                k[e].mZ2 = mZ2.v[e];
            }
        }
        double w[E];
        bool live[E];
#pragma unroll
        for (int e = 0; e < E; ++e) {
            live[e] = i0 + e < nlive;
            w[e] = is_norm ? wv.v[e] : 0.0;
            const double S0 = fma(k[e].Ap.x, k[e].Ap.x, fma(k[e].Ap.y, k[e].Ap.y, fma(k[e].Am.x, k[e].Am.x, k[e].Am.y * k[e].Am.y)));
            k[e].S0 = S0;
            k[e].Sguard = DELTA_CANCEL * S0;
            if (is_norm) {
                bad |= live[e] && !isfinite(S0);
                acc0N = fma(w[e], S0, acc0N);
            } else {
                const bool ok = S0 > 0.0 && isfinite(S0);
                bad |= live[e] && !ok;
                double f; int x1, x2;
                split_exp((live[e] && ok) ? S0 : 1.0, &f, &x1);
                split_exp(acc0F * f, &acc0F, &x2);   // running product of mantissas, renormalised to [0.5, 1)
                acc0E += x1 + x2;
            }
        }
        // ---- the points, 32 per block; lane totals go to the per-lane accumulators
        SlotVal sv[E];
#pragma unroll
        for (int e = 0; e < E; ++e) { sv[e].Sp = sv[e].Sm = sv[e].bw0 = sv[e].T2 = make_double2(0.0, 0.0); sv[e].n = 0.0; }
        int it = 0;
        for (int b = 0; b < nblk; ++b) {
            double v; int x;
            const int slot = b * THREADS + tid;
            if (is_norm) {
                eval_block<true, FAST>(a, prog, slots, it, k, fg, zst, sv, w, live, bad, lane, &v, &x);
                accN[slot] += v;
            } else {
                eval_block<false, FAST>(a, prog, slots, it, k, fg, zst, sv, w, live, bad, lane, &v, &x);
                double f; int x2;
                split_exp(accF[slot] * v, &f, &x2);
                accF[slot] = f;
                accE[slot] += x + x2;
            }
        }
        __syncthreads();   // Z region (and the group factors) no longer needed: stream the next tile's Z columns
        if (have_z && tid == 0 && has_next) issue(tile + gridDim.x, 1);
    }
    for (int b = 0; b < nblk; ++b) bad |= !isfinite(accN[b * THREADS + tid]);   // a non-finite S on the normalisation side
    if (bad & 1) atomicOr(a.flag, 2);
    if (bad & 2) atomicOr(a.flag, 1024);

    // ---- per-CTA partials: partial[(seg * rows + row) * stride + cta], seg 0 = sum log S (data), 1 = sum w S (norm);
    //      row 0 = point 0, row 1 + s = point s of this launch
    const double LN2 = 0.69314718055994530942;
    const int rows = 1 + d.nsorted;
    {
        const double t0 = block_sum(log(acc0F) + (double)acc0E * LN2, sm);
        const double t1 = block_sum(acc0N, sm);
        if (tid == 0) { d.partial[(size_t)0 * d.stride + blockIdx.x] = t0; d.partial[(size_t)rows * d.stride + blockIdx.x] = t1; }
    }
    __syncthreads();
    for (int idx = tid; idx < d.nsorted; idx += THREADS) {
        const int b = idx >> 5, l = idx & 31;
        double sN = 0.0, sL = 0.0;
        for (int wv = 0; wv < THREADS / 32; ++wv) {   // the warp totals in warp order
            const int slot = b * THREADS + wv * 32 + l;
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
    double* tot = accN;   // [2 rows]: the accumulators are dead (2 * 129 doubles fit)
    for (int r = tid; r < 2 * rows; r += THREADS) {
        const double* p = d.partial + (size_t)r * d.stride;
        double s = 0.0;
        for (unsigned c = 0; c < gridDim.x; ++c) s += __ldcg(p + c);
        tot[r] = s;
    }
    __syncthreads();
    if (FAST) {
        // quads of coupling points (eval_block): the four normalisation rows hold sum w T2.re, sum w T2.im, sum w n, 0 of the
        // quad's slot; point j of the quad is sum w S(0) + Re(coef_j T2) + |coef_j|^2 n.  Thread q takes the q-th group of four.
        __shared__ int s_first[DELTA_MAX_SORTED / 4];   // first contribution of each aligned group of four points
        if (tid == 0) {
            int it = 0;
            for (int idx = 0; idx < d.nsorted; ++idx) {
                if ((idx & 3) == 0) s_first[idx >> 2] = it;
                while (!(prog[it++].hdr & 4)) {}
            }
        }
        __syncthreads();
        if (tid < d.nsorted / 4) {
            const DeltaContrib* c = prog + s_first[tid];
            if ((c[0].hdr & 64) && (c[0].hdr & 3) == 0) {
                double* row = tot + rows + 1 + 4 * tid;
                const double t2r = row[0], t2i = row[1], nn = row[2], s0 = tot[rows];
#pragma unroll
                for (int j = 0; j < 4; ++j) row[j] = fma(c[j].c, nn, fma(c[j].a, t2r, fma(-c[j].b, t2i, s0)));
            }
        }
        __syncthreads();
    }
    for (int r = tid; r < rows; r += THREADS) {
        const int p = r == 0 ? 0 : d.point_of_sorted[r - 1];
        if (p < 0) continue;
        const double I = tot[rows + r] / a.wsum;
        d.result[d.P + p] = I;
        d.result[2 * d.P + 1 + p] = tot[r];
        d.result[3 * d.P + 1 + p] = tot[rows + r];
        double v = -(tot[r] + a.sum_log_eff) + (double)a.n * log(I);
        if (!isfinite(v) || !(I > 0.0)) v = INFINITY;
        d.result[p] = d.want_nll ? v : 0.0;
    }
    if (tid == 0) {
        const double fl = (double)atomicExch(a.flag, 0);   // domain flag of this launch, cleared for the next one
        d.result[2 * d.P] = d.first_chunk ? fl : d.result[2 * d.P] + fl;
        *a.ticket = 0u;
    }
}

namespace {

size_t delta_smem(bool have_z, int ngrp) {
    return (size_t)((have_z ? NCOL_ALL : NCOL_K) + 1) * TILE * sizeof(double) + (size_t)ngrp * TILE * sizeof(double2) +
           (size_t)DBLK * THREADS * (2 * sizeof(double) + sizeof(int)) + (size_t)DELTA_MAX_CONTRIB * sizeof(DeltaContrib) +
           (size_t)DELTA_MAX_SLOTWORDS * sizeof(double) + 2 * sizeof(uint64_t);
}

template <class SH, bool FAST>
cudaError_t launch_delta_shape(const DeltaArgs& d, int grid, cudaStream_t s) {
    static DeviceOnce attr_done;
    cudaError_t e = cudaSuccess;
    if (attr_done.first()) { e = cudaFuncSetAttribute(k_delta<SH, FAST>, cudaFuncAttributeMaxDynamicSharedMemorySize, 224 * 1024); }
    if (e != cudaSuccess) return e;
    const bool have_z = d.a.gstart[NSPIN] > d.a.gstart[5];
    k_delta<SH, FAST><<<grid, THREADS, delta_smem(have_z, d.a.gstart[NSPIN]), s>>>(d);
    return cudaGetLastError();
}

}  // namespace

bool delta_fits(int ngrp) { return delta_smem(true, ngrp) <= (size_t)224 * 1024; }

int delta_grid(long long n_data, long long n_norm) {
    const long long ntiles = (n_data + TILE - 1) / TILE + (n_norm + TILE - 1) / TILE;
    return (int)(ntiles < 1 ? 1 : (ntiles > sm_count() ? sm_count() : ntiles));   // persistent: one CTA per SM
}

// the paper's model (ten K* + one Z, one radius per spin) runs the unrolled shape; anything else the generic loops.
// exact: the repeat of a call whose expansion guard tripped — amplitudes summed term by term, generic kernel.
cudaError_t launch_delta(const DeltaArgs& d, int grid, cudaStream_t s, bool exact) {
    if (exact) return launch_delta_shape<Generic, false>(d, grid, s);
    const int* n = d.a.shape;
    if (d.a.shape_fixed && n[0] == 3 && n[1] == 3 && n[2] == 2 && n[3] == 1 && n[4] == 1 && n[5] == 1 && n[6] + n[7] + n[8] + n[9] == 0)
        return launch_delta_shape<Shape<3, 3, 2, 1, 1, 1>, true>(d, grid, s);
    return launch_delta_shape<Generic, true>(d, grid, s);
}

}  // namespace amp
