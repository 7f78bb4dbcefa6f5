// delta_core.cuh — pieces shared by the point-loop kernels built on the streaming core (delta.cu: gradient batches;
// grad.cu: analytic gradient): what a thread keeps of its event, the angular factors of Eqs. 4 and 10 for one
// (spin, helicity) term, and the recursive-halving exchange that reduces 32 per-lane values per lane to one total per lane.
// Include after stream_core.cuh (uses its E / TILE).
#pragma once
#include "stream_core.cuh"

namespace amp {

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

struct EvK {   // what the point loop keeps of one event in registers
    double2 Ap, Am;                 // A_xi(0)
    double S0, Sguard;              // |A_+(0)|^2 + |A_-(0)|^2 (delta.cu: expansion point of the single-contribution points) and its guard level
    double m2, mZ2;
    double cK, sK;
    double h0, a1, a2, a3, a4;      // d^1_{0,+}(theta_psi); hp cos phi, hp sin phi, hm cos phi, hm sin phi
};
// Angular factor g_{J,lambda,xi} of one term for one event (Eq. 4 for a K*, Eq. 10 for the Z), given the d functions of the
// term's spin: (d0, d1) = (d^J_{00}, d^J_{+1,0}) at theta_K* for a K*, at theta_Z for a Z (where d^J_{0,+1} = -d^J_{+1,0}).
// zst: this event's element of the staged tile (the Z-chain angles stay there during the point loop).
__device__ __forceinline__ void term_angular_d(double d0, double d1, int lam, bool isz, const EvK& k, const double* zst, double2* gp, double2* gm) {
    const double RSQRT2 = 0.70710678118654752440;
    if (!isz) {
        if (lam == 0) {
            const double t = d0 * k.h0;
            *gp = make_double2(t, 0.0);
            *gm = make_double2(-t, 0.0);
        } else if (lam > 0) {                     // e^{+i phi} (hp, hm)
            *gp = make_double2(d1 * k.a1, d1 * k.a2);
            *gm = make_double2(d1 * k.a3, d1 * k.a4);
        } else {                                  // e^{-i phi} (hm, hp); d^J_{-1,0} = -d^J_{+1,0}
            *gp = make_double2(-d1 * k.a3, d1 * k.a4);
            *gm = make_double2(-d1 * k.a1, d1 * k.a2);
        }
        return;
    }
    // d^J_{0 l'}(theta_Z) e^{i l' phi~} d^1_{l' xi}(theta~) e^{i xi alpha};  d^J_{0,+1} = -d^J_{+1,0}, d^J_{0,-1} = d^J_{+1,0}
    const double ct = zst[C_CT * TILE], st = zst[C_ST * TILE];
    const double cpt = zst[C_CPT * TILE], spt = zst[C_SPT * TILE], ca = zst[C_CA * TILE], sa = zst[C_SA * TILE];
    const double zf = lam == 0 ? d0 : (lam > 0 ? -d1 : d1);
    const double dp = lam == 0 ? RSQRT2 * st : (lam > 0 ? 0.5 * (1.0 + ct) : 0.5 * (1.0 - ct));
    const double dm = lam == 0 ? -RSQRT2 * st : (lam > 0 ? 0.5 * (1.0 - ct) : 0.5 * (1.0 + ct));
    const double2 eph = lam == 0 ? make_double2(1.0, 0.0) : make_double2(cpt, lam > 0 ? spt : -spt);
    *gp = cscale(zf * dp, cmul(eph, make_double2(ca, sa)));
    *gm = cscale(zf * dm, cmul(eph, make_double2(ca, -sa)));
}
// the same with the d functions evaluated here.  Z1P: every Z of the model is a 1+ (the gradient-batch kernel's plans)
template <bool Z1P = false>
__device__ __forceinline__ void term_angular(int J, int lam, bool isz, const EvK& k, const double* zst, double2* gp, double2* gm) {
    double d0, d1;
    if (!isz) dJ(J, k.cK, k.sK, &d0, &d1);
    else if (Z1P) { d0 = zst[C_CZ * TILE]; d1 = -0.70710678118654752440 * zst[C_SZ * TILE]; }
    else dJ(J, zst[C_CZ * TILE], zst[C_SZ * TILE], &d0, &d1);
    term_angular_d(d0, d1, lam, isz, k, zst, gp, gm);
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

}  // namespace amp
