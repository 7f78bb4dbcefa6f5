// stream.cu — steps a2 + a3 + a5 (and the direct-sum form of a4) for ONE parameter point: lineshapes,
// streaming amplitude combine and the -log L / normalisation reduction fused in one pass over the cache.
//
// Per event (Eqs. 2-5, 10, 12), with c_k the couplings and BW_R the lineshape
// of resonance R:
//   K* chain   V_l   = sum_J d^J_{l0}(theta_K*) sum_{R in J} c_{R,l} BW_R          l = -1, 0, +1
//              A_xi  = sum_l e^{i l phi} d^1_{l xi}(theta_psi) V_l
//   Z chain    T_l'  = d^1_{0 l'}(theta_Z) e^{i l' phi~} sum_Z c_{Z,l'} BW_Z
//              A_xi += e^{i xi alpha} sum_l' d^1_{l' xi}(theta~) T_l'
//   S = |A_+|^2 + |A_-|^2
// The coherent sum is grouped by spin so the d-functions multiply a partial sum once (the dense
// contraction events x basis x couplings with its angular factors pulled out).
//
// Lineshapes are evaluated in registers (no HBM round trip) unless an entry points at a pool column.
// On B200 the FP64 pipe and HBM are balanced such that recomputing a Breit-Wigner (about 14 FP64
// instructions once the barrier factors are shared, see BarrierGroup) is cheaper than reading its 16 B
// column, so for P = 1 the in-register form is the default.  The spin loop
// is unrolled at compile time: L_R = J and L_B are constants inside it, so barrier polynomials and
// momentum powers are straight-line code.
//
// Reduction: per-thread running sum over a grid-stride loop -> fixed xor-shuffle tree -> fixed-order sum
// of the 8 warp values -> one partial per block; k_finalize adds the block partials in a fixed order.
// No floating-point atomics: bitwise reproducible.
#include "amp_internal.cuh"

namespace amp {

// A^R = kN F / (M2 - m2 - i kG G)
__device__ __forceinline__ double2 bw_from_factors(const ResEntry& e, double m2, double F, double G) {
    const double MG = e.kG * G, dre = e.M2 - m2;
    const double s = e.kN * F * fast_rcp(fma(dre, dre, MG * MG));
    return make_double2(s * dre, s * MG);
}

// Partial sums U_l = sum_{R in spin-J groups} c_{R,l} BW_R for one spin (compile-time J).
template <int J>
__device__ __forceinline__ void spin_sum(const StreamArgs& a, long long i, double m2, double invm, double q, double pB, double2& Um,
                                         double2& U0, double2& Up) {
    constexpr int LB = (J == 0) ? 1 : J - 1;   // lowest allowed L_B
    for (int g = a.gstart[J]; g < a.gstart[J + 1]; ++g) {
        const BarrierGroup grp = a.grp[g];
        double F, G;
        group_factors<J, LB>(grp.r2, invm, q, pB, &F, &G);
        for (int t = grp.first; t < grp.first + grp.count; ++t) {
            const ResEntry& e = a.ent[t];
            const double2 bw = (e.column >= 0) ? a.cols[(size_t)e.column * a.npad + i] : bw_from_factors(e, m2, F, G);
            if (J == 0) {
                U0 = cfma(a.c[e.c0], bw, U0);
            } else {
                Um = cfma(a.c[e.c0], bw, Um);
                U0 = cfma(a.c[e.c0 + 1], bw, U0);
                Up = cfma(a.c[e.c0 + 2], bw, Up);
            }
        }
    }
}

template <int MODE>
__global__ void __launch_bounds__(256, 3) k_stream(const __grid_constant__ StreamArgs a) {
    const double RSQRT2 = 0.70710678118654752440;
    const bool have_z = a.gstart[6] > a.gstart[5];
    double acc = 0.0;
    bool bad = false;
    for (long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x; i < a.n; i += (long long)gridDim.x * blockDim.x) {
        const double* col = a.cache + i;
        const double m2 = col[C_M2 * a.npad], invm = col[C_INVM * a.npad], q = col[C_Q * a.npad], pB = col[C_PB * a.npad];
        const double cK = col[C_CK * a.npad], sK = col[C_SK * a.npad];
        const double cpsi = col[C_CPSI * a.npad], spsi = col[C_SPSI * a.npad];
        const double cphi = col[C_CPHI * a.npad], sphi = col[C_SPHI * a.npad];
        const double c2 = cK * cK;

        double2 V0 = make_double2(0, 0), Vp = V0, Vm = V0;
        for (int t = 0; t < a.nconst; ++t) V0 = cadd(V0, a.c[a.const_c0[t]]);   // constant term: lineshape 1, d^0_00 = 1
        // d^J_{00} = P_J(cK), d^J_{+1,0} = -sK P_J'(cK) / sqrt(J(J+1)), d^J_{-1,0} = -d^J_{+1,0}
        {
            double2 Um = make_double2(0, 0), U0 = Um, Up = Um;
            spin_sum<0>(a, i, m2, invm, q, pB, Um, U0, Up);
            V0 = cadd(V0, U0);
        }
        {
            double2 Um = make_double2(0, 0), U0 = Um, Up = Um;
            spin_sum<1>(a, i, m2, invm, q, pB, Um, U0, Up);
            const double d1 = -RSQRT2 * sK;
            V0 = cadd(V0, cscale(cK, U0)); Vp = cadd(Vp, cscale(d1, Up)); Vm = cadd(Vm, cscale(-d1, Um));
        }
        {
            double2 Um = make_double2(0, 0), U0 = Um, Up = Um;
            spin_sum<2>(a, i, m2, invm, q, pB, Um, U0, Up);
            const double d1 = -1.2247448713915890491 * sK * cK;                      // sqrt(3/2)
            V0 = cadd(V0, cscale(fma(1.5, c2, -0.5), U0)); Vp = cadd(Vp, cscale(d1, Up)); Vm = cadd(Vm, cscale(-d1, Um));
        }
        {
            double2 Um = make_double2(0, 0), U0 = Um, Up = Um;
            spin_sum<3>(a, i, m2, invm, q, pB, Um, U0, Up);
            const double d1 = -0.43301270189221932338 * sK * fma(5.0, c2, -1.0);     // sqrt(3)/4
            V0 = cadd(V0, cscale(cK * fma(2.5, c2, -1.5), U0)); Vp = cadd(Vp, cscale(d1, Up)); Vm = cadd(Vm, cscale(-d1, Um));
        }
        {
            double2 Um = make_double2(0, 0), U0 = Um, Up = Um;
            spin_sum<4>(a, i, m2, invm, q, pB, Um, U0, Up);
            const double d1 = -0.55901699437494742410 * sK * cK * fma(7.0, c2, -3.0);   // sqrt(5)/4
            V0 = cadd(V0, cscale(fma(fma(4.375, c2, -3.75), c2, 0.375), U0)); Vp = cadd(Vp, cscale(d1, Up)); Vm = cadd(Vm, cscale(-d1, Um));
        }
        // A_xi = sum_l e^{i l phi} d^1_{l xi}(theta_psi) V_l ; d^1_{0,+-1} = +-s/sqrt2, d^1_{11} = d^1_{-1-1} = (1+c)/2, d^1_{1-1} = d^1_{-11} = (1-c)/2
        const double2 Wp = cmul(make_double2(cphi, sphi), Vp), Wm = cmul(make_double2(cphi, -sphi), Vm);
        const double hp = 0.5 * (1.0 + cpsi), hm = 0.5 * (1.0 - cpsi), h0 = RSQRT2 * spsi;
        double2 Ap = make_double2(h0 * V0.x + hp * Wp.x + hm * Wm.x, h0 * V0.y + hp * Wp.y + hm * Wm.y);
        double2 Am = make_double2(-h0 * V0.x + hm * Wp.x + hp * Wm.x, -h0 * V0.y + hm * Wp.y + hp * Wm.y);

        if (have_z) {
            const double mZ2 = col[C_MZ2 * a.npad], invmZ = col[C_INVMZ * a.npad], qZ = col[C_QZ * a.npad], pBZ = col[C_PBZ * a.npad];
            const double cZ = col[C_CZ * a.npad], sZ = col[C_SZ * a.npad], ct = col[C_CT * a.npad], st = col[C_ST * a.npad];
            const double cpt = col[C_CPT * a.npad], spt = col[C_SPT * a.npad], ca = col[C_CA * a.npad], sa = col[C_SA * a.npad];
            double2 U0 = make_double2(0, 0), Up = U0, Um = U0;
            for (int g = a.gstart[5]; g < a.gstart[6]; ++g) {
                const BarrierGroup grp = a.grp[g];
                double F, G;
                group_factors<0, 1>(grp.r2, invmZ, qZ, pBZ, &F, &G);   // 1+ Z: L_R = 0, L_B = 1
                for (int t = grp.first; t < grp.first + grp.count; ++t) {
                    const ResEntry& e = a.ent[t];
                    const double2 bw = (e.column >= 0) ? a.cols[(size_t)e.column * a.npad + i] : bw_from_factors(e, mZ2, F, G);
                    Um = cfma(a.c[e.c0], bw, Um);
                    U0 = cfma(a.c[e.c0 + 1], bw, U0);
                    Up = cfma(a.c[e.c0 + 2], bw, Up);
                }
            }
            // T_l' = d^1_{0 l'}(theta_Z) e^{i l' phi~} U_l' ; d^1_{00} = cZ, d^1_{0,+-1} = +-sZ/sqrt2
            const double z1 = RSQRT2 * sZ;
            const double2 T0 = cscale(cZ, U0);
            const double2 Tp = cscale(z1, cmul(make_double2(cpt, spt), Up));
            const double2 Tm = cscale(-z1, cmul(make_double2(cpt, -spt), Um));
            const double gp = 0.5 * (1.0 + ct), gm = 0.5 * (1.0 - ct), g0 = RSQRT2 * st;
            const double2 Zp = make_double2(g0 * T0.x + gp * Tp.x + gm * Tm.x, g0 * T0.y + gp * Tp.y + gm * Tm.y);
            const double2 Zm = make_double2(-g0 * T0.x + gm * Tp.x + gp * Tm.x, -g0 * T0.y + gm * Tp.y + gp * Tm.y);
            Ap = cfma(make_double2(ca, sa), Zp, Ap);    // e^{+i alpha}
            Am = cfma(make_double2(ca, -sa), Zm, Am);   // e^{-i alpha}
        }
        const double S = fma(Ap.x, Ap.x, fma(Ap.y, Ap.y, fma(Am.x, Am.x, Am.y * Am.y)));
        if (MODE == MODE_DATA) {
            bad |= !(S > 0.0) || !isfinite(S);
            acc += log(S);
        } else if (MODE == MODE_NORM) {
            bad |= !isfinite(S);
            acc = fma(a.weight[i], S, acc);
        } else {
            a.out[i] = a.weight[i] * S;
        }
    }
    if (MODE == MODE_EVAL) return;
    if (bad) atomicOr(a.flag, 2);
    __shared__ double sm[8];
#pragma unroll
    for (int o = 16; o; o >>= 1) acc += __shfl_xor_sync(0xffffffffu, acc, o);
    if ((threadIdx.x & 31) == 0) sm[threadIdx.x >> 5] = acc;
    __syncthreads();
    if (threadIdx.x == 0) {
        double t = 0.0;
        for (int wv = 0; wv < 8; ++wv) t += sm[wv];
        a.partial[blockIdx.x] = t;
    }
}

int stream_grid(long long n) {
    long long blocks = (n + 255) / 256;
    const long long cap = 148 * 3 * 4;   // a multiple of 148 SMs x 3 resident CTAs
    return (int)(blocks < 1 ? 1 : (blocks > cap ? cap : blocks));
}

cudaError_t launch_stream(const StreamArgs& a, int grid, cudaStream_t s) {
    switch (a.mode) {
        case MODE_DATA: k_stream<MODE_DATA><<<grid, 256, 0, s>>>(a); break;
        case MODE_NORM: k_stream<MODE_NORM><<<grid, 256, 0, s>>>(a); break;
        default: k_stream<MODE_EVAL><<<grid, 256, 0, s>>>(a); break;
    }
    return cudaGetLastError();
}

}  // namespace amp
