// gradf.cu — the NLL and its analytic gradient in all complex couplings, shape-specialised form of grad.cu
// for the paper's resonance lists (ten K* with and without 1+ Z's): same sums, same partial rows and
// the same last-CTA finish (grad_tail.cuh), but every gradient component lives in a REGISTER of the thread that owns the event.
//
// With A_xi = sum_k c_k B_k,xi and S = sum_xi |A_xi|^2 (Eqs. 4, 5, 10, 12),
//   dNLL/dconj(c_k) = - sum_i u_i sum_xi conj(B_k,xi(i)) A_xi(i)  + N [sum_j w_j sum_xi conj(B_k,xi(j)) A_xi(j)] / [sum_j w_j S_j],  u_i = 1/S_i
// and B_k,xi = BW_R d^J_{lambda 0}(theta_K*) e^{i lambda phi} d^1_{lambda xi}(theta_psi), so per event
//   W_lambda = u sum_xi conj(e^{i lambda phi} d^1_{lambda xi}) A_xi            three complex numbers, once per event
//   X_{J,lambda} = d^J_{lambda 0} W_lambda                                      one real scaling per spin
//   leaf (R, lambda) += conj(BW_R) X_{J(R),lambda}                              four FMAs per coupling slot
// (the Z chain of Eq. 10 likewise with its own angles).  The 2 K running sums (54 doubles for the ten K* and one Z) stay in
// registers for the whole kernel: no shuffle, no shared-memory accumulator and no index arithmetic per slot, because the
// model shape is a template argument and every loop unrolls.  grad.cu reduces every leaf across the warp for every event
// instead (it cannot index registers at run time); this kernel reduces once per CTA.
//
// Thread = one event of a 256-event unit (half a cache block); four units in flight per CTA (cp.async.bulk + full / empty
// mbarrier ring, one 2 KB copy per cache column issued by the lanes of warp 0, no CTA-wide barrier in the loop); the lineshapes
// of the event stay in registers between the forward pass and the gradient pass.  One CTA of 256 threads per SM (the
// accumulators take 108 registers), data units first, then the normalisation units; fixed order everywhere: bit-reproducible.
#define AMP_STREAM_E 2
#define AMP_STREAM_THREADS 256
#define AMP_STREAM_MINB 1
#include "stream_core.cuh"
#include "grad_tail.cuh"

namespace amp {

namespace {

constexpr int UNIT = THREADS;   // events per pipeline unit (half a cache block)
constexpr int NSTAGE = 4;
static_assert(2 * UNIT == CACHE_TILE, "two units per cache block");

__device__ __forceinline__ void mbar_arrive(uint64_t* bar) {
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(smem_u32(bar)) : "memory");
}

template <class SH>
struct Lay {
    static constexpr int NENT = SH::oz + SH::nz;                        // Breit-Wigner entries, spin-class order
    static constexpr int NACC = SH::n0 + 3 * (NENT - SH::n0);           // complex accumulators = coupling slots
    __host__ __device__ static constexpr int base(int t) { return t < SH::n0 ? t : SH::n0 + 3 * (t - SH::n0); }
};

// lineshapes of one spin class: U_l += c BW (couplings carry kN), BW / kN kept (bwr: registers, every index a constant after unrolling)
template <int J, int LRv, int LBv, int CNT, int OFF, int SPIN>
__device__ __forceinline__ void class_forward(const StreamArgs& a, double m2, double invm, double pR, double pB, double2* bwr, double2& Um,
                                              double2& U0, double2& Up) {
    double F, G;
    group_factors<LRv, LBv>(a.r2_spin[SPIN], invm, pR, pB, &F, &G);
#pragma unroll
    for (int t = 0; t < CNT; ++t) {
        const ResEntry& en = a.ent[OFF + t];
        const double2 bw = bw_unscaled(en, m2, F, G);
        bwr[OFF + t] = bw;
        U0 = cfma(en.c0, bw, U0);
        if (J) { Um = cfma(en.cm, bw, Um); Up = cfma(en.cp, bw, Up); }
    }
}

// acc += conj(bw) x
__device__ __forceinline__ void conj_fma(double2 bw, double2 x, double2& acc) {
    acc.x = fma(bw.x, x.x, fma(bw.y, x.y, acc.x));
    acc.y = fma(bw.x, x.y, fma(-bw.y, x.x, acc.y));
}

// gradient leaves of one spin class: slots (lambda = -1, 0, +1) of entry OFF + t are accumulators base(OFF + t) + 0, 1, 2
template <class SH, int J, int CNT, int OFF, int NACC>
__device__ __forceinline__ void class_leaves(const double2* bwr, double2 Xm, double2 X0, double2 Xp, double2 (&acc)[NACC]) {
#pragma unroll
    for (int t = 0; t < CNT; ++t) {
        const double2 bw = bwr[OFF + t];
        const int b = Lay<SH>::base(OFF + t);
        if (J == 0) {
            conj_fma(bw, X0, acc[b]);
        } else {
            conj_fma(bw, Xm, acc[b]);
            conj_fma(bw, X0, acc[b + 1]);
            conj_fma(bw, Xp, acc[b + 2]);
        }
    }
}

}  // namespace

template <class SH>
__global__ void __launch_bounds__(THREADS, 1) k_gradf(const __grid_constant__ GradArgs g) {
    using L = Lay<SH>;
    constexpr int NENT = L::NENT, NACC = L::NACC;
    constexpr bool have_z = SH::nz > 0;
    const StreamArgs& a = g.a;
    const double RSQRT2 = 0.70710678118654752440, LN2 = 0.69314718055994530942;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int ncolw = a.ncolw;                      // cache columns per block, the weight last
    const int nleaf = 2 * g.npairs;

    extern __shared__ __align__(128) unsigned char smem_raw[];
    double* stage0 = reinterpret_cast<double*>(smem_raw);                                        // [NSTAGE][ncolw][UNIT]
    double* red = stage0 + (size_t)NSTAGE * ncolw * UNIT;                                        // the flushes: [NWARPS][2 NACC]; the finish: 3 + 2 nleaf
    uint64_t* full = reinterpret_cast<uint64_t*>(red + NWARPS * 2 * NACC);
    __shared__ double sm[NWARPS];
    __shared__ bool s_last;
    uint64_t* empty = full + NSTAGE;   // a stage is free again once every warp has read its event's columns
    if (tid == 0) {
        for (int s = 0; s < NSTAGE; ++s) { mbar_init(&full[s], 1); mbar_init(&empty[s], NWARPS); }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();
    // units: the halves of the data blocks, then the halves of the normalisation blocks
    const long long nud = 2 * ((a.n + CACHE_TILE - 1) / CACHE_TILE), nunits = nud + 2 * ((a.n2 + CACHE_TILE - 1) / CACHE_TILE);
    auto issue = [&](long long unit, int s) {   // warp 0: one 2 KB copy per cache column
        const bool nrm = unit >= nud;
        const long long lu = nrm ? unit - nud : unit;
        const double* src = (nrm ? a.cache2 : a.cache) + (size_t)(lu >> 1) * ncolw * CACHE_TILE + (size_t)(lu & 1) * UNIT;
        if (lane == 0) mbar_expect_tx(&full[s], (uint32_t)ncolw * UNIT * sizeof(double));
        __syncwarp();
        if (lane < ncolw) bulk_g2s(stage0 + ((size_t)s * ncolw + lane) * UNIT, src + (size_t)lane * CACHE_TILE, UNIT * sizeof(double), &full[s]);
    };
    if (warp == 0)
        for (int s = 0; s < NSTAGE; ++s)
            if (blockIdx.x + (long long)s * gridDim.x < nunits) issue(blockIdx.x + (long long)s * gridDim.x, s);

    double2 acc[NACC];
#pragma unroll
    for (int q = 0; q < NACC; ++q) acc[q] = make_double2(0.0, 0.0);
    double accF = 1.0, accW = 0.0;   // sum log S as mantissa product / exponent sum; sum w S
    int accE = 0;
    bool bad = false, in_norm = false;

    // per-CTA partial rows of the leaves held in acc: scaled by kN (the records hold BW / kN), summed over the warp by a fixed
    // xor tree, then over the warps in warp order
    auto flush = [&](int row0) {
        __syncthreads();
#pragma unroll
        for (int t = 0; t < NENT; ++t) {
            const double kN = a.ent[t].kN;
            const int b = L::base(t);
#pragma unroll
            for (int j = 0; j < (t < SH::n0 ? 1 : 3); ++j) {
                double x = acc[b + j].x * kN, y = acc[b + j].y * kN;
#pragma unroll
                for (int o = 16; o; o >>= 1) { x += __shfl_xor_sync(0xffffffffu, x, o); y += __shfl_xor_sync(0xffffffffu, y, o); }
                if (lane == 0) { red[warp * 2 * NACC + 2 * (b + j)] = x; red[warp * 2 * NACC + 2 * (b + j) + 1] = y; }
                acc[b + j] = make_double2(0.0, 0.0);
            }
        }
        __syncthreads();
        for (int idx = tid; idx < nleaf; idx += THREADS) {
            double s = 0.0;
            int row = idx;                                        // padding pairs: rows past the slots, zero
            if (idx < 2 * NACC) {
                for (int wv = 0; wv < NWARPS; ++wv) s += red[wv * 2 * NACC + idx];
                row = 2 * g.acc_pair[idx >> 1] + (idx & 1);
            }
            g.partial[(size_t)(row0 + row) * g.stride + blockIdx.x] = s;
        }
        __syncthreads();
    };

    long long k = 0;
    for (long long unit = blockIdx.x; unit < nunits; unit += gridDim.x, ++k) {
        const int s = (int)(k % NSTAGE);
        const uint32_t parity = (uint32_t)((k / NSTAGE) & 1);
        const bool is_norm = unit >= nud;
        if (is_norm && !in_norm) {   // this CTA's data units are complete
            const double t0 = block_sum(log(accF) + (double)accE * LN2, sm);
            if (tid == 0) g.partial[(size_t)0 * g.stride + blockIdx.x] = t0;
            flush(2);
            in_norm = true;
        }
        const long long lu = is_norm ? unit - nud : unit;
        const bool live = lu * UNIT + tid < (is_norm ? a.n2 : a.n);
        mbar_wait(&full[s], parity);
        const double* st = stage0 + (size_t)s * ncolw * UNIT + tid;
        // ---- the point: K* chain (Eq. 4)
        const double m2 = st[C_M2 * UNIT], invm = st[C_INVM * UNIT], q = st[C_Q * UNIT], pB = st[C_PB * UNIT];
        const double cK = st[C_CK * UNIT], sK = st[C_SK * UNIT], cK2 = cK * cK;
        // d^J_{00} = P_J(cK), d^J_{+1,0} = -sK P_J'(cK) / sqrt(J(J+1))
        const double d10 = cK, d11 = -RSQRT2 * sK;
        const double d20 = fma(1.5, cK2, -0.5), d21 = -1.2247448713915890491 * sK * cK;
        const double d30 = cK * fma(2.5, cK2, -1.5), d31 = -0.43301270189221932338 * sK * fma(5.0, cK2, -1.0);
        const double d40 = fma(fma(4.375, cK2, -3.75), cK2, 0.375), d41 = -0.55901699437494742410 * sK * cK * fma(7.0, cK2, -3.0);
        double2 V0 = make_double2(0, 0), Vp = V0, Vm = V0;
        double2 rec[NENT];   // BW_R / kN of this event
#define AMP_FSPIN(J, LB, CNT, OFF, D0, D1)                                                  \
        if (CNT > 0) {                                                                       \
            double2 Um = make_double2(0, 0), U0 = Um, Up = Um;                               \
            class_forward<J, J, LB, CNT, OFF, J>(a, m2, invm, q, pB, rec, Um, U0, Up);       \
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
        // ---- the point: Z chain (Eq. 10), 1+ only in the specialised shapes
        double zc0 = 0, zcp = 0, gp = 0, gm = 0, g0 = 0, cpt = 0, spt = 0, ca = 0, sa = 0;
        if (have_z) {
            const double mZ2 = st[C_MZ2 * UNIT], invmZ = st[C_INVMZ * UNIT], qZ = st[C_QZ * UNIT], pBZ = st[C_PBZ * UNIT];
            zc0 = st[C_CZ * UNIT];                       // d^1_{00}(theta_Z)
            zcp = RSQRT2 * st[C_SZ * UNIT];              // d^1_{0,+1}(theta_Z) = -d^1_{0,-1}
            const double ct = st[C_CT * UNIT], stt = st[C_ST * UNIT];
            cpt = st[C_CPT * UNIT]; spt = st[C_SPT * UNIT]; ca = st[C_CA * UNIT]; sa = st[C_SA * UNIT];
            double2 Um = make_double2(0, 0), U0 = Um, Up = Um;
            class_forward<1, 0, 1, SH::nz, SH::oz, 5>(a, mZ2, invmZ, qZ, pBZ, rec, Um, U0, Up);
            const double2 T0 = cscale(zc0, U0);
            const double2 Tp = cmul(make_double2(cpt, spt), cscale(zcp, Up));      // e^{+i phi~}
            const double2 Tm = cmul(make_double2(cpt, -spt), cscale(-zcp, Um));    // e^{-i phi~}
            gp = 0.5 * (1.0 + ct); gm = 0.5 * (1.0 - ct); g0 = RSQRT2 * stt;
            const double2 Zp = make_double2(g0 * T0.x + gp * Tp.x + gm * Tm.x, g0 * T0.y + gp * Tp.y + gm * Tm.y);
            const double2 Zm = make_double2(-g0 * T0.x + gm * Tp.x + gp * Tm.x, -g0 * T0.y + gm * Tp.y + gp * Tm.y);
            Ap = cfma(make_double2(ca, sa), Zp, Ap);      // e^{+i alpha}
            Am = cfma(make_double2(ca, -sa), Zm, Am);     // e^{-i alpha}
        }
        const double wgt = st[(ncolw - 1) * UNIT];
        __syncwarp();
        if (lane == 0) mbar_arrive(&empty[s]);   // this warp has read everything it needs from the stage
        // Refill the stage of the PREVIOUS unit (every warp released it before its gradient pass, so this rarely waits) with the
        // unit NSTAGE steps after it.  The warps take turns: a fixed producer warp would fall behind the others by its extra work
        // until they run into the end of the ring and wait for a whole memory latency every unit.  No CTA-wide barrier in the loop.
        if (k > 0 && warp == (int)(k & (NWARPS - 1)) && unit + (long long)(NSTAGE - 1) * gridDim.x < nunits) {
            const int ps = (int)((k - 1) % NSTAGE);
            mbar_wait(&empty[ps], (uint32_t)(((k - 1) / NSTAGE) & 1));
            issue(unit + (long long)(NSTAGE - 1) * gridDim.x, ps);
        }
        const double S = fma(Ap.x, Ap.x, fma(Ap.y, Ap.y, fma(Am.x, Am.x, Am.y * Am.y)));
        double u;   // weight of this event in the gradient sums
        if (is_norm) {
            bad |= live && !isfinite(S);
            accW = fma(wgt, S, accW);        // padding events carry w = 0
            u = wgt;
        } else {
            const bool ok = S > 0.0 && isfinite(S);
            bad |= live && !ok;
            double f; int x1, x2;
            split_exp((live && ok) ? S : 1.0, &f, &x1);
            split_exp(accF * f, &accF, &x2);
            accE += x1 + x2;
            u = (live && ok) ? fast_rcp(S) : 0.0;
        }
        // ---- gradient leaves, K* chain: W_l = u sum_xi conj(g_{l,xi}) A_xi
        {
            const double2 uAp = cscale(u, Ap), uAm = cscale(u, Am);
            const double2 W0 = make_double2(h0 * (uAp.x - uAm.x), h0 * (uAp.y - uAm.y));
            // conj(x + i y) A = (x A.x + y A.y, x A.y - y A.x)
            const double2 Wp = make_double2(fma(a1, uAp.x, fma(a2, uAp.y, fma(a3, uAm.x, a4 * uAm.y))),
                                            fma(a1, uAp.y, fma(-a2, uAp.x, fma(a3, uAm.y, -a4 * uAm.x))));
            // lambda = -1: g_+ = -a3 + i a4, g_- = -a1 + i a2 (the sign of d^J_{-1,0} folded in, so X_{J,-1} = d^J_{+1,0} Wm)
            const double2 Wm = make_double2(fma(-a3, uAp.x, fma(a4, uAp.y, fma(-a1, uAm.x, a2 * uAm.y))),
                                            fma(-a3, uAp.y, fma(-a4, uAp.x, fma(-a1, uAm.y, -a2 * uAm.x))));
            class_leaves<SH, 0, SH::n0, 0, NACC>(rec, W0, W0, W0, acc);
            class_leaves<SH, 1, SH::n1, SH::o1, NACC>(rec, cscale(d11, Wm), cscale(d10, W0), cscale(d11, Wp), acc);
            class_leaves<SH, 2, SH::n2, SH::o2, NACC>(rec, cscale(d21, Wm), cscale(d20, W0), cscale(d21, Wp), acc);
            class_leaves<SH, 3, SH::n3, SH::o3, NACC>(rec, cscale(d31, Wm), cscale(d30, W0), cscale(d31, Wp), acc);
            class_leaves<SH, 4, SH::n4, SH::o4, NACC>(rec, cscale(d41, Wm), cscale(d40, W0), cscale(d41, Wp), acc);
            // ---- Z chain: B_{l',xi} = BW_Z d^1_{0 l'}(theta_Z) e^{i l' phi~} d^1_{l' xi}(theta~) e^{i xi alpha}
            if (have_z) {
                const double2 Bp = make_double2(fma(ca, uAp.x, sa * uAp.y), fma(ca, uAp.y, -sa * uAp.x));    // conj(e^{+i alpha}) u A+
                const double2 Bm = make_double2(fma(ca, uAm.x, -sa * uAm.y), fma(ca, uAm.y, sa * uAm.x));    // conj(e^{-i alpha}) u A-
                const double2 Y0 = make_double2(zc0 * g0 * (Bp.x - Bm.x), zc0 * g0 * (Bp.y - Bm.y));
                const double2 Rp = make_double2(fma(gp, Bp.x, gm * Bm.x), fma(gp, Bp.y, gm * Bm.y));         // l' = +1: d^1_{1,+} = gp, d^1_{1,-} = gm
                const double2 Rm = make_double2(fma(gm, Bp.x, gp * Bm.x), fma(gm, Bp.y, gp * Bm.y));         // l' = -1
                // conj(e^{+-i phi~}) R, times d^1_{0,+-1}(theta_Z) = +-zcp
                const double2 Yp = make_double2(zcp * fma(cpt, Rp.x, spt * Rp.y), zcp * fma(cpt, Rp.y, -spt * Rp.x));
                const double2 Ym = make_double2(-zcp * fma(cpt, Rm.x, -spt * Rm.y), -zcp * fma(cpt, Rm.y, spt * Rm.x));
                class_leaves<SH, 1, SH::nz, SH::oz, NACC>(rec, Ym, Y0, Yp, acc);
            }
        }
    }
    if (bad) atomicOr(a.flag, 2);

    // ---- per-CTA partials: rows 0, 1 = sum log S, sum w S; rows 2 + j = data-side leaf j; rows 2 + nleaf + j = normalisation side
    if (!in_norm) {   // this CTA saw data units only
        const double t0 = block_sum(log(accF) + (double)accE * LN2, sm);
        if (tid == 0) g.partial[(size_t)0 * g.stride + blockIdx.x] = t0;
        flush(2);
    }
    flush(2 + nleaf);   // zeros if no normalisation unit was walked
    {
        const double t1 = block_sum(accW, sm);
        if (tid == 0) {
            g.partial[(size_t)1 * g.stride + blockIdx.x] = t1;
            g.partial[(size_t)(2 + 2 * nleaf) * g.stride + blockIdx.x] = 0.0;
        }
    }
    // ---- the last CTA to finish adds the partials of every row in CTA order and forms NLL, I and the gradient
    __threadfence();
    __syncthreads();
    if (tid == 0) s_last = atomicAdd(a.ticket, 1u) == gridDim.x - 1;
    __syncthreads();
    if (!s_last) return;
    __threadfence();
    grad_finish(g, red, nleaf, tid, THREADS, gridDim.x);
}

namespace {

size_t gradf_smem(int ncolw, int nacc) {
    return (size_t)NSTAGE * ncolw * UNIT * sizeof(double) + (size_t)NWARPS * 2 * nacc * sizeof(double) + 2 * NSTAGE * sizeof(uint64_t);
}

template <class SH>
cudaError_t launch_gradf_shape(const GradArgs& g, int grid, cudaStream_t s) {
    static DeviceOnce attr_done;
    cudaError_t e = cudaSuccess;
    if (attr_done.first()) { e = cudaFuncSetAttribute(k_gradf<SH>, cudaFuncAttributeMaxDynamicSharedMemorySize, 224 * 1024); }
    if (e != cudaSuccess) return e;
    k_gradf<SH><<<grid, THREADS, gradf_smem(g.a.ncolw, Lay<SH>::NACC), s>>>(g);
    return cudaGetLastError();
}

}  // namespace

int gradf_grid(long long n_data, long long n_norm) {
    const long long nunits = 2 * ((n_data + CACHE_TILE - 1) / CACHE_TILE) + 2 * ((n_norm + CACHE_TILE - 1) / CACHE_TILE);
    return (int)(nunits < 1 ? 1 : (nunits > sm_count() ? sm_count() : nunits));   // persistent: one CTA per SM
}

// 1 if the point is one of the specialised shapes (one radius per spin class, no constant or LASS term, no background, Z's
// of spin-parity 1+ only) — the caller then fills g.acc_pair and launches this kernel instead of k_grad
bool gradf_supports(const GradArgs& g) {
    const StreamArgs& a = g.a;
    const int* n = a.shape;
    if (!a.shape_fixed || a.nlass > 0 || a.bkg || a.cconst.x != 0.0 || a.cconst.y != 0.0) return false;
    if (n[6] + n[7] + n[8] + n[9] != 0) return false;
    if (!(n[0] == 3 && n[1] == 3 && n[2] == 2 && n[3] == 1 && n[4] == 1 && n[5] >= 0 && n[5] <= 2)) return false;
    if (a.ncolw != (n[5] > 0 ? NCOL_ALL : NCOL_K) + 1) return false;
    for (int p = 0; p < g.npairs; ++p)
        if (g.pair_ent[p] == -1) return false;
    return true;
}

cudaError_t launch_gradf(const GradArgs& g, int grid, cudaStream_t s) {
    switch (g.a.shape[5]) {
        case 0: return launch_gradf_shape<Shape<3, 3, 2, 1, 1, 0>>(g, grid, s);
        case 1: return launch_gradf_shape<Shape<3, 3, 2, 1, 1, 1>>(g, grid, s);
        default: return launch_gradf_shape<Shape<3, 3, 2, 1, 1, 2>>(g, grid, s);
    }
}

}  // namespace amp
