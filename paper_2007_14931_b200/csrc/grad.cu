// grad.cu — the NLL and its ANALYTIC gradient in all complex couplings in one pass over the data and the normalisation
// events (replaces the 2 x ~50 finite-difference points a MINUIT gradient step spends on the couplings).
//
// With A_xi = sum_k c_k B_k,xi and S = sum_xi |A_xi|^2 (Eqs. 4, 5, 10, 12),
//   dNLL/dconj(c_k) = - sum_i [sum_xi conj(B_k,xi(i)) A_xi(i)] / S_i + N [sum_j w_j sum_xi conj(B_k,xi(j)) A_xi(j)] / [sum_j w_j S_j]
// and B_k,xi = BW_R g_{J,lambda,xi}, so per event and slot the work is conj(BW_R) * T with T = sum_xi conj(g_xi) A_xi — two
// complex multiply-adds — times u = 1/S (data) or u = w (normalisation): the SAME kernel serves both sums.
//
// Thread = one event (512 threads, 16 warps per SM).  Per tile: the point as the streaming kernel does it (TMA-fed tile,
// lineshapes in registers, kept in a thread-private shared-memory record), then the 2 K gradient components as leaves of the
// recursive-halving exchange of delta_core.cuh: after every block of 32 leaves lane l holds the warp total of leaf 32 b + l.
// Fixed order everywhere: bit-reproducible.  The last CTA forms the NLL, the integral and the gradient.
#define AMP_STREAM_E 1
#define AMP_STREAM_THREADS 512
#include "stream_core.cuh"
#include "delta_core.cuh"
#include "grad_tail.cuh"

namespace amp {

namespace {

constexpr int GBLK = 2 * GRAD_MAX_PAIRS / 32;   // blocks of 32 leaves

// lineshapes of one spin class (runtime group loops): U_l += c BW, and BW itself (with its constant kN) into bw_rec
template <int J, int LR, int LB>
__device__ __forceinline__ void spin_class(const StreamArgs& a, int sp, double m2, double invm, double pR, double pB, double2* bw_rec,
                                           double2& Um, double2& U0, double2& Up) {
    for (int g = a.gstart[sp]; g < a.gstart[sp + 1]; ++g) {
        double F, G;
        group_factors<LR, LB>(a.grp[g].r2, invm, pR, pB, &F, &G);
        for (int t = a.grp[g].first; t < a.grp[g].first + a.grp[g].count; ++t) {
            const double2 bw = bw_unscaled(a.ent[t], m2, F, G);          // the entry's couplings carry kN
            bw_rec[t * TILE] = cscale(a.ent[t].kN, bw);
            U0 = cfma(a.ent[t].c0, bw, U0);
            if (J) { Um = cfma(a.ent[t].cm, bw, Um); Up = cfma(a.ent[t].cp, bw, Up); }
        }
    }
}

}  // namespace

__global__ void __launch_bounds__(THREADS, 1) k_grad(const __grid_constant__ GradArgs g) {
    const StreamArgs& a = g.a;
    const double RSQRT2 = 0.70710678118654752440, LN2 = 0.69314718055994530942;
    const int tid = threadIdx.x, lane = tid & 31;
    const bool have_z = a.gstart[NSPIN] > a.gstart[5];
    const int ncache = have_z ? NCOL_ALL : NCOL_K;
    int nent = a.nlass;   // Breit-Wigner entries of all spin classes + the LASS terms (stored after them)
    for (int sp = 0; sp < NSPIN; ++sp) nent += a.shape[sp];
    const int nleaf = 2 * g.npairs, nblk = nleaf / 32;

    extern __shared__ __align__(128) unsigned char smem_raw[];
    double* stage = reinterpret_cast<double*>(smem_raw);                                 // [ncache + 1][TILE]
    double2* bw_base = reinterpret_cast<double2*>(stage + (size_t)(ncache + 1) * TILE);   // [nent][TILE]
    double* accD = reinterpret_cast<double*>(bw_base + (size_t)nent * TILE);              // [GBLK][THREADS] data-side leaf totals
    double* accN = accD + GBLK * THREADS;                                                 // [GBLK][THREADS] normalisation side
    uint64_t* full = reinterpret_cast<uint64_t*>(accN + GBLK * THREADS);
    __shared__ double sm[NWARPS];
    __shared__ bool s_last;
    for (int b = 0; b < GBLK; ++b) { accD[b * THREADS + tid] = 0.0; accN[b * THREADS + tid] = 0.0; }
    if (tid == 0) {
        mbar_init(&full[0], 1);
        mbar_init(&full[1], 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();
    const long long ntd = (a.n + TILE - 1) / TILE;
    const long long ntiles = ntd + (a.n2 + TILE - 1) / TILE;
    auto issue = [&](long long tile, int region) {
        const bool nrm = tile >= ntd;
        const double* cache = nrm ? a.cache2 : a.cache;
        const long long lt = nrm ? tile - ntd : tile;
        if (region == 0) issue_cols(cache, a.ncolw, lt, stage, &full[0], 0, NCOL_K, true);
        else issue_cols(cache, a.ncolw, lt, stage, &full[1], NCOL_K, NCOL_ALL, false);
    };
    if (tid == 0 && (long long)blockIdx.x < ntiles) {
        issue(blockIdx.x, 0);
        if (have_z) issue(blockIdx.x, 1);
    }
    // Eq. 14 (background + purity): f_i = ps eps_i S_i + qb b_i with ps = purity / I, I = W / sum_j w_j, W = sum_j w_j S_j.  W is needed
    // before the first data event: from the held matrix (c^H M c, every CTA the same fixed-order sum) or from the normalisation
    // launch the host ran before this one.
    double bkg_ps = 0.0, bkg_qb = 0.0;
    if (a.bkg) {
        __shared__ double s_W;
        if (a.qf_G) {
            double r = 0.0;
            if (tid < a.qf_nent) {
                double2 acc = make_double2(0.0, 0.0);
                for (int f = 0; f < a.qf_nent; ++f) {
                    const double2 cf = a.qf_c[f];
                    const double* gm = a.qf_G + (size_t)(2 * tid) * a.qf_KP + 2 * f;
                    const double mre = gm[0] + gm[a.qf_KP + 1], mim = gm[1] - gm[a.qf_KP];
                    acc.x += mre * cf.x - mim * cf.y;
                    acc.y += mre * cf.y + mim * cf.x;
                }
                r = a.qf_c[tid].x * acc.x + a.qf_c[tid].y * acc.y;
            }
            const double t = block_sum(r, sm);
            if (tid == 0) s_W = t;
        } else if (tid == 0) {
            s_W = __ldcg(a.sum_wS);
        }
        __syncthreads();
        bkg_ps = a.purity * a.wsum / s_W;
        bkg_qb = 1.0 - a.purity;
    }
    double2* bw_rec = bw_base + tid;
    const double* st = stage + tid;
    double accF = 1.0, accW = 0.0;   // sum log S (log f with a background) as mantissa product / exponent sum; sum w S
    double accT = 0.0;               // background: sum_i u_i S_i, u_i = ps eps_i / f_i (= N without a background)
    int accE = 0;
    bool bad = false;
    uint32_t parity = 0;
    for (long long tile = blockIdx.x; tile < ntiles; tile += gridDim.x, parity ^= 1) {
        const bool has_next = tile + gridDim.x < ntiles;
        const bool is_norm = tile >= ntd;
        const long long lt = is_norm ? tile - ntd : tile;
        const bool live = lt * TILE + tid < (is_norm ? a.n2 : a.n);
        // ---- the point: K* chain
        mbar_wait(&full[0], parity);
        EvK k;
        k.m2 = st[C_M2 * TILE];
        k.cK = st[C_CK * TILE]; k.sK = st[C_SK * TILE];
        const double invm = st[C_INVM * TILE], q = st[C_Q * TILE], pB = st[C_PB * TILE];
        const double cpsi = st[C_CPSI * TILE], spsi = st[C_SPSI * TILE], cphi = st[C_CPHI * TILE], sphi = st[C_SPHI * TILE];
        const double wgt = st[ncache * TILE];
        __syncthreads();   // K* region (and the weights) consumed: stream the next tile into it
        if (tid == 0 && has_next) issue(tile + gridDim.x, 0);
        double2 V0 = a.cconst, Vp = make_double2(0, 0), Vm = Vp;
#define AMP_GSPIN(J, LB)                                                                        \
        if (a.gstart[J + 1] > a.gstart[J]) {                                                      \
            double2 Um = make_double2(0, 0), U0 = Um, Up = Um;                                    \
            spin_class<J, J, LB>(a, J, k.m2, invm, q, pB, bw_rec, Um, U0, Up);                    \
            double d0, d1;                                                                        \
            dJ(J, k.cK, k.sK, &d0, &d1);                                                          \
            V0 = cadd(V0, cscale(d0, U0));                                                        \
            if (J) { Vp = cadd(Vp, cscale(d1, Up)); Vm = cadd(Vm, cscale(-d1, Um)); }             \
        }
        AMP_GSPIN(0, 1)
        AMP_GSPIN(1, 0)
        AMP_GSPIN(2, 1)
        AMP_GSPIN(3, 2)
        AMP_GSPIN(4, 3)
#undef AMP_GSPIN
        for (int t = a.lass0; t < a.lass0 + a.nlass; ++t) {   // LASS S-wave terms (Eq. 7): J = 0, lambda = 0, no constant folded in
            const double2 bw = lass_eval(a.ent[t].M2, a.ent[t].kG, k.m2, invm, q);
            bw_rec[t * TILE] = bw;
            V0 = cfma(a.ent[t].c0, bw, V0);
        }
        {
            const double hp = 0.5 * (1.0 + cpsi), hm = 0.5 * (1.0 - cpsi);
            k.h0 = RSQRT2 * spsi;
            k.a1 = hp * cphi; k.a2 = hp * sphi; k.a3 = hm * cphi; k.a4 = hm * sphi;
            k.Ap = make_double2(k.h0 * V0.x, k.h0 * V0.y);
            k.Am = make_double2(-k.Ap.x, -k.Ap.y);
            k.Ap = cfma(Vp, make_double2(k.a1, k.a2), k.Ap);
            k.Am = cfma(Vp, make_double2(k.a3, k.a4), k.Am);
            k.Ap = cfma(Vm, make_double2(k.a3, -k.a4), k.Ap);
            k.Am = cfma(Vm, make_double2(k.a1, -k.a2), k.Am);
        }
        // ---- the point: Z chain (its staged columns stay in place: the gradient leaves of the Z slots read the angles)
        k.mZ2 = 0.0;
        if (have_z) {
            mbar_wait(&full[1], parity);
            k.mZ2 = st[C_MZ2 * TILE];
            const double invmZ = st[C_INVMZ * TILE], qZ = st[C_QZ * TILE], pBZ = st[C_PBZ * TILE];
            const double cZ = st[C_CZ * TILE], sZ = st[C_SZ * TILE], ct = st[C_CT * TILE], stt = st[C_ST * TILE];
            const double cpt = st[C_CPT * TILE], spt = st[C_SPT * TILE], ca = st[C_CA * TILE], sa = st[C_SA * TILE];
            // sum over the Z spin classes of d^J_{0 l'}(theta_Z) U_l' (d^J_{0,+1} = -d^J_{+1,0}), then the phi~ phases
            double2 T0 = make_double2(0, 0), Tp = T0, Tm = T0;
#define AMP_GZ(ZC, J, LR, LB)                                                                   \
            if (a.gstart[5 + ZC + 1] > a.gstart[5 + ZC]) {                                        \
                double2 Um = make_double2(0, 0), U0 = Um, Up = Um;                                \
                spin_class<J, LR, LB>(a, 5 + ZC, k.mZ2, invmZ, qZ, pBZ, bw_rec, Um, U0, Up);      \
                double d0, d1;                                                                    \
                dJ(J, cZ, sZ, &d0, &d1);                                                          \
                T0 = cadd(T0, cscale(d0, U0));                                                    \
                if (J) { Tp = cadd(Tp, cscale(-d1, Up)); Tm = cadd(Tm, cscale(d1, Um)); }         \
            }
            AMP_GZ(0, 1, 0, 1)   // 1+
            AMP_GZ(1, 2, 2, 2)   // 2+
            AMP_GZ(2, 0, 1, 0)   // 0-
            AMP_GZ(3, 1, 1, 1)   // 1-
            AMP_GZ(4, 2, 1, 2)   // 2-
#undef AMP_GZ
            Tp = cmul(make_double2(cpt, spt), Tp);
            Tm = cmul(make_double2(cpt, -spt), Tm);
            const double gp = 0.5 * (1.0 + ct), gm = 0.5 * (1.0 - ct), g0 = RSQRT2 * stt;
            const double2 Zp = make_double2(g0 * T0.x + gp * Tp.x + gm * Tm.x, g0 * T0.y + gp * Tp.y + gm * Tm.y);
            const double2 Zm = make_double2(-g0 * T0.x + gm * Tp.x + gp * Tm.x, -g0 * T0.y + gm * Tp.y + gp * Tm.y);
            k.Ap = cfma(make_double2(ca, sa), Zp, k.Ap);
            k.Am = cfma(make_double2(ca, -sa), Zm, k.Am);
        }
        const double S = fma(k.Ap.x, k.Ap.x, fma(k.Ap.y, k.Ap.y, fma(k.Am.x, k.Am.x, k.Am.y * k.Am.y)));
        double u;   // weight of this event in the gradient sums
        if (is_norm) {
            bad |= live && !isfinite(S);
            accW = fma(wgt, S, accW);        // padding events carry w = 0
            u = wgt;
        } else if (a.bkg) {
            const double f0 = fma(bkg_ps * wgt, S, bkg_qb * (live ? a.bkg[lt * TILE + tid] : 1.0));
            const bool ok = f0 > 0.0 && isfinite(f0);
            bad |= live && !ok;
            double f; int x1, x2;
            split_exp((live && ok) ? f0 : 1.0, &f, &x1);
            split_exp(accF * f, &accF, &x2);
            accE += x1 + x2;
            u = (live && ok) ? bkg_ps * wgt / f0 : 0.0;
            accT = fma(u, S, accT);
        } else {
            const bool ok = S > 0.0 && isfinite(S);
            bad |= live && !ok;
            double f; int x1, x2;
            split_exp((live && ok) ? S : 1.0, &f, &x1);
            split_exp(accF * f, &accF, &x2);
            accE += x1 + x2;
            u = (live && ok) ? fast_rcp(S) : 0.0;
        }
        // ---- gradient leaves: slot pair p -> (Re, Im) of u conj(BW) sum_xi conj(g_xi) A_xi
        int Jc = -1;             // spin code of the d functions held in (d0c, d1c): the slots of one resonance follow each other
        double d0c = 0.0, d1c = 0.0;
        auto pair_value = [&](int p, double* re, double* im) {
            const int ent = g.pair_ent[p];
            if (ent == -2) { *re = 0.0; *im = 0.0; return; }
            const int J = g.pair_J[p];   // 8 + J: a Z slot of spin J
            if (J != Jc) {
                if (J >= 8) dJ(J - 8, st[C_CZ * TILE], st[C_SZ * TILE], &d0c, &d1c);
                else dJ(J, k.cK, k.sK, &d0c, &d1c);
                Jc = J;
            }
            double2 gp, gm;
            term_angular_d(d0c, d1c, g.pair_lam[p], J >= 8, k, st, &gp, &gm);
            // T = conj(g+) A+ + conj(g-) A-
            double2 T = make_double2(fma(gp.x, k.Ap.x, gp.y * k.Ap.y), fma(gp.x, k.Ap.y, -gp.y * k.Ap.x));
            T.x = fma(gm.x, k.Am.x, fma(gm.y, k.Am.y, T.x));
            T.y = fma(gm.x, k.Am.y, fma(-gm.y, k.Am.x, T.y));
            if (ent >= 0) {
                const double2 bw = bw_rec[ent * TILE];
                T = make_double2(fma(bw.x, T.x, bw.y * T.y), fma(bw.x, T.y, -bw.y * T.x));   // conj(BW) T
            }
            *re = u * T.x;
            *im = u * T.y;
        };
        for (int b = 0; b < nblk; ++b) {
            double s2 = 0, s3 = 0, s4 = 0, v = 0;
            int dummy;
#pragma unroll 1
            for (int i = 0; i < 8; ++i) {
                double y[4];
                pair_value(16 * b + 2 * i, &y[0], &y[1]);
                pair_value(16 * b + 2 * i + 1, &y[2], &y[3]);
                double x, w2;
                halve<true>(0, lane, y[0], 0, y[1], 0, &w2, &dummy);
                halve<true>(0, lane, y[2], 0, y[3], 0, &x, &dummy);
                halve<true>(1, lane, w2, 0, x, 0, &x, &dummy);
                if (!(i & 1)) { s2 = x; continue; }
                halve<true>(2, lane, s2, 0, x, 0, &x, &dummy);
                if (!(i & 2)) { s3 = x; continue; }
                halve<true>(3, lane, s3, 0, x, 0, &x, &dummy);
                if (!(i & 4)) { s4 = x; continue; }
                halve<true>(4, lane, s4, 0, x, 0, &v, &dummy);
            }
            (is_norm ? accN : accD)[b * THREADS + tid] += v;
        }
        __syncthreads();   // Z region and the lineshape records no longer needed: stream the next tile's Z columns
        if (have_z && tid == 0 && has_next) issue(tile + gridDim.x, 1);
    }
    for (int b = 0; b < nblk; ++b) bad |= !isfinite(accD[b * THREADS + tid]) || !isfinite(accN[b * THREADS + tid]);
    if (bad) atomicOr(a.flag, 2);

    // ---- per-CTA partials: rows 0, 1 = sum log S, sum w S; rows 2 + j = data-side leaf j; rows 2 + nleaf + j = normalisation side
    {
        const double t0 = block_sum(log(accF) + (double)accE * LN2, sm);
        const double t1 = block_sum(accW, sm);
        const double t2 = block_sum(accT, sm);
        if (tid == 0) {
            g.partial[(size_t)0 * g.stride + blockIdx.x] = t0;
            g.partial[(size_t)1 * g.stride + blockIdx.x] = t1;
            g.partial[(size_t)(2 + 2 * nleaf) * g.stride + blockIdx.x] = t2;
        }
    }
    __syncthreads();
    for (int idx = tid; idx < nleaf; idx += THREADS) {
        const int b = idx >> 5, l = idx & 31;
        double sD = 0.0, sN = 0.0;
        for (int wv = 0; wv < NWARPS; ++wv) {   // the warp totals in warp order
            sD += accD[b * THREADS + wv * 32 + l];
            sN += accN[b * THREADS + wv * 32 + l];
        }
        g.partial[(size_t)(2 + idx) * g.stride + blockIdx.x] = sD;
        g.partial[(size_t)(2 + nleaf + idx) * g.stride + blockIdx.x] = sN;
    }
    // ---- the last CTA to finish adds the partials of every row in CTA order and forms NLL, I and the gradient
    __threadfence();
    __syncthreads();
    if (tid == 0) s_last = atomicAdd(a.ticket, 1u) == gridDim.x - 1;
    __syncthreads();
    if (!s_last) return;
    __threadfence();
    grad_finish(g, accD, nleaf, tid, THREADS, gridDim.x);   // accD: the accumulators are dead (3 + 2 nleaf <= 195 doubles)
}

namespace {

size_t grad_smem(bool have_z, int nent) {
    return (size_t)((have_z ? NCOL_ALL : NCOL_K) + 1) * TILE * sizeof(double) + (size_t)nent * TILE * sizeof(double2) +
           (size_t)2 * GBLK * THREADS * sizeof(double) + 2 * sizeof(uint64_t);
}

}  // namespace

bool grad_fits(int nent, int ngrp) { (void)ngrp; return grad_smem(true, nent) <= (size_t)224 * 1024; }

int grad_grid(long long n_data, long long n_norm) {
    const long long ntiles = (n_data + TILE - 1) / TILE + (n_norm + TILE - 1) / TILE;
    return (int)(ntiles < 1 ? 1 : (ntiles > sm_count() ? sm_count() : ntiles));   // persistent: one CTA per SM
}

cudaError_t launch_grad(const GradArgs& g, int grid, cudaStream_t s) {
    static DeviceOnce attr_done;
    cudaError_t e = cudaSuccess;
    if (attr_done.first()) { e = cudaFuncSetAttribute(k_grad, cudaFuncAttributeMaxDynamicSharedMemorySize, 224 * 1024); }
    if (e != cudaSuccess) return e;
    int nent = g.a.nlass;
    for (int sp = 0; sp < NSPIN; ++sp) nent += g.a.shape[sp];
    k_grad<<<grid, THREADS, grad_smem(g.a.gstart[NSPIN] > g.a.gstart[5], nent), s>>>(g);
    return cudaGetLastError();
}

}  // namespace amp
