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
#include "stream_core.cuh"

namespace amp {



// A warp has read its part of a staged region into registers.  True in lane 0 of the LAST warp of the CTA to say so for
// this tile (it resets the count and may overwrite the region): the warps never wait for one another here, and the count
// cannot be touched again before the refill this warp issues has landed (the next mbarrier phase).
__device__ __forceinline__ bool region_released(int* count) {
    __syncwarp();
    bool last = false;
    if ((threadIdx.x & 31) == 0) {
        __threadfence_block();                       // this warp's shared-memory reads are done before the count moves
        last = atomicAdd(count, 1) == NWARPS - 1;
        if (last) {
            *count = 0;
            __threadfence_block();                   // ... and every other warp's, before the bulk copy is issued
        }
    }
    return last;
}

template <int MODE, class SH>
__global__ void __launch_bounds__(THREADS, AMP_STREAM_MINB) k_stream(const __grid_constant__ StreamArgs a) {
    const double RSQRT2 = 0.70710678118654752440;
    const bool have_z = SH::nz > 0 || (SH::nz < 0 && a.gstart[NSPIN] > a.gstart[5]);
    // sum w S (normalisation tiles) lives in `acc`; sum log S (data tiles) as a running product of mantissas in `acc` and a
    // sum of exponents in `accE` (split_exp: integer ops + one multiply per event instead of a ~35-instruction FP64 log)
    const double LN2 = 0.69314718055994530942;
    double acc = (MODE == MODE_DATA || MODE == MODE_FUSED || MODE == MODE_DATA_BKG || MODE == MODE_DATA_M) ? 1.0 : 0.0;
    // Eq. 14: f = (purity / I) eps S + (1 - purity) b, I = sum_wS / wsum from the normalisation pass that ran before
    const double bkg_ps = MODE == MODE_DATA_BKG ? a.purity * a.wsum / __ldg(a.sum_wS) : 0.0, bkg_qb = 1.0 - a.purity;
    int accE = 0;
    bool bad = false;
    // One staged tile per CTA, split in two regions with their own mbarrier: the K*-chain columns (+ weight) are
    // copied to registers at the top of an iteration and their region is refilled at once with the next tile;
    // the Z-chain region is refilled as soon as its values have been read, a little past the middle.  A region
    // therefore has a whole iteration to arrive, and two CTAs (16 warps) fit on an SM.
    extern __shared__ __align__(128) unsigned char smem_raw[];
    const int ncache = have_z ? NCOL_ALL : NCOL_K;
    const bool with_w = MODE != MODE_DATA && MODE != MODE_DATA_M;   // the K* region carries the weight column (MODE_FUSED: only for normalisation tiles)
    double* stage = reinterpret_cast<double*>(smem_raw);
    uint64_t* full = reinterpret_cast<uint64_t*>(smem_raw + (size_t)(ncache + 1) * TILE * sizeof(double));   // [0]: K* region, [1]: Z region
    __shared__ int consumed[2];   // warps that have taken their values of the region's current tile into registers
    if (threadIdx.x == 0) {
        mbar_init(&full[0], 1);
        mbar_init(&full[1], 1);
        consumed[0] = consumed[1] = 0;
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();
    // npad is a multiple of TILE: every tile is fully backed by memory
    const long long ntd = (a.n + TILE - 1) / TILE;                                              // tiles of the first dataset
    const long long ntiles = MODE == MODE_FUSED ? ntd + (a.n2 + TILE - 1) / TILE : ntd;
    if (threadIdx.x == 0 && (long long)blockIdx.x < ntiles) {
        issue_tile<MODE>(a, ntd, blockIdx.x, stage, &full[0], 0, NCOL_K, true);
        if (have_z) issue_tile<MODE>(a, ntd, blockIdx.x, stage, &full[1], NCOL_K, NCOL_ALL, false);
    }
    __shared__ double sm[NWARPS];
    uint32_t parity = 0;
    bool in_norm = false;   // MODE_FUSED: this CTA has passed from the data tiles to the normalisation tiles
    for (long long tile = blockIdx.x; tile < ntiles; tile += gridDim.x, parity ^= 1) {
        const bool has_next = tile + gridDim.x < ntiles;
        const bool is_norm = MODE == MODE_FUSED ? tile >= ntd : MODE == MODE_NORM;
        if (MODE == MODE_FUSED && is_norm && !in_norm) {   // sum log S of this CTA's data tiles is complete
            const double t = block_sum(log(acc) + (double)accE * LN2, sm);
            if (threadIdx.x == 0) a.partial[blockIdx.x] = t;
            acc = 0.0;
            in_norm = true;
        }
        const long long lt = (MODE == MODE_FUSED && is_norm) ? tile - ntd : tile;
        const long long nlive = (MODE == MODE_FUSED && is_norm) ? a.n2 : a.n;
        const long long i0 = lt * TILE + threadIdx.x * E;     // first of the E events of this thread
        mbar_wait(&full[0], parity);
        const Ev m2 = load_col(stage, C_M2), invm = load_col(stage, C_INVM);
        const Ev q = load_col(stage, C_Q), pB = load_col(stage, C_PB);
        const Ev cK = load_col(stage, C_CK), sK = load_col(stage, C_SK);
        const Ev cpsi = load_col(stage, C_CPSI), spsi = load_col(stage, C_SPSI);
        const Ev cphi = load_col(stage, C_CPHI), sphi = load_col(stage, C_SPHI);
        Ev w;
        if (MODE == MODE_FUSED ? is_norm : with_w) w = load_col(stage, ncache);
        // K* region consumed by this warp; the last warp to say so streams the next tile into it (no CTA-wide barrier)
        if (region_released(&consumed[0]) && has_next) issue_tile<MODE>(a, ntd, tile + gridDim.x, stage, &full[0], 0, NCOL_K, true);

        double2 V0[E], Vp[E], Vm[E];
#pragma unroll
        for (int e = 0; e < E; ++e) { V0[e] = a.cconst; Vp[e] = make_double2(0, 0); Vm[e] = make_double2(0, 0); }   // constant terms: lineshape 1, d^0_00 = 1
        // d^J_{00} = P_J(cK), d^J_{+1,0} = -sK P_J'(cK) / sqrt(J(J+1)), d^J_{-1,0} = -d^J_{+1,0}
#define AMP_SPIN(J, LB, CNT, OFF, D0, D1)                                                              \
        if (CNT != 0 && (CNT > 0 || a.gstart[J + 1] > a.gstart[J])) {                                  \
            double2 Um[E], U0[E], Up[E];                                                               \
            _Pragma("unroll") for (int e = 0; e < E; ++e) Um[e] = U0[e] = Up[e] = make_double2(0, 0);  \
            spin_sum<J, J, LB, CNT, OFF, J>(a, i0, m2, invm, q, pB, Um, U0, Up);                       \
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
        AMP_SPIN(2, 1, SH::n2, SH::o2, fma(1.5, c2, -0.5), -1.2247448713915890491 * s * c)                                  // sqrt(3/2)
        AMP_SPIN(3, 2, SH::n3, SH::o3, c * fma(2.5, c2, -1.5), -0.43301270189221932338 * s * fma(5.0, c2, -1.0))            // sqrt(3)/4
        AMP_SPIN(4, 3, SH::n4, SH::o4, fma(fma(4.375, c2, -3.75), c2, 0.375), -0.55901699437494742410 * s * c * fma(7.0, c2, -3.0))   // sqrt(5)/4
#undef AMP_SPIN
        if (SH::nl != 0) {   // LASS S-wave terms (shapes compiled with them): J = 0, lambda = 0, lineshape of Eq. 7
            for (int t = a.lass0; t < a.lass0 + a.nlass; ++t) {
#pragma unroll
                for (int e = 0; e < E; ++e) {
                    const double2 bw = a.ent[t].column >= 0 ? a.cols[(size_t)a.ent[t].column * a.npad + i0 + e]
                                                            : lass_eval(a.ent[t].M2, a.ent[t].kG, m2.v[e], invm.v[e], q.v[e]);
                    V0[e] = cfma(a.ent[t].c0, bw, V0[e]);
                }
            }
        }
        // A_xi = sum_l e^{i l phi} d^1_{l xi}(theta_psi) V_l ; d^1_{0,+-1} = +-s/sqrt2, d^1_{11} = d^1_{-1-1} = (1+c)/2, d^1_{1-1} = d^1_{-11} = (1-c)/2
        double2 Ap[E], Am[E];
#pragma unroll
        for (int e = 0; e < E; ++e) {
            const double2 Wp = cmul(make_double2(cphi.v[e], sphi.v[e]), Vp[e]), Wm = cmul(make_double2(cphi.v[e], -sphi.v[e]), Vm[e]);
            const double hp = 0.5 * (1.0 + cpsi.v[e]), hm = 0.5 * (1.0 - cpsi.v[e]), h0 = RSQRT2 * spsi.v[e];
            Ap[e] = make_double2(h0 * V0[e].x + hp * Wp.x + hm * Wm.x, h0 * V0[e].y + hp * Wp.y + hm * Wm.y);
            Am[e] = make_double2(-h0 * V0[e].x + hm * Wp.x + hp * Wm.x, -h0 * V0[e].y + hm * Wp.y + hp * Wm.y);
        }
        if (have_z) {
            mbar_wait(&full[1], parity);
            const Ev mZ2 = load_col(stage, C_MZ2), invmZ = load_col(stage, C_INVMZ);
            const Ev qZ = load_col(stage, C_QZ), pBZ = load_col(stage, C_PBZ);
            const Ev cZ = load_col(stage, C_CZ), sZ = load_col(stage, C_SZ);
            const Ev ct = load_col(stage, C_CT), st = load_col(stage, C_ST);
            const Ev cpt = load_col(stage, C_CPT), spt = load_col(stage, C_SPT);
            const Ev ca = load_col(stage, C_CA), sa = load_col(stage, C_SA);
            // Z region consumed: the last warp refills it with the next tile
            if (region_released(&consumed[1]) && has_next) issue_tile<MODE>(a, ntd, tile + gridDim.x, stage, &full[1], NCOL_K, NCOL_ALL, false);
            // T_l' = sum over the Z spin classes of d^J_{0 l'}(theta_Z) U_l' ; d^J_{0,+1} = -d^J_{+1,0}, d^J_{0,-1} = -d^J_{0,+1}
            double2 T0[E], Tp[E], Tm[E];
#pragma unroll
            for (int e = 0; e < E; ++e) T0[e] = Tp[e] = Tm[e] = make_double2(0, 0);
#define AMP_ZCLASS(ZC, J, LR, LB, CNT, OFF, D0, D1)                                                    \
            if (CNT != 0 && (CNT > 0 || a.gstart[5 + ZC + 1] > a.gstart[5 + ZC])) {                    \
                double2 Um[E], U0[E], Up[E];                                                           \
                _Pragma("unroll") for (int e = 0; e < E; ++e) Um[e] = U0[e] = Up[e] = make_double2(0, 0); \
                spin_sum<J, LR, LB, CNT, OFF, 5 + ZC>(a, i0, mZ2, invmZ, qZ, pBZ, Um, U0, Up);         \
                _Pragma("unroll") for (int e = 0; e < E; ++e) {                                        \
                    const double c = cZ.v[e], s = sZ.v[e], c2 = c * c;                                 \
                    (void)s; (void)c2;                                                                 \
                    const double d0 = (D0), d1 = (D1);                                                 \
                    T0[e] = cadd(T0[e], cscale(d0, U0[e]));                                            \
                    if (J) { Tp[e] = cadd(Tp[e], cscale(d1, Up[e])); Tm[e] = cadd(Tm[e], cscale(-d1, Um[e])); } \
                }                                                                                      \
            }
            AMP_ZCLASS(0, 1, 0, 1, SH::nz, SH::oz, c, RSQRT2 * s)                                       // 1+ : L_R = 0, L_B = 1
            if (SH::nz < 0) {   // the other spin-parities run in the generic kernel only
                AMP_ZCLASS(1, 2, 2, 2, -1, 0, fma(1.5, c2, -0.5), 1.2247448713915890491 * s * c)        // 2+ : 2, 2
                AMP_ZCLASS(2, 0, 1, 0, -1, 0, 1.0, 0.0)                                                 // 0- : 1, 0
                AMP_ZCLASS(3, 1, 1, 1, -1, 0, c, RSQRT2 * s)                                            // 1- : 1, 1
                AMP_ZCLASS(4, 2, 1, 2, -1, 0, fma(1.5, c2, -0.5), 1.2247448713915890491 * s * c)        // 2- : 1, 2
            }
#undef AMP_ZCLASS
#pragma unroll
            for (int e = 0; e < E; ++e) {
                Tp[e] = cmul(make_double2(cpt.v[e], spt.v[e]), Tp[e]);     // e^{+i phi~}
                Tm[e] = cmul(make_double2(cpt.v[e], -spt.v[e]), Tm[e]);    // e^{-i phi~}
                const double gp = 0.5 * (1.0 + ct.v[e]), gm = 0.5 * (1.0 - ct.v[e]), g0 = RSQRT2 * st.v[e];
                const double2 Zp = make_double2(g0 * T0[e].x + gp * Tp[e].x + gm * Tm[e].x, g0 * T0[e].y + gp * Tp[e].y + gm * Tm[e].y);
                const double2 Zm = make_double2(-g0 * T0[e].x + gm * Tp[e].x + gp * Tm[e].x, -g0 * T0[e].y + gm * Tp[e].y + gp * Tm[e].y);
                Ap[e] = cfma(make_double2(ca.v[e], sa.v[e]), Zp, Ap[e]);    // e^{+i alpha}
                Am[e] = cfma(make_double2(ca.v[e], -sa.v[e]), Zm, Am[e]);   // e^{-i alpha}
            }
        }
#pragma unroll
        for (int e = 0; e < E; ++e) {
            const double S = fma(Ap[e].x, Ap[e].x, fma(Ap[e].y, Ap[e].y, fma(Am[e].x, Am[e].x, Am[e].y * Am[e].y)));
            const bool live = i0 + e < nlive;   // the last thread may hold padding events (weight 0)
            if (MODE == MODE_DATA_BKG) {
                const double f0 = fma(bkg_ps * w.v[e], S, bkg_qb * (live ? a.bkg[i0 + e] : 1.0));
                const bool ok = f0 > 0.0 && isfinite(f0);
                bad |= live && !ok;
                double f; int x;
                split_exp((live && ok) ? f0 : 1.0, &f, &x);
                acc *= f;
                accE += x;
            } else if (MODE == MODE_DATA || MODE == MODE_DATA_M || (MODE == MODE_FUSED && !is_norm)) {
                const bool ok = S > 0.0 && isfinite(S);
                bad |= live && !ok;
                double f; int x;
                split_exp((live && ok) ? S : 1.0, &f, &x);
                acc *= f;
                accE += x;
            } else if (MODE == MODE_NORM || MODE == MODE_FUSED) {
                if (live) { bad |= !isfinite(S); acc = fma(w.v[e], S, acc); }
            } else {
                if (live) a.out[i0 + e] = w.v[e] * S;
            }
        }
        if (MODE == MODE_DATA || MODE == MODE_DATA_BKG || MODE == MODE_DATA_M || (MODE == MODE_FUSED && !is_norm)) {   // running product back to [0.5, 1) once per tile
            int x;
            split_exp(acc, &acc, &x);
            accE += x;
        }
    }
    if (MODE == MODE_EVAL) return;
    if (bad) atomicOr(a.flag, 2);
    {
        const bool logs = MODE == MODE_DATA || MODE == MODE_DATA_BKG || MODE == MODE_DATA_M || (MODE == MODE_FUSED && !in_norm);
        const double t = block_sum(logs ? log(acc) + (double)accE * LN2 : acc, sm);
        if (threadIdx.x == 0) {
            if (MODE == MODE_FUSED && !in_norm) { a.partial[blockIdx.x] = t; a.partial2[blockIdx.x] = 0.0; }   // this CTA saw data tiles only
            else (MODE == MODE_FUSED ? a.partial2 : a.partial)[blockIdx.x] = t;
        }
    }
    if (MODE != MODE_FUSED && MODE != MODE_DATA_M) return;
    // The last CTA to finish (integer ticket) adds the per-CTA partials in a fixed order and forms the NLL: the result
    // does not depend on which CTA that is, so it stays bit-reproducible; no second launch, no host round trip.
    __shared__ bool s_last;
    if (threadIdx.x == 0) {
        __threadfence();
        s_last = atomicAdd(a.ticket, 1u) == gridDim.x - 1;
    }
    __syncthreads();
    if (!s_last) return;
    __threadfence();
    const double slog = partial_sum(a.partial, gridDim.x, sm);
    double swS;
    if (MODE == MODE_DATA_M) {
        // sum_j w_j S_j = c^H M c from the held matrix (Re M_ef = G'[2e][2f] + G'[2e+1][2f+1], Im M_ef = G'[2e][2f+1] - G'[2e+1][2f]):
        // K^2 terms, thread t takes idx = t, t + 256, ... in a fixed order
        double q = 0.0;
        for (int idx = threadIdx.x; idx < a.qf_nent * a.qf_nent; idx += THREADS) {
            const int e = idx / a.qf_nent, f = idx % a.qf_nent;
            const double2 ce = a.qf_c[e], cf = a.qf_c[f];
            if ((ce.x == 0.0 && ce.y == 0.0) || (cf.x == 0.0 && cf.y == 0.0)) continue;
            const double* gm = a.qf_G + (size_t)(2 * e) * a.qf_KP + 2 * f;
            const double mre = gm[0] + gm[a.qf_KP + 1], mim = gm[1] - gm[a.qf_KP];
            q += ce.x * (mre * cf.x - mim * cf.y) + ce.y * (mre * cf.y + mim * cf.x);
        }
        swS = block_sum(q, sm);
    } else {
        swS = partial_sum(a.partial2, gridDim.x, sm);
    }
    if (threadIdx.x == 0) {
        const double I = swS / a.wsum;
        double v = -(slog + a.sum_log_eff) + (double)a.n * log(I);
        if (!isfinite(v) || !(I > 0.0)) v = INFINITY;
        a.result[0] = v;
        a.result[1] = I;
        a.result[3] = slog;
        a.result[4] = swS;
        a.result[2] = (double)atomicExch(a.flag, 0);   // domain flag of this call, cleared for the next one
        *a.ticket = 0u;
        // the result block may live in mapped host memory: the host spins on the stamp instead of paying a copy + stream sync
        __threadfence_system();
        *reinterpret_cast<volatile double*>(a.result + 5) = a.seq;
    }
}

static size_t stream_smem(bool have_z, int mode) {
    (void)mode;
    return (size_t)((have_z ? NCOL_ALL : NCOL_K) + 1) * TILE * sizeof(double) + 2 * sizeof(uint64_t);
}

// persistent grid: one CTA per resident slot (as many CTAs per SM as the staged tiles leave room for, at most
// AMP_STREAM_MINB), never more than there are tiles
int stream_grid(long long n, bool have_z, int mode) {
    const long long ntiles = (n + TILE - 1) / TILE;
    long long per_sm = (long long)((224 * 1024) / (stream_smem(have_z, mode) + 1024));
    if (per_sm > AMP_STREAM_MINB) per_sm = AMP_STREAM_MINB;
    if (per_sm < 1) per_sm = 1;
    const long long cap = (long long)sm_count() * per_sm;
    return (int)(ntiles < 1 ? 1 : (ntiles > cap ? cap : ntiles));
}

int stream_grid_fused(long long n1, long long n2, bool have_z) {
    const long long t1 = (n1 + TILE - 1) / TILE, t2 = (n2 + TILE - 1) / TILE;
    return stream_grid((t1 + t2) * TILE, have_z, MODE_FUSED);
}

long long stream_pad(long long n) { return (n + 511) / 512 * 512; }   // whole tiles of every streaming kernel (k_stream, k_delta: 512 events)

template <class SH>
static cudaError_t launch_shape(const StreamArgs& a, int grid, cudaStream_t s) {
    const bool have_z = SH::nz > 0 || (SH::nz < 0 && a.gstart[NSPIN] > a.gstart[5]);
    const size_t smem = stream_smem(have_z, a.mode);
    cudaError_t e = cudaSuccess;
#define AMP_LAUNCH(M)                                                                                              \
    {                                                                                                              \
        static DeviceOnce attr_done;                                                                             \
        if (attr_done.first()) { e = cudaFuncSetAttribute(k_stream<M, SH>, cudaFuncAttributeMaxDynamicSharedMemorySize, 224 * 1024); } \
        if (e == cudaSuccess) k_stream<M, SH><<<grid, THREADS, smem, s>>>(a);                                      \
    }
    switch (a.mode) {
        case MODE_DATA: AMP_LAUNCH(MODE_DATA) break;
        case MODE_NORM: AMP_LAUNCH(MODE_NORM) break;
        case MODE_FUSED: AMP_LAUNCH(MODE_FUSED) break;
        case MODE_DATA_BKG: AMP_LAUNCH(MODE_DATA_BKG) break;
        case MODE_DATA_M: AMP_LAUNCH(MODE_DATA_M) break;
        default: AMP_LAUNCH(MODE_EVAL) break;
    }
#undef AMP_LAUNCH
    return e;
}

// Shapes with a fully unrolled kernel: the paper's ten K* (three J = 0, three J = 1, two J = 2, one J = 3, one
// J = 4) with and without one Z, and the single K*(892) of configs[0].  Any other resonance list
// (or different radii within one spin) runs the generic kernel.
cudaError_t launch_stream(const StreamArgs& a, int grid, cudaStream_t s) {
    const int* n = a.shape;
    auto is = [&](int a0, int a1, int a2, int a3, int a4, int az) {
        return a.shape_fixed && n[0] == a0 && n[1] == a1 && n[2] == a2 && n[3] == a3 && n[4] == a4 && n[5] == az &&
               n[6] + n[7] + n[8] + n[9] == 0;   // Z's of another spin-parity than 1+: generic kernel
    };
    cudaError_t e;
    if (a.nlass > 0) {   // the paper's LASS variant: LASS + K0*(1950) in the S wave, the other eight K*, one Z
        if (a.nlass == 1 && is(1, 3, 2, 1, 1, 1)) e = launch_shape<Shape<1, 3, 2, 1, 1, 1, 1>>(a, grid, s);
        else e = launch_shape<Generic>(a, grid, s);
    }
    else if (is(3, 3, 2, 1, 1, 1)) e = launch_shape<Shape<3, 3, 2, 1, 1, 1>>(a, grid, s);
    else if (is(3, 3, 2, 1, 1, 2)) e = launch_shape<Shape<3, 3, 2, 1, 1, 2>>(a, grid, s);   // "ten K*s and two Zs"
    else if (is(3, 3, 2, 1, 1, 0)) e = launch_shape<Shape<3, 3, 2, 1, 1, 0>>(a, grid, s);
    else if (is(0, 1, 0, 0, 0, 0)) e = launch_shape<Shape<0, 1, 0, 0, 0, 0>>(a, grid, s);
    else e = launch_shape<Generic>(a, grid, s);
    return e != cudaSuccess ? e : cudaGetLastError();
}

}  // namespace amp
