// lineshape.cu — step a2: recompute only the lineshape columns whose (resonance, mass, width) is not
// already held in the column pool.  A^R(m) of Eqs. 2-3: relativistic Breit-Wigner with
// Blatt-Weisskopf barrier factors, momentum powers and running width.
//
// One launch handles all missing columns of one dataset: a thread reads the four running-mass
// quantities of each chain once (32 B per chain per event) and writes one double2 (16 B) per column.
#include <algorithm>

#include "amp_internal.cuh"

namespace amp {

struct LineshapeArgs {
    LineshapeJob job[MAX_LINE_JOBS];   // sorted so that the jobs of one barrier group (chain, L_R, L_B, radius) are consecutive
    unsigned long long group_first;    // bit j: job j starts a group
    int njobs;
    int any_k, any_z;
    const double* cache;
    int ncolw;
    double2* cols;
    long long n, npad;
};

// Resonances that share (chain, L_R, L_B, radius) share the barrier factors and momentum powers (amp_internal.cuh, BarrierGroup):
//   A^R = kN F / (M2 - m^2 - i kG G),  F = rs pB^LB (pR/m)^LR,  G = pR^(2LR+1) (1/m) rs^2 B_LB(zB),  rs = 1 / sqrt(B_LR(zR) B_LB(zB))
// so F and G (the square root, the polynomials and the powers with their run-time orbital momenta) are formed once per event and
// group, and a column costs one reciprocal and ten FP64 operations.
__global__ void __launch_bounds__(256) k_lineshape(const __grid_constant__ LineshapeArgs a) {
    for (long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x; i < a.n; i += (long long)gridDim.x * blockDim.x) {
        const double* col = a.cache + cache_idx(a.ncolw, 0, i);
        double m2 = 0, invm = 0, q = 0, pB = 0, mZ2 = 0, invmZ = 0, qZ = 0, pBZ = 0;
        if (a.any_k) { m2 = col[C_M2 * CACHE_TILE]; invm = col[C_INVM * CACHE_TILE]; q = col[C_Q * CACHE_TILE]; pB = col[C_PB * CACHE_TILE]; }
        if (a.any_z) { mZ2 = col[C_MZ2 * CACHE_TILE]; invmZ = col[C_INVMZ * CACHE_TILE]; qZ = col[C_QZ * CACHE_TILE]; pBZ = col[C_PBZ * CACHE_TILE]; }
        double F = 0.0, G = 0.0;
        for (int j = 0; j < a.njobs; ++j) {
            const LineConst& lc = a.job[j].lc;
            const bool z = lc.chain == 1;
            double2 A;
            if (lc.chain == 2 || lc.kind == AMP_LASS) {
                A = z ? lineshape_eval(lc, mZ2, invmZ, qZ, pBZ) : lineshape_eval(lc, m2, invm, q, pB);
            } else {
                if ((a.group_first >> j) & 1ull) {
                    const double pR = z ? qZ : q, pBc = z ? pBZ : pB, im = z ? invmZ : invm;
                    switch (lc.LR * 8 + lc.LB) {   // (warp-uniform) the pairs of the paper's resonance lists with their powers unrolled
                        case 0 * 8 + 1: group_factors<0, 1>(lc.r2, im, pR, pBc, &F, &G); break;   // K* J = 0; 1+ Z
                        case 1 * 8 + 0: group_factors<1, 0>(lc.r2, im, pR, pBc, &F, &G); break;   // K* J = 1
                        case 2 * 8 + 1: group_factors<2, 1>(lc.r2, im, pR, pBc, &F, &G); break;
                        case 3 * 8 + 2: group_factors<3, 2>(lc.r2, im, pR, pBc, &F, &G); break;
                        case 4 * 8 + 3: group_factors<4, 3>(lc.r2, im, pR, pBc, &F, &G); break;
                        default: {
                            const double DB = bw_poly(lc.LB, lc.r2 * pBc * pBc);
                            const double rs = rsqrt(bw_poly(lc.LR, lc.r2 * pR * pR) * DB);
                            F = rs * powi(pBc, lc.LB) * powi(pR * im, lc.LR);
                            G = powi(pR, 2 * lc.LR + 1) * im * (rs * rs) * DB;
                        }
                    }
                }
                A = bw_from_consts(lc.kN, lc.kG, lc.M2, z ? mZ2 : m2, F, G);
            }
            a.cols[(size_t)a.job[j].column * a.npad + i] = A;
        }
    }
}

cudaError_t launch_lineshape(const Dataset& d, const LineshapeJob* jobs, int njobs, cudaStream_t s) {
    for (int j0 = 0; j0 < njobs; j0 += MAX_LINE_JOBS) {
        LineshapeArgs a;
        a.njobs = (njobs - j0 < MAX_LINE_JOBS) ? njobs - j0 : MAX_LINE_JOBS;
        a.any_k = a.any_z = 0;
        for (int j = 0; j < a.njobs; ++j) {
            a.job[j] = jobs[j0 + j];
            if (a.job[j].lc.chain == 0) a.any_k = 1;
            if (a.job[j].lc.chain == 1) a.any_z = 1;
        }
        auto key_less = [](const LineshapeJob& x, const LineshapeJob& y) {
            const LineConst &p = x.lc, &q = y.lc;
            if (p.chain != q.chain) return p.chain < q.chain;
            if (p.LR != q.LR) return p.LR < q.LR;
            if (p.LB != q.LB) return p.LB < q.LB;
            return p.r2 < q.r2;
        };
        std::stable_sort(a.job, a.job + a.njobs, key_less);
        a.group_first = 0;
        int prev = -1;   // the last Breit-Wigner job (constant and LASS terms take no part in the groups)
        for (int j = 0; j < a.njobs; ++j) {
            if (a.job[j].lc.chain == 2 || a.job[j].lc.kind == AMP_LASS) continue;
            if (prev < 0 || key_less(a.job[prev], a.job[j]) || key_less(a.job[j], a.job[prev])) a.group_first |= 1ull << j;
            prev = j;
        }
        a.cache = d.cache;
        a.ncolw = d.ncache + 1;
        a.cols = d.cols;
        a.n = d.n;
        a.npad = d.npad;
        long long blocks = (d.n + 255) / 256;
        const long long cap = (long long)sm_count() * 8;
        const int grid = (int)(blocks < 1 ? 1 : (blocks > cap ? cap : blocks));
        k_lineshape<<<grid, 256, 0, s>>>(a);
        cudaError_t e = cudaGetLastError();
        if (e != cudaSuccess) return e;
    }
    return cudaSuccess;
}

}  // namespace amp
