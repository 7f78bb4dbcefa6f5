// lineshape.cu — step a2: recompute only the lineshape columns whose (resonance, mass, width) is not
// already held in the column pool.  A^R(m) of Eqs. 2-3: relativistic Breit-Wigner with
// Blatt-Weisskopf barrier factors, momentum powers and running width.
//
// One launch handles all missing columns of one dataset: a thread reads the four running-mass
// quantities of each chain once (32 B per chain per event) and writes one double2 (16 B) per column.
#include "amp_internal.cuh"

namespace amp {

struct LineshapeArgs {
    LineshapeJob job[MAX_LINE_JOBS];
    int njobs;
    int any_k, any_z;
    const double* cache;
    int ncolw;
    double2* cols;
    long long n, npad;
};

__global__ void __launch_bounds__(256) k_lineshape(const __grid_constant__ LineshapeArgs a) {
    for (long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x; i < a.n; i += (long long)gridDim.x * blockDim.x) {
        const double* col = a.cache + cache_idx(a.ncolw, 0, i);
        double m2 = 0, invm = 0, q = 0, pB = 0, mZ2 = 0, invmZ = 0, qZ = 0, pBZ = 0;
        if (a.any_k) { m2 = col[C_M2 * CACHE_TILE]; invm = col[C_INVM * CACHE_TILE]; q = col[C_Q * CACHE_TILE]; pB = col[C_PB * CACHE_TILE]; }
        if (a.any_z) { mZ2 = col[C_MZ2 * CACHE_TILE]; invmZ = col[C_INVMZ * CACHE_TILE]; qZ = col[C_QZ * CACHE_TILE]; pBZ = col[C_PBZ * CACHE_TILE]; }
        for (int j = 0; j < a.njobs; ++j) {
            const LineConst& lc = a.job[j].lc;
            const double2 A = (lc.chain == 1) ? lineshape_eval(lc, mZ2, invmZ, qZ, pBZ) : lineshape_eval(lc, m2, invm, q, pB);
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
