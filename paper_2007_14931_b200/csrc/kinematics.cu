// kinematics.cu — step a1: the once-per-dataset kinematics cache.
//
// For every event (m_Kpi, cos theta_K*, cos theta_psi, phi) (Eq. 1) compute everything
// in Eqs. 4 and 10 that does not depend on fit parameters: the running-mass quantities the lineshapes
// need, the sines of the input helicity angles, the phi phase, and the Z-chain
// variables m_psipi, theta_Z, theta~_psi, phi~, alpha.
//
// The Z chain is derived from planar closed forms, not by boosting
// 3D 4-vectors: in the J/psi rest frame every hadron lies in the x-z plane (z = K* direction, K on the
// +x side), so only z components change under the boost along z, the two dihedral angles reduce to
// ratios of components of the mu+ direction, and the Z frame is one more boost along the pion.
//
// HBM-bound: reads 32-40 B, writes 88-184 B per event; one thread per event, fully coalesced.  The cache is written in
// the tiled layout of amp_internal.cuh (blocks of 512 events, one 4 KB column per quantity, the weight last).
#include "amp_internal.cuh"

namespace amp {

__device__ __forceinline__ double two_body(double M, double a, double b) {
    const double s = a + b, d = a - b;
    return sqrt((M - s) * (M + s) * (M - d) * (M + d)) / (2.0 * M);
}

__global__ void __launch_bounds__(256) k_kinematics(const KinArgs a) {
    const double MB = a.dk.MB, mpsi = a.dk.mpsi, mK = a.dk.mK, mpi = a.dk.mpi;
    double acc = 0.0;
    bool bad = false;
    for (long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x; i < a.npad; i += (long long)gridDim.x * blockDim.x) {
        double* col = a.cache + cache_idx(a.ncolw, 0, i);   // this event's element of column 0; column c is CACHE_TILE * c further
        if (i >= a.n) {   // padding: benign values, weight 0
            for (int c = 0; c < a.ncolw - 1; ++c) col[c * CACHE_TILE] = 1.0;
            col[(a.ncolw - 1) * CACHE_TILE] = 0.0;
            continue;
        }
        const double m = a.x[i], cK = a.x[a.n + i], cpsi = a.x[2 * a.n + i], phi = a.x[3 * a.n + i];
        const double w = a.w ? a.w[i] : 1.0;
        // domain: strictly inside phase space, finite inputs, positive efficiency / non-negative weight
        const bool ok = (m > mK + mpi) && (m < MB - mpsi) && (fabs(cK) <= 1.0) && (fabs(cpsi) <= 1.0) && isfinite(phi) &&
                        isfinite(w) && (a.weight_positive ? (w > 0.0) : (w >= 0.0));
        if (!ok) { bad = true; continue; }
        col[(a.ncolw - 1) * CACHE_TILE] = w;
        acc += a.weight_positive ? log(w) : w;

        const double m2 = m * m, invm = 1.0 / m;
        const double q = two_body(m, mK, mpi);
        const double pB = two_body(MB, m, mpsi);
        const double sK = sqrt((1.0 - cK) * (1.0 + cK)), spsi = sqrt((1.0 - cpsi) * (1.0 + cpsi));
        double sphi, cphi;
        sincos(phi, &sphi, &cphi);
        col[C_M2 * CACHE_TILE] = m2;
        col[C_INVM * CACHE_TILE] = invm;
        col[C_Q * CACHE_TILE] = q;
        col[C_PB * CACHE_TILE] = pB;
        col[C_CK * CACHE_TILE] = cK;
        col[C_SK * CACHE_TILE] = sK;
        col[C_CPSI * CACHE_TILE] = cpsi;
        col[C_SPSI * CACHE_TILE] = spsi;
        col[C_CPHI * CACHE_TILE] = cphi;
        col[C_SPHI * CACHE_TILE] = sphi;
        if (!a.with_z) continue;

        // From the K pi rest frame (K along (sK, 0, cK), the J/psi along -z with energy E*_psi and momentum p*_psi = pB MB / m)
        // straight to the J/psi rest frame, a boost along z: for (E, p_z) there, p_z' = (E*_psi p_z + p*_psi E) / m_psi and
        // E' = (E*_psi E + p*_psi p_z) / m_psi; p_x is unchanged.  Every hadron stays in the x-z plane.
        const double Epi_r = (m2 - mK * mK + mpi * mpi) * (0.5 * invm), EK_r = (m2 + mK * mK - mpi * mpi) * (0.5 * invm);
        const double Eps = (MB * MB - m2 - mpsi * mpsi) * (0.5 * invm), pps = pB * MB * invm;
        const double qc = q * cK, qs = q * sK, impsi = 1.0 / mpsi;
        const double pz = (pps * Epi_r - Eps * qc) * impsi, px = -qs;          // pion
        const double Epi_p = (Eps * Epi_r - pps * qc) * impsi;
        const double kz = (pps * EK_r + Eps * qc) * impsi, kx = qs;            // kaon
        const double EK_p = (Eps * EK_r + pps * qc) * impsi;
        // m_psipi^2 = (P_psi + P_pi)^2 = m_psi^2 + m_pi^2 + 2 m_psi E'_pi, linear in cos theta_K*
        const double mZ2 = mpsi * mpsi + mpi * mpi + 2.0 * mpsi * Epi_p;
        const double mZ = sqrt(mZ2), invmZ = 1.0 / mZ;
        // pion direction n_pi = (nx, 0, nz) and momentum p' in the J/psi rest frame
        const double pp2 = pz * pz + px * px;
        const double inorm = rsqrt(pp2), pp = pp2 * inorm;
        const double nx = px * inorm, nz = pz * inorm;
        // mu+ direction n_mu = (spsi cphi, spsi sphi, cpsi); theta~ = angle(mu+, pi)
        const double ct = spsi * cphi * nx + cpsi * nz;
        // components of n_mu perpendicular to n_pi: along x_Z = y x n_pi = (nz, 0, -nx) and along y
        const double ax = spsi * cphi * nz - cpsi * nx, ay = spsi * sphi;
        const double st = sqrt(ax * ax + ay * ay);
        const double ist = 1.0 / st;
        // phi~: azimuth of mu+ about n_pi from the K side; alpha: from the (mu+,pi) to the (mu+,K*) plane about n_mu
        const double cpt = ax * ist, spt = ay * ist;
        const double ca = (spsi * nz - cpsi * cphi * nx) * ist, sa = -sphi * nx * ist;
        // Z rest frame = the J/psi frame boosted along n_pi (gamma = (m_psi + E'_pi)/m_Z, gamma v = p'/m_Z): the pion keeps its
        // direction, |p_pi^Z| = p' m_psi / m_Z; the kaon's components along and across n_pi give theta_Z = angle(K, pi) and |p_K^Z|
        // directly.  No momentum is formed from m_psipi minus a threshold: within 1e-3 MeV of m_psi + m_pi or m_B - m_K that
        // subtraction loses 1e-10 of the angle and of the barrier momenta, these component forms 1e-13.
        const double nk = nx * kx + nz * kz;
        const double apar = ((mpsi + Epi_p) * nk - pp * EK_p) * invmZ;
        const double aperp = fabs(nz * kx - nx * kz);    // (n_pi x p_K)_y > 0: the kaon is on the +x side
        const double pKZ = sqrt(apar * apar + aperp * aperp), iden = 1.0 / pKZ;
        const double cZ = apar * iden, sZ = aperp * iden;
        const double qZ = pp * mpsi * invmZ;             // pi momentum in the Z frame (p_R of the Z)
        const double pBZ = pKZ * mZ / MB;                // Z (and K) momentum in the B frame (p_B of the Z)
        // degenerate Z-chain geometry (reading A17): mu+ exactly along the pion (st = 0: phi~ and alpha undefined), m_psipi exactly at
        // one of its thresholds (theta_Z undefined), the pion at rest in the J/psi frame.  Measure zero; refused at load instead of
        // caching NaN that would only surface in a later amp_nll.
        if (!isfinite(ist * iden * inorm * invmZ)) { bad = true; continue; }
        col[C_MZ2 * CACHE_TILE] = mZ2;
        col[C_INVMZ * CACHE_TILE] = invmZ;
        col[C_QZ * CACHE_TILE] = qZ;
        col[C_PBZ * CACHE_TILE] = pBZ;
        col[C_CZ * CACHE_TILE] = cZ;
        col[C_SZ * CACHE_TILE] = sZ;
        col[C_CT * CACHE_TILE] = ct;
        col[C_ST * CACHE_TILE] = st;
        col[C_CPT * CACHE_TILE] = cpt;
        col[C_SPT * CACHE_TILE] = spt;
        col[C_CA * CACHE_TILE] = ca;
        col[C_SA * CACHE_TILE] = sa;
    }
    if (bad) atomicOr(a.flag, 1);
    // deterministic block reduction of acc (fixed shuffle tree, fixed warp order)
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

int sm_count() {
    static int cache[AMP_MAX_DEVICES] = {};
    const int d = current_device();
    if (!cache[d]) {
        int v = 0;
        if (cudaDeviceGetAttribute(&v, cudaDevAttrMultiProcessorCount, d) != cudaSuccess || v < 1) v = 148;   // B200
        cache[d] = v;
    }
    return cache[d];
}

int kinematics_grid(long long n) {
    long long blocks = (n + 255) / 256;
    const long long cap = (long long)sm_count() * 8;
    return (int)(blocks < 1 ? 1 : (blocks > cap ? cap : blocks));
}

cudaError_t launch_kinematics(const KinArgs& a, int grid, cudaStream_t s) {
    k_kinematics<<<grid, 256, 0, s>>>(a);
    return cudaGetLastError();
}

// out[j] = sum_b partial[j * stride + b], b < nblocks, in a fixed order: thread t adds b = t, t+256, ...
// then a fixed shuffle/shared tree.  One block per row.
__global__ void __launch_bounds__(256) k_finalize(const double* __restrict__ partial, int nblocks, int stride, double* __restrict__ out) {
    const double* p = partial + (size_t)blockIdx.x * stride;
    double acc = 0.0;
    for (int b = threadIdx.x; b < nblocks; b += 256) acc += p[b];
    __shared__ double sm[8];
#pragma unroll
    for (int o = 16; o; o >>= 1) acc += __shfl_xor_sync(0xffffffffu, acc, o);
    if ((threadIdx.x & 31) == 0) sm[threadIdx.x >> 5] = acc;
    __syncthreads();
    if (threadIdx.x == 0) {
        double t = 0.0;
        for (int wv = 0; wv < 8; ++wv) t += sm[wv];
        out[blockIdx.x] = t;
    }
}

cudaError_t launch_finalize(const double* partial, int nblocks, int stride, int nrows, double* out, cudaStream_t s) {
    k_finalize<<<nrows, 256, 0, s>>>(partial, nblocks, stride, out);
    return cudaGetLastError();
}

}  // namespace amp
