// amp_internal.cuh — shared declarations of the CUDA path (product code; shares nothing with oracle/).
//
// Data layout in HBM:
//   kinematics cache  double[npad/512][NCOL + 1][512]   tiled structure-of-arrays: blocks of 512 events, inside a block
//                                          one 4 KB column per cached quantity and the event weights as the last
//                                          column.  A streaming tile is ONE contiguous block (94 KB with the Z
//                                          chain): a CTA reads it with three bulk copies and HBM sees long sequential
//                                          bursts instead of 23 scattered 4 KB pieces.  npad = n rounded up to 512.
//   lineshape columns double2[ncol][npad]  complex A^R(m_i) (re, im) interleaved: one 128-bit load
//                                          per (event, column)
// One thread owns one event at a time; a warp reads 32 consecutive doubles (256 B) of a cache
// column or 32 consecutive double2 (512 B) of a lineshape column.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include "../../include/amp.h"

namespace amp {

// ---- kinematics cache columns (a1) -------------------------------------------------------------
enum CacheCol {
    // K* chain: running mass and momenta (Eqs. 2-3), helicity-angle cosines/sines and phi phase (Eq. 4)
    C_M2 = 0,   // m_Kpi^2
    C_INVM,     // 1 / m_Kpi
    C_Q,        // K momentum in the K pi frame (p_R of a K*)
    C_PB,       // K pi momentum in the B frame (p_B of a K*)
    C_CK, C_SK,         // cos, sin theta_K*
    C_CPSI, C_SPSI,     // cos, sin theta_J/psi
    C_CPHI, C_SPHI,     // cos, sin phi
    NCOL_K = 10,
    // Z chain (Eq. 10): running mass m_psipi and momenta, theta_Z, theta~_psi, phi~, alpha
    C_MZ2 = 10, // m_psipi^2
    C_INVMZ,    // 1 / m_psipi
    C_QZ,       // pi momentum in the Z frame (p_R of the Z)
    C_PBZ,      // Z momentum in the B frame (p_B of the Z)
    C_CZ, C_SZ,         // cos, sin theta_Z
    C_CT, C_ST,         // cos, sin theta~_psi
    C_CPT, C_SPT,       // cos, sin phi~
    C_CA, C_SA,         // cos, sin alpha
    NCOL_ALL = 22
};

struct DecayConst {
    double MB, mpsi, mK, mpi;
};

// Per-(resonance, mass, width) constants of Eqs. 2-3, prepared on the host once per lineshape column
// (O(1) work; every per-event step runs on the device).  With z = (r p)^2, B_L the Blatt-Weisskopf
// polynomial and rs = 1/sqrt(B_LR(zR) B_LB(zB)):
//   F_B F_R          = kF rs                      kF  = sqrt(B_LR(zR0) B_LB(zB0))
//   numerator        = kN rs pB^LB (pR/m)^LR      kN  = kF / MB^LB
//   M_R Gamma(m)     = kG pR^(2LR+1) (1/m) rs^2 B_LB(zB),   kG = M_R^2 Gamma0 B_LR(zR0) / pR0^(2LR+1)
// Spin classes of the streaming kernels: the K* spins J = 0..4, then the Z spin-parities (A24):
//   class 5: 1+ (the paper's default)   6: 2+   7: 0-   8: 1-   9: 2-
// B -> Z K has L_B = J; Z -> psi pi takes the lowest L_R with (-1)^L_R = P and |L_R - 1| <= J <= L_R + 1.
constexpr int NZCLASS = 5, NSPIN = 5 + NZCLASS;
__host__ __device__ __forceinline__ bool kind_is_z(int kind) { return kind == AMP_Z || kind == AMP_ZM; }
__host__ __device__ __forceinline__ int z_class(int kind, int J) { return kind == AMP_Z ? (J == 1 ? 0 : 1) : 2 + J; }
__host__ __device__ __forceinline__ int z_class_kind(int zc) { return zc < 2 ? AMP_Z : AMP_ZM; }
__host__ __device__ __forceinline__ int z_class_J(int zc) { return zc == 0 ? 1 : (zc == 1 ? 2 : zc - 2); }
__host__ __device__ __forceinline__ int z_class_LR(int zc) { return zc == 0 ? 0 : (zc == 1 ? 2 : 1); }

struct LineConst {
    int kind, LR, LB, chain;  // chain: 0 = K pi (K*), 1 = psi pi (Z), 2 = constant
    double M2, r2, kN, kG;
};

struct Dataset {
    long long n = 0, npad = 0;
    double* cache = nullptr;   // [npad / 512][ncache + 1][512]; last column: eps_i (data) or w_j (norm), 1 if the caller gave none
    double2* cols = nullptr;   // lineshape column pool [capacity][npad]
    int ncache = 0;            // columns present (NCOL_K or NCOL_ALL)
    double wsum = 0;           // sum_j w_j (norm) ; sum_i log eps_i (data)
    bool loaded = false;
};

static inline long long pad32(long long n) { return (n + 31) / 32 * 32; }

// ---- per-device host state -------------------------------------------------------------------------------
// One process may drive several devices (one amp_model per device): the SM count that sizes the persistent grids and the
// opt-in to more than 48 KB of dynamic shared memory (cudaFuncSetAttribute applies to the CURRENT device only) are kept
// per device, not per process.
enum { AMP_MAX_DEVICES = 64 };
static inline int current_device() {
    int d = 0;
    if (cudaGetDevice(&d) != cudaSuccess || d < 0 || d >= AMP_MAX_DEVICES) d = 0;
    return d;
}
int sm_count();   // multiprocessors of the current device (kinematics.cu)
// first() is true the first time it is called on the current device; one function-local static per kernel instantiation
struct DeviceOnce {
    bool seen[AMP_MAX_DEVICES] = {};
    bool first() { const int d = current_device(); const bool f = !seen[d]; seen[d] = true; return f; }
};

// ---- tiled cache addressing --------------------------------------------------------------------------
constexpr int CACHE_TILE = 512;
// element (col, i) of a cache with ncolw = ncache + 1 columns per block (the weight is column ncache)
__host__ __device__ __forceinline__ size_t cache_idx(int ncolw, int col, long long i) {
    return ((size_t)(i / CACHE_TILE) * ncolw + col) * CACHE_TILE + (size_t)(i % CACHE_TILE);
}

// ---- device helpers ------------------------------------------------------------------------------
__device__ __forceinline__ double2 cmul(double2 a, double2 b) { return make_double2(a.x * b.x - a.y * b.y, a.x * b.y + a.y * b.x); }
__device__ __forceinline__ double2 cfma(double2 a, double2 b, double2 c) {   // a*b + c
    return make_double2(fma(a.x, b.x, fma(-a.y, b.y, c.x)), fma(a.x, b.y, fma(a.y, b.x, c.y)));
}
__device__ __forceinline__ double2 cscale(double s, double2 a) { return make_double2(s * a.x, s * a.y); }
__device__ __forceinline__ double2 cadd(double2 a, double2 b) { return make_double2(a.x + b.x, a.y + b.y); }

// 1/d and 1/sqrt(d) for normal positive d: hardware seed (MUFU.RCP64H / RSQ64H, about 20 good bits) followed by
// one third-order correction, error ~ seed_error^3 ~ 1e-18 before rounding: a few 1e-16 relative in the end
// (not correctly rounded — the parity bar is 1e-11).
__device__ __forceinline__ double fast_rcp(double d) {
    double r;
    asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(r) : "d"(d));
    const double e = fma(-d, r, 1.0);               // 1 - d r ~ 1e-6
    return fma(r, fma(e, e, e), r);                 // r (1 + e + e^2)
}
__device__ __forceinline__ double fast_rsqrt(double d) {
    double y;
    asm("rsqrt.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(d));
    const double e = fma(-d * y, y, 1.0);           // 1 - d y^2 ~ 1e-6
    return fma(y * fma(0.375, e, 0.5), e, y);       // y (1 + e/2 + 3 e^2 / 8)
}
// Sums of logs without a log per event: S = f 2^e with f in [0.5, 1) for positive finite S (integer ops on the exponent field)
__device__ __forceinline__ void split_exp(double S, double* f, int* e) {
    int e0 = 0;
    if (S < 1e-290) { S *= 1.3407807929942597e154; e0 = -512; }   // 2^512: keeps subnormals out of the bit trick
    const int hi = __double2hiint(S), lo = __double2loint(S);
    *e = e0 + ((hi >> 20) & 0x7ff) - 1022;
    *f = __hiloint2double((hi & 0x800fffff) | 0x3fe00000, lo);
}

template <int L>
__device__ __forceinline__ double bw_poly_c(double z) {
    if (L == 0) return 1.0;
    if (L == 1) return 1.0 + z;
    if (L == 2) return fma(z + 3.0, z, 9.0);
    if (L == 3) return fma(fma(z + 6.0, z, 45.0), z, 225.0);
    return fma(fma(fma(z + 10.0, z, 135.0), z, 1575.0), z, 11025.0);
}
template <int N>
__device__ __forceinline__ double powc(double x) {
    if (N == 0) return 1.0;
    if (N == 1) return x;
    const double h = powc<N / 2>(x);
    return (N & 1) ? h * h * x : h * h;
}
// Per-event factors of a barrier group with compile-time orbital momenta (see BarrierGroup).
template <int LR, int LB>
__device__ __forceinline__ void group_factors(double r2, double invm, double pR, double pB, double* F, double* G) {
    const double DB = bw_poly_c<LB>(r2 * (pB * pB));   // (pB pB), (pR pR): shared by every spin group of the event
    const double DR = bw_poly_c<LR>(r2 * (pR * pR));
    const double rs = (LR == 0 && LB == 0) ? 1.0 : fast_rsqrt(DR * DB);
    *F = rs * powc<LB>(pB) * powc<LR>(pR * invm);
    // G = pR^(2LR+1) (1/m) / B_LR(zR); rs^2 B_LB(zB) = 1 / B_LR(zR), which is 1 for L_R = 0
    *G = (LR == 0) ? pR * invm : powc<2 * LR + 1>(pR) * invm * (rs * rs) * DB;
}
// Blatt-Weisskopf polynomial B_L(z), z = (r p)^2 (ref. [35]); L is warp-uniform.
__device__ __forceinline__ double bw_poly(int L, double z) {
    switch (L) {
        case 0: return 1.0;
        case 1: return 1.0 + z;
        case 2: return fma(z + 3.0, z, 9.0);
        case 3: return fma(fma(z + 6.0, z, 45.0), z, 225.0);
        default: return fma(fma(fma(z + 10.0, z, 135.0), z, 1575.0), z, 11025.0);
    }
}
__device__ __forceinline__ double powi(double x, int n) {   // n in 0..9, warp-uniform
    double r = 1.0;
#pragma unroll 1
    for (int i = 0; i < n; ++i) r *= x;
    return r;
}

// LASS S-wave, Eqs. 7-8, in rational form (no angle is ever formed): with t = cot(theta_B) =
// 1/(a q) + b q/2,  sin(th) e^{i th} = (t + i)/(t^2 + 1),  e^{2 i th} = (t + i)^2/(t^2 + 1), and M0 Gamma(m) = kG q/m,
// kG = M0^2 Gamma0 / q0 (also the numerator constant of the resonant term):
//   A_LASS = (m/q) (t + i)/(t^2 + 1) + 2 kG (t + i)^2/(t^2 + 1) / (M0^2 - m^2 - i kG q/m)
__device__ __forceinline__ double2 lass_eval(double M2, double kG, double m2, double invm, double q) {
    const double a = 1.95e-3, b = 1.76e-3;                    // MeV^-1
    const double t = fast_rcp(a * q) + 0.5 * b * q;
    const double n1 = fast_rcp(fma(t, t, 1.0));
    const double x = q * invm, mq = fast_rcp(x);
    const double2 s1 = make_double2(t * n1, n1);              // sin(th) e^{i th}
    const double2 e2 = make_double2(fma(t, t, -1.0) * n1, 2.0 * t * n1);   // e^{2 i th}
    const double MG = kG * x, dre = M2 - m2;
    const double r = 2.0 * kG * fast_rcp(fma(dre, dre, MG * MG));
    const double2 bw = make_double2(r * dre, r * MG);         // 2 kG / (M0^2 - m^2 - i M0 Gamma(m))
    const double2 second = cmul(e2, bw);
    return make_double2(fma(mq, s1.x, second.x), fma(mq, s1.y, second.y));
}

// Lineshape A^R(m) of Eqs. 2-3 from the cached running-mass quantities of its chain.
__device__ __forceinline__ double2 lineshape_eval(const LineConst& c, double m2, double invm, double pR, double pB) {
    if (c.chain == 2) return make_double2(1.0, 0.0);
    if (c.kind == AMP_LASS) return lass_eval(c.M2, c.kG, m2, invm, pR);
    const double zR = c.r2 * pR * pR, zB = c.r2 * pB * pB;
    const double DB = bw_poly(c.LB, zB);
    const double rs = rsqrt(bw_poly(c.LR, zR) * DB);
    const double x = pR * invm;
    const double num = c.kN * rs * powi(pB, c.LB) * powi(x, c.LR);
    const double MG = c.kG * powi(pR, 2 * c.LR + 1) * invm * (rs * rs) * DB;   // M_R Gamma(m), Eq. 3
    const double dre = c.M2 - m2;
    const double s = num / fma(dre, dre, MG * MG);
    return make_double2(s * dre, s * MG);   // num / (M^2 - m^2 - i M Gamma), Eq. 2
}

// ---- launchers (one translation unit per kernel family) -------------------------------------------
struct KinArgs {
    DecayConst dk;
    const double* x;      // [4][n] input events (borrowed)
    const double* w;      // [n] or null
    double* cache;        // tiled, ncolw columns per block (the last one receives the weight)
    int ncolw;
    long long n, npad;
    int with_z;           // also fill the Z-chain columns
    int weight_positive;  // 1: weights must be > 0 (eps), 0: >= 0 (norm weights)
    int* flag;            // device int: set to 1 on a domain error
    double* partial;      // [grid] per-block partial of sum(log w) (data) or sum(w) (norm)
};
cudaError_t launch_kinematics(const KinArgs& a, int grid, cudaStream_t s);
int kinematics_grid(long long n);

struct LineshapeJob {
    LineConst lc;
    int column;   // index into the column pool
};
enum { MAX_LINE_JOBS = 64 };
cudaError_t launch_lineshape(const Dataset& d, const LineshapeJob* jobs, int njobs, cudaStream_t s);

// Streaming combine + reduce for one parameter point (a3 + a5, P = 1)
enum StreamMode { MODE_DATA = 0, MODE_NORM = 1, MODE_EVAL = 2, MODE_FUSED = 3, MODE_DATA_BKG = 4, MODE_DATA_M = 5 };   // FUSED: data (sum log S) then norm (sum w S) in one launch + final NLL;
                                                                                              // DATA_BKG: sum log(purity eps S / I + (1 - purity) b), Eq. 14
                                                                                              // DATA_M: data tiles only; the last CTA takes I = c^H M c from the held matrix + final NLL
// One resonance as the streaming kernel sees it: the three per-(mass,width) constants of LineConst,
// its first coupling slot, and either a pool column to read or -1 = evaluate in registers.
struct ResEntry {
    double kN, kG, M2;
    double2 cm, c0, cp;   // couplings of lambda = -1, 0, +1 (J = 0: only c0); times kN when the lineshape is evaluated in
                          // registers (column < 0): the kernels then form A^R / kN (bw_unscaled)
    int column;
};
// Resonances that share (chain, L_R, L_B, radius) share the barrier factors and momentum powers:
//   A^R = kN F / (M2 - m^2 - i kG G),  F = rs pB^LB (pR/m)^LR,  G = pR^(2LR+1) (1/m) rs^2 B_LB(zB)
// F and G are computed once per event and group; entries [first, first+count) belong to the group.
struct BarrierGroup {
    double r2;
    int first, count;
};
// A^R = kN F / (M2 - m2 - i kG G)
__device__ __forceinline__ double2 bw_from_consts(double kN, double kG, double M2, double m2, double F, double G) {
    const double MG = kG * G, dre = M2 - m2;
    const double s = kN * F * fast_rcp(fma(dre, dre, MG * MG));
    return make_double2(s * dre, s * MG);
}
__device__ __forceinline__ double2 bw_from_factors(const ResEntry& e, double m2, double F, double G) {
    return bw_from_consts(e.kN, e.kG, e.M2, m2, F, G);
}
// A^R / kN: the streaming kernels multiply it with couplings that the host has scaled by kN (one multiply less per resonance)
__device__ __forceinline__ double2 bw_unscaled(const ResEntry& e, double m2, double F, double G) {
    const double MG = e.kG * G, dre = e.M2 - m2;
    const double s = F * fast_rcp(fma(dre, dre, MG * MG));
    return make_double2(s * dre, s * MG);
}
struct StreamArgs {
    ResEntry ent[AMP_MAX_RESONANCES];
    BarrierGroup grp[AMP_MAX_RESONANCES];
    int lass0, nlass;               // LASS terms: entries ent[lass0 .. lass0 + nlass) (kG, M2 and c0 used), after the K* and Z entries
    int gstart[NSPIN + 1];          // groups of spin class sp: grp[gstart[sp] .. gstart[sp+1]); sp = J for the K* (0..4), 5 + z_class for the Z's
    int shape[NSPIN];               // resonances per spin class; entries are stored in that order
    int shape_fixed;                // 1: one radius per spin class, r2_spin valid: a shape-specialised kernel may run
    double r2_spin[NSPIN];
    double2 cconst;                 // sum of the couplings of the constant (lineshape == 1) terms
    const double* cache;            // tiled cache of the (first) sample, ncolw columns per 512-event block
    int ncolw;
    const double2* cols;
    long long n, npad;
    double* partial;                // [grid] (MODE_DATA: sum log S; MODE_NORM: sum w S)
    double* out;                    // MODE_EVAL: [n] eps_i S_i
    int* flag;
    int mode;
    // MODE_FUSED: the normalisation sample (second dataset), its partials, and what the last CTA needs to finish the NLL
    const double* cache2;
    long long n2, npad2;
    double* partial2;               // [grid] sum w S
    unsigned int* ticket;           // device counter, 0 between launches
    double* result;                 // [6]: NLL, I, domain flag, sum log S, sum w S, sequence stamp; may be mapped HOST memory
    double seq;                     // written to result[5] after a system-wide fence once the other five are in place
    double sum_log_eff, wsum;
    // MODE_DATA_BKG (Eq. 14): background density at the data events, signal purity, and the device location of sum_j w_j S_j
    // of this point (the normalisation pass runs first on the same stream)
    const double* bkg;
    const double* sum_wS;
    double purity;
    // MODE_DATA_M (static lineshapes): the held realified Gram matrix G' [KP][KP] (herk.cu) and the couplings in its entry
    // order (slot order, zero-padded to qf_nent): the last CTA evaluates sum_j w_j S_j = c^H M c itself
    const double* qf_G;
    int qf_KP, qf_nent;
    double2 qf_c[AMP_MAX_COUPLINGS];
};
cudaError_t launch_stream(const StreamArgs& a, int grid, cudaStream_t s);
int stream_grid(long long n, bool have_z, int mode);
int stream_grid_fused(long long n_data, long long n_norm, bool have_z);
long long stream_pad(long long n);   // events per column rounded up to whole pipeline tiles

// Gradient batches (P > 1 points that differ from point 0 in a few resonances), see delta.cu.
// The host compiles a batch into a small program the kernel keeps in shared memory:
//   A_xi(p) = A_xi(0) + sum over the point's contributions of  coef * SLOT_xi
// SLOT = a complex pair (xi = +1, -1) per event, a sum of terms  weight * [BW_ent(0)] * g_{J,lambda,xi}  (the angular
// factors of Eq. 4 or Eq. 10); consecutive contributions that use the same slot reuse it from registers.
//   coupling change of slot k:              coef = c_k(p) - c_k(0),      SLOT = BW_R(0) g_k          (1 term, unit weight)
//   mass/width change of resonance R:       coef = BW_R(p) - BW_R(0),    SLOT = sum_l c_{R,l}(0) g_{R,l}
//   both at once:                           coef = BW_R(p), SLOT = sum_l c_{R,l}(p) g_{R,l}   and   coef = -1, SLOT = sum_l c_{R,l}(0) BW_R(0) g_{R,l}
struct DeltaContrib {   // 32 bytes
    int hdr;            // bits 0-1: coef kind (0 explicit (a, b), c = a^2 + b^2; 1 BW(kN=a, kG=b, M2=c) - BW_ent(0) of the slot; 2 BW(a, b, c));
                        // bit 2: last contribution of its point; bit 3: slot differs from the previous contribution's;
                        // bit 4: empty (point equal to point 0 / padding); bit 5: the BW runs on the Z chain; bit 6: first of four
                        // single-contribution points of one kind (0 or 1) on one slot (host-marked); bits 8-11: barrier group
    int slot;           // offset of the slot record in the slot area, in 8-byte words
    double a, b, c;
};
// slot record: int2 {nterms, bw0 spec (ent | grp << 8 | isZ << 12, or -1: no BW(0) needed by kind-1 contributions)}, then
// per term: int2 {hdr, 0}, double w_re, double w_im;  term hdr: bits 0-7 ent (255: no BW factor), 8-11 grp, 12-14 J,
// 15-16 lambda + 1, 17 Z-chain term, 18 unit weight
enum { DELTA_MAX_SORTED = 128, DELTA_MAX_CONTRIB = 320, DELTA_MAX_SLOTWORDS = 1536 };   // per launch: points besides point 0; program sizes
struct DeltaArgs {
    StreamArgs a;                   // point 0 as the streaming kernel sees it (cache/weight/n/npad: data; cache2/...: norm)
    const DeltaContrib* contrib;    // [ncontrib] device
    const double* slots;            // [nslotwords] device
    int ncontrib, nslotwords;
    int nsorted;                    // points of this launch, padded to a multiple of 32 with empty points
    const int* point_of_sorted;     // [nsorted] -> point index 1..P-1 of this call, -1: padding
    int P;
    double* partial;                // [2][1 + nsorted][stride] per-CTA partials: sum log S (data) and sum w S (norm); row 0 = point 0
    int stride;
    double* result;                 // [4 P + 1]: NLL[P], I[P], domain flag, sum log S [P], sum w S [P]
    int want_nll;
    int first_chunk;                // 0: a later launch of the same call: the domain flag adds to the earlier launches'
};
cudaError_t launch_delta(const DeltaArgs& d, int grid, cudaStream_t s, bool exact = false);
int delta_grid(long long n_data, long long n_norm);
bool delta_fits(int ngrp);

// Gradient batches of the paper's resonance lists, shape-specialised form (deltaf.cu): every point besides point 0 is ONE coupling
// change (position = a coupling slot, or the tied pair of a Z's helicities +-1) or ONE lineshape change (mass / width of an entry);
// at most four points per position / entry.  All tables live in kernel parameter space (constant bank operands).
enum { DELTAF_MAX_POS = 32, DELTAF_MAX_ENT = 12 };
struct DeltaFArgs {
    StreamArgs a;                                 // point 0 as the streaming kernel sees it (cache/n: data; cache2/n2: norm)
    double cq[DELTAF_MAX_POS][4][3];              // coupling points of a position: Re, Im, |.|^2 of (c_k(p) - c_k(0)) kN_R(0)
    double cmax[DELTAF_MAX_POS][2];               // largest |Re|, |Im| and largest |.|^2 of cq[pos] (the guard on r)
    double mw[DELTAF_MAX_ENT][4][3];              // lineshape points of an entry: kN(p) / kN(0), kG(p), M2(p)
    unsigned pos_active, ent_active;              // bit per position / entry with at least one point
    short val_of_point[AMP_MAX_POINTS];           // point -> value slot 4 quad + j in the kernel's value order (DeltaFLayout); -1: equal to point 0
    short pos_of_point[AMP_MAX_POINTS];           // point -> its coupling position, -1 for a lineshape point
    int P;
    double* partial;                              // [2 + 2 NVAL][stride] per-CTA partials
    int stride;
    double* result;                               // [4 P + 2]: NLL[P], I[P], domain flag, sum log S [P], sum w S [P] (as DeltaArgs), stamp; may be mapped HOST memory
    double seq;                                   // written to result[4 P + 1] after a system-wide fence once the rest is in place
    int want_nll;
    // The normalisation events in a kernel of their own (deltan.cu; launched first on the same stream): its per-CTA partials,
    // the totals its last CTA leaves — [0] sum w S0, [1 + v] the normalisation-side value row v of k_deltaf's layout — and the
    // layout it scatters them by.  norm_tot == nullptr: k_deltaf walks the normalisation events itself.
    double* npartial;                             // [1 + 2 NSLOT + 8 NENT][stride]
    double* norm_tot;                             // [1 + NVAL]
    short quad_of_pos[DELTAF_MAX_POS], quad_of_ent[DELTAF_MAX_ENT];
};
cudaError_t launch_deltaf(const DeltaFArgs& d, int grid, cudaStream_t s);
int deltaf_grid(long long n_data, long long n_norm);
cudaError_t launch_deltan(const DeltaFArgs& d, int grid, int pass, cudaStream_t s);
int deltan_grid(long long n_norm);
struct DeltaFLayout { int nslot, npos, nent, nquad; int quad_of_pos[DELTAF_MAX_POS], quad_of_ent[DELTAF_MAX_ENT]; };
bool deltaf_layout(const StreamArgs& a, DeltaFLayout* lay);   // false: not one of the compiled shapes

// Analytic gradient of the NLL in the couplings (grad.cu): one pair of leaves (real, imaginary part) per coupling slot
enum { GRAD_MAX_PAIRS = 48 };
struct GradArgs {
    StreamArgs a;                       // the point, as the streaming kernel sees it (cache/n: data; cache2/n2: norm)
    int npairs;                         // coupling slots, padded to a multiple of 16 (2 npairs leaves = whole 32-leaf blocks)
    signed char pair_ent[GRAD_MAX_PAIRS];   // entry of StreamArgs::ent whose lineshape the slot carries; -1: lineshape == 1; -2: padding
    signed char pair_lam[GRAD_MAX_PAIRS];   // helicity -1, 0, +1
    signed char pair_J[GRAD_MAX_PAIRS];     // spin of a K* (0 for a constant term); 8: Z
    signed char pair_grp[GRAD_MAX_PAIRS];   // barrier group of the entry
    short pair_slot[GRAD_MAX_PAIRS];        // coupling slot k the pair belongs to, -1: padding
    signed char acc_pair[GRAD_MAX_PAIRS];   // gradf.cu: pair of accumulator q (entry order; lambda = -1, 0, +1 within an entry of spin >= 1)
    int K;
    double* partial;                    // [2][2 + 2 npairs][stride]: per-CTA partials; rows 0, 1 = sum log S / sum w S
    int stride;
    double* result;                     // [3 + 2 K]: NLL, I, domain flag, then (dNLL/dRe c_k, dNLL/dIm c_k); may be mapped host memory
};
cudaError_t launch_grad(const GradArgs& g, int grid, cudaStream_t s);
// gradf.cu: the shape-specialised form (gradient components in registers)
bool gradf_supports(const GradArgs& g);
int gradf_grid(long long n_data, long long n_norm);
cudaError_t launch_gradf(const GradArgs& g, int grid, cudaStream_t s);

// toy.cu — accept-reject toy generator: one block of candidates
struct ToyArgs {
    unsigned long long seed, first;   // Philox key; number of this block's first candidate
    long long n;                      // candidates in the block
    double m_lo, m_span, cos_max, f_max;
    double* x;                        // [4][n] candidate points (written by k_toy_candidates)
    double* u;                        // [n] acceptance uniforms
    const double* S;                  // [n] signal density of the candidates (streaming kernel, MODE_EVAL, weight 1)
    const double* cache;              // the candidates' kinematics cache (q and p_B columns are read)
    int ncolw;
    int* count;                       // [blocks + 1] accepted per block -> exclusive offsets, total last
    unsigned long long* f_seen;       // bits of the largest weight seen
    int* flag;
    double* x_out;                    // [4][capacity] accepted events, candidate order
    long long* index_out;             // [capacity] their candidate numbers, or null
    long long capacity, out_base;     // out_base: accepted before this block
};
int toy_blocks(long long n);
cudaError_t launch_toy_candidates(const ToyArgs& t, cudaStream_t s);
cudaError_t launch_toy_select(const ToyArgs& t, cudaStream_t s);
int grad_grid(long long n_data, long long n_norm);
bool grad_fits(int nent, int ngrp);

// Batched combine (P > 1) on the FP64 tensor cores, see batch.cu
enum { BATCH_NKT = 14, BATCH_POINTS = 128, BATCH_MAX_COLS = 48 };   // dense k-tiles (2K <= 56 realified rows) and points per launch
struct BatchArgs {
    const double* cache;    // tiled cache, ncolw columns per block (weight last)
    int ncolw;
    const double2* cols;
    long long n, npad;
    const double* Adense;   // [16 octets][re/im][BATCH_NKT][32 lanes]: coefficient fragments of the K base entries
    const int2* entries;    // [nent] (index into colu | -1 empty | -2 lineshape == 1, angular code) per complex basis entry
    int colu[BATCH_MAX_COLS];   // distinct pool columns the entries use (staged per tile)
    int ncolu;
    const int2* items;      // [nitems] (first realified row of an extended k-tile, octet 0/1 within the warp)
    const double* itemA;    // [nitems][re/im][32 lanes]
    int item_start[9];      // items of warp w: [item_start[w], item_start[w+1])
    short point_of_row[BATCH_POINTS];   // GEMM row (16 per warp) -> point of this launch, -1: unused row
    int nent;               // complex basis entries (base, padded to BATCH_NKT * 2, then extended), even
    int nkt;
    int P;                  // points in this launch (<= BATCH_POINTS)
    int have_z;
    int mode;               // MODE_DATA: sum_i log S(p,i); MODE_NORM: sum_j w_j S(p,j)
    double* partial;        // [P][partial_stride]
    int partial_stride;
    int* flag;
};
// Gram / normalisation matrix on the FP64 tensor cores, see herk.cu.  `b` carries the tile source (cache, weight,
// cols, n, npad, entries, nent (a multiple of 4), colu, ncolu, have_z); its GEMM fields are unused.
struct HerkArgs {
    BatchArgs b;
    const int4* runs;       // [8 warps][nrun] (row tile I, column tiles J0, J1, unused); 8 realified rows per tile
    const int2* runs_out;   // [8 warps][nrun] index of (I,J0), (I,J1) in the tile list, -1: padding (result dropped)
    int nrun;               // runs per warp (padded to the kernel's unroll count by launch_herk's choice: even numbers up to 12)
    int ntile;
    double* partial;        // [grid][ntile][64]
};
cudaError_t launch_herk(const HerkArgs& h, int grid, cudaStream_t s);
cudaError_t launch_herk_finish(const double* partial, int ncta, int ntile, const int2* tiles, int KP, double* gt, double* G, cudaStream_t s);
cudaError_t launch_quadform(const double* G, int KP, const double2* C, int nent, int P, double* out, cudaStream_t s);
int herk_max_runs();
int herk_grid(long long n, int nent, int ncolu);
int herk_grid_max();
cudaError_t launch_batch(const BatchArgs& a, int grid, cudaStream_t s);
int batch_grid(long long n);
bool batch_fits(int nent, int ncolu);

// fixed-order final reduction of per-block partials: out[j] = sum_b partial[j][b], j < nrows
cudaError_t launch_finalize(const double* partial, int nblocks, int stride, int nrows, double* out, cudaStream_t s);

cudaError_t probe_fp64(int kind, int iters, double* flops, cudaStream_t s);
cudaError_t probe_hbm_read(long long bytes, double* gbs, cudaStream_t s);

}  // namespace amp
