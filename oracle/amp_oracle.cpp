// amp_oracle.cpp — TEST INFRASTRUCTURE, NOT PRODUCT CODE.
//
// Plain, slow, event-by-event CPU oracle (FP64; an 80-bit `long double` twin is
// instantiated from the same template as a tie-breaker) of the per-event unbinned
// negative log-likelihood of the 4D amplitude model of Sur et al., "A GPU based
// multidimensional amplitude analysis to search for tetraquark candidates"
// (PAPER.md, Methodology, Eqs. 1-12 and 14).
//
// Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference
// legs may load this.  It shares no code, header, table or constant with the CUDA
// path under paper_2007_14931_b200/csrc and neither includes the other.
//
// The method is exact inside one NLL evaluation, so every function below is the
// paper's definition written out in the paper's order; where the paper is silent
// the reading (A1..A18) is the one listed in DESIGN.md §"Readings".
//
// Parity pins: every function here is pinned by tests/test_oracle_pins.py (P1-P23), and tests/test_oracle_mutations.py
// applies the one-line mistakes of tests/oracle_mutants.py to a copy of this file and requires a pin to fail for each.
// The orientation
// of theta_Z (reading A10: literal "angle between K and pi momenta in the Z rest frame",
// PAPER.md:176) is pinned by P22: it is the Jacob-Wick helicity angle of the psi from the Z's line
// of flight, which Eq. 10's d^{J}_{0 lambda'} requires; its supplement would only relabel the
// couplings H_lambda' -> (-1)^{J+lambda'} H_lambda' (same family of PDFs).
//
// Units: MeV; Blatt-Weisskopf radius in MeV^-1.

#include <cmath>
#include <complex>
#include <cstdint>
#include <cstring>
#include <limits>
#include <vector>
#ifdef _OPENMP
#include <omp.h>
#endif

namespace {

enum Kind { KSTAR = 0, ZRES = 1, CONSTANT = 2, LASS = 3, ZNEG = 4 };
// ZRES: an exotic Z -> J/psi pi of POSITIVE parity (the paper's default 1+; also 2+); ZNEG: of negative parity (0-, 1-, 2-).
// PAPER.md:171 ("J(Z) is the spin of the Z"), 314 ("any combination of their spin-parity values"); reading A24.
inline bool is_z(int kind) { return kind == ZRES || kind == ZNEG; }

template <typename T>
struct Decay {
    T MB, mpsi, mK, mpi;  // parent, J/psi, K, pi masses
};

template <typename T>
struct Resonance {
    int kind, J;
    T mass, width, radius;
};

// ---------------------------------------------------------------------------------
// O1. Two-body breakup momentum of M -> a b ("momenta ... calculated
// from the running and pole mass").  Fully factored Kallen form, differences first.
// Returns NaN below threshold.
template <typename T>
T breakup_momentum(T M, T a, T b) {
    const T s = a + b, d = a - b;
    const T k = (M - s) * (M + s) * (M - d) * (M + d);
    if (!(M > 0) || k < 0) return std::numeric_limits<T>::quiet_NaN();
    return std::sqrt(k) / (2 * M);
}

// ---------------------------------------------------------------------------------
// O2. Blatt-Weisskopf barrier factor (ref. [35]; reading A2): z = (r p)^2,
// F^(L)(p, p0) = sqrt(B_L(z0) / B_L(z)), normalised to 1 at the pole momentum p0.
template <typename T>
T barrier_polynomial(int L, T z) {
    switch (L) {
        case 0: return T(1);
        case 1: return 1 + z;
        case 2: return 9 + 3 * z + z * z;
        case 3: return 225 + 45 * z + 6 * z * z + z * z * z;
        case 4: return 11025 + 1575 * z + 135 * z * z + 10 * z * z * z + z * z * z * z;
    }
    return std::numeric_limits<T>::quiet_NaN();
}

template <typename T>
T blatt_weisskopf(int L, T p, T p0, T r) {
    const T z = (r * p) * (r * p), z0 = (r * p0) * (r * p0);
    return std::sqrt(barrier_polynomial(L, z0) / barrier_polynomial(L, z));
}

// ---------------------------------------------------------------------------------
// Orbital angular momenta ("lowest L_B is taken as the default"; readings A5, A6).
// Z chain (reading A24): B(0-) -> Z(J) K(0-) has L_B = J (angular momentum alone; the weak decay does not conserve parity);
// Z(J^P) -> psi(1-) pi(0-) is a strong decay: P = (+1)(-1)^L_R with |L_R - 1| <= J <= L_R + 1, lowest such L_R taken:
//   1+: 0,  2+: 2,  0-: 1,  1-: 1,  2-: 1   (0+ cannot decay to psi pi).
inline void orbital_L(int kind, int J, int* LB, int* LR) {
    if (is_z(kind)) {
        *LB = J;
        *LR = (kind == ZRES) ? (J == 1 ? 0 : 2) : 1;
        return;
    }
    *LR = J;                                           // K* -> K pi
    *LB = (J == 0) ? 1 : J - 1;                        // B(0-) -> psi(1-) K*(J): lowest allowed
}

// ---------------------------------------------------------------------------------
// O3. Lineshape, Eqs. (2)-(3) (readings A1, A4).
//   Gamma(m) = Gamma0 (pR/pR0)^(2LR+1) (MR/m) FR^2
//   A^R(m)   = FB (pB/MB)^LB FR (pR/m)^LR / (MR^2 - m^2 - i MR Gamma(m))
// m is the running mass of the resonance's daughters: m_Kpi for a K*, m_psipi for the Z.
// O3b. LASS parametrisation of the K pi S-wave, Eqs. (7)-(8) (readings A21, A22):
//   A_LASS = (m/q) sin(theta_B) e^{i theta_B} + 2 e^{2 i theta_B} (M0^2/q0) Gamma0 / (M0^2 - m^2 - i M0 Gamma(m))
//   cot(theta_B) = 1/(a q) + b q / 2,   a = 1.95 GeV^-1, b = 1.76 GeV^-1
// q = K momentum in the K pi frame at the running mass, q0 at the K0*(1430) mass M0; Gamma(m) is Eq. (3) with L_R = 0.
template <typename T>
std::complex<T> lass_lineshape(const Decay<T>& dk, const Resonance<T>& R, T m, T* gamma_out) {
    const T a = T(1.95e-3L), b = T(1.76e-3L);                 // MeV^-1
    const T q = breakup_momentum(m, dk.mK, dk.mpi), q0 = breakup_momentum(R.mass, dk.mK, dk.mpi);
    const T cot = 1 / (a * q) + b * q / 2;                      // Eq. (8)
    const T theta = std::atan2(T(1), cot);                      // theta_B in (0, pi)
    const T gamma = R.width * (q / q0) * (R.mass / m);          // Eq. (3), L_R = 0 (F^(0) = 1)
    if (gamma_out) *gamma_out = gamma;
    const std::complex<T> first = (m / q) * std::sin(theta) * std::polar(T(1), theta);
    const std::complex<T> den(R.mass * R.mass - m * m, -R.mass * gamma);
    const std::complex<T> second = T(2) * std::polar(T(1), 2 * theta) * ((R.mass * R.mass / q0) * R.width) / den;
    return first + second;                                       // Eq. (7)
}

template <typename T>
std::complex<T> lineshape(const Decay<T>& dk, const Resonance<T>& R, T m, T* gamma_out = nullptr) {
    if (R.kind == CONSTANT) { if (gamma_out) *gamma_out = 0; return {T(1), T(0)}; }
    if (R.kind == LASS) return lass_lineshape(dk, R, m, gamma_out);
    int LB, LR;
    orbital_L(R.kind, R.J, &LB, &LR);
    T pB, pB0, pR, pR0;
    if (R.kind == KSTAR) {
        pB  = breakup_momentum(dk.MB, m, dk.mpsi);        // K* momentum in the B frame
        pB0 = breakup_momentum(dk.MB, R.mass, dk.mpsi);
        pR  = breakup_momentum(m, dk.mK, dk.mpi);         // K momentum in the K* frame
        pR0 = breakup_momentum(R.mass, dk.mK, dk.mpi);
    } else {
        pB  = breakup_momentum(dk.MB, m, dk.mK);          // Z momentum in the B frame
        pB0 = breakup_momentum(dk.MB, R.mass, dk.mK);
        pR  = breakup_momentum(m, dk.mpsi, dk.mpi);       // pi momentum in the Z frame
        pR0 = breakup_momentum(R.mass, dk.mpsi, dk.mpi);
    }
    const T FB = blatt_weisskopf(LB, pB, pB0, R.radius);
    const T FR = blatt_weisskopf(LR, pR, pR0, R.radius);
    const T gamma = R.width * std::pow(pR / pR0, 2 * LR + 1) * (R.mass / m) * FR * FR;   // Eq. (3)
    if (gamma_out) *gamma_out = gamma;
    const T num = FB * std::pow(pB / dk.MB, LB) * FR * std::pow(pR / m, LR);
    const std::complex<T> den(R.mass * R.mass - m * m, -R.mass * gamma);
    return std::complex<T>(num, 0) / den;                                                 // Eq. (2)
}

// ---------------------------------------------------------------------------------
// O4. Wigner small-d, d^j_{m'm}(beta) = <j m'| exp(-i beta J_y) |j m>, Wigner's factorial sum
// ("Wigner small-d functions").
template <typename T>
T factorial(int n) { T f = 1; for (int i = 2; i <= n; ++i) f *= i; return f; }

template <typename T>
T wigner_d(int j, int mp, int m, T beta) {
    const T ch = std::cos(beta / 2), sh = std::sin(beta / 2);
    T sum = 0;
    for (int k = 0; k <= 2 * j; ++k) {
        const int a = j + m - k, b = j - mp - k, c = k, d = k + mp - m;
        if (a < 0 || b < 0 || c < 0 || d < 0) continue;
        const T sign = ((k + mp - m) % 2 == 0) ? T(1) : T(-1);
        sum += sign / (factorial<T>(a) * factorial<T>(b) * factorial<T>(c) * factorial<T>(d)) *
               std::pow(ch, 2 * j - 2 * k + m - mp) * std::pow(sh, 2 * k - m + mp);
    }
    return sum * std::sqrt(factorial<T>(j + m) * factorial<T>(j - m) * factorial<T>(j + mp) * factorial<T>(j - mp));
}

// ---------------------------------------------------------------------------------
// plain 4-vector algebra for O6 ("Lorentz boosts and rotations to go from one rest frame to
// another")
template <typename T> struct V3 { T x, y, z; };
template <typename T> struct V4 { T E; V3<T> p; };
template <typename T> T dot(V3<T> a, V3<T> b) { return a.x * b.x + a.y * b.y + a.z * b.z; }
template <typename T> V3<T> cross(V3<T> a, V3<T> b) { return {a.y * b.z - a.z * b.y, a.z * b.x - a.x * b.z, a.x * b.y - a.y * b.x}; }
template <typename T> V3<T> scale(T s, V3<T> a) { return {s * a.x, s * a.y, s * a.z}; }
template <typename T> V3<T> add(V3<T> a, V3<T> b) { return {a.x + b.x, a.y + b.y, a.z + b.z}; }
template <typename T> V3<T> sub(V3<T> a, V3<T> b) { return {a.x - b.x, a.y - b.y, a.z - b.z}; }
template <typename T> T norm(V3<T> a) { return std::sqrt(dot(a, a)); }
template <typename T> V3<T> unit(V3<T> a) { return scale(1 / norm(a), a); }
template <typename T> V4<T> add4(V4<T> a, V4<T> b) { return {a.E + b.E, add(a.p, b.p)}; }

// 4-momentum p seen from a frame that moves with velocity beta (|beta| < 1) relative to the
// frame in which p is given.
template <typename T>
V4<T> boost_to_frame(V4<T> p, V3<T> beta) {
    const T b2 = dot(beta, beta);
    if (b2 == 0) return p;
    const T g = 1 / std::sqrt(1 - b2);
    const T bp = dot(beta, p.p);
    V4<T> out;
    out.E = g * (p.E - bp);
    out.p = add(p.p, scale((g - 1) * bp / b2 - g * p.E, beta));
    return out;
}

// signed dihedral angle about the unit axis a from the direction u to the direction v
template <typename T>
T dihedral(V3<T> a, V3<T> u, V3<T> v) {
    const V3<T> up = sub(u, scale(dot(u, a), a)), vp = sub(v, scale(dot(v, a), a));
    return std::atan2(dot(a, cross(up, vp)), dot(up, vp));
}

template <typename T>
struct ZKinematics {
    T mZ, cosZ, sinZ, cosT, sinT, phiT, alpha;   // m_psipi, theta_Z, theta~_psi, phi~, alpha
    V4<T> K_B, pi_B, psi_B;                       // B-frame 4-momenta (diagnostics, pin P5)
    V3<T> nK, npi, nKst, nmu;                     // unit vectors in the psi rest frame (pin P7)
};

// O6. Z-chain kinematics from (m_Kpi, cos theta_K*, cos theta_psi, phi)
// (definitions; readings A7-A11).
template <typename T>
ZKinematics<T> z_kinematics(const Decay<T>& dk, T m, T cK, T cpsi, T phi) {
    ZKinematics<T> k;
    const T pB = breakup_momentum(dk.MB, m, dk.mpsi);
    const T q = breakup_momentum(m, dk.mK, dk.mpi);
    // 1. B rest frame, z along the K pi system
    const T EKpi = (dk.MB * dk.MB + m * m - dk.mpsi * dk.mpsi) / (2 * dk.MB);
    const V4<T> Kpi_B{EKpi, {0, 0, pB}};
    k.psi_B = V4<T>{dk.MB - EKpi, {0, 0, -pB}};
    // 2. K pi rest frame: theta_K* is the angle of the K from the K* flight direction
    const T sK = std::sqrt((1 - cK) * (1 + cK));
    const V4<T> K_R{std::sqrt(q * q + dk.mK * dk.mK), {q * sK, 0, q * cK}};
    const V4<T> pi_R{std::sqrt(q * q + dk.mpi * dk.mpi), {-q * sK, 0, -q * cK}};
    const V3<T> vKpi{0, 0, pB / EKpi};
    k.K_B = boost_to_frame(K_R, scale(T(-1), vKpi));
    k.pi_B = boost_to_frame(pi_R, scale(T(-1), vKpi));
    // 3. J/psi rest frame
    const V3<T> vpsi = scale(1 / k.psi_B.E, k.psi_B.p);
    const V4<T> K_P = boost_to_frame(k.K_B, vpsi), pi_P = boost_to_frame(k.pi_B, vpsi), Kst_P = boost_to_frame(Kpi_B, vpsi);
    k.nK = unit(K_P.p); k.npi = unit(pi_P.p); k.nKst = unit(Kst_P.p);
    // 4. mu+ direction: polar angle theta_psi from n_K* (A7), azimuth phi about n_K* from the K side (A8)
    const V3<T> ez = k.nKst;
    const V3<T> ex = unit(sub(k.nK, scale(dot(k.nK, ez), ez)));
    const V3<T> ey = cross(ez, ex);
    const T spsi = std::sqrt((1 - cpsi) * (1 + cpsi));
    k.nmu = add(add(scale(spsi * std::cos(phi), ex), scale(spsi * std::sin(phi), ey)), scale(cpsi, ez));
    // 5. Z = psi pi; theta_Z = angle between K and pi momenta in the Z rest frame (A10)
    const V4<T> Z_B = add4(k.psi_B, k.pi_B);
    k.mZ = std::sqrt(Z_B.E * Z_B.E - dot(Z_B.p, Z_B.p));
    const V3<T> vZ = scale(1 / Z_B.E, Z_B.p);
    const V3<T> uK = unit(boost_to_frame(k.K_B, vZ).p), upi = unit(boost_to_frame(k.pi_B, vZ).p);
    k.cosZ = dot(uK, upi);
    k.sinZ = norm(cross(uK, upi));
    // 6. theta~_psi = angle between mu+ and pi in the psi rest frame (A11)
    k.cosT = dot(k.nmu, k.npi);
    k.sinT = norm(cross(k.nmu, k.npi));
    // 7. phi~: between the (mu, pi) and (K, pi) planes about n_pi; alpha: between the (mu+, pi) and
    //    (mu+, K pi) planes about n_mu (A9)
    k.phiT = dihedral(k.npi, k.nK, k.nmu);
    k.alpha = dihedral(k.nmu, k.npi, k.nKst);
    return k;
}

// ---------------------------------------------------------------------------------
// Model = decay constants + resonance list; coupling slots in resonance order, lambda = -1,0,+1
// for J >= 1 K* and for the Z, lambda = 0 only for J = 0 K* and the constant term.
template <typename T>
struct Model {
    Decay<T> dk;
    std::vector<Resonance<T>> res;
    int num_couplings() const {
        int K = 0;
        for (auto& r : res) K += (is_z(r.kind) || (r.kind == KSTAR && r.J >= 1)) ? 3 : 1;
        return K;
    }
};

// Parameter-independent part of one event: the angles of both decay chains and the Wigner d's and
// phases Eqs. (4) and (10) need.  Computed once per event and reused for every parameter point
// (hoisting only: each entry is the same call the equations spell out).
template <typename T>
struct EventAngles {
    T m;                              // m_Kpi
    T dK[5][3];                       // d^J_{lambda 0}(theta_K*), J = 0..4, lambda = -1,0,+1 (index lambda+1)
    std::complex<T> ephi[3];          // e^{i lambda phi}
    T dpsi[3][2];                     // d^1_{lambda xi}(theta_psi), xi = +1 (index 0), -1 (index 1)
    bool haveZ = false;
    T mZ;                             // m_psipi
    T dZ[5][3];                       // d^J_{0 lambda'}(theta_Z)
    std::complex<T> ephiT[3];         // e^{i lambda' phi~}
    T dT[3][2];                       // d^1_{lambda' xi}(theta~_psi)
    std::complex<T> ealpha[2];        // e^{i xi alpha}
};

template <typename T>
EventAngles<T> event_angles(const Model<T>& M, const T x[4]) {
    EventAngles<T> a;
    const int xis[2] = {+1, -1};
    const T m = x[0], cK = x[1], cpsi = x[2], phi = x[3];
    a.m = m;
    const T thK = std::atan2(std::sqrt((1 - cK) * (1 + cK)), cK);
    const T thpsi = std::atan2(std::sqrt((1 - cpsi) * (1 + cpsi)), cpsi);
    for (const auto& R : M.res) {
        if (is_z(R.kind)) {
            if (!a.haveZ) {
                const ZKinematics<T> zk = z_kinematics(M.dk, m, cK, cpsi, phi);
                const T thT = std::atan2(zk.sinT, zk.cosT);
                a.haveZ = true;
                a.mZ = zk.mZ;
                for (int lp = -1; lp <= 1; ++lp) {
                    a.ephiT[lp + 1] = std::polar(T(1), lp * zk.phiT);
                    for (int ix = 0; ix < 2; ++ix) a.dT[lp + 1][ix] = wigner_d<T>(1, lp, xis[ix], thT);
                }
                for (int ix = 0; ix < 2; ++ix) a.ealpha[ix] = std::polar(T(1), xis[ix] * zk.alpha);
                const T thZ = std::atan2(zk.sinZ, zk.cosZ);
                for (int J = 0; J <= 4; ++J)
                    for (int lp = -1; lp <= 1; ++lp) a.dZ[J][lp + 1] = (std::abs(lp) <= J) ? wigner_d<T>(J, 0, lp, thZ) : T(0);
            }
        }
    }
    for (int J = 0; J <= 4; ++J)
        for (int l = -1; l <= 1; ++l) a.dK[J][l + 1] = (std::abs(l) <= J) ? wigner_d<T>(J, l, 0, thK) : T(0);
    for (int l = -1; l <= 1; ++l) {
        a.ephi[l + 1] = std::polar(T(1), l * phi);
        for (int ix = 0; ix < 2; ++ix) a.dpsi[l + 1][ix] = wigner_d<T>(1, l, xis[ix], thpsi);
    }
    return a;
}

// O5 + O7. Basis terms B_{k,xi}(event): everything in Eqs. (4) and (10) except the coupling H.
// out[k][0] is xi = +1, out[k][1] is xi = -1.
template <typename T>
void basis_terms(const Model<T>& M, const EventAngles<T>& a, std::complex<T>* out /* [K][2] */) {
    using C = std::complex<T>;
    int k = 0;
    for (const auto& R : M.res) {
        if (is_z(R.kind)) {
            const C A = lineshape(M.dk, R, a.mZ);
            for (int lp = -1; lp <= 1; ++lp, ++k)
                for (int ix = 0; ix < 2; ++ix)
                    // Eq. (10): A^Z d^J_{0 lambda'}(theta_Z) e^{i lambda' phi~} d^1_{lambda' xi}(theta~) e^{i xi alpha}
                    out[2 * k + ix] = A * a.dZ[R.J][lp + 1] * a.ephiT[lp + 1] * a.dT[lp + 1][ix] * a.ealpha[ix];
        } else {
            const C A = lineshape(M.dk, R, a.m);
            const int lmax = (R.kind == KSTAR && R.J >= 1) ? 1 : 0;
            for (int l = -lmax; l <= lmax; ++l, ++k)
                for (int ix = 0; ix < 2; ++ix)
                    // Eq. (4): A^K* d^J_{lambda 0}(theta_K*) e^{i lambda phi} d^1_{lambda xi}(theta_psi)
                    out[2 * k + ix] = A * a.dK[R.J][l + 1] * a.ephi[l + 1] * a.dpsi[l + 1][ix];
        }
    }
}

template <typename T>
void basis_terms(const Model<T>& M, const T x[4], std::complex<T>* out) {
    basis_terms(M, event_angles(M, x), out);
}

// O8. Signal density, Eq. (12): S = sum_xi | sum_k c_k B_{k xi} |^2
template <typename T>
T signal_density(const Model<T>& M, const std::complex<T>* c, const EventAngles<T>& a) {
    const int K = M.num_couplings();
    std::vector<std::complex<T>> B(2 * K);
    basis_terms(M, a, B.data());
    T S = 0;
    for (int ix = 0; ix < 2; ++ix) {
        std::complex<T> A(0, 0);
        for (int k = 0; k < K; ++k) A += c[k] * B[2 * k + ix];
        S += std::norm(A);
    }
    return S;
}

template <typename T>
T signal_density(const Model<T>& M, const std::complex<T>* c, const T x[4]) {
    return signal_density(M, c, event_angles(M, x));
}

// Neumaier-compensated running sum
template <typename T>
struct Neumaier {
    T s = 0, c = 0;
    void add(T v) { const T t = s + v; c += (std::fabs(s) >= std::fabs(v)) ? (s - t) + v : (v - t) + s; s = t; }
    T value() const { return s + c; }
};

template <typename T>
Model<T> make_model(const double* decay, int n_res, const int* kinds, const int* Js, const double* mass,
                    const double* width, const double* radius) {
    Model<T> M;
    M.dk = Decay<T>{T(decay[0]), T(decay[1]), T(decay[2]), T(decay[3])};
    for (int r = 0; r < n_res; ++r) M.res.push_back(Resonance<T>{kinds[r], Js[r], T(mass[r]), T(width[r]), T(radius[r])});
    return M;
}

template <typename T>
std::vector<std::complex<T>> make_couplings(const double* c, int K) {
    std::vector<std::complex<T>> v(K);
    for (int k = 0; k < K; ++k) v[k] = std::complex<T>(T(c[2 * k]), T(c[2 * k + 1]));
    return v;
}

// per-event v_i = eff_i * S_i (Eq. 14 with purity p = 1); x is SoA [4][n]
template <typename T>
void eval_events(const Model<T>& M, const std::complex<T>* c, const double* x, const double* eff, long long n, double* out) {
#pragma omp parallel for schedule(static)
    for (long long i = 0; i < n; ++i) {
        const T xi[4] = {T(x[i]), T(x[n + i]), T(x[2 * n + i]), T(x[3 * n + i])};
        const T S = signal_density(M, c, xi);
        out[i] = double((eff ? T(eff[i]) : T(1)) * S);
    }
}

// O9 pieces.  For every parameter point p: sum over events of w*S_p and of w (normalisation) or of
// log(eff*S_p) (data), each Neumaier-compensated, in event order (per-thread chunks are contiguous and
// combined in thread order: the result depends on the thread count only, not on scheduling).  The
// parameter loop sits inside the event loop so the angles of an event are computed once.
template <typename T>
void weighted_sums(const std::vector<Model<T>>& Ms, const std::vector<std::vector<std::complex<T>>>& cs, const double* x,
                   const double* w, long long n, bool take_log, std::vector<T>& sum_out, T* wsum_out) {
    const int P = (int)Ms.size();
    int nt = 1;
#ifdef _OPENMP
    nt = omp_get_max_threads();
#endif
    std::vector<std::vector<Neumaier<T>>> acc(nt, std::vector<Neumaier<T>>(P));
    std::vector<Neumaier<T>> wacc(nt);
#pragma omp parallel num_threads(nt)
    {
        int t = 0;
#ifdef _OPENMP
        t = omp_get_thread_num();
#endif
        const long long lo = n * t / nt, hi = n * (t + 1) / nt;
        for (long long i = lo; i < hi; ++i) {
            const T xi[4] = {T(x[i]), T(x[n + i]), T(x[2 * n + i]), T(x[3 * n + i])};
            const EventAngles<T> a = event_angles(Ms[0], xi);
            const T wi = w ? T(w[i]) : T(1);
            for (int p = 0; p < P; ++p) {
                const T S = signal_density(Ms[p], cs[p].data(), a);
                acc[t][p].add(take_log ? std::log(wi * S) : wi * S);
            }
            wacc[t].add(wi);
        }
    }
    sum_out.assign(P, T(0));
    for (int p = 0; p < P; ++p) {
        Neumaier<T> tot;
        for (int t = 0; t < nt; ++t) { tot.add(acc[t][p].s); tot.add(acc[t][p].c); }
        sum_out[p] = tot.value();
    }
    Neumaier<T> wtot;
    for (int t = 0; t < nt; ++t) { wtot.add(wacc[t].s); wtot.add(wacc[t].c); }
    *wsum_out = wtot.value();
}

template <typename T>
int nll_impl(const double* decay, int n_res, const int* kinds, const int* Js, const double* mass, const double* width,
             const double* radius, int P, const double* couplings /*[P][K][2]*/, const double* mass_width /*[P][R][2] or null*/,
             const double* x, const double* eff, long long n, const double* xn, const double* wn, long long mn,
             double* nll_out, double* integral_out) {
    std::vector<Model<T>> Ms;
    std::vector<std::vector<std::complex<T>>> cs;
    for (int p = 0; p < P; ++p) {
        Model<T> M = make_model<T>(decay, n_res, kinds, Js, mass, width, radius);
        if (mass_width)
            for (int r = 0; r < n_res; ++r) { M.res[r].mass = T(mass_width[(p * n_res + r) * 2]); M.res[r].width = T(mass_width[(p * n_res + r) * 2 + 1]); }
        const int K = M.num_couplings();
        cs.push_back(make_couplings<T>(couplings + (size_t)p * K * 2, K));
        Ms.push_back(M);
    }
    std::vector<T> wS, slog;
    T wsum, dummy;
    weighted_sums(Ms, cs, xn, wn, mn, false, wS, &wsum);
    if (nll_out) weighted_sums(Ms, cs, x, eff, n, true, slog, &dummy);
    for (int p = 0; p < P; ++p) {
        const T I = wS[p] / wsum;                                   // MC integral (A15)
        if (integral_out) integral_out[p] = double(I);
        if (nll_out) nll_out[p] = double(-(slog[p] - T(n) * std::log(I)));   // -sum_i log(eff_i S_i / I)
    }
    return 0;
}

// Gradient of the NLL with respect to the complex couplings (the derivative of O9 written out).
// With A_xi = sum_k c_k B_k,xi and S = sum_xi |A_xi|^2:  dS/dconj(c_k) = sum_xi conj(B_k,xi) A_xi, so
//   dNLL/dconj(c_k) = - sum_i [sum_xi conj(B_k,xi(i)) A_xi(i)] / S_i  +  N [sum_j w_j sum_xi conj(B_k,xi(j)) A_xi(j)] / [sum_j w_j S_j]
// and for the real parameters dNLL/dRe(c_k) = 2 Re(.), dNLL/dIm(c_k) = 2 Im(.).  grad_out is [K][2] = (d/dRe, d/dIm).
template <typename T>
void nll_gradient_impl(const Model<T>& M, const std::complex<T>* c, const double* x, const double* eff, long long n, const double* xn,
                       const double* wn, long long mn, double* nll_out, double* grad_out) {
    using C = std::complex<T>;
    const int K = M.num_couplings();
    std::vector<C> B(2 * K), D(K, C(0, 0)), Nk(K, C(0, 0));
    Neumaier<T> slog, swS, sw;
    for (long long i = 0; i < n; ++i) {
        const T xi[4] = {T(x[i]), T(x[n + i]), T(x[2 * n + i]), T(x[3 * n + i])};
        basis_terms(M, xi, B.data());
        C A[2] = {C(0, 0), C(0, 0)};
        for (int k = 0; k < K; ++k) { A[0] += c[k] * B[2 * k]; A[1] += c[k] * B[2 * k + 1]; }
        const T S = std::norm(A[0]) + std::norm(A[1]);
        slog.add(std::log((eff ? T(eff[i]) : T(1)) * S));
        for (int k = 0; k < K; ++k) D[k] += (std::conj(B[2 * k]) * A[0] + std::conj(B[2 * k + 1]) * A[1]) / S;
    }
    for (long long j = 0; j < mn; ++j) {
        const T xj[4] = {T(xn[j]), T(xn[mn + j]), T(xn[2 * mn + j]), T(xn[3 * mn + j])};
        basis_terms(M, xj, B.data());
        C A[2] = {C(0, 0), C(0, 0)};
        for (int k = 0; k < K; ++k) { A[0] += c[k] * B[2 * k]; A[1] += c[k] * B[2 * k + 1]; }
        const T w = wn ? T(wn[j]) : T(1);
        swS.add(w * (std::norm(A[0]) + std::norm(A[1])));
        sw.add(w);
        for (int k = 0; k < K; ++k) Nk[k] += w * (std::conj(B[2 * k]) * A[0] + std::conj(B[2 * k + 1]) * A[1]);
    }
    *nll_out = double(-(slog.value() - T(n) * std::log(swS.value() / sw.value())));
    for (int k = 0; k < K; ++k) {
        const C g = -D[k] + T(n) * Nk[k] / swS.value();
        grad_out[2 * k] = double(2 * g.real());
        grad_out[2 * k + 1] = double(2 * g.imag());
    }
}

// Gradient with background and purity, Eq. 14: NLL = - sum_i log f_i, f_i = (p / I) eps_i S_i + (1 - p) b_i,
// I = W / sum_j w_j, W = sum_j w_j S_j.  With u_i = (p / I) eps_i / f_i:
//   dNLL/dconj(c_k) = - sum_i u_i [sum_xi conj(B_k,xi(i)) A_xi(i)]  +  [sum_i u_i S_i] [sum_j w_j sum_xi conj(B_k,xi(j)) A_xi(j)] / W
// (the second term is the derivative of 1/I); without background u_i = 1 / S_i and sum_i u_i S_i = N: nll_gradient_impl.
template <typename T>
void nll_gradient_bkg_impl(const Model<T>& M, const std::complex<T>* c, const double* x, const double* eff, const double* bkg, double purity,
                           long long n, const double* xn, const double* wn, long long mn, double* nll_out, double* grad_out) {
    using C = std::complex<T>;
    const int K = M.num_couplings();
    std::vector<C> B(2 * K), D(K, C(0, 0)), Nk(K, C(0, 0));
    Neumaier<T> slog, swS, sw, suS;
    for (long long j = 0; j < mn; ++j) {
        const T xj[4] = {T(xn[j]), T(xn[mn + j]), T(xn[2 * mn + j]), T(xn[3 * mn + j])};
        basis_terms(M, xj, B.data());
        C A[2] = {C(0, 0), C(0, 0)};
        for (int k = 0; k < K; ++k) { A[0] += c[k] * B[2 * k]; A[1] += c[k] * B[2 * k + 1]; }
        const T w = wn ? T(wn[j]) : T(1);
        swS.add(w * (std::norm(A[0]) + std::norm(A[1])));
        sw.add(w);
        for (int k = 0; k < K; ++k) Nk[k] += w * (std::conj(B[2 * k]) * A[0] + std::conj(B[2 * k + 1]) * A[1]);
    }
    const T I = swS.value() / sw.value(), p = T(purity);
    for (long long i = 0; i < n; ++i) {
        const T xi[4] = {T(x[i]), T(x[n + i]), T(x[2 * n + i]), T(x[3 * n + i])};
        basis_terms(M, xi, B.data());
        C A[2] = {C(0, 0), C(0, 0)};
        for (int k = 0; k < K; ++k) { A[0] += c[k] * B[2 * k]; A[1] += c[k] * B[2 * k + 1]; }
        const T S = std::norm(A[0]) + std::norm(A[1]), e = eff ? T(eff[i]) : T(1);
        const T f = (p / I) * e * S + (1 - p) * T(bkg[i]);
        slog.add(std::log(f));
        const T u = (p / I) * e / f;
        suS.add(u * S);
        for (int k = 0; k < K; ++k) D[k] += u * (std::conj(B[2 * k]) * A[0] + std::conj(B[2 * k + 1]) * A[1]);
    }
    *nll_out = double(-slog.value());
    for (int k = 0; k < K; ++k) {
        const C g = -D[k] + suS.value() * Nk[k] / swS.value();
        grad_out[2 * k] = double(2 * g.real());
        grad_out[2 * k + 1] = double(2 * g.imag());
    }
}

// Hermitian normalisation matrix M_kl = sum_j w_j sum_xi conj(B_k xi) B_l xi / sum_j w_j (pin P10,
// fit fractions Eq. 13).  out is [K][K][2] row-major.
template <typename T>
void norm_matrix_impl(const Model<T>& M, const double* xn, const double* wn, long long mn, double* out) {
    const int K = M.num_couplings();
    std::vector<std::complex<T>> acc((size_t)K * K, std::complex<T>(0, 0));
    std::vector<std::complex<T>> B(2 * K);
    T wsum = 0;
    for (long long j = 0; j < mn; ++j) {
        const T xj[4] = {T(xn[j]), T(xn[mn + j]), T(xn[2 * mn + j]), T(xn[3 * mn + j])};
        basis_terms(M, xj, B.data());
        const T w = wn ? T(wn[j]) : T(1);
        wsum += w;
        for (int k = 0; k < K; ++k)
            for (int l = 0; l < K; ++l)
                for (int ix = 0; ix < 2; ++ix) acc[(size_t)k * K + l] += w * std::conj(B[2 * k + ix]) * B[2 * l + ix];
    }
    for (size_t i = 0; i < acc.size(); ++i) { out[2 * i] = double(acc[i].real() / wsum); out[2 * i + 1] = double(acc[i].imag() / wsum); }
}

}  // namespace

// ---------------------------------------------------------------------------------
// C ABI for ctypes (tests and the bench's cpu_baseline leg).  `prec` = 0: double, 1: long double.
#define DISPATCH(prec, CALL_D, CALL_L) do { if (prec) { CALL_L; } else { CALL_D; } } while (0)

extern "C" {

int orc_num_threads() {
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}
void orc_set_num_threads(int n) {
#ifdef _OPENMP
    omp_set_num_threads(n);
#else
    (void)n;
#endif
}

double orc_breakup_momentum(double M, double a, double b, int prec) {
    if (prec) return double(breakup_momentum<long double>(M, a, b));
    return breakup_momentum<double>(M, a, b);
}
double orc_barrier_polynomial(int L, double z) { return barrier_polynomial<double>(L, z); }
double orc_blatt_weisskopf(int L, double p, double p0, double r) { return blatt_weisskopf<double>(L, p, p0, r); }
double orc_wigner_d(int j, int mp, int m, double beta, int prec) {
    if (prec) return double(wigner_d<long double>(j, mp, m, beta));
    return wigner_d<double>(j, mp, m, beta);
}
void orc_orbital_L(int kind, int J, int* LB, int* LR) { orbital_L(kind, J, LB, LR); }

// out[0..1] = A^R(m) (re, im), out[2] = Gamma(m)
void orc_lineshape(const double* decay, int kind, int J, double mass, double width, double radius, double m, int prec, double* out) {
    if (prec) {
        Decay<long double> dk{decay[0], decay[1], decay[2], decay[3]};
        Resonance<long double> R{kind, J, mass, width, radius};
        long double g; auto A = lineshape<long double>(dk, R, m, &g);
        out[0] = double(A.real()); out[1] = double(A.imag()); out[2] = double(g);
    } else {
        Decay<double> dk{decay[0], decay[1], decay[2], decay[3]};
        Resonance<double> R{kind, J, mass, width, radius};
        double g; auto A = lineshape<double>(dk, R, m, &g);
        out[0] = A.real(); out[1] = A.imag(); out[2] = g;
    }
}

// A^R at an EVENT: the running mass of the resonance's chain (m_Kpi, or m_psipi from O6) is formed from the event in the working
// precision and handed to O3 without passing through a double — plumbing of z_kinematics + lineshape for the long-double
// arbitration of the parity tests near the m_psipi thresholds (no arithmetic of its own).  out[0..1] = A^R (re, im), out[2] = running mass
}  // extern "C"
template <typename T>
static void lineshape_at_event_fill(const double* decay, int kind, int J, double mass, double width, double radius, const double* x, double* out) {
    Decay<T> dk{T(decay[0]), T(decay[1]), T(decay[2]), T(decay[3])};
    Resonance<T> R{kind, J, T(mass), T(width), T(radius)};
    const T m = is_z(kind) ? z_kinematics<T>(dk, T(x[0]), T(x[1]), T(x[2]), T(x[3])).mZ : T(x[0]);
    const std::complex<T> A = lineshape<T>(dk, R, m);
    out[0] = double(A.real()); out[1] = double(A.imag()); out[2] = double(m);
}
extern "C" {
void orc_lineshape_at_event(const double* decay, int kind, int J, double mass, double width, double radius, const double* x /*[4]*/, int prec, double* out /*[3]*/) {
    DISPATCH(prec, lineshape_at_event_fill<double>(decay, kind, J, mass, width, radius, x, out),
             lineshape_at_event_fill<long double>(decay, kind, J, mass, width, radius, x, out));
}

// out[0..6] = mZ, cosZ, sinZ, cosT, sinT, phiT, alpha; out[7..18] = K_B, pi_B, psi_B (E,px,py,pz);
// out[19..30] = nK, npi, nKst, nmu (unit 3-vectors in the psi rest frame)
}  // extern "C"
template <typename T>
static void zkin_fill(const double* decay, const double* x, double* out) {
    Decay<T> dk{T(decay[0]), T(decay[1]), T(decay[2]), T(decay[3])};
    auto k = z_kinematics<T>(dk, T(x[0]), T(x[1]), T(x[2]), T(x[3]));
    const T v[31] = {k.mZ, k.cosZ, k.sinZ, k.cosT, k.sinT, k.phiT, k.alpha,
                     k.K_B.E, k.K_B.p.x, k.K_B.p.y, k.K_B.p.z, k.pi_B.E, k.pi_B.p.x, k.pi_B.p.y, k.pi_B.p.z,
                     k.psi_B.E, k.psi_B.p.x, k.psi_B.p.y, k.psi_B.p.z,
                     k.nK.x, k.nK.y, k.nK.z, k.npi.x, k.npi.y, k.npi.z, k.nKst.x, k.nKst.y, k.nKst.z, k.nmu.x, k.nmu.y, k.nmu.z};
    for (int i = 0; i < 31; ++i) out[i] = double(v[i]);
}
extern "C" {
void orc_z_kinematics(const double* decay, const double* x /*[4]*/, int prec, double* out /*[31]*/) {
    DISPATCH(prec, zkin_fill<double>(decay, x, out), zkin_fill<long double>(decay, x, out));
}

int orc_num_couplings(int n_res, const int* kinds, const int* Js) {
    int K = 0;
    for (int r = 0; r < n_res; ++r) K += (is_z(kinds[r]) || (kinds[r] == KSTAR && Js[r] >= 1)) ? 3 : 1;
    return K;
}

// basis terms of one event: out [K][2 (xi=+1,-1)][2 (re,im)]
}  // extern "C"
template <typename T>
static void basis_fill(const double* decay, int n_res, const int* kinds, const int* Js, const double* mass, const double* width,
                       const double* radius, const double* x, double* out) {
    auto M = make_model<T>(decay, n_res, kinds, Js, mass, width, radius);
    const int K = M.num_couplings();
    std::vector<std::complex<T>> B(2 * K);
    const T xx[4] = {T(x[0]), T(x[1]), T(x[2]), T(x[3])};
    basis_terms(M, xx, B.data());
    for (int i = 0; i < 2 * K; ++i) { out[2 * i] = double(B[i].real()); out[2 * i + 1] = double(B[i].imag()); }
}
extern "C" {
void orc_basis_terms(const double* decay, int n_res, const int* kinds, const int* Js, const double* mass, const double* width,
                     const double* radius, const double* x, int prec, double* out) {
    DISPATCH(prec, basis_fill<double>(decay, n_res, kinds, Js, mass, width, radius, x, out),
             basis_fill<long double>(decay, n_res, kinds, Js, mass, width, radius, x, out));
}

// v_i = eff_i S_i for n events, x SoA [4][n]; eff may be null (= 1)
void orc_eval_events(const double* decay, int n_res, const int* kinds, const int* Js, const double* mass, const double* width,
                     const double* radius, const double* couplings, const double* x, const double* eff, long long n, int prec,
                     double* out) {
    if (prec) {
        auto M = make_model<long double>(decay, n_res, kinds, Js, mass, width, radius);
        auto c = make_couplings<long double>(couplings, M.num_couplings());
        eval_events(M, c.data(), x, eff, n, out);
    } else {
        auto M = make_model<double>(decay, n_res, kinds, Js, mass, width, radius);
        auto c = make_couplings<double>(couplings, M.num_couplings());
        eval_events(M, c.data(), x, eff, n, out);
    }
}

// NLL(p) = -sum_i log(eff_i S_i(p) / I(p)), I(p) = sum_j w_j S_j(p) / sum_j w_j, for P parameter points.
// nll_out and/or integral_out may be null.
int orc_nll(const double* decay, int n_res, const int* kinds, const int* Js, const double* mass, const double* width,
            const double* radius, int P, const double* couplings, const double* mass_width, const double* x, const double* eff,
            long long n, const double* xn, const double* wn, long long mn, int prec, double* nll_out, double* integral_out) {
    if (prec) return nll_impl<long double>(decay, n_res, kinds, Js, mass, width, radius, P, couplings, mass_width, x, eff, n, xn, wn, mn, nll_out, integral_out);
    return nll_impl<double>(decay, n_res, kinds, Js, mass, width, radius, P, couplings, mass_width, x, eff, n, xn, wn, mn, nll_out, integral_out);
}

void orc_nll_gradient(const double* decay, int n_res, const int* kinds, const int* Js, const double* mass, const double* width,
                      const double* radius, const double* couplings, const double* x, const double* eff, long long n, const double* xn,
                      const double* wn, long long mn, double* nll_out, double* grad_out) {
    auto M = make_model<double>(decay, n_res, kinds, Js, mass, width, radius);
    auto c = make_couplings<double>(couplings, M.num_couplings());
    nll_gradient_impl(M, c.data(), x, eff, n, xn, wn, mn, nll_out, grad_out);
}

void orc_nll_gradient_bkg(const double* decay, int n_res, const int* kinds, const int* Js, const double* mass, const double* width,
                          const double* radius, const double* couplings, const double* x, const double* eff, const double* bkg,
                          double purity, long long n, const double* xn, const double* wn, long long mn, double* nll_out, double* grad_out) {
    auto M = make_model<double>(decay, n_res, kinds, Js, mass, width, radius);
    auto c = make_couplings<double>(couplings, M.num_couplings());
    nll_gradient_bkg_impl(M, c.data(), x, eff, bkg, purity, n, xn, wn, mn, nll_out, grad_out);
}

void orc_norm_matrix(const double* decay, int n_res, const int* kinds, const int* Js, const double* mass, const double* width,
                     const double* radius, const double* xn, const double* wn, long long mn, double* out) {
    auto M = make_model<double>(decay, n_res, kinds, Js, mass, width, radius);
    norm_matrix_impl(M, xn, wn, mn, out);
}

}  // extern "C"
