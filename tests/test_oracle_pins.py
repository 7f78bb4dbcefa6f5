"""Pins of the CPU oracle (oracle/amp_oracle.cpp) against what the paper and the mathematics fix.

None of these re-types an oracle formula: each compares against a library routine (sympy Wigner d,
scipy spherical Bessel / quadrature / Legendre), a closed form, an invariant, or an identity that a
dropped term, wrong sign, wrong index or transposed operand breaks.  Pin numbers P1..P12 are those of
DESIGN.md §"Oracle pins".
"""
import functools
import math

import numpy as np
import pytest
from numpy.polynomial import legendre as npleg
from scipy import integrate, special

from oracle import oracle as O
from paper_2007_14931_b200 import workloads as W

DEC = W.DECAY
MB, MPSI, MK, MPI = DEC
R16 = W.RADIUS


@functools.lru_cache(maxsize=None)
def _sympy_d_function(j, mp, m):
    import sympy
    from sympy.physics.quantum.spin import Rotation
    b = sympy.Symbol("beta", real=True)
    f = sympy.lambdify(b, Rotation.d(j, mp, m, b).doit(), "math")
    return lambda beta: float(f(beta))


def model(cfg):
    return O.Model(DEC, W.resonances(cfg))


# ------------------------------------------------------------------ P1: Wigner d closed forms / library
def test_P1_wigner_d_matches_sympy_and_tables():
    for beta in (0.3, 1.1, 2.9):
        for j in (1, 2, 3, 4):
            for mp in range(-j, j + 1):
                for m in (-1, 0, 1):
                    ref = _sympy_d(j, mp, m, beta)
                    assert abs(O.wigner_d(j, mp, m, beta) - ref) < 2e-15, (j, mp, m, beta)
    # PDG table, j = 1 (valid for any beta, also negative)
    for b in np.linspace(-3.0, 3.0, 13):
        c, s = math.cos(b), math.sin(b)
        assert abs(O.wigner_d(1, 1, 1, b) - (1 + c) / 2) < 1e-15
        assert abs(O.wigner_d(1, -1, -1, b) - (1 + c) / 2) < 1e-15
        assert abs(O.wigner_d(1, 1, -1, b) - (1 - c) / 2) < 1e-15
        assert abs(O.wigner_d(1, -1, 1, b) - (1 - c) / 2) < 1e-15
        assert abs(O.wigner_d(1, 1, 0, b) + s / math.sqrt(2)) < 1e-15
        assert abs(O.wigner_d(1, 0, 1, b) - s / math.sqrt(2)) < 1e-15
        assert abs(O.wigner_d(1, 0, -1, b) + s / math.sqrt(2)) < 1e-15
        assert abs(O.wigner_d(1, 0, 0, b) - c) < 1e-15
        assert abs(O.wigner_d(2, 1, 0, b) + math.sqrt(1.5) * s * c) < 1e-15
        assert abs(O.wigner_d(2, 0, 0, b) - (3 * c * c - 1) / 2) < 1e-15
    # d^J_00 = P_J(cos), d^J_{10} = -sin P_J'(cos)/sqrt(J(J+1)) (Legendre from numpy)
    for J in range(0, 5):
        PJ = npleg.Legendre.basis(J)
        for b in (0.2, 1.3, 2.7):
            assert abs(O.wigner_d(J, 0, 0, b) - PJ(math.cos(b))) < 2e-15
            if J:
                ref = -math.sin(b) * PJ.deriv()(math.cos(b)) / math.sqrt(J * (J + 1))
                assert abs(O.wigner_d(J, 1, 0, b) - ref) < 4e-15
                assert abs(O.wigner_d(J, -1, 0, b) + ref) < 4e-15
    assert abs(O.wigner_d(3, 1, 0, 0.9, prec=1) - O.wigner_d(3, 1, 0, 0.9)) < 1e-15


# ------------------------------------------------------------------ P2: orthogonality
def test_P2_wigner_d_orthogonality():
    xs, ws = npleg.leggauss(24)
    for lam in (0, 1):
        for J in range(lam, 5):
            for Jp in range(lam, 5):
                val = sum(w * O.wigner_d(J, lam, 0, math.acos(x)) * O.wigner_d(Jp, lam, 0, math.acos(x)) for x, w in zip(xs, ws))
                assert abs(val - (2.0 / (2 * J + 1) if J == Jp else 0.0)) < 1e-13
    for lam in (-1, 0, 1):
        val = sum(w * sum(O.wigner_d(1, lam, xi, math.acos(x)) ** 2 for xi in (1, -1)) for x, w in zip(xs, ws))
        assert abs(val - 4.0 / 3.0) < 1e-13


# ------------------------------------------------------------------ P3: lineshape at the pole; optical-theorem identity
@pytest.mark.parametrize("cfg", [1, 2])
def test_P3_lineshape_pole_and_phase(cfg):
    M = model(cfg)
    for r, (kind, J, mass, width, rad) in enumerate(W.resonances(cfg)):
        A, gam = M.lineshape(r, mass)
        assert abs(gam - width) < 1e-12 * width                       # Gamma(M_R) = Gamma0
        LB, LR = O.orbital_L(kind, J)
        if kind == O.KSTAR:
            pB0, pR0 = O.breakup_momentum(MB, mass, MPSI), O.breakup_momentum(mass, MK, MPI)
        else:
            pB0, pR0 = O.breakup_momentum(MB, mass, MK), O.breakup_momentum(mass, MPSI, MPI)
        # F = 1 at the pole, so A = i (pB0/MB)^LB (pR0/M)^LR / (M Gamma0): bare propagator modulus 1/(M Gamma0)
        bare = A / ((pB0 / MB) ** LB * (pR0 / mass) ** LR)
        assert abs(bare.real) < 1e-12 * abs(bare)
        assert abs(bare.imag - 1.0 / (mass * width)) < 1e-12 / (mass * width)
        # phase rises through pi/2 at the pole; imaginary part positive everywhere (Gamma > 0)
        lo, hi = (MK + MPI + 1, MB - MPSI - 1) if kind == O.KSTAR else (MPSI + MPI + 1, MB - MK - 1)
        ms = np.linspace(lo, hi, 400)
        ph = np.unwrap([np.angle(M.lineshape(r, m)[0]) for m in ms])
        assert np.all(np.diff(ph) > 0) and np.all((ph > 0) & (ph < np.pi))
        assert (ph[ms < mass] < np.pi / 2).all() and (ph[ms > mass] > np.pi / 2).all()


def test_P3b_running_width_scaling_from_optical_identity():
    """Im(1/D) = M Gamma(m)/|D|^2 gives Gamma(m) from the complex output alone.  With r -> 0 the barrier
    factors are 1, so Gamma(m) m / (M Gamma0) must be an exact power (2L+1) of the breakup momentum and the
    numerator an exact power law — fixes the exponents and the M_R/m factor of Eq. 3 and the momentum powers
    of Eq. 2 (reading A4)."""
    for kind, J, mass, width in [(O.KSTAR, 0, 1425.0, 270.0), (O.KSTAR, 1, 895.55, 47.3), (O.KSTAR, 2, 1432.4, 109.0),
                                 (O.KSTAR, 3, 1776.0, 159.0), (O.KSTAR, 4, 2045.0, 198.0), (O.ZRES, 1, 4196.0, 370.0)]:
        M = O.Model(DEC, [(kind, J, mass, width, 0.0)])
        LB, LR = O.orbital_L(kind, J)
        assert (LB, LR) == ((1, 0) if kind == O.ZRES else (1 if J == 0 else J - 1, J))
        mom = (lambda m: (O.breakup_momentum(MB, m, MPSI), O.breakup_momentum(m, MK, MPI))) if kind == O.KSTAR else \
              (lambda m: (O.breakup_momentum(MB, m, MK), O.breakup_momentum(m, MPSI, MPI)))
        pB0, pR0 = mom(mass)
        for m in np.linspace(mass - 200, mass + 130, 7):
            A, gam = M.lineshape(0, m)
            pB, pR = mom(m)
            num = (pB / MB) ** LB * (pR / m) ** LR                    # r = 0: |A| |D| = numerator
            D = num / A                                               # M^2 - m^2 - i M Gamma
            assert abs(D.real - (mass * mass - m * m)) < 1e-9 * mass * mass
            g = -D.imag / mass
            assert abs(g - gam) < 1e-10 * width
            assert abs(g * m / (mass * width) - (pR / pR0) ** (2 * LR + 1)) < 1e-11 * (pR / pR0) ** (2 * LR + 1)


# ------------------------------------------------------------------ P4: Blatt-Weisskopf polynomials = x^(2L+2) |h_L(x)|^2
def test_P4_barrier_polynomials_are_spherical_hankel_moduli():
    for L in range(5):
        for x in (0.05, 0.4, 1.0, 2.5, 7.0):
            h2 = special.spherical_jn(L, x) ** 2 + special.spherical_yn(L, x) ** 2
            ref = x ** (2 * L + 2) * h2
            assert abs(O.barrier_polynomial(L, x * x) - ref) < 1e-11 * ref, (L, x)
    for L in range(5):
        assert O.blatt_weisskopf(L, 321.0, 321.0, R16) == 1.0          # F(p0) = 1
        assert O.blatt_weisskopf(0, 100.0, 300.0, R16) == 1.0          # F^(0) = 1
        # monotone: F decreases with p for L > 0; limit F -> (p0/p)^L (B_L(z0)/z0^L)^(1/2) ... ratio check at r -> 0
        if L:
            assert O.blatt_weisskopf(L, 400.0, 300.0, R16) < 1.0 < O.blatt_weisskopf(L, 200.0, 300.0, R16)
            assert abs(O.blatt_weisskopf(L, 400.0, 300.0, 1e-9) - 1.0) < 1e-9


def _hankel_B(L, x):
    """x^(2L+2) |h_L^(1)(x)|^2 from scipy's spherical Bessel functions: the Blatt-Weisskopf polynomial B_L(x^2) (pin P4)"""
    return x ** (2 * L + 2) * (special.spherical_jn(L, x) ** 2 + special.spherical_yn(L, x) ** 2)


# ------------------------------------------------------------------ P4b: the barrier FACTOR at r != 0 (square root, normalisation)
def test_P4b_blatt_weisskopf_factor_at_finite_radius():
    """F^(L)(p, p0) = sqrt(B_L(z0)/B_L(z)) (reading A2) with B_L from scipy's spherical Hankel functions, at the
    radii and momenta of the configs; for L = 1 also the textbook closed form sqrt((1 + z0)/(1 + z)).  A missing square root, a
    swapped (p, p0) or z = r p instead of (r p)^2 fails here (at r = 1.6e-3, p ~ 300-1500 MeV: z = 0.2-6, nowhere near 1)."""
    for r in (R16, 3.0e-3):
        for L in range(5):
            for p, p0 in ((291.0, 642.0), (642.0, 291.0), (1204.0, 88.0), (35.0, 1377.0)):
                ref = math.sqrt(_hankel_B(L, r * p0) / _hankel_B(L, r * p))
                got = O.blatt_weisskopf(L, p, p0, r)
                assert abs(got - ref) < 1e-12 * ref, (L, p, p0, r, got, ref)
                if L == 1:
                    z, z0 = (r * p) ** 2, (r * p0) ** 2
                    assert abs(got - math.sqrt((1 + z0) / (1 + z))) < 1e-14 * got
                if L:
                    assert abs(got * got - ref) > 1e-3 * ref          # the square root is not optional at these momenta


# ------------------------------------------------------------------ P3c: Eqs. 2-3 at r != 0 from the complex output alone
@pytest.mark.parametrize("radius", [R16, 3.0e-3])
def test_P3c_barrier_factors_in_numerator_and_running_width(radius):
    """A = num / (M^2 - m^2 - i M Gamma(m)) with num real, so 1/A gives both back without any model input:
    num = (M^2 - m^2)/Re(1/A) and Gamma(m) = -Im(1/A) num / M.  Then, with B_L from scipy's Hankel functions (pin P4),
        Gamma(m) m / (M Gamma0 (p_R/p_R0)^(2 L_R + 1)) = B_LR(z_R0)/B_LR(z_R)                  [F_R SQUARED in Eq. 3, PAPER.md:94]
        num / ((p_B/M_B)^L_B (p_R/m)^L_R) = sqrt(B_LB(z_B0)/B_LB(z_B)) sqrt(B_LR(z_R0)/B_LR(z_R)) [F_B F_R in Eq. 2, PAPER.md:89]
    for every resonance of the full model off the pole.  Dropping F_B or F_R from the numerator, F_R instead of F_R^2 in the
    width, or a barrier factor without its square root each fail one of the two lines."""
    res = [(k, J, m, w, radius) for (k, J, m, w, _) in W.resonances(2)]
    M = O.Model(DEC, res)
    for r, (kind, J, mass, width, rad) in enumerate(res):
        LB, LR = O.orbital_L(kind, J)
        if kind == O.KSTAR:
            mom = lambda m: (O.breakup_momentum(MB, m, MPSI), O.breakup_momentum(m, MK, MPI))
            lo, hi = MK + MPI + 5, MB - MPSI - 5
        else:
            mom = lambda m: (O.breakup_momentum(MB, m, MK), O.breakup_momentum(m, MPSI, MPI))
            lo, hi = MPSI + MPI + 5, MB - MK - 5
        pB0, pR0 = mom(mass)
        for m in np.linspace(lo, hi, 9):
            if abs(m - mass) < 1.0:
                continue
            A, gam = M.lineshape(r, m)
            inv = 1.0 / A
            num = (mass * mass - m * m) / inv.real
            g = -inv.imag * num / mass
            assert abs(g - gam) < 1e-9 * abs(gam)
            pB, pR = mom(m)
            ratioR = _hankel_B(LR, radius * pR0) / _hankel_B(LR, radius * pR)
            ratioB = _hankel_B(LB, radius * pB0) / _hankel_B(LB, radius * pB)
            lhs_w = g * m / (mass * width * (pR / pR0) ** (2 * LR + 1))
            assert abs(lhs_w - ratioR) < 1e-9 * ratioR, (r, m, lhs_w, ratioR)
            lhs_n = num / ((pB / MB) ** LB * (pR / m) ** LR)
            assert abs(lhs_n - math.sqrt(ratioB * ratioR)) < 1e-9 * lhs_n, (r, m, lhs_n, math.sqrt(ratioB * ratioR))
        # the factors are not trivially 1 for this resonance (else the two lines above pin nothing); L = 0 factors are 1
        pB, pR = mom(0.5 * (lo + mass) if mass - lo > 50 else 0.5 * (hi + mass))
        if LB:
            assert abs(_hankel_B(LB, radius * pB0) / _hankel_B(LB, radius * pB) - 1.0) > 1e-3


# ------------------------------------------------------------------ P5: kinematic invariants
def test_P5_kinematic_invariants():
    M = model(2)
    rng = np.random.default_rng(5)
    x = W.phase_space_events(rng, 300)
    for i in range(x.shape[1]):
        k = M.z_kinematics(x[:, i])
        K, pi, psi = k["K_B"], k["pi_B"], k["psi_B"]
        tot = K + pi + psi
        assert abs(tot[0] - MB) < 1e-9 and np.abs(tot[1:]).max() < 1e-9          # 4-momentum conservation
        m2 = lambda p: p[0] ** 2 - p[1:] @ p[1:]
        assert abs(m2(K) - MK ** 2) < 1e-6 and abs(m2(pi) - MPI ** 2) < 1e-6 and abs(m2(psi) - MPSI ** 2) < 1e-5
        assert abs(math.sqrt(m2(K + pi)) - x[0, i]) < 1e-9
        s_kpi, s_psipi, s_psik = m2(K + pi), m2(psi + pi), m2(psi + K)
        assert abs(s_kpi + s_psipi + s_psik - (MB ** 2 + MPSI ** 2 + MK ** 2 + MPI ** 2)) < 1e-6   # Dalitz identity
        assert abs(k["mZ"] - math.sqrt(s_psipi)) < 1e-9
        assert MPSI + MPI <= k["mZ"] <= MB - MK
        assert abs(k["cosZ"] ** 2 + k["sinZ"] ** 2 - 1) < 1e-12 and k["sinZ"] >= 0
        assert abs(k["cosT"] ** 2 + k["sinT"] ** 2 - 1) < 1e-12 and k["sinT"] >= 0
        # the helicity angle of the K in the K pi frame is recovered from B-frame invariants:
        # m_psipi^2 is linear in cos theta_K* with slope -2 q pB MB / m  (two-body kinematics)
        pB, q = O.breakup_momentum(MB, x[0, i], MPSI), O.breakup_momentum(x[0, i], MK, MPI)
        k0 = M.z_kinematics([x[0, i], 0.0, x[2, i], x[3, i]])
        slope = (k["mZ"] ** 2 - k0["mZ"] ** 2) / x[1, i]
        assert abs(slope + 2 * q * pB * MB / x[0, i]) < 1e-7 * abs(slope)
    # independent of (cos theta_psi, phi): the Z mass and theta_Z only depend on the hadronic variables
    a, b = M.z_kinematics([1200.0, 0.3, 0.5, 1.0]), M.z_kinematics([1200.0, 0.3, -0.7, -2.0])
    assert abs(a["mZ"] - b["mZ"]) < 1e-10 and abs(a["cosZ"] - b["cosZ"]) < 1e-13


# ------------------------------------------------------------------ P6: theta_Z from Lorentz invariants
def test_P6_theta_Z_from_invariants():
    """cos theta_Z via Lorentz invariants only (energies in the Z frame from two-body kinematics, p_K.p_pi
    from m_Kpi) must agree with the oracle's explicit boosts; sin theta_Z via the Gram determinant."""
    M = model(2)
    x = W.phase_space_events(np.random.default_rng(6), 500)
    for i in range(x.shape[1]):
        m, cK = x[0, i], x[1, i]
        k = M.z_kinematics(x[:, i])
        mZ = k["mZ"]
        EK, Epi = (MB ** 2 - mZ ** 2 - MK ** 2) / (2 * mZ), (mZ ** 2 + MPI ** 2 - MPSI ** 2) / (2 * mZ)
        pK, ppi = math.sqrt(EK ** 2 - MK ** 2), math.sqrt(Epi ** 2 - MPI ** 2)
        cZ = (EK * Epi - (m * m - MK ** 2 - MPI ** 2) / 2) / (pK * ppi)
        assert abs(cZ - k["cosZ"]) < 5e-11
        pB, q = O.breakup_momentum(MB, m, MPSI), O.breakup_momentum(m, MK, MPI)
        sZ = MB * q * pB * math.sqrt((1 - cK) * (1 + cK)) / (mZ * pK * ppi)
        assert abs(sZ - k["sinZ"]) < 5e-11


# ------------------------------------------------------------------ P7: rotation-composition identity
def test_P7_rotation_composition_pins_Z_angles():
    """The J/psi helicity state quantised along n_K* (K* chain, Eq. 4) re-expressed along n_pi (Z chain, Eq. 10):
    sum_l d^1_{l l'}(beta) e^{i l phi} d^1_{l xi}(theta_psi) = e^{i l' phi~} d^1_{l' xi}(theta~) e^{i xi alpha},
    beta the rotation angle about y from n_K* to n_pi.  Fixes theta~, phi~, alpha and the sign in e^{+i xi alpha};
    flipping any of those signs breaks it at O(1)."""
    M = model(2)
    x = W.phase_space_events(np.random.default_rng(7), 200)
    d1 = lambda a, b, ang: O.wigner_d(1, a, b, ang)
    worst, worst_flip = 0.0, [10.0, 10.0, 10.0]
    for i in range(x.shape[1]):
        m, cK, cpsi, phi = x[:, i]
        k = M.z_kinematics(x[:, i])
        # the frame (x, y, z = n_K*) of reading A7/A8: everything hadronic lies in the x-z plane, K on the +x side
        ez = k["nKst"]
        ex = k["nK"] - (k["nK"] @ ez) * ez
        ex /= np.linalg.norm(ex)
        ey = np.cross(ez, ex)
        assert abs(k["npi"] @ ey) < 1e-12 and k["nK"] @ ex > 0
        spsi = math.sqrt(1 - cpsi * cpsi)
        assert np.allclose(k["nmu"], spsi * math.cos(phi) * ex + spsi * math.sin(phi) * ey + cpsi * ez, atol=1e-13)
        beta = math.atan2(k["npi"] @ ex, k["npi"] @ ez)
        th, tht = math.acos(cpsi), math.atan2(k["sinT"], k["cosT"])
        for lp in (-1, 0, 1):
            for xi in (-1, 1):
                lhs = sum(d1(l, lp, beta) * np.exp(1j * l * phi) * d1(l, xi, th) for l in (-1, 0, 1))
                f = lambda s1, s2: np.exp(1j * lp * s1 * k["phiT"]) * d1(lp, xi, tht) * np.exp(1j * xi * s2 * k["alpha"])
                worst = max(worst, abs(lhs - f(1, 1)))
                if lp:
                    for j, (s1, s2) in enumerate([(-1, 1), (1, -1), (-1, -1)]):
                        worst_flip[j] = min(worst_flip[j], 10.0) if abs(lhs - f(s1, s2)) > 0.05 else 0.0
    assert worst < 1e-13
    # the three other sign choices fail for (almost) every event
    for j, (s1, s2) in enumerate([(-1, 1), (1, -1), (-1, -1)]):
        bad = 0
        for i in range(50):
            m, cK, cpsi, phi = x[:, i]
            k = M.z_kinematics(x[:, i])
            beta = math.atan2(k["npi"][0], k["npi"][2])
            th, tht = math.acos(cpsi), math.atan2(k["sinT"], k["cosT"])
            lhs = sum(d1(l, 1, beta) * np.exp(1j * l * phi) * d1(l, 1, th) for l in (-1, 0, 1))
            rhs = np.exp(1j * s1 * k["phiT"]) * d1(1, 1, tht) * np.exp(1j * s2 * k["alpha"])
            bad += abs(lhs - rhs) > 1e-3
        assert bad > 40


# ------------------------------------------------------------------ helpers: tensor quadrature grid as weighted "norm events"
def quadrature_events(nm, ncK, ncpsi, nphi, m_lo=None, m_hi=None):
    m_lo = MK + MPI if m_lo is None else m_lo
    m_hi = MB - MPSI if m_hi is None else m_hi
    xm, wm = npleg.leggauss(nm)
    mm = 0.5 * (m_hi - m_lo) * xm + 0.5 * (m_hi + m_lo)
    wm = wm * 0.5 * (m_hi - m_lo)
    pq = np.array([O.breakup_momentum(MB, m, MPSI) * O.breakup_momentum(m, MK, MPI) for m in mm])
    xk, wk = npleg.leggauss(ncK)
    xp, wp = npleg.leggauss(ncpsi)
    ph = -np.pi + 2 * np.pi * (np.arange(nphi) + 0.5) / nphi
    G = np.meshgrid(mm, xk, xp, ph, indexing="ij")
    Wt = np.einsum("i,j,k,l->ijkl", wm * pq, wk, wp, np.full(nphi, 2 * np.pi / nphi))
    return np.stack([g.ravel() for g in G]), Wt.ravel()


# ------------------------------------------------------------------ P8: K*-only angular average; spin-0 normalisation
def test_P8_kstar_angular_average_closed_form():
    """<S>_angles = (2/3) sum_lambda sum_J |sum_{R in J} H^R_lambda A^R(m)|^2 / (2J+1) (orthogonality of the d's),
    checked per mass point on a Gauss-Legendre x uniform grid — pins Eq. 4/5's angular structure, the slot order
    and which sums are coherent."""
    res = W.resonances(1)
    M = model(1)
    c = W.couplings(1)
    slots = W.slot_table(res)
    xk, wk = npleg.leggauss(8)
    xp, wp = npleg.leggauss(4)
    nphi = 8
    ph = -np.pi + 2 * np.pi * (np.arange(nphi) + 0.5) / nphi
    for m in (700.0, 895.55, 1432.0, 1800.0, 2100.0):
        G = np.meshgrid([m], xk, xp, ph, indexing="ij")
        x = np.stack([g.ravel() for g in G])
        w = np.einsum("j,k,l->jkl", wk, wp, np.full(nphi, 2 * np.pi / nphi)).ravel()
        avg = np.sum(w * M.eval_events(c, x)) / np.sum(w)
        amp = {}
        for k, (r, lam) in enumerate(slots):
            amp[(res[r][1], lam)] = amp.get((res[r][1], lam), 0) + c[k] * M.lineshape(r, m)[0]
        ref = (2.0 / 3.0) * sum(abs(a) ** 2 / (2 * J + 1) for (J, lam), a in amp.items())
        assert abs(avg - ref) < 1e-13 * ref


def test_P8b_spin0_normalisation_vs_quadrature():
    """north_star pin: a single spin-0 resonance's MC normalisation against brute-force quadrature.
    I = (2/3) |H|^2 int |A(m)|^2 pB q dm / int pB q dm (scipy.integrate.quad on the oracle's pinned 1D pieces)
    against the oracle's weighted-event normalisation over a 4D tensor grid."""
    res = [(O.KSTAR, 0, 1425.0, 270.0, R16)]
    M = O.Model(DEC, res)
    H = 0.7 - 1.1j
    x, w = quadrature_events(512, 3, 3, 4)   # sqrt end-point behaviour of pB q: GL error ~ n^-3
    I4d = M.norm_integral(np.array([H]), x, w)[0]
    lo, hi = MK + MPI, MB - MPSI
    pq = lambda m: O.breakup_momentum(MB, m, MPSI) * O.breakup_momentum(m, MK, MPI)
    num = integrate.quad(lambda m: abs(M.lineshape(0, m)[0]) ** 2 * pq(m), lo, hi, epsabs=0, epsrel=1e-12, limit=400, points=[1425.0])[0]
    den = integrate.quad(pq, lo, hi, epsabs=0, epsrel=1e-12, limit=400)[0]
    ref = (2.0 / 3.0) * abs(H) ** 2 * num / den
    assert abs(I4d - ref) < 5e-8 * ref
    # and brute force: plain 4D midpoint rule in (m, cK, cpsi, phi), no Gauss weights
    n = 24
    mm = lo + (hi - lo) * (np.arange(400) + 0.5) / 400
    cc = -1 + 2 * (np.arange(n) + 0.5) / n
    G = np.meshgrid(mm, cc[::6], cc, [0.3], indexing="ij")
    xb = np.stack([g.ravel() for g in G])
    wb = np.array([pq(m) for m in xb[0]])
    Ib = M.norm_integral(np.array([H]), xb, wb)[0]
    assert abs(Ib - ref) < 2e-3 * ref


# ------------------------------------------------------------------ P9: Z-only integral over K*-chain phase space
def test_P9_z_only_phase_space_integral():
    """Z-only density integrated over the (m_Kpi, cosK, cospsi, phi) phase space equals (2/9) sum|H|^2 times the
    1D integral of |A^Z|^2 over m_psipi with the Z-chain phase-space weight — exercises m_psipi, theta~, phi~ and
    |d(theta_Z)| through the change of variables; and Z-only S does not depend on alpha."""
    res = [(O.ZRES, 1, 4196.0, 370.0, R16)]
    M = O.Model(DEC, res)
    H = np.array([0.8 * np.exp(0.4j), 1.3 * np.exp(-2.0j), 0.6 * np.exp(1.9j)])
    x, w = quadrature_events(64, 64, 4, 8)
    I = M.norm_integral(H, x, w)[0]
    pqZ = lambda mz: O.breakup_momentum(MB, mz, MK) * O.breakup_momentum(mz, MPSI, MPI)
    lo, hi = MPSI + MPI, MB - MK
    num = integrate.quad(lambda mz: abs(M.lineshape(0, mz)[0]) ** 2 * pqZ(mz), lo, hi, epsabs=0, epsrel=1e-11, limit=400)[0]
    den = integrate.quad(pqZ, lo, hi, epsabs=0, epsrel=1e-11, limit=400)[0]
    ref = (2.0 / 9.0) * np.sum(np.abs(H) ** 2) * num / den
    assert abs(I - ref) < 1e-5 * ref          # quadrature-limited (sqrt end points), converges with the grid
    # each helicity separately (catches a d^1_{0 lambda'} / d^1_{lambda' xi} mix-up that the sum hides)
    for l in range(3):
        Hl = np.zeros(3, complex)
        Hl[l] = 1.0
        Il = M.norm_integral(Hl, x, w)[0]
        assert abs(Il - (2.0 / 9.0) * num / den) < 1e-5 * Il


# ------------------------------------------------------------------ P10: c^H M c = direct sum
def test_P10_norm_matrix_quadratic_form():
    M = model(2)
    c = W.couplings(2)
    xn, wn = W.norm_events(2, 3000)
    Mat = M.norm_matrix(xn, wn)
    assert np.abs(Mat - Mat.conj().T).max() < 1e-16 * np.abs(Mat).max() + 1e-30
    assert np.linalg.eigvalsh(Mat).min() > -1e-14 * np.abs(Mat).max()
    direct = M.norm_integral(c, xn, wn)[0]
    quad = (c.conj() @ Mat @ c).real
    assert abs(quad - direct) < 1e-13 * direct


# ------------------------------------------------------------------ P11: invariances
def test_P11_invariances():
    M = model(2)
    c = W.couplings(2)
    xn, wn = W.norm_events(2, 2000)
    x, eff = xn[:, :500].copy(), wn[:500].copy()
    v = M.eval_events(c, x, eff)
    assert np.all(v > 0)
    assert np.allclose(M.eval_events(np.exp(0.77j) * c, x, eff), v, rtol=1e-13, atol=0)       # global phase
    assert np.allclose(M.eval_events(3.0 * c, x, eff), 9.0 * v, rtol=1e-13, atol=0)
    nll0 = M.nll(c, x, eff, xn, wn)[0][0]
    nll1 = M.nll((0.3 - 2.0j) * c, x, eff, xn, wn)[0][0]
    assert abs(nll0 - nll1) < 1e-12 * abs(nll0)
    x2 = x.copy()
    x2[3] += 2 * np.pi
    assert np.allclose(M.eval_events(c, x2, eff), v, rtol=1e-12, atol=0)                      # periodic in phi
    # K*-only with all H_{+-1} = 0: no phi dependence at all
    M1, c1 = model(1), W.couplings(1).copy()
    for k, (r, lam) in enumerate(W.slot_table(W.resonances(1))):
        if lam:
            c1[k] = 0
    x3 = x.copy()
    x3[3] = np.random.default_rng(1).uniform(-np.pi, np.pi, x.shape[1])
    assert np.allclose(M1.eval_events(c1, x3), M1.eval_events(c1, x), rtol=1e-13, atol=0)
    # Z-only: S independent of alpha is equivalent to: S(xi=+1)+S(xi=-1) unchanged under phi -> shifts that keep
    # theta~, phi~ fixed — checked through the basis: |B_{k,xi}| carries no alpha
    B = M.basis_terms(x[:, 0])
    kZ = [k for k, (r, lam) in enumerate(W.slot_table(W.resonances(2))) if W.resonances(2)[r][0] == O.ZRES]
    k0 = M.z_kinematics(x[:, 0])
    for k, lp in zip(kZ, (-1, 0, 1)):
        for ix, xi in enumerate((1, -1)):
            expect = B[k, ix] * np.exp(-1j * xi * k0["alpha"]) * np.exp(-1j * lp * k0["phiT"])
            ratio = expect / M.lineshape(10, k0["mZ"])[0]
            assert abs(ratio.imag) < 1e-13                                # what is left is real: d * d


# ------------------------------------------------------------------ P12: PDF properties, summation, closure
def test_P12_normalisation_and_exact_summation():
    M = model(1)
    c = W.couplings(1)
    xn, wn = W.norm_events(1, 4000)
    I = M.norm_integral(c, xn, wn)[0]
    S = M.eval_events(c, xn)                      # eff = 1 -> S_j
    assert np.all(S >= 0)
    assert abs(math.fsum(wn * S / I) / math.fsum(wn) - 1.0) < 1e-13
    x, eff = xn[:, :1500], wn[:1500]
    nll = M.nll(c, x, eff, xn, wn)[0][0]
    v = M.eval_events(c, x, eff)
    ref = -math.fsum(math.log(vi / I) for vi in v)   # exactly rounded sum of the same terms
    assert abs(nll - ref) < 1e-13 * abs(ref)
    # long double twin agrees
    nllL = M.nll(c, x, eff, xn, wn, prec=1)[0][0]
    assert abs(nll - nllL) < 1e-12 * abs(nll)


def test_P12b_closure_true_parameters_beat_wrong_ones():
    cfg = 0
    M = model(cfg)
    c = W.couplings(cfg)
    xn, wn = W.norm_events(cfg, 20000)
    x, eff = W.data_events(cfg, lambda xx, ee: M.eval_events(c, xx, ee), n=4000)
    nll_true = M.nll(c, x, eff, xn, wn)[0][0]
    rng = np.random.default_rng(3)
    for _ in range(4):
        c2 = c.copy()
        c2[:3] *= 1 + 0.5 * rng.uniform(-1, 1, 3)
        c2[:3] *= np.exp(1j * rng.uniform(-1, 1, 3))
        assert M.nll(c2, x, eff, xn, wn)[0][0] > nll_true
    # and a wrong mass: K*(892) moved by one width
    mw = np.array([[[895.55 + 47.3, 47.3], [0, 0]]])
    assert M.nll(c, x, eff, xn, wn, mass_width=mw)[0][0] > nll_true + 100


def test_mass_width_override_equals_new_model():
    res = W.resonances(2)
    M = O.Model(DEC, res)
    c = W.couplings(2)
    xn, wn = W.norm_events(2, 500)
    mw = W.step_mass_width(3, 1)
    res2 = [(r[0], r[1], mw[i, 0], mw[i, 1], r[4]) for i, r in enumerate(res)]
    a = M.nll(c, xn[:, :100], wn[:100], xn, wn, mass_width=mw[None])[0][0]
    b = O.Model(DEC, res2).nll(c, xn[:, :100], wn[:100], xn, wn)[0][0]
    assert a == b


# ------------------------------------------------------------------ LASS S-wave, Eqs. 7-8
def test_P14_lass_lineshape():
    """Eqs. 7-8.  The oracle returns the sum of the two terms; they are separated by letting the width
    go to zero (the resonant term vanishes away from the pole).  Pins: (i) the effective-range term is (m/q) sin(th) e^{i th}
    with cot(th) = 1/(a q) + b q/2: modulus, phase, and the scattering-length limit A -> a m at threshold; (ii) the resonant
    term is 2 (m/q) e^{2 i th} sin(dR) e^{i dR} with tan(dR) = M0 Gamma(m)/(M0^2 - m^2) and Gamma(m) = Gamma0 (q/q0)(M0/m):
    modulus and phase, and its value 2 i e^{2 i th} M0/q0 at the pole; (iii) with the resonant term at HALF its printed
    strength the sum is the elastic-unitary amplitude (m/q) sin(th + dR) e^{i (th + dR)} — the form the 'similar
    parametrization' of LASS descends from — which fixes the relative phase e^{2 i th} and the running width together."""
    a, b = 1.95e-3, 1.76e-3
    M0, G0 = 1425.0, 270.0
    lass = O.Model(DEC, [(O.LASS, 0, M0, G0, R16)])
    bare = O.Model(DEC, [(O.LASS, 0, M0, 1e-30, R16)])
    q0 = O.breakup_momentum(M0, MK, MPI)
    assert lass.K == 1
    for m in (640.0, 700.0, 900.0, 1200.0, 1424.0, 1500.0, 1900.0, 2150.0):
        q = O.breakup_momentum(m, MK, MPI)
        th = math.atan2(1.0, 1.0 / (a * q) + 0.5 * b * q)
        A, gam = lass.lineshape(0, m)
        A1 = bare.lineshape(0, m)[0]
        assert abs(gam - G0 * (q / q0) * (M0 / m)) < 1e-12 * gam
        assert abs(abs(A1) * q / m - math.sin(th)) < 1e-13 and abs(np.angle(A1) - th) < 1e-13
        dR = math.atan2(M0 * gam, M0 * M0 - m * m)
        T2 = A - A1
        ref2 = 2.0 * (m / q) * np.exp(2j * th) * math.sin(dR) * np.exp(1j * dR)
        assert abs(T2 - ref2) < 1e-12 * abs(ref2)
        unitary = A1 + 0.5 * T2
        assert abs(unitary - (m / q) * math.sin(th + dR) * np.exp(1j * (th + dR))) < 1e-12 * abs(unitary)
        assert abs(unitary) * q / m <= 1.0 + 1e-12
    m_thr = MK + MPI + 1e-6
    q_thr = O.breakup_momentum(m_thr, MK, MPI)
    assert abs(bare.lineshape(0, m_thr)[0] - a * m_thr) < 2.0 * a * q_thr * a * m_thr   # scattering length: A = a m (1 + O(a q))
    qp = O.breakup_momentum(M0, MK, MPI)
    thp = math.atan2(1.0, 1.0 / (a * qp) + 0.5 * b * qp)
    Ap = lass.lineshape(0, M0)[0] - (M0 / qp) * math.sin(thp) * np.exp(1j * thp)   # (at the pole the resonant term survives width -> 0)
    assert abs(Ap - 2j * np.exp(2j * thp) * M0 / q0) < 1e-12 * abs(Ap)
    # in the model: one lambda = 0 slot with the J = 0 angular factor d^1_{0 xi}(theta_psi), Eq. 9
    x = np.array([1000.0, 0.3, -0.4, 1.1])
    B = lass.basis_terms(x)
    A1000 = lass.lineshape(0, 1000.0)[0]
    s = math.sqrt(1 - 0.16) / math.sqrt(2)
    assert abs(B[0, 0] - A1000 * s) < 1e-14 * abs(A1000) and abs(B[0, 1] + A1000 * s) < 1e-14 * abs(A1000)
    assert abs(lass.lineshape(0, 1000.0, prec=1)[0] - A1000) < 1e-13 * abs(A1000)


# ------------------------------------------------------------------ gradient of the NLL in the couplings
def test_P16_nll_gradient():
    """(i) central finite differences of the oracle's own NLL (an independent route: no derivative formula involved);
    (ii) Euler identities from pin P11: the NLL is invariant under c -> s c for any complex s, so
    sum_k conj(c_k) dNLL/dconj(c_k) = 0 exactly (real part: scale, imaginary part: global phase);
    (iii) at fixed normalisation events, the data term alone is homogeneous of degree -... checked through (ii) with n_norm >> n."""
    cfg = 2
    M = model(cfg)
    c = W.couplings(cfg)
    xn, wn = W.norm_events(cfg, 3000)
    x, eff = W.data_events(cfg, lambda xx, ee: M.eval_events(c, xx, ee), n=400)
    nll, g = M.nll_gradient(c, x, eff, xn, wn)
    assert abs(nll - M.nll(c, x, eff, xn, wn)[0][0]) < 1e-12 * abs(nll)
    gc = 0.5 * (g[:, 0] + 1j * g[:, 1])                       # dNLL/dconj(c_k)
    euler = np.sum(np.conj(c) * gc)
    assert abs(euler) < 1e-10 * np.sum(np.abs(c) * np.abs(gc))
    for k in (0, 4, 11, 24, 26):                              # J = 0 slot, K*(892) lambda = 0, a J = 2 slot, Z lambda' = -1, +1
        for part, d in ((0, 1.0), (1, 1j)):
            h = 1e-4 * max(abs(c[k]), 1.0)        # NLL ~ 1e4 to 1e-16 relative: rounding 1e-8, truncation O(h^2)
            cp, cm = c.copy(), c.copy()
            cp[k] += h * d
            cm[k] -= h * d
            fd = (M.nll(cp, x, eff, xn, wn)[0][0] - M.nll(cm, x, eff, xn, wn)[0][0]) / (2 * h)
            assert abs(fd - g[k, part]) < 1e-6 * np.abs(g).max(), (k, part, fd, g[k, part])


# ------------------------------------------------------------------ background and purity, Eq. 14
def test_P15_background_and_purity():
    """Eq. 14.  (i) purity 1 gives the signal-only NLL; (ii) a background with the signal's own shape,
    b_i = eps_i S_i / I, gives the signal-only NLL at ANY purity (fixes where I divides and that p weights the normalised
    signal); (iii) purity 0 gives -sum log b_i; (iv) f is linear in purity: exp(-NLL) per event interpolates — checked through
    the single-event case; (v) the mixture is a normalised density: sum_j w_j f(x_j) / sum_j w_j = 1 on the MC sample when b is
    normalised on it."""
    cfg = 2
    M = model(cfg)
    c = W.couplings(cfg)
    xn, wn = W.norm_events(cfg, 4000)
    x, eff = W.data_events(cfg, lambda xx, ee: M.eval_events(c, xx, ee), n=300)
    base, I = M.nll(c, x, eff, xn, wn)
    rng = np.random.default_rng(4)
    b = rng.uniform(0.2, 2.0, x.shape[1])
    assert abs(M.nll_background(c, x, eff, b, 1.0, xn, wn)[0] - base[0]) < 1e-12 * abs(base[0])
    b_sig = M.eval_events(c, x, eff) / I[0]
    for p in (0.15, 0.85):
        assert abs(M.nll_background(c, x, eff, b_sig, p, xn, wn)[0] - base[0]) < 1e-12 * abs(base[0])
    assert abs(M.nll_background(c, x, eff, b, 0.0, xn, wn)[0] + np.sum(np.log(b))) < 1e-12 * abs(np.sum(np.log(b)))
    x1, e1, b1 = x[:, :1], eff[:1], b[:1]
    f = lambda p: math.exp(-M.nll_background(c, x1, e1, b1, p, xn, wn)[0])
    assert abs(f(0.4) - (0.4 * f(1.0) + 0.6 * f(0.0))) < 1e-13 * f(0.4)
    # normalisation of the mixture on the MC sample: signal part integrates to 1 (pin P12), background given normalised
    bn = rng.uniform(0.5, 1.5, xn.shape[1])
    bn /= np.sum(wn * bn / wn) / xn.shape[1]                        # mean of b over the (uniform phase-space) sample = 1
    sig = M.eval_events(c, xn, None) / I[0]                         # S_j / I ; sum_j w_j S_j / I / sum w = 1
    mix = 0.85 * np.sum(wn * sig) / np.sum(wn) + 0.15 * np.mean(bn)
    assert abs(mix - 1.0) < 1e-12


# ------------------------------------------------------------------ fit fractions, Eq. 13
def test_P13_fit_fractions():
    """Eq. 13.  (i) a model with one resonance has FF = 1; (ii) on a full-angle quadrature grid with
    eps = 1 the interference between K* of different spin integrates to zero (orthogonality of the d^J, pin P2), so the
    fractions of the SPIN GROUPS add up to exactly 1 while the per-resonance fractions do not ("the sum of
    all the fit fractions is not constrained to 100%"); (iii) FF is invariant under a common rescaling of all couplings
    and linear in |H_j|^2 for the numerator alone."""
    xq, wq = quadrature_events(24, 6, 4, 8)
    one = O.Model(DEC, [W.resonances(1)[4]])
    assert abs(one.fit_fractions(np.array([0.3 + 0.1j, 1.0, -0.7j]), xq, wq)[0] - 1.0) < 1e-14
    res = W.resonances(1)
    M = model(1)
    c = W.couplings(1)
    ff = M.fit_fractions(c, xq, wq)
    assert np.all(ff > 0) and abs(ff.sum() - 1.0) > 1e-3                       # interference between same-spin K*
    groups = [[r for r, rr in enumerate(res) if rr[1] == J] for J in range(5)]
    ffJ = M.fit_fractions(c, xq, wq, groups=groups)
    assert abs(ffJ.sum() - 1.0) < 1e-12
    assert np.max(np.abs(M.fit_fractions((2.0 - 1.5j) * c, xq, wq) - ff)) < 1e-14
    slots = W.slot_table(res)
    c2 = np.array([2.0 * v if slots[k][0] == 4 else v for k, v in enumerate(c)])   # K2*(1430) amplitudes doubled
    I1, I2 = M.norm_integral(c, xq, wq)[0], M.norm_integral(c2, xq, wq)[0]
    assert abs(M.fit_fractions(c2, xq, wq)[4] * I2 - 4.0 * ff[4] * I1) < 1e-13 * ff[4] * I1


# ------------------------------------------------------------------ golden fixtures (tests/golden/)
GOLDEN = __import__("os").path.join(__import__("os").path.dirname(__import__("os").path.abspath(__file__)), "golden")


def test_golden_wigner_d_exact_values():
    """tests/golden/wigner_d_exact.txt: exact surd values of the PDG d-function table at pi/3 and pi/2 (hand-written
    expressions, evaluated here with math.sqrt) against the oracle's factorial sum."""
    n = 0
    for line in open(__import__("os").path.join(GOLDEN, "wigner_d_exact.txt")):
        if line.startswith("#") or not line.strip():
            continue
        j, mp, m, b, expr = line.split(None, 4)
        beta = eval(b, {"pi": math.pi})
        val = eval(expr, {"sqrt": math.sqrt})
        assert abs(O.wigner_d(int(j), int(mp), int(m), beta) - val) < 3e-16 + 1e-15 * abs(val), line
        n += 1
    assert n >= 20


def test_golden_oracle_regression():
    """tests/golden/oracle_regression.json (written by make_golden.py from oracle/ only): the oracle still gives the stored
    values — guards against silent drift of its arithmetic; correctness is pinned by P1-P12 above."""
    import json
    g = json.load(open(__import__("os").path.join(GOLDEN, "oracle_regression.json")))
    for cfg in (0, 1, 2):
        e = g["configs"][str(cfg)]
        Mo = model(cfg)
        c = W.couplings(cfg)
        xn, wn = W.norm_events(cfg, e["n_norm"])
        x, eff = W.data_events(cfg, lambda xx, ee: Mo.eval_events(c, xx, ee), n=e["n_data"])
        assert [float(t).hex() for t in x[:, 0]] == e["x0"]            # the seeded generators are unchanged
        v = Mo.eval_events(c, x, eff)
        ref = np.array([float.fromhex(t) for t in e["eps_S"]])
        assert np.max(np.abs(v[:12] - ref) / ref) < 1e-13
        B = Mo.basis_terms(x[:, 0]).ravel()
        Bref = np.array([complex(float.fromhex(a), float.fromhex(b)) for a, b in e["basis_terms_event0"]])
        assert np.max(np.abs(B - Bref)) < 1e-13 * np.max(np.abs(Bref))
        nll, integral = Mo.nll(c, x, eff, xn, wn)
        assert abs(nll[0] - float.fromhex(e["nll"])) < 1e-12 * abs(nll[0])
        assert abs(integral[0] - float.fromhex(e["integral"])) < 1e-13 * integral[0]


# ------------------------------------------------------------------ P17-P19: toy generator (oracle/toy.py)
def test_P17_philox_known_answers():
    """the counter-based generator against the publication's known-answer vectors (tests/golden/philox4x32_10_kat.txt)"""
    import os
    from oracle import toy
    rows = [l.split() for l in open(os.path.join(os.path.dirname(__file__), "golden", "philox4x32_10_kat.txt")) if l.strip() and not l.startswith("#")]
    assert len(rows) == 3
    for r in rows:
        v = [int(t, 16) for t in r]
        out = toy.philox4x32_10(np.array([v[0:4]], dtype=np.uint64), (v[4], v[5]))[0]
        assert [int(o) for o in out] == v[6:10]
    # vectorised call = row-by-row calls; distinct counters give distinct outputs
    ctr = np.array([[i, 7, j, 0] for i in range(5) for j in range(3)], dtype=np.uint64)
    allr = toy.philox4x32_10(ctr, (123, 456))
    for k in range(len(ctr)):
        assert np.array_equal(allr[k], toy.philox4x32_10(ctr[k:k + 1], (123, 456))[0])
    assert len({tuple(int(v) for v in r) for r in allr}) == len(ctr)


def test_P18_uniform53_range_and_resolution():
    from oracle import toy
    F = 0xFFFFFFFF
    assert toy.uniform53([0], [0])[0] == 0.0
    assert toy.uniform53([F], [F])[0] == 1.0 - 2.0 ** -53          # largest value: strictly below 1
    assert toy.uniform53([1 << 5], [0])[0] == 2.0 ** -27            # lowest kept bit of the first word
    assert toy.uniform53([0], [1 << 6])[0] == 2.0 ** -53            # lowest kept bit of the second word
    assert toy.uniform53([31], [63])[0] == 0.0                      # dropped bits
    # candidate map: ranges, and the stream does not depend on how it is cut into calls
    lo, hi, cm = MK + MPI + 1e-3, 2182.0, 1 - 1e-9
    x, u = toy.candidates(99, 0, 20000, lo, hi, cm)
    assert x[0].min() >= lo and x[0].max() < hi and np.abs(x[1:3]).max() <= cm and x[3].min() >= -np.pi and x[3].max() < np.pi
    assert u.min() >= 0 and u.max() < 1
    x2, u2 = toy.candidates(99, 5000, 100, lo, hi, cm)
    assert np.array_equal(x2, x[:, 5000:5100]) and np.array_equal(u2, u[5000:5100])
    xb, _ = toy.candidates(99 + (1 << 32), 0, 100, lo, hi, cm)      # the high seed word is part of the key
    assert not np.array_equal(xb, x[:, :100])
    # uniformity of each of the five streams and independence of neighbours (means, variances, lag-1 and cross correlations)
    U = np.vstack([(x[0] - lo) / (hi - lo), (x[1] / cm + 1) / 2, (x[2] / cm + 1) / 2, (x[3] / np.pi + 1) / 2, u])
    n = U.shape[1]
    assert np.all(np.abs(U.mean(1) - 0.5) < 5 * math.sqrt(1 / 12 / n))
    assert np.all(np.abs(U.var(1) - 1 / 12) < 5 * math.sqrt(1 / 180 / n))
    cc = np.corrcoef(U)
    assert np.all(np.abs(cc - np.eye(5)) < 5 / math.sqrt(n))
    for k in range(5):
        assert abs(np.corrcoef(U[k, :-1], U[k, 1:])[0, 1]) < 5 / math.sqrt(n)


def test_P19_toy_of_constant_spin0_model_follows_phase_space():
    """one constant spin-0 term: S = |c|^2 sum_xi |d^1_{0 xi}(theta_psi)|^2 = |c|^2 sin^2 theta_psi, so the accepted events follow
    p_B(m) q(m) in m_Kpi (compared with scipy quadrature of the textbook two-body momenta), (1 - c^2) in cos theta_psi,
    and are flat in cos theta_K* and phi"""
    from oracle import toy
    M = O.Model(DEC, [(W.CONST, 0, 0.0, 0.0, 0.0)])
    c = np.array([0.7 - 0.4j])
    lo, hi, cm = MK + MPI + 1e-3, 2182.0, 1 - 1e-9

    def pq(m):
        pB = math.sqrt((MB * MB - (m + MPSI) ** 2) * (MB * MB - (m - MPSI) ** 2)) / (2 * MB)
        q = math.sqrt((m * m - (MK + MPI) ** 2) * (m * m - (MK - MPI) ** 2)) / (2 * m)
        return pB * q

    grid = np.linspace(lo, hi, 20001)
    fmax = 1.0001 * abs(c[0]) ** 2 * max(pq(m) for m in grid)
    n = 300_000
    g = toy.generate(M, c, 4242, 0, n, fmax, lo, hi, cm)
    assert g["f_seen_max"] <= fmax
    x = g["x"]
    nacc = x.shape[1]
    # acceptance = mean f / f_max;  mean f = |c|^2 <pq> <sin^2> = |c|^2 * (int pq dm / (hi - lo)) * 2/3
    ipq = integrate.quad(pq, lo, hi, epsabs=0, epsrel=1e-10, limit=200)[0]
    p_acc = abs(c[0]) ** 2 * ipq / (hi - lo) * (2 / 3) / fmax
    assert abs(nacc - n * p_acc) < 5 * math.sqrt(n * p_acc * (1 - p_acc)), (nacc, n * p_acc)
    assert np.array_equal(x, toy.candidates(4242, 0, n, lo, hi, cm)[0][:, g["index"]])
    # m_Kpi histogram against the integral of p_B q per bin
    edges = np.linspace(lo, hi, 41)
    obs = np.histogram(x[0], edges)[0]
    exp = np.array([integrate.quad(pq, a, b, epsabs=0, epsrel=1e-10)[0] for a, b in zip(edges[:-1], edges[1:])]) / ipq * nacc
    chi2 = float(np.sum((obs - exp) ** 2 / exp))
    assert chi2 < 39 + 5 * math.sqrt(2 * 39), chi2
    # angular moments: <cos^2 theta_psi> = 1/5 for a sin^2 law, 1/3 for a flat one; phi flat
    assert abs(np.mean(x[2] ** 2) - 0.2) < 5 * math.sqrt((3 / 35 - 1 / 25) / nacc)
    assert abs(np.mean(x[1] ** 2) - 1 / 3) < 5 * math.sqrt((1 / 5 - 1 / 9) / nacc)
    assert abs(np.mean(x[1])) < 5 * math.sqrt(1 / 3 / nacc) and abs(np.mean(x[2])) < 5 * math.sqrt(0.2 / nacc)
    assert abs(np.mean(np.cos(x[3]))) < 5 * math.sqrt(0.5 / nacc) and abs(np.mean(np.cos(2 * x[3]))) < 5 * math.sqrt(0.5 / nacc)
    # a model WITH structure must not pass the flat-phi test: K*(892) with helicity +-1 couplings modulates cos(2 phi)
    M2 = O.Model(DEC, W.resonances(0))
    c2 = W.couplings(0)
    x2p, _ = toy.candidates(7, 0, 50_000, lo, hi, cm)
    f2 = toy.weights(M2, c2, x2p)
    g2 = toy.generate(M2, c2, 7, 0, 50_000, float(f2.max()), lo, hi, cm)
    assert g2["x"].shape[1] > 300
    # accepted events are denser where the weight is larger: mean weight of accepted = <f^2>/<f> > <f>
    assert np.mean(f2[g2["index"]]) > 1.5 * np.mean(f2)
    assert abs(np.mean(f2[g2["index"]]) / (np.mean(f2 ** 2) / np.mean(f2)) - 1) < 5 * math.sqrt(np.var(f2[g2["index"]]) / g2["x"].shape[1]) / np.mean(f2[g2["index"]])


# ------------------------------------------------------------------ P20: Z of any spin-parity (reading A24)
Z_CLASSES = [(O.ZRES, 1), (O.ZRES, 2), (O.ZNEG, 0), (O.ZNEG, 1), (O.ZNEG, 2)]


def test_P20_z_orbital_momenta_from_selection_rules():
    """L_B, L_R of each J^P by brute-force enumeration of the selection rules: L_B couples spin J and spin 0 to the B's spin 0;
    L_R couples the psi's spin 1 to J with parity P = P_psi P_pi (-1)^L = (-1)^L; the lowest allowed value is taken"""
    for kind, J in Z_CLASSES:
        P = +1 if kind == O.ZRES else -1
        LBs = [L for L in range(0, 8) if abs(L - J) <= 0 <= L + J]                     # |L - J| <= 0 <= L + J
        LRs = [L for L in range(0, 8) if abs(L - 1) <= J <= L + 1 and (-1) ** L == P]
        assert O.orbital_L(kind, J) == (min(LBs), min(LRs)), (kind, J)
    assert [L for L in range(0, 8) if abs(L - 1) <= 0 <= L + 1 and (-1) ** L == +1] == []   # 0+ -> psi pi is forbidden


@pytest.mark.parametrize("kind,J", Z_CLASSES)
def test_P20_z_spin_parity_lineshape_and_integral(kind, J):
    res = [(kind, J, 4196.0, 370.0, R16)]
    M = O.Model(DEC, res)
    LB, LR = O.orbital_L(kind, J)
    # pole: Gamma(M) = Gamma0 and A = (pB0/MB)^LB (pR0/M)^LR i/(M Gamma0) (the barrier factors are 1 at the pole)
    A, G = M.lineshape(0, 4196.0)
    pB0, pR0 = O.breakup_momentum(MB, 4196.0, MK), O.breakup_momentum(4196.0, MPSI, MPI)
    assert abs(G - 370.0) < 1e-12 * 370.0
    ref = (pB0 / MB) ** LB * (pR0 / 4196.0) ** LR * 1j / (4196.0 * 370.0)
    assert abs(A - ref) < 1e-13 * abs(ref)
    # threshold behaviour of the momentum powers: |A| ~ pR^LR near the psi pi threshold
    m1, m2 = MPSI + MPI + 0.02, MPSI + MPI + 0.08
    r = abs(M.lineshape(0, m2)[0]) / abs(M.lineshape(0, m1)[0])
    p1, p2 = O.breakup_momentum(m1, MPSI, MPI), O.breakup_momentum(m2, MPSI, MPI)
    assert abs(r - (p2 / p1) ** LR) < 2e-3 * r
    # phase-space integral of the Z-only density: (2/3) (1/(2J+1)) sum_{|l'| <= J} |H_l'|^2 <|A^Z|^2>  (orthogonality of the d's)
    H = np.array([0.8 * np.exp(0.4j), 1.3 * np.exp(-2.0j), 0.6 * np.exp(1.9j)])
    x, w = quadrature_events(64, 64, 4, 8)
    pqZ = lambda mz: O.breakup_momentum(MB, mz, MK) * O.breakup_momentum(mz, MPSI, MPI)
    lo, hi = MPSI + MPI, MB - MK
    num = integrate.quad(lambda mz: abs(M.lineshape(0, mz)[0]) ** 2 * pqZ(mz), lo, hi, epsabs=0, epsrel=1e-11, limit=400)[0]
    den = integrate.quad(pqZ, lo, hi, epsabs=0, epsrel=1e-11, limit=400)[0]
    for l in range(3):
        Hl = np.zeros(3, complex)
        Hl[l] = H[l]
        Il = M.norm_integral(Hl, x, w)[0]
        ref = (2.0 / 3.0) / (2 * J + 1) * abs(H[l]) ** 2 * num / den if abs(l - 1) <= J else 0.0
        assert abs(Il - ref) <= 2e-5 * max(ref, 1e-300), (l, Il, ref)
    # helicities do not interfere in the integral
    Iall = M.norm_integral(H, x, w)[0]
    assert abs(Iall - sum(M.norm_integral(np.where(np.arange(3) == l, H, 0), x, w)[0] for l in range(3))) < 1e-9 * Iall


def test_P20_spin0_z_density_closed_form():
    """0- Z alone: S = |H_0 A^Z(m_psipi)|^2 sin^2(theta~) — no dependence on theta_Z, phi~ or alpha; the lambda' = +-1 slots are inert"""
    M = O.Model(DEC, [(O.ZNEG, 0, 4196.0, 370.0, R16)])
    xn, _ = W.norm_events(2, 400)
    H = np.array([0.3 + 0.2j, 0.9 - 0.5j, -0.7j])
    S = M.eval_events(H, xn)
    for i in range(0, 400, 7):
        zk = M.z_kinematics(xn[:, i])
        A = M.lineshape(0, zk["mZ"])[0]
        ref = abs(H[1] * A) ** 2 * zk["sinT"] ** 2
        assert abs(S[i] - ref) < 1e-12 * ref
    assert np.array_equal(S, M.eval_events(np.array([0, H[1], 0]), xn))
    # spin 2: d^2_{00}(theta_Z)^2 sin^2(theta~) for lambda' = 0 alone (sympy value of the d function)
    from sympy import N
    from sympy.physics.quantum.spin import Rotation
    M2 = O.Model(DEC, [(O.ZRES, 2, 4196.0, 370.0, R16)])
    S2 = M2.eval_events(np.array([0, 1.0, 0]), xn)
    S2p = M2.eval_events(np.array([0, 0, 1.0]), xn)
    for i in range(0, 400, 41):
        zk = M2.z_kinematics(xn[:, i])
        A = M2.lineshape(0, zk["mZ"])[0]
        thZ, thT = math.atan2(zk["sinZ"], zk["cosZ"]), math.atan2(zk["sinT"], zk["cosT"])
        d200 = float(N(Rotation.d(2, 0, 0, thZ).doit(), 30))
        d201 = float(N(Rotation.d(2, 0, 1, thZ).doit(), 30))
        assert abs(S2[i] - abs(A) ** 2 * d200 ** 2 * zk["sinT"] ** 2) < 1e-11 * S2[i] + 1e-40
        d1p = sum(float(N(Rotation.d(1, 1, xi, thT).doit(), 30)) ** 2 for xi in (1, -1))
        assert abs(S2p[i] - abs(A) ** 2 * d201 ** 2 * d1p) < 1e-11 * S2p[i] + 1e-40


# ------------------------------------------------------------------ P21: gradient with background and purity (Eq. 14)
def test_P21_background_gradient():
    """(i) central finite differences of the plain-definition NLL of Eq. 14 (Model.nll_background: a different code path, python +
    fsum) in every coupling; (ii) purity 1: the signal-only gradient; (iii) a background of the signal's own shape leaves the NLL
    stationary in the overall scale of the couplings at any purity (Euler: sum_k conj(c_k) dNLL/dconj(c_k) = 0 still holds, since
    f is homogeneous of degree 0 in c)"""
    cfg = 2
    M = model(cfg)
    c = W.couplings(cfg)
    xn, wn = W.norm_events(cfg, 3000)
    x, eff = W.data_events(cfg, lambda xx, ee: M.eval_events(c, xx, ee), n=250)
    rng = np.random.default_rng(14)
    b = rng.uniform(0.2, 2.0, x.shape[1]) * np.mean(M.eval_events(c, x, eff)) / M.norm_integral(c, xn, wn)[0]
    for purity in (0.85, 0.4):
        nll, g = M.nll_gradient_background(c, x, eff, b, purity, xn, wn)
        assert abs(nll - M.nll_background(c, x, eff, b, purity, xn, wn)[0]) < 1e-12 * abs(nll)
        gmax = np.max(np.abs(g))
        for k in range(len(c)):
            for part, d in ((0, 1.0), (1, 1.0j)):
                h = 1e-4 * max(abs(c[k]), 0.1)
                cp, cm = c.copy(), c.copy()
                cp[k] += h * d
                cm[k] -= h * d
                fd = (M.nll_background(cp, x, eff, b, purity, xn, wn)[0] - M.nll_background(cm, x, eff, b, purity, xn, wn)[0]) / (2 * h)
                assert abs(fd - g[k, part]) < 2e-6 * gmax, (purity, k, part, fd, g[k, part])
        euler = np.sum(np.conj(c) * (g[:, 0] + 1j * g[:, 1]) / 2)
        assert abs(euler) < 1e-10 * gmax * np.max(np.abs(c))
    n1, g1 = M.nll_gradient_background(c, x, eff, b, 1.0, xn, wn)
    n0, g0 = M.nll_gradient(c, x, eff, xn, wn)
    assert abs(n1 - n0) < 1e-12 * abs(n0) and np.max(np.abs(g1 - g0)) < 1e-11 * np.max(np.abs(g0))


# ------------------------------------------------------------------ P22: orientation of theta_Z (reading A10)
def _boost(p, v):
    """4-vector p = (E, px, py, pz) seen from a frame that moves with velocity v (c = 1)"""
    v = np.asarray(v, float)
    v2 = v @ v
    g = 1.0 / math.sqrt(1.0 - v2)
    vp = v @ p[1:]
    return np.concatenate([[g * (p[0] - vp)], p[1:] + ((g - 1.0) * vp / v2 - g * p[0]) * v])


def test_P22_theta_Z_is_the_helicity_angle_of_the_psi_from_the_Z_line_of_flight():
    """Eq. 10's d^{J(Z)}_{0 lambda'}(theta_Z) is the Jacob-Wick two-body amplitude of a Z of helicity 0 (B and K are spinless)
    into a psi of helicity lambda': its angle is the polar angle of the psi, in the Z rest frame, from the Z's line of flight
    in the B frame.  There p_psi = -p_pi and the Z's line of flight is opposite to p_K, so that angle IS the literal
    'angle between K and pi momenta in the Z rest frame' and not its supplement."""
    M = model(2)
    x = W.phase_space_events(np.random.default_rng(22), 300)
    for i in range(x.shape[1]):
        k = M.z_kinematics(x[:, i])
        Z = k["psi_B"] + k["pi_B"]
        nZ = Z[1:] / np.linalg.norm(Z[1:])                       # the Z's line of flight in the B rest frame
        vZ = Z[1:] / Z[0]
        psi_Z, pi_Z, K_Z = _boost(k["psi_B"], vZ), _boost(k["pi_B"], vZ), _boost(k["K_B"], vZ)
        assert np.abs(psi_Z[1:] + pi_Z[1:]).max() < 1e-8         # Z rest frame: back to back
        assert np.linalg.norm(np.cross(K_Z[1:], nZ)) < 1e-9 * np.linalg.norm(K_Z[1:]) and K_Z[1:] @ nZ < 0
        c_hel = psi_Z[1:] @ nZ / np.linalg.norm(psi_Z[1:])
        assert abs(c_hel - k["cosZ"]) < 1e-11
        c_sup = pi_Z[1:] @ nZ / np.linalg.norm(pi_Z[1:])         # the supplement: the pion's polar angle
        assert abs(c_sup + k["cosZ"]) < 1e-11


@pytest.mark.parametrize("kind,J", [(O.ZRES, 1), (O.ZRES, 2), (O.ZNEG, 1), (O.ZNEG, 2)])
def test_P22_supplement_of_theta_Z_is_a_relabelling_of_the_couplings(kind, J):
    """Had the paper meant the supplement, d^J_{0 l'}(pi - theta) = (-1)^{J + l'} d^J_{0 l'}(theta): the density with couplings
    H_l' under one reading is the density with (-1)^{J + l'} H_l' under the other, K* interference included — the two readings
    span the same family of PDFs, with the same likelihood minimum, fit fractions and significances.  The Z basis terms are
    rebuilt here from the oracle's separately pinned pieces (lineshape P3/P20, d functions P1, angles P5-P7)."""
    res = W.resonances(1)[:4] + [(kind, J, 4196.0, 370.0, R16)]
    M = O.Model(DEC, res)
    K = M.K
    rng = np.random.default_rng(220 + J)
    c = rng.normal(size=K) + 1j * rng.normal(size=K)
    sign = np.array([(-1.0) ** (J + lp) for lp in (-1, 0, 1)])
    c_flip = c.copy()
    c_flip[K - 3:] *= sign
    x = W.phase_space_events(rng, 60)
    S, S_flip = M.eval_events(c, x), M.eval_events(c_flip, x)
    d = O.wigner_d
    for i in range(x.shape[1]):
        zk = M.z_kinematics(x[:, i])
        A = M.lineshape(len(res) - 1, zk["mZ"])[0]
        thZ, thT = math.atan2(zk["sinZ"], zk["cosZ"]), math.atan2(zk["sinT"], zk["cosT"])
        B = M.basis_terms(x[:, i])

        def z_terms(theta):
            return np.array([[A * d(J, 0, lp, theta) * np.exp(1j * lp * zk["phiT"]) * d(1, lp, xi, thT) * np.exp(1j * xi * zk["alpha"])
                              if abs(lp) <= J else 0.0 for xi in (1, -1)] for lp in (-1, 0, 1)])

        lit, sup = z_terms(thZ), z_terms(math.pi - thZ)
        scale = np.abs(lit).max()
        assert np.abs(B[K - 3:] - lit).max() < 1e-12 * scale      # the oracle's terms are Eq. 10 with the literal angle
        assert np.abs(sup - sign[:, None] * lit).max() < 1e-12 * scale
        Bs = B.copy()
        Bs[K - 3:] = sup
        S_sup = sum(abs(c @ Bs[:, j]) ** 2 for j in range(2))     # supplement reading, couplings c
        S_sup_flip = sum(abs(c_flip @ Bs[:, j]) ** 2 for j in range(2))
        assert abs(S_sup - S_flip[i]) < 1e-11 * S[i] and abs(S_sup_flip - S[i]) < 1e-11 * S[i]
    assert (np.abs(S - S_flip) / S).max() > 1e-3                   # the relabelling is not trivial: the sign matters at fixed H


# ------------------------------------------------------------------ P23: the K* branch of the basis terms (Eq. 4) and its frame relative to the Z's
def _sympy_d(j, mp, m, beta):
    """sympy's Wigner small-d (sympy.physics.quantum.spin.Rotation.d), its symbolic form compiled once per (j, m', m)"""
    return _sympy_d_function(j, mp, m)(beta)


def test_P23_kstar_basis_terms_are_eq4_with_library_d_functions():
    """Eq. 4: B_(R,lambda),xi = A^R(m) d^J_{lambda 0}(theta_K*) e^{i lambda phi} d^1_{lambda xi}(theta_psi), rebuilt in the
    test from the separately pinned lineshape (P3, P3c) and sympy's d functions (a few events) / the Legendre forms
    d^J_{+-1 0} = -+ sin P_J'(cos)/sqrt(J(J+1)), d^J_00 = P_J (numpy, more events), against the oracle's `basis_terms` for the full
    K* + Z model: slot order, the index order of d^J_{lambda 0}, the sign of the phi phase and the helicity index of d^1."""
    res = W.resonances(2)
    M = model(2)
    slots = W.slot_table(res)
    x = W.phase_space_events(np.random.default_rng(23), 40)
    for i in range(x.shape[1]):
        m, cK, cpsi, phi = x[:, i]
        thK, thpsi = math.acos(cK), math.acos(cpsi)
        B = M.basis_terms(x[:, i])
        for k, (r, lam) in enumerate(slots):
            kind, J = res[r][0], res[r][1]
            if kind != O.KSTAR:
                continue
            A = M.lineshape(r, m)[0]
            if i < 4:
                dJ = _sympy_d(J, lam, 0, thK)
                d1 = [_sympy_d(1, lam, xi, thpsi) for xi in (1, -1)]
            else:
                PJ = npleg.Legendre.basis(J)
                dJ = PJ(cK) if lam == 0 else -lam * math.sin(thK) * PJ.deriv()(cK) / math.sqrt(J * (J + 1))
                d1 = [{(1, 1): (1 + cpsi) / 2, (1, -1): (1 - cpsi) / 2, (-1, 1): (1 - cpsi) / 2, (-1, -1): (1 + cpsi) / 2,
                       (0, 1): math.sin(thpsi) / math.sqrt(2), (0, -1): -math.sin(thpsi) / math.sqrt(2)}[(lam, xi)] for xi in (1, -1)]   # PDG table
            for ix in range(2):
                ref = A * dJ * np.exp(1j * lam * phi) * d1[ix]
                assert abs(B[k, ix] - ref) < 1e-13 * abs(A), (i, k, r, lam, ix, B[k, ix], ref)


def test_P23_kstar_and_z_basis_terms_share_one_jpsi_frame():
    """Pin P7's rotation identity applied to the ORACLE'S OWN basis terms (PAPER.md:111 Eq. 4, :167 Eq. 10): the J/psi-side factor
    u_{lambda xi} = B_(K*,lambda),xi / (A^K* d^J_{lambda 0}(theta_K*)) of the K* chain, rotated by the spin-1 matrix of the rotation that
    takes the K* axes (z = n_K*) into the Z axes (z = n_pi), must equal the Z chain's v_{lambda' xi} = B_(Z,lambda'),xi / (A^Z
    d^1_{0 lambda'}(theta_Z)):   sum_lambda d^1_{lambda lambda'}(beta) u_{lambda xi} = v_{lambda' xi}.
    Fixes the sign of e^{i lambda phi} and the index order of d^J_{lambda 0} RELATIVE to the Z chain — what decides the K*-Z
    interference (Eq. 12).  Library d functions throughout (sympy); the oracle supplies only B, A and the angles."""
    res = [W.resonances(2)[i] for i in (1, 4, 6, 10)]           # K*(892) J=1, K2*(1430) J=2, K3*(1780) J=3, Z(4200)
    assert [r[1] for r in res] == [1, 2, 3, 1] and res[3][0] == O.ZRES
    M = O.Model(DEC, res)
    x = W.phase_space_events(np.random.default_rng(2323), 25)
    worst, wrong_phi, wrong_idx = 0.0, 0, 0
    for i in range(x.shape[1]):
        m, cK, cpsi, phi = x[:, i]
        zk = M.z_kinematics(x[:, i])
        B = M.basis_terms(x[:, i])
        thK, thZ = math.acos(cK), math.atan2(zk["sinZ"], zk["cosZ"])
        ez = zk["nKst"]
        ex = zk["nK"] - (zk["nK"] @ ez) * ez
        ex /= np.linalg.norm(ex)
        beta = math.atan2(zk["npi"] @ ex, zk["npi"] @ ez)
        AZ = M.lineshape(3, zk["mZ"])[0]
        v = np.array([[B[9 + lp + 1, ix] / (AZ * _sympy_d(1, 0, lp, thZ)) for ix in range(2)] for lp in (-1, 0, 1)])
        D = np.array([[_sympy_d(1, l, lp, beta) for lp in (-1, 0, 1)] for l in (-1, 0, 1)])          # D[l, lp]
        for r, J in ((0, 1), (1, 2), (2, 3)):
            A = M.lineshape(r, m)[0]
            u = np.array([[B[3 * r + l + 1, ix] / (A * _sympy_d(J, l, 0, thK)) for ix in range(2)] for l in (-1, 0, 1)])
            worst = max(worst, np.abs(D.T @ u - v).max())
            # what the two plausible mistakes would give: e^{-i lambda phi}, and d^J_{0 lambda} = (-1)^lambda d^J_{lambda 0}
            u_phi = np.conj(u * np.exp(-1j * np.array([-1, 0, 1])[:, None] * phi)) * np.exp(-1j * np.array([-1, 0, 1])[:, None] * phi)
            u_idx = u * np.array([-1.0, 1.0, -1.0])[:, None]
            wrong_phi += np.abs(D.T @ u_phi - v).max() > 1e-2
            wrong_idx += np.abs(D.T @ u_idx - v).max() > 1e-2
    assert worst < 1e-12, worst
    assert wrong_phi > 60 and wrong_idx > 60                      # of 75: either mistake breaks the identity at O(1)


def test_P23_kstar_phase_convention_changes_the_density_when_a_z_interferes():
    """The two K* conventions pinned by P23 are not relabellings once a Z is present at FIXED couplings: S rebuilt with
    e^{-i lambda phi} (or d^J_{0 lambda}) in the K* terms and the oracle's own Z terms differs from the oracle's S at O(10 %)."""
    res = W.resonances(2)
    M = model(2)
    c = W.couplings(2)
    slots = W.slot_table(res)
    x = W.phase_space_events(np.random.default_rng(233), 30)
    S = M.eval_events(c, x)
    lam = np.array([l for (_, l) in slots], dtype=float)
    isK = np.array([res[r][0] == O.KSTAR for (r, _) in slots])
    dphi, didx = [], []
    for i in range(x.shape[1]):
        B = M.basis_terms(x[:, i])
        assert abs(sum(abs(c @ B[:, j]) ** 2 for j in range(2)) - S[i]) < 1e-13 * S[i]      # Eq. 12 from the basis terms
        Bp = np.where(isK[:, None], B * np.exp(-2j * lam * x[3, i])[:, None], B)          # e^{i lambda phi} -> e^{-i lambda phi}
        Bi = np.where(isK[:, None], B * ((-1.0) ** lam)[:, None], B)                        # d^J_{lambda 0} -> d^J_{0 lambda}
        dphi.append(abs(sum(abs(c @ Bp[:, j]) ** 2 for j in range(2)) / S[i] - 1))
        didx.append(abs(sum(abs(c @ Bi[:, j]) ** 2 for j in range(2)) / S[i] - 1))
    assert np.median(dphi) > 1e-2 and np.median(didx) > 1e-2
