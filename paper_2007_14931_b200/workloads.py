"""Seeded synthetic inputs for BASELINE.json's five configs (recipe: DESIGN.md §"Input recipe").

This module serves both the oracle tests and the CUDA path and therefore holds NONE of the
method's arithmetic: it draws events, couplings, efficiencies and parameter points.  Anything
that needs the model density (accept-reject sampling of data events) takes it as a callback.
The only kinematics here is the two-body momentum that shapes the phase-space proposal density
(dm2_Kpi dm2_psipi = 4 M_B p_B q dm dcosK — the input distribution, not a model output).

The paper's pseudo-data are not public; these inputs stand in for them and take
their shapes: 4 FP64 variables per event, 1e4-1e6 data events, several 1e6 normalisation
points.
"""
import numpy as np

SEED = 2007014931
# m_B0, m_J/psi, m_K+, m_pi- in MeV (BASELINE.json configs[0])
DECAY = (5279.65, 3096.9, 493.677, 139.570)
RADIUS = 1.6e-3  # MeV^-1 (1.6 GeV^-1; reading A3)
KSTAR, ZRES, CONST, LASS, ZNEG = 0, 1, 2, 3, 4   # ZRES: a Z of positive parity (1+, 2+), ZNEG: of negative parity (0-, 1-, 2-)

# (name, kind, J, mass, width) — BASELINE.json configs[1], configs[2] for the Z
KSTARS = [
    ("kappa(800)", KSTAR, 0, 682.0, 547.0),
    ("K*(892)", KSTAR, 1, 895.55, 47.3),
    ("K*(1410)", KSTAR, 1, 1414.0, 232.0),
    ("K0*(1430)", KSTAR, 0, 1425.0, 270.0),
    ("K2*(1430)", KSTAR, 2, 1432.4, 109.0),
    ("K*(1680)", KSTAR, 1, 1717.0, 322.0),
    ("K3*(1780)", KSTAR, 3, 1776.0, 159.0),
    ("K0*(1950)", KSTAR, 0, 1945.0, 201.0),
    ("K2*(1980)", KSTAR, 2, 1973.0, 373.0),
    ("K4*(2045)", KSTAR, 4, 2045.0, 198.0),
]
ZPLUS = ("Z(4200)", ZRES, 1, 4196.0, 370.0)
Z_COUPLING_SCALE = 6.0   # |H^Z| scale so that the Z fit fraction is a few percent
CONST_SCALE = 0.05       # constant S-wave coupling = CONST_SCALE / (M Gamma) of K*(892): ~40 % of the rate (A13)

M_LO_MARGIN = 1e-3     # MeV above threshold (reading A17)
M_HI = 2182.0          # MeV (BASELINE.json configs[0]; reading A12)
COS_MAX = 1.0 - 1e-9   # |cos theta| cap (reading A17)

# data / normalisation sizes per config (cfg 3 is a sweep; its headline point is 2M / 10M)
SIZES = {0: (10_000, 100_000), 1: (200_000, 1_000_000), 2: (500_000, 2_000_000),
         3: (2_000_000, 10_000_000), 4: (2_000_000, 10_000_000)}


def _rng(cfg, purpose):
    tag = {"couplings": 0, "efficiency": 1, "norm": 2, "data": 3, "steps": 4}[purpose]
    return np.random.default_rng(np.random.SeedSequence([SEED, int(cfg), tag]))


def resonances(cfg):
    """[(kind, J, mass, width, radius)] of a config; cfg 0: K*(892) + constant S-wave (reading A13)."""
    if cfg == 0:
        k = KSTARS[1]
        return [(k[1], k[2], k[3], k[4], RADIUS), (CONST, 0, 0.0, 0.0, 0.0)]
    res = [(k[1], k[2], k[3], k[4], RADIUS) for k in KSTARS]
    if cfg >= 2:
        res.append((ZPLUS[1], ZPLUS[2], ZPLUS[3], ZPLUS[4], RADIUS))
    return res


def resonances_lass(with_z=True):
    """The paper's LASS variant of the model (Eq. 9): the low-mass K pi S-wave — kappa(800) and K0*(1430)
    — is replaced by ONE LASS term built on the K0*(1430) mass and width (Eq. 7); the other eight K* (and the Z) stay."""
    k1430 = KSTARS[3]
    res = [(LASS, 0, k1430[3], k1430[4], RADIUS)]
    res += [(k[1], k[2], k[3], k[4], RADIUS) for i, k in enumerate(KSTARS) if i not in (0, 3)]
    if with_z:
        res.append((ZPLUS[1], ZPLUS[2], ZPLUS[3], ZPLUS[4], RADIUS))
    return res


def couplings_lass(with_z=True):
    """seeded couplings of the LASS model: as `couplings`, the LASS amplitude scaled to the size of a Breit-Wigner peak
    (A_LASS is O(1-10), a K* lineshape O(1e-6)), Eq. 6 on K*(892), Eq. 11 on the Z"""
    res = resonances_lass(with_z)
    slots = slot_table(res)
    rng = np.random.default_rng(np.random.SeedSequence([SEED, 7, 0]))
    c = rng.uniform(0.5, 1.5, len(slots)) * np.exp(1j * rng.uniform(-np.pi, np.pi, len(slots)))
    for k, (r, lam) in enumerate(slots):
        if res[r][0] == LASS:
            c[k] *= 0.3 / (KSTARS[1][3] * KSTARS[1][4])
        if res[r][0] == KSTAR and abs(res[r][2] - KSTARS[1][3]) < 1e-9 and lam == 0:
            c[k] = 1.0
        if res[r][0] == ZRES:
            c[k] *= Z_COUPLING_SCALE
    for k, (r, lam) in enumerate(slots):
        if res[r][0] == ZRES and lam == +1:
            c[k] = c[k - 2]
    return c


def slot_table(res):
    """[(resonance index, lambda)] in coupling-slot order (include/amp.h: amp_num_couplings)."""
    slots = []
    for r, (kind, J, *_rest) in enumerate(res):
        if kind in (ZRES, ZNEG) or (kind == KSTAR and J >= 1):
            slots += [(r, -1), (r, 0), (r, +1)]
        else:
            slots += [(r, 0)]
    return slots


def couplings(cfg):
    """complex [K]: |H| ~ U[0.5,1.5], arg ~ U(-pi,pi) per slot, then Eq. 6 (K*(892) lambda=0 fixed to 1),
    Eq. 11 (H^Z_+1 = H^Z_-1 for 1+) and, for cfg 0, the constant term fixed to 0.05/(M Gamma) of K*(892)."""
    res = resonances(cfg)
    slots = slot_table(res)
    rng = _rng(min(cfg, 2), "couplings")      # cfg 3, 4 are cfg 2 scaled up
    c = rng.uniform(0.5, 1.5, len(slots)) * np.exp(1j * rng.uniform(-np.pi, np.pi, len(slots)))
    i892 = 0 if cfg == 0 else 1
    for k, (r, lam) in enumerate(slots):
        kind = res[r][0]
        if r == i892 and lam == 0:
            c[k] = 1.0                                    # Eq. 6
        if kind == CONST:
            c[k] = CONST_SCALE / (KSTARS[1][3] * KSTARS[1][4])    # reading A13
        if kind == ZRES:
            c[k] *= Z_COUPLING_SCALE
    for k, (r, lam) in enumerate(slots):
        if res[r][0] == ZRES and lam == +1:
            c[k] = c[k - 2]                               # Eq. 11: H_+1 = H_-1
    return c


def _legendre3(a, u):
    return a[0] + a[1] * u + a[2] * 0.5 * (3 * u * u - 1) + a[3] * 0.5 * (5 * u ** 3 - 3 * u)


def efficiency(cfg, x):
    """eps(x) for x SoA [4][n]: 1 for cfg 0, else a seeded product of four degree-3 Legendre series in the
    affine-mapped variables, clipped to [0.05, 1] (BASELINE.json configs[1])."""
    x = np.asarray(x, dtype=np.float64)
    if cfg == 0:
        return np.ones(x.shape[1])
    rng = _rng(1, "efficiency")
    a = rng.uniform(-0.08, 0.08, (4, 4))
    a[:, 0] = 0.85
    m_lo = DECAY[2] + DECAY[3]
    u = [2 * (x[0] - m_lo) / (M_HI - m_lo) - 1, x[1], x[2], x[3] / np.pi]
    e = np.ones(x.shape[1])
    for d in range(4):
        e = e * _legendre3(a[d], u[d])
    return np.clip(e, 0.05, 1.0)


def _two_body_momentum(M, a, b):
    return np.sqrt(np.maximum((M - (a + b)) * (M + (a + b)) * (M - (a - b)) * (M + (a - b)), 0.0)) / (2 * M)


def phase_space_events(rng, n):
    """x SoA [4][n] = (m_Kpi, cos theta_K*, cos theta_psi, phi) uniform over B -> psi K pi phase space:
    density in m proportional to p_B(m) q(m) on [m_K + m_pi + 1e-3, 2182] MeV (reading A15), cosines
    uniform in [-1, 1] capped at |c| <= 1 - 1e-9, phi uniform in [-pi, pi)."""
    MB, mpsi, mK, mpi = DECAY
    lo, hi = mK + mpi + M_LO_MARGIN, M_HI
    grid = np.linspace(lo, hi, 4001)
    fmax = 1.02 * np.max(_two_body_momentum(MB, grid, mpsi) * _two_body_momentum(grid, mK, mpi))
    m = np.empty(n)
    filled = 0
    while filled < n:
        k = int(1.7 * (n - filled)) + 64
        mm = rng.uniform(lo, hi, k)
        keep = mm[rng.uniform(0, fmax, k) < _two_body_momentum(MB, mm, mpsi) * _two_body_momentum(mm, mK, mpi)]
        take = min(len(keep), n - filled)
        m[filled:filled + take] = keep[:take]
        filled += take
    x = np.empty((4, n))
    x[0] = m
    x[1] = np.clip(rng.uniform(-1, 1, n), -COS_MAX, COS_MAX)
    x[2] = np.clip(rng.uniform(-1, 1, n), -COS_MAX, COS_MAX)
    x[3] = rng.uniform(-np.pi, np.pi, n)
    return x


def norm_events(cfg, m=None):
    """(x [4][m], w [m] = efficiency): the phase-space Monte Carlo sample of a config."""
    m = SIZES[cfg][1] if m is None else m
    x = phase_space_events(_rng(cfg, "norm"), m)
    return x, efficiency(cfg, x)


def _mass_proposal(rng, k):
    """m drawn from an equal mixture of the phase-space density and a truncated Cauchy peak at the K*(892)
    (a proposal shape only: it flattens the narrow peak so that accept-reject wastes fewer model evaluations);
    returns (m [k], ratio [k] = phase-space density / proposal density, up to a common constant)."""
    MB, mpsi, mK, mpi = DECAY
    lo, hi = mK + mpi + M_LO_MARGIN, M_HI
    M0, G0 = KSTARS[1][3], 0.5 * KSTARS[1][4]
    grid = np.linspace(lo, hi, 20001)
    fps = _two_body_momentum(MB, grid, mpsi) * _two_body_momentum(grid, mK, mpi)
    zps = np.sum(0.5 * (fps[1:] + fps[:-1])) * (grid[1] - grid[0])          # normalisation of the phase-space density
    a_lo, a_hi = np.arctan((lo - M0) / G0), np.arctan((hi - M0) / G0)
    n_ps = rng.binomial(k, 0.5)
    m = np.concatenate([phase_space_events(rng, n_ps)[0], M0 + G0 * np.tan(rng.uniform(a_lo, a_hi, k - n_ps))])
    m = m[rng.permutation(k)]
    g_ps = _two_body_momentum(MB, m, mpsi) * _two_body_momentum(m, mK, mpi) / zps
    g_c = (G0 / ((m - M0) ** 2 + G0 ** 2)) / (a_hi - a_lo)
    return m, g_ps / (0.5 * g_ps + 0.5 * g_c)


def _proposal_events(rng, k):
    m, ratio = _mass_proposal(rng, k)
    x = np.empty((4, k))
    x[0] = m
    x[1] = np.clip(rng.uniform(-1, 1, k), -COS_MAX, COS_MAX)
    x[2] = np.clip(rng.uniform(-1, 1, k), -COS_MAX, COS_MAX)
    x[3] = rng.uniform(-np.pi, np.pi, k)
    return x, ratio


def data_events(cfg, density, n=None, chunk=None):
    """(x [4][n], eff [n]) accept-reject sampled from eff * S over phase space.

    ``density(x, eff) -> eff(x) * S(x)`` for x SoA [4][k] is the model evaluation handed in by the caller
    (the oracle in tests; the product's amp_eval_events in bench.py, as the paper generates its pseudo-data
    with the fitter itself).  Proposals: angles uniform, m from `_mass_proposal`; a proposal is accepted
    with probability density * ratio / envelope, envelope = 1.5 x the maximum of density * ratio over a
    1e5-event pilot (values above the envelope are accepted with probability 1: the sample is a valid
    input either way)."""
    n = SIZES[cfg][0] if n is None else n
    rng = _rng(cfg, "data")
    pilot, ratio = _proposal_events(rng, 100_000)
    fmax = 1.5 * float(np.max(density(pilot, efficiency(cfg, pilot)) * ratio))
    chunk = chunk or int(max(100_000, min(2 * n, 4_000_000)))
    out, filled = np.empty((4, n)), 0
    while filled < n:
        xx, ratio = _proposal_events(rng, chunk)
        f = density(xx, efficiency(cfg, xx)) * ratio
        keep = xx[:, rng.uniform(0, fmax, chunk) < f]
        take = min(keep.shape[1], n - filled)
        out[:, filled:filled + take] = keep[:, :take]
        filled += take
    return out, efficiency(cfg, out)


def floating_resonances(cfg):
    """indices of resonances whose mass and width float: cfg 2: Z; cfg 3: all; cfg 4: Z + first four K* (A14)."""
    res = resonances(cfg)
    if cfg == 2:
        return [len(res) - 1]
    if cfg == 3:
        return list(range(len(res)))
    if cfg == 4:
        return [0, 1, 2, 3, len(res) - 1]
    return []


def step_mass_width(cfg, step):
    """[R][2] masses and widths of timed call `step`: floating ones moved by a seeded 1e-4 relative step
    (cfg 3 call pattern: every lineshape column is recomputed on every call)."""
    res = resonances(cfg)
    mw = np.array([[r[2], r[3]] for r in res], dtype=np.float64)
    rng = np.random.default_rng(np.random.SeedSequence([SEED, int(cfg), 4, int(step)]))
    for r in floating_resonances(cfg):
        mw[r] *= 1.0 + 1e-4 * rng.uniform(-1, 1, 2)
    return mw


def fit_parameters(cfg=4):
    """Polar fit parameters of cfg 4 (reading A14): theta [60], and a function theta -> (couplings [K],
    mass_width [R][2]).  46 K* moduli/phases (K*(892) lambda=0 fixed, Eq. 6), Z: |H_-1|, arg, |H_0|, arg
    (H_+1 tied by Eq. 11), Z mass and width, mass and width of the first four K*."""
    res = resonances(cfg)
    slots = slot_table(res)
    c0 = couplings(cfg)
    mw0 = np.array([[r[2], r[3]] for r in res], dtype=np.float64)
    free = []          # (kind, index) kind: 'mod', 'arg' on slot k; 'mass', 'width' on resonance r
    for k, (r, lam) in enumerate(slots):
        if res[r][0] == KSTAR and not (r == 1 and lam == 0):
            free += [("mod", k), ("arg", k)]
    for k, (r, lam) in enumerate(slots):
        if res[r][0] == ZRES and lam in (-1, 0):
            free += [("mod", k), ("arg", k)]
    zr = len(res) - 1
    free += [("mass", zr), ("width", zr)]
    for r in range(4):
        free += [("mass", r), ("width", r)]
    theta = np.array([abs(c0[i]) if t == "mod" else np.angle(c0[i]) if t == "arg" else mw0[i, 0] if t == "mass" else mw0[i, 1]
                      for t, i in free])

    def unpack(th):
        mod, arg, mw = np.abs(c0).copy(), np.angle(c0).copy(), mw0.copy()
        for v, (t, i) in zip(th, free):
            if t == "mod":
                mod[i] = v
            elif t == "arg":
                arg[i] = v
            elif t == "mass":
                mw[i, 0] = v
            else:
                mw[i, 1] = v
        c = mod * np.exp(1j * arg)
        for k, (r, lam) in enumerate(slots):
            if r == 1 and lam == 0:
                c[k] = 1.0                    # Eq. 6
            if res[r][0] == ZRES and lam == +1:
                c[k] = c[k - 2]               # Eq. 11
        return c, mw

    return theta, unpack, free


def fit_points(cfg=4, step=0):
    """(couplings [P][K] complex, mass_width [P][R][2]) for one MINUIT-style gradient step: the central
    point then theta_k +- h_k, h_k = 1e-4 max(|theta_k|, 1e-3) (reading A14); P = 2*60 + 1 = 121.
    `step` moves the central point by a seeded 1e-3 relative amount so successive calls differ."""
    theta, unpack, _free = fit_parameters(cfg)
    if step:
        rng = np.random.default_rng(np.random.SeedSequence([SEED, int(cfg), 4, int(step)]))
        theta = theta * (1.0 + 1e-3 * rng.uniform(-1, 1, theta.size))
    pts = [theta]
    for k in range(theta.size):
        h = 1e-4 * max(abs(theta[k]), 1e-3)
        for s in (+1, -1):
            t = theta.copy()
            t[k] += s * h
            pts.append(t)
    cs, mws = zip(*(unpack(t) for t in pts))
    return np.array(cs), np.array(mws)
