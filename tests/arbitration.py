"""Long-double arbitration for the GPU parity tests and seeded event samples at the ill-conditioned loci.

Where the method itself is ill-conditioned in FP64 — m_psipi within an MeV of m_psi + m_pi (the pion at rest in the Z frame) or of
m_B - m_K (the kaon at rest), and |cos| -> 1 — neither FP64 route is "the truth": the oracle's 80-bit `long double` twin is.  A
parity assertion there reads
    |GPU - long double| <= max(tol, 4 |double oracle - long double|)        (relative, per element)
i.e. the north_star tolerance holds wherever the FP64 oracle itself achieves it, and where it does not the GPU may be no more than
four times further from the truth than the oracle is, on that very element.  The worst element is reported with its event.
Holds none of the method's arithmetic: references come from oracle/, inputs are numbers.
"""
import numpy as np

from paper_2007_14931_b200 import workloads as W

MB, MPSI, MK, MPI = W.DECAY


def check(gpu, ref_double, ref_ld, tol, what, events=None, oracle_model=None, scale=None, factor=4.0):
    """assert the arbitrated bound element by element; returns (worst GPU error, worst double-oracle error)"""
    gpu, rd, rl = (np.asarray(a) for a in (gpu, ref_double, ref_ld))
    sc = np.abs(rl) if scale is None else np.broadcast_to(np.asarray(scale, dtype=np.float64), rl.shape)
    eg, eo = np.abs(gpu - rl) / sc, np.abs(rd - rl) / sc
    bound = np.maximum(tol, factor * eo)
    ratio = eg / bound
    i = int(np.argmax(ratio))
    msg = f"{what}: worst element {i}: |gpu - ld| = {eg.flat[i]:.3e}, |double oracle - ld| = {eo.flat[i]:.3e}, bound {bound.flat[i]:.3e}"
    if events is not None:
        x = np.asarray(events)[:, i % np.asarray(events).shape[1]]
        msg += f", event (m_Kpi, cosK, cosPsi, phi) = {tuple(float(v) for v in x)}"
        if oracle_model is not None:
            mz = oracle_model.z_kinematics(x, prec=1)["mZ"]
            msg += f", m_Z - m_psi - m_pi = {mz - MPSI - MPI:.6g} MeV, m_B - m_K - m_Z = {MB - MK - mz:.6g} MeV"
    assert ratio.flat[i] <= 1.0, msg
    return float(eg.max()), float(eo.max()), msg


def threshold_events(oracle_model, which, n, dmax, seed):
    """n seeded events whose m_psipi lies within dmax MeV of m_psi + m_pi (which = 0) or of m_B - m_K (which = 1), the other
    two variables uniform (|cos| <= COS_MAX).  m_psipi^2 is linear in cos theta_K* at fixed m_Kpi (pin P5), so the cosine that puts an
    event at a target m_psipi follows from two oracle evaluations; the threshold itself is reached at a single point of the
    Dalitz boundary (cos theta_K* = +1 resp. -1 at one m_Kpi), found by a golden-section search on the oracle's m_psipi."""
    rng = np.random.default_rng(np.random.SeedSequence([W.SEED, 7700 + which, int(seed)]))
    cb = W.COS_MAX if which == 0 else -W.COS_MAX
    sgn = 1.0 if which == 0 else -1.0
    thr = MPSI + MPI if which == 0 else MB - MK
    mz = lambda m, c: oracle_model.z_kinematics([m, c, 0.1, 0.2], prec=1)["mZ"]
    dist = lambda m: sgn * (mz(m, cb) - thr)                       # distance from the threshold along the boundary, >= 0
    lo, hi = MK + MPI + 1.0, W.M_HI
    g = (np.sqrt(5.0) - 1.0) / 2.0
    a, b = lo, hi
    for _ in range(80):
        c1, c2 = b - g * (b - a), a + g * (b - a)
        if dist(c1) < dist(c2):
            b = c2
        else:
            a = c1
    m_star = 0.5 * (a + b)
    d_star = dist(m_star)                                          # > 0: COS_MAX keeps the boundary a hair away from the threshold
    curv = max((dist(m_star + 1.0) - d_star), (dist(m_star - 1.0) - d_star))          # distance grows ~ curv (m - m*)^2
    out = []
    while len(out) < n:
        d_t = d_star + rng.uniform(0.0, 1.0) * max(dmax - d_star, 0.0)
        w = np.sqrt(max(d_t - d_star, 0.0) / curv)
        m = m_star + w * rng.uniform(-1.0, 1.0)
        if not (lo < m < hi):
            continue
        z0, z1 = mz(m, 0.0) ** 2, mz(m, cb) ** 2                    # linear in cos theta_K*
        tgt = (thr + sgn * d_t) ** 2
        cK = cb * (tgt - z0) / (z1 - z0)
        if abs(cK) > W.COS_MAX:
            continue
        out.append([m, cK, rng.uniform(-1, 1) * W.COS_MAX, rng.uniform(-np.pi, np.pi)])
    return np.array(out).T
