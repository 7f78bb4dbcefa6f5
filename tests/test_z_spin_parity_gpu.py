"""Z resonances of any spin-parity ("J(Z) is the spin of the Z", 314 "testing any combination of their spin-parity
values"): 1+, 2+ (kind AMP_Z), 0-, 1-, 2- (kind AMP_ZM) — alone with the ten K*, and mixed (two Zs of different
J^P).  Every evaluation path against the oracle: per-event density, fused NLL with moved lineshapes, analytic gradient (floating
and fixed lineshapes), a parameter batch (dense tensor-core path), the normalisation matrix and fit fractions."""
import numpy as np
import pytest

torch = pytest.importorskip("torch")

from oracle import oracle as O
from paper_2007_14931_b200 import workloads as W

pytestmark = pytest.mark.gpu

Z4200, Z4430 = (4196.0, 370.0), (4478.0, 181.0)
CLASSES = {"1+": (W.ZRES, 1), "2+": (W.ZRES, 2), "0-": (W.ZNEG, 0), "1-": (W.ZNEG, 1), "2-": (W.ZNEG, 2)}


def dev(a):
    return torch.as_tensor(np.ascontiguousarray(a), dtype=torch.float64).cuda()


def build(zs, seed):
    """ten K* + the listed Zs [(J^P name, (mass, width))]; couplings seeded, Eq. 11 applied per J^P"""
    res = [(k[1], k[2], k[3], k[4], W.RADIUS) for k in W.KSTARS]
    for name, (mass, width) in zs:
        kind, J = CLASSES[name]
        res.append((kind, J, mass, width, W.RADIUS))
    slots = W.slot_table(res)
    rng = np.random.default_rng(seed)
    c = rng.uniform(0.5, 1.5, len(slots)) * np.exp(1j * rng.uniform(-np.pi, np.pi, len(slots)))
    for k, (r, lam) in enumerate(slots):
        kind, J = res[r][0], res[r][1]
        if kind in (W.ZRES, W.ZNEG):
            # size: a few per cent of the rate whatever the momentum powers of the class (L_B = J, L_R)
            LB, LR = O.orbital_L(kind, J)
            c[k] *= 6.0 * (3.0 ** LB) * (6.0 ** LR)
            P = +1 if kind == W.ZRES else -1
            sign = -P * (-1) ** J                       # Eq. 11: H_l' = -P (-1)^J H_-l'
            if lam == +1:
                c[k] = sign * c[k - 2]
            if lam == 0 and sign < 0:
                c[k] = 0.0                              # H_0 = -H_0
    return res, c


MODELS = [[(n, Z4200)] for n in CLASSES] + [[("1+", Z4200), ("0-", Z4430)], [("2-", Z4200), ("1-", Z4430)], [("2+", Z4200), ("1+", Z4430), ("1+", (4300.0, 250.0))]]


@pytest.mark.parametrize("zs", MODELS, ids=lambda zs: "_".join(n for n, _ in zs))
def test_z_spin_parity_all_paths(zs):
    from paper_2007_14931_b200 import binding as B
    res, c = build(zs, 17 + len(zs))
    Mo, Mg = O.Model(W.DECAY, res), B.Model(W.DECAY, res)
    K, R = len(c), len(res)
    assert Mg.K == Mo.K == K
    n, m = 6001, 20_003
    xn, wn = W.norm_events(2, m)
    x, eff = W.data_events(2, lambda xx, ee: Mo.eval_events(c, xx, ee), n=n)
    Mg.load_events(dev(x), dev(eff))
    Mg.load_norm(dev(xn), dev(wn))
    Mg.set_params(c)
    v, vref = Mg.eval_events(0).cpu().numpy(), Mo.eval_events(c, x, eff)
    assert np.max(np.abs(v - vref) / vref) < 1e-11
    # the Z is a visible part of the density (the test would not see a wrong Z term otherwise)
    cK = c.copy()
    cK[24:] = 0
    assert np.max(np.abs(Mo.eval_events(cK, x, eff) - vref) / vref) > 0.05
    rng = np.random.default_rng(3)
    mw = np.array([[r[2], r[3]] for r in res]) * (1 + 2e-3 * rng.uniform(-1, 1, (R, 2)))
    Mg.set_params(c, mw[None])
    nll = Mg.nll()[0]
    only_1p = all(nm == "1+" for nm, _ in zs)
    assert Mg.last_call_stats()["norm_path"] == 4
    ref, refI = Mo.nll(c, x, eff, xn, wn, mass_width=mw[None])
    assert abs(nll - ref[0]) < 1e-9 * abs(ref[0])
    assert abs(Mg.norm_integral()[0] - refI[0]) < 1e-12 * refI[0]
    # analytic gradient, lineshapes just moved (both samples walked) and then fixed (normalisation side from the matrix M)
    res2 = [(r[0], r[1], mw[i, 0], mw[i, 1], r[4]) for i, r in enumerate(res)]
    Mo2 = O.Model(W.DECAY, res2)
    nllg, g = Mg.nll_grad()
    rn, rg = Mo2.nll_gradient(c, x, eff, xn, wn)
    assert abs(nllg - rn) < 1e-9 * abs(rn)
    assert np.max(np.abs(g - rg)) < 1e-9 * np.max(np.abs(rg))
    c2 = c * (1 + 0.03 * np.cos(np.arange(K)))
    Mg.set_params(c2, mw[None])
    nllg, g = Mg.nll_grad()
    rn, rg = Mo2.nll_gradient(c2, x, eff, xn, wn)
    assert abs(nllg - rn) < 1e-9 * abs(rn)
    assert np.max(np.abs(g - rg)) < 1e-9 * np.max(np.abs(rg))
    # a parameter batch: couplings and lineshapes of the Z (and two K*) move
    zslots = [k for k, (r, lam) in enumerate(W.slot_table(res)) if res[r][0] in (W.ZRES, W.ZNEG)]
    P = 1 + 2 * len(zslots) + 2 * (R - 10) + 4
    cs, mws = np.tile(c, (P, 1)), np.tile(mw, (P, 1, 1))
    p = 1
    for k in zslots:
        cs[p, k] = cs[p, k] * (1 + 1e-3) + 1e-3; p += 1
        cs[p, k] = cs[p, k] * np.exp(-1e-3j) - 1e-3j; p += 1
    for r in list(range(10, R)) + [1, 4]:
        mws[p, r, 0] *= 1 + 1e-4
        mws[p + 1, r, 1] *= 1 - 1e-4
        p += 2
    assert p == P
    Mg.set_params(cs, mws)
    nb = Mg.nll()
    path = Mg.last_call_stats()["norm_path"]
    assert path in (5, 9) if only_1p else path in (1, 2, 3), path   # 1+ Zs: a gradient-batch kernel (9: the paper's shape); other spin-parities: dense path
    rb, rI = Mo.nll(cs, x, eff, xn, wn, mass_width=mws)
    assert np.max(np.abs(nb - rb) / np.abs(rb)) < 1e-9
    assert np.max(np.abs(Mg.norm_integral() - rI) / rI) < 1e-12
    # normalisation matrix (FP64 tensor-core Gram kernel) and fit fractions (Eq. 13)
    Mg.set_norm_mode(2)
    Mg.set_params(c)
    nll_m = Mg.nll()[0]
    ref0 = Mo.nll(c, x, eff, xn, wn)[0][0]
    assert abs(nll_m - ref0) < 1e-9 * abs(ref0)
    ff = Mg.fit_fractions(0)
    ffo = Mo.fit_fractions(c, xn, wn)
    assert np.max(np.abs(ff - ffo)) < 1e-11
    assert all(ff[r] > 1e-4 for r in range(10, R)), ff[10:]


def test_zero_plus_z_is_rejected():
    from paper_2007_14931_b200 import binding as B
    for kind, J in [(W.ZRES, 0), (W.ZRES, 3), (W.ZNEG, 3), (W.ZNEG, -1)]:
        with pytest.raises(Exception):
            B.Model(W.DECAY, [(W.KSTAR, 1, 895.55, 47.3, W.RADIUS), (kind, J, 4196.0, 370.0, W.RADIUS)])


def test_toy_of_a_spin_parity_model():
    """the generator runs the same kernels: accepted set of a 0- + 1+ model against the oracle"""
    from oracle import toy as T
    from paper_2007_14931_b200 import binding as B
    res, c = build([("1+", Z4200), ("0-", Z4430)], 5)
    Mo, Mg = O.Model(W.DECAY, res), B.Model(W.DECAY, res)
    Mg.set_params(c)
    lo, hi, cm = W.DECAY[2] + W.DECAY[3] + W.M_LO_MARGIN, W.M_HI, W.COS_MAX
    n = 30_000
    xp, _ = T.candidates(8, 0, n, lo, hi, cm)
    fmax = 0.7 * float(T.weights(Mo, c, xp).max())
    g = T.generate(Mo, c, 8, 0, n, fmax, lo, hi, cm)
    x, idx, nacc, fseen = Mg.generate(8, 0, n, fmax, lo, hi, cm, n, with_index=True)
    border = np.nonzero(np.abs(g["u"] * fmax - g["f"]) <= 1e-9 * g["f"])[0]
    assert len(border) <= 2
    assert np.array_equal(np.setdiff1d(idx.cpu().numpy()[:nacc], border), np.setdiff1d(g["index"], border))
    assert abs(fseen - g["f_seen_max"]) <= 1e-11 * fseen
