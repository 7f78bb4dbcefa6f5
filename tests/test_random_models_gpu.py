"""Randomised resonance lists through the GENERIC kernels (runtime loops over barrier groups): different radii inside one
spin (several barrier groups per spin), missing spins, zero / one / two Zs, constant terms, a LASS term.  For every model:
per-event density, the fused NLL with moved masses and widths, the analytic gradient (where defined), a gradient batch
through the gradient-batch kernel (or the dense path where that one does not apply) — all against the oracle."""
import numpy as np
import pytest

torch = pytest.importorskip("torch")

from oracle import oracle as O
from paper_2007_14931_b200 import workloads as W

pytestmark = pytest.mark.gpu

RADII = (1.6e-3, 3.0e-3, 4.5e-3)


def dev(a):
    return torch.as_tensor(np.ascontiguousarray(a), dtype=torch.float64).cuda()


def random_model(seed):
    rng = np.random.default_rng(seed)
    res = []
    for k in W.KSTARS:
        if rng.uniform() < 0.7:
            res.append((W.KSTAR, k[2], k[3] * (1 + 0.01 * rng.uniform(-1, 1)), k[4] * (1 + 0.05 * rng.uniform(-1, 1)), RADII[rng.integers(3)]))
    if not res:
        res.append((W.KSTAR, 1, 895.55, 47.3, RADII[0]))
    nz = int(rng.integers(3))
    for z in range(nz):
        res.append((W.ZRES, 1, (4196.0, 4478.0)[z], (370.0, 181.0)[z], RADII[rng.integers(3)]))
    for _ in range(int(rng.integers(3))):
        res.append((W.CONST, 0, 0.0, 0.0, 0.0))
    lass = rng.uniform() < 0.3
    if lass:
        res.append((W.LASS, 0, 1425.0, 270.0, 0.0))
    order = rng.permutation(len(res))
    res = [res[i] for i in order]
    slots = W.slot_table(res)
    c = rng.uniform(0.5, 1.5, len(slots)) * np.exp(1j * rng.uniform(-np.pi, np.pi, len(slots)))
    for k, (r, lam) in enumerate(slots):
        if res[r][0] == W.CONST:
            c[k] *= 2e-6
        if res[r][0] == W.LASS:
            c[k] *= 7e-6
        if res[r][0] == W.ZRES:
            c[k] *= 5.0
    return res, c, lass, nz


@pytest.mark.parametrize("seed", list(range(1, 21)))
def test_random_model_all_paths(seed):
    from paper_2007_14931_b200 import binding as B
    res, c, lass, nz = random_model(seed)
    Mo, Mg = O.Model(W.DECAY, res), B.Model(W.DECAY, res)
    K, R = len(c), len(res)
    assert Mg.K == Mo.K == K
    rng = np.random.default_rng(100 + seed)
    n, m = int(rng.integers(900, 4000)), int(rng.integers(3000, 9000))
    xn, wn = W.norm_events(2, m)
    x, eff = W.data_events(2, lambda xx, ee: Mo.eval_events(c, xx, ee), n=n)
    Mg.load_events(dev(x), dev(eff))
    Mg.load_norm(dev(xn), dev(wn))
    Mg.set_params(c)
    v, vref = Mg.eval_events(0).cpu().numpy(), Mo.eval_events(c, x, eff)
    assert np.max(np.abs(v - vref) / vref) < 1e-11, (seed, res)
    mw = np.array([[r[2], r[3]] for r in res]) * (1 + 2e-3 * rng.uniform(-1, 1, (R, 2)))
    Mg.set_params(c, mw[None])
    nll = Mg.nll()[0]
    assert Mg.last_call_stats()["norm_path"] == 4
    ref = Mo.nll(c, x, eff, xn, wn, mass_width=mw[None])[0][0]
    assert abs(nll - ref) < 1e-9 * abs(ref), (seed, nll, ref)
    if not lass:
        nllg, g = Mg.nll_grad()
        res2 = [(r[0], r[1], mw[i, 0], mw[i, 1], r[4]) for i, r in enumerate(res)]
        rn, rg = O.Model(W.DECAY, res2).nll_gradient(c, x, eff, xn, wn)
        assert abs(nllg - rn) < 1e-9 * abs(rn)
        assert np.max(np.abs(g - rg)) < 1e-9 * np.max(np.abs(rg)), seed
    # a gradient-style batch: one coupling or one (mass, width) changes per point
    nonconst = [k for k, (r, lam) in enumerate(W.slot_table(res)) if res[r][0] != W.CONST]
    P = 1 + 2 * min(len(nonconst), 9) + 2 * min(R, 4)
    cs, mws = np.tile(c, (P, 1)), np.tile(mw, (P, 1, 1))
    p = 1
    for k in nonconst[:9]:
        cs[p, k] *= 1 + 1e-3; p += 1
        cs[p, k] *= np.exp(-1e-3j); p += 1
    for r in range(min(R, 4)):
        if res[r][0] != W.CONST:
            mws[p, r, 0] *= 1 + 1e-4
            mws[p + 1, r, 1] *= 1 - 1e-4
        p += 2
    assert p == P
    Mg.set_params(cs, mws)
    nb = Mg.nll()
    path = Mg.last_call_stats()["norm_path"]
    # gradient-batch kernel; LASS models or more barrier groups than its shared memory holds: dense DMMA path (P >= 24) or
    # the loop of single-point launches
    assert path in ((1, 2, 3) if lass else (5, 9, 1, 2, 3)), (seed, path)
    rb, rI = Mo.nll(cs, x, eff, xn, wn, mass_width=mws)
    assert np.max(np.abs(nb - rb) / np.abs(rb)) < 1e-9, seed
    assert np.max(np.abs(Mg.norm_integral() - rI) / rI) < 1e-12, seed
