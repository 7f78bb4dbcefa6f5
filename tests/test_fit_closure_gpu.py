"""Closure test of the fit loop at reduced scale (the paper's validation method: generate pseudo-data
from the model, fit, compare with the generated values) — on the GPU path end to end: amp_nll_grad drives an L-BFGS loop.

Data: accept-reject sampled from the TRUE couplings by the oracle (no oracle input comes from the CUDA path).  Checks:
the fit converges from a perturbed start, NLL(fit) <= NLL(true), the likelihood-ratio 2 (NLL(true) - NLL(fit)) is of the size
Wilks' theorem gives for the number of free parameters, the fitted couplings sit within a few per cent of the true ones,
and the per-resonance fit fractions (Eq. 13) of the fitted and true parameters agree.  A fit takes ~150 launches of k_grad (< 0.1 s)."""
import numpy as np
import pytest

torch = pytest.importorskip("torch")

from oracle import oracle as O
from paper_2007_14931_b200 import workloads as W

pytestmark = pytest.mark.gpu


def dev(a):
    return torch.as_tensor(np.ascontiguousarray(a), dtype=torch.float64).cuda()


@pytest.mark.parametrize("cfg", [1, 2])
def test_fit_recovers_generated_couplings(cfg):
    from paper_2007_14931_b200 import binding as B
    from paper_2007_14931_b200 import fit as F
    res = W.resonances(cfg)
    slots = W.slot_table(res)
    c_true = W.couplings(cfg)
    Mo = O.Model(W.DECAY, res)
    n, m = 150_000, 600_000
    xn, wn = W.norm_events(cfg, m)
    x, eff = W.data_events(cfg, lambda xx, ee: Mo.eval_events(c_true, xx, ee), n=n)
    Mg = B.Model(W.DECAY, res)
    Mg.load_events(dev(x), dev(eff))
    Mg.load_norm(dev(xn), dev(wn))
    fixed = [k for k, (r, lam) in enumerate(slots) if r == 1 and lam == 0]                       # Eq. 6
    ties = [(k, k - 2) for k, (r, lam) in enumerate(slots) if res[r][0] == W.ZRES and lam == +1]   # Eq. 11
    n_free = 2 * (len(c_true) - len(fixed) - len(ties))
    Mg.set_params(c_true)
    nll_true = Mg.nll()[0]
    rng = np.random.default_rng(5)
    start = c_true * (1 + 0.3 * rng.uniform(-1, 1, c_true.size)) * np.exp(0.3j * rng.uniform(-1, 1, c_true.size))
    for k in fixed:
        start[k] = c_true[k]
    for d, s in ties:
        start[d] = start[s]
    Mg.set_params(start)
    assert Mg.nll()[0] > nll_true + 100.0                       # the start is far away
    r = F.fit_couplings(Mg, start, fixed=fixed, ties=ties)
    assert r.converged, r
    assert r.nll <= nll_true + 1e-6
    lr = 2.0 * (nll_true - r.nll)                              # ~ chi2(n_free) by Wilks' theorem
    assert lr < n_free + 6.0 * np.sqrt(2.0 * n_free), (lr, n_free)
    # the likelihood is what the fit reports, and it is a stationary point
    Mg.set_params(r.couplings)
    nll_fit, g = Mg.nll_grad()
    assert abs(nll_fit - r.nll) < 1e-9 * abs(nll_fit)
    # fit fractions (Eq. 13) of fitted and generated parameters agree
    Mg.set_norm_mode(2)
    Mg.set_params(r.couplings)
    ff_fit = Mg.fit_fractions(0)
    Mg.set_params(c_true)
    ff_true = Mg.fit_fractions(0)
    assert np.max(np.abs(ff_fit - ff_true)) < 0.02, (ff_fit, ff_true)
    # fitted couplings near the generated ones: typically a few per cent with 150k events; the amplitudes of resonances
    # with a sizeable fit fraction individually (a K4*(2045) helicity at the edge of phase space is a flat direction)
    dev_rel = np.abs(r.couplings - c_true) / np.abs(c_true)
    assert np.median(dev_rel) < 0.12, np.median(dev_rel)
    sizeable = np.array([ff_true[slots[k][0]] > 0.05 for k in range(len(c_true))])
    assert np.max(dev_rel[sizeable]) < 0.3, dev_rel[sizeable]


def test_generate_on_device_then_fit_one_million_events():
    """The paper's validation at its own size ("a pseudo-data sample of one million events is generated with the ten
    K*s ... masses and widths fixed"), generated AND fitted on the device: amp_generate draws the toy from the true couplings,
    the host thins it by the efficiency (a detector simulation's job), the fit starts from perturbed couplings."""
    from paper_2007_14931_b200 import binding as B
    from paper_2007_14931_b200 import fit as F
    cfg = 1
    res = W.resonances(cfg)
    slots = W.slot_table(res)
    c_true = W.couplings(cfg)
    lo, hi, cm = W.DECAY[2] + W.DECAY[3] + W.M_LO_MARGIN, W.M_HI, W.COS_MAX
    Mg = B.Model(W.DECAY, res)
    Mg.set_params(c_true)
    xt, used, fmax, fseen = Mg.generate_toy(2_100_000, 20210301, lo, hi, cm)
    assert fseen <= fmax
    xt = xt.cpu().numpy()
    eps = W.efficiency(cfg, xt)
    keep = np.random.default_rng(11).uniform(0, 1, xt.shape[1]) < eps          # eps <= 1
    x, eff = xt[:, keep][:, :1_000_000], eps[keep][:1_000_000]
    assert x.shape[1] == 1_000_000
    xn, wn = W.norm_events(cfg, 2_000_000)
    Mg.load_events(dev(x), dev(eff))
    Mg.load_norm(dev(xn), dev(wn))
    fixed = [k for k, (r, lam) in enumerate(slots) if r == 1 and lam == 0]
    n_free = 2 * (len(c_true) - len(fixed))
    Mg.set_params(c_true)
    nll_true = Mg.nll()[0]
    rng = np.random.default_rng(6)
    start = c_true * (1 + 0.3 * rng.uniform(-1, 1, c_true.size)) * np.exp(0.3j * rng.uniform(-1, 1, c_true.size))
    for k in fixed:
        start[k] = c_true[k]
    r = F.fit_couplings(Mg, start, fixed=fixed)
    assert r.converged, r
    lr = 2.0 * (nll_true - r.nll)
    # Wilks: chi2(n_free), plus the bias of a finite normalisation sample (2e6 points for 1e6 events), which the bound leaves room for
    assert -1e-6 < lr < n_free + 8.0 * np.sqrt(2.0 * n_free) + 40.0, (lr, n_free)
    Mg.set_norm_mode(2)
    Mg.set_params(r.couplings)
    ff_fit = Mg.fit_fractions(0)
    Mg.set_params(c_true)
    ff_true = Mg.fit_fractions(0)
    assert np.max(np.abs(ff_fit - ff_true)) < 0.01, (ff_fit, ff_true)
    dev_rel = np.abs(r.couplings - c_true) / np.abs(c_true)
    assert np.median(dev_rel) < 0.06, np.median(dev_rel)


def test_native_fit_agrees_with_scipy_bfgs():
    """amp_fit (BFGS in the library, csrc/minimize.cu) against scipy's BFGS on the same device gradient: same minimum, same
    covariance; constraints of Eq. 6 (fixed slot) and Eq. 11 (tie) in force"""
    import time
    from paper_2007_14931_b200 import binding as B
    from paper_2007_14931_b200 import fit as F
    cfg = 2
    res = W.resonances(cfg)
    slots = W.slot_table(res)
    c_true = W.couplings(cfg)
    Mo = O.Model(W.DECAY, res)
    xn, wn = W.norm_events(cfg, 400_000)
    x, eff = W.data_events(cfg, lambda xx, ee: Mo.eval_events(c_true, xx, ee), n=100_000)
    Mg = B.Model(W.DECAY, res)
    Mg.load_events(dev(x), dev(eff))
    Mg.load_norm(dev(xn), dev(wn))
    fixed = [k for k, (r, lam) in enumerate(slots) if r == 1 and lam == 0]
    ties = [(k, k - 2) for k, (r, lam) in enumerate(slots) if res[r][0] == W.ZRES and lam == +1]
    rng = np.random.default_rng(8)
    start = c_true * (1 + 0.3 * rng.uniform(-1, 1, c_true.size)) * np.exp(0.3j * rng.uniform(-1, 1, c_true.size))
    for k in fixed:
        start[k] = c_true[k]
    for d, s in ties:
        start[d] = start[s]
    Mg.set_params(start)
    Mg.nll_grad()
    t0 = time.perf_counter()
    rn = Mg.fit(start, fixed=fixed, ties=ties, errors=True, gtol=1e-4)
    t_native = time.perf_counter() - t0
    t0 = time.perf_counter()
    rs = F.fit_couplings(Mg, start, fixed=fixed, ties=ties, errors=True, gtol=1e-4)
    t_scipy = time.perf_counter() - t0
    print(f"\nnative: {rn['n_calls']} calls {t_native * 1e3:.1f} ms;  scipy: {rs.n_calls} calls {t_scipy * 1e3:.1f} ms")
    assert rn["converged"] and rs.converged
    assert rn["grad_max"] < 1e-4
    assert abs(rn["nll"] - rs.nll) < 1e-6                                   # same minimum (NLL ~ 1e6; both stop at |g| < 1e-4)
    assert rn["free"] == rs.free
    for d, s in ties:
        assert rn["couplings"][d] == rn["couplings"][s]
    for k in fixed:
        assert rn["couplings"][k] == c_true[k]
    big = np.abs(c_true) > 0
    assert np.max(np.abs(rn["couplings"] - rs.couplings)[big] / np.abs(c_true)[big]) < 1e-3 * 50      # within a small fraction of the errors
    err_n, err_s = rn["errors"], rs.errors
    assert np.max(np.abs(err_n.real - err_s.real) / err_s.real) < 1e-3 and np.max(np.abs(err_n.imag - err_s.imag) / err_s.imag) < 1e-3
    assert np.max(np.abs(rn["couplings"] - rs.couplings)[rn["free"]] / np.abs(err_s)) < 0.01           # 1 % of a standard deviation
    # the model is left at the fitted point
    nll_now, g = Mg.nll_grad()
    Mg.set_params(rn["couplings"])
    assert abs(Mg.nll()[0] - rn["nll"]) < 1e-9 * abs(rn["nll"])
    # bad arguments
    with pytest.raises(B.AmpError):
        Mg.fit(start, fixed=[99])
    with pytest.raises(B.AmpError):
        Mg.fit(start, ties=[(3, 3)])


def test_fit_with_floating_z_mass_and_width():
    """the paper's exotic-state fit ("floating masses/widths"): the Z's mass and width float with the couplings.  Toy
    generated on the device at M = 4196, Gamma = 370; the fit starts 34 MeV / 40 MeV away.  Checks: recovery within the Hessian
    errors, and the errors themselves against the profile likelihood (M moved by one sigma, everything else refitted: 2 dNLL = 1)"""
    from paper_2007_14931_b200 import binding as B
    cfg = 2
    res = W.resonances(cfg)
    slots = W.slot_table(res)
    c_true = W.couplings(cfg)
    R = len(res)
    iz = R - 1
    lo, hi, cm = W.DECAY[2] + W.DECAY[3] + W.M_LO_MARGIN, W.M_HI, W.COS_MAX
    Mg = B.Model(W.DECAY, res)
    Mg.set_params(c_true)
    x, _, fmax, fseen = Mg.generate_toy(300_000, 4196370, lo, hi, cm)
    assert fseen <= fmax
    Mg.load_events(x.contiguous())
    Mg.load_norm(torch.as_tensor(W.phase_space_events(np.random.default_rng(5), 3_000_000)).cuda())
    fixed = [k for k, (r, lam) in enumerate(slots) if r == 1 and lam == 0]
    ties = [(k, k - 2) for k, (r, lam) in enumerate(slots) if res[r][0] == W.ZRES and lam == +1]
    mw_true = np.array([[r[2], r[3]] for r in res])
    Mg.set_params(c_true, mw_true[None])
    nll_true = Mg.nll()[0]
    rng = np.random.default_rng(12)
    start = c_true * (1 + 0.2 * rng.uniform(-1, 1, c_true.size)) * np.exp(0.2j * rng.uniform(-1, 1, c_true.size))
    for k in fixed:
        start[k] = c_true[k]
    for d, s in ties:
        start[d] = start[s]
    mw_start = mw_true.copy()
    mw_start[iz] = (4230.0, 330.0)
    r = Mg.fit(start, fixed=fixed, ties=ties, mass_width=mw_start, float_mw=[(iz, 0), (iz, 1)], errors=True, gtol=1e-3)
    assert r["converged"] and r["errors"] is not None, {k: r[k] for k in ("nll", "grad_max", "converged", "n_calls", "iterations")}
    assert r["nll"] <= nll_true + 1e-6
    Mfit, Gfit = r["mass_width"][iz]
    sM, sG = r["mw_errors"]
    assert 1.0 < sM < 30.0 and 2.0 < sG < 80.0, (sM, sG)
    assert abs(Mfit - 4196.0) < 4.5 * sM and abs(Gfit - 370.0) < 4.5 * sG, (Mfit, sM, Gfit, sG)
    assert np.array_equal(r["mass_width"][:iz], mw_true[:iz])                  # the K* lineshapes did not move
    n_free = len(r["free"]) * 2 + 2
    lr = 2 * (nll_true - r["nll"])
    assert lr < n_free + 6 * np.sqrt(2 * n_free) + 20, (lr, n_free)
    # profile likelihood: M fixed one sigma up, width and couplings refitted -> NLL rises by 1/2 (parabolic regime)
    mw_p = r["mass_width"].copy()
    mw_p[iz, 0] = Mfit + sM
    rp = Mg.fit(r["couplings"], fixed=fixed, ties=ties, mass_width=mw_p, float_mw=[(iz, 1)], gtol=1e-3)
    assert rp["converged"]
    assert 0.35 < rp["nll"] - r["nll"] < 0.7, rp["nll"] - r["nll"]
    # and the derivative the fit used for M agrees with a symmetric difference of amp_nll at a larger step
    Mg.set_params(np.tile(r["couplings"], (2, 1)), np.stack([mw_p, r["mass_width"]]))
    assert Mg.nll()[0] - Mg.nll()[1] > 0
