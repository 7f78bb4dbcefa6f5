"""Parity of the device toy generator (amp_generate, toy.cu) with its oracle (oracle/toy.py) — SURVEY.md 8(f)-4.

Integer / bit work is compared exactly: the candidate stream (Philox words -> uniforms -> points) bit for bit, the accepted
candidates as an index set and in order.  The acceptance itself is a floating-point decision (U f_max < p_B q S, S agreeing
with the oracle to ~1e-12): candidates whose two sides agree to 1e-9 relative are listed as borderline and left out of the
set comparison (there are none at these sizes unless something is wrong; at most a handful are allowed)."""
import numpy as np
import pytest

torch = pytest.importorskip("torch")

from oracle import oracle as O
from oracle import toy as T
from paper_2007_14931_b200 import workloads as W

pytestmark = pytest.mark.gpu

LO, HI, CM = W.DECAY[2] + W.DECAY[3] + W.M_LO_MARGIN, W.M_HI, W.COS_MAX


def dev(a):
    return torch.as_tensor(np.ascontiguousarray(a), dtype=torch.float64).cuda()


def gpu_model(res, c):
    from paper_2007_14931_b200 import binding as B
    M = B.Model(W.DECAY, res)
    M.set_params(c)
    return M


@pytest.mark.parametrize("seed,first,n", [(7, 0, 5000), ((3 << 32) + 11, (1 << 32) - 1500, 3333), (2 ** 64 - 1, 2 ** 40 + 3, 1025), (5, 0, 1)])
def test_candidate_stream_is_bit_exact(seed, first, n):
    """f_max = 0 accepts every candidate: the output IS the candidate stream (ragged sizes, the 32-bit counter carry, a full-width seed)"""
    Mg = gpu_model(W.resonances(2), W.couplings(2))
    x, idx, nacc, fseen = Mg.generate(seed, first, n, 0.0, LO, HI, CM, n, with_index=True)
    assert nacc == n
    xo, _ = T.candidates(seed, first, n, LO, HI, CM)
    assert np.array_equal(x.cpu().numpy(), xo)
    assert np.array_equal(idx.cpu().numpy(), first + np.arange(n, dtype=np.int64))
    f = T.weights(O.Model(W.DECAY, W.resonances(2)), W.couplings(2), xo)
    assert abs(fseen - f.max()) <= 1e-11 * f.max()


@pytest.mark.parametrize("cfg,lass", [(0, False), (1, False), (2, False), (2, True)])
def test_accepted_set_matches_oracle(cfg, lass):
    res = W.resonances_lass(True) if lass else W.resonances(cfg)
    c = W.couplings_lass(True) if lass else W.couplings(cfg)
    Mo = O.Model(W.DECAY, res)
    Mg = gpu_model(res, c)
    seed, first, n = 20070149 + cfg, 12345, 70_001
    # envelope from the oracle's own pilot (no oracle input comes from the CUDA path); 0.6 x: some weights exceed it, as a user's might
    xp, _ = T.candidates(seed, first, n, LO, HI, CM)
    fmax = 0.6 * float(T.weights(Mo, c, xp).max())
    g = T.generate(Mo, c, seed, first, n, fmax, LO, HI, CM)
    cap = n
    x, idx, nacc, fseen = Mg.generate(seed, first, n, fmax, LO, HI, CM, cap, with_index=True)
    assert abs(fseen - g["f_seen_max"]) <= 1e-11 * g["f_seen_max"]
    border = np.nonzero(np.abs(g["u"] * fmax - g["f"]) <= 1e-9 * g["f"])[0]
    assert len(border) <= 3
    got = idx.cpu().numpy()[:nacc] - first
    assert np.all(np.diff(got) > 0)                                      # candidate order
    want = g["index"]
    assert np.array_equal(np.setdiff1d(got, border), np.setdiff1d(want, border))
    assert abs(nacc - len(want)) <= len(border)
    assert 0.01 * n < nacc < 0.9 * n
    assert np.array_equal(x.cpu().numpy()[:, :nacc], xp[:, got])        # the accepted points, bit for bit
    # a smaller output buffer: the first `capacity` accepted are written, all are counted
    cap2 = nacc // 3
    x2, idx2, nacc2, _ = Mg.generate(seed, first, n, fmax, LO, HI, CM, cap2, with_index=True)
    assert nacc2 == nacc
    assert np.array_equal(idx2.cpu().numpy(), idx.cpu().numpy()[:cap2]) and np.array_equal(x2.cpu().numpy(), x.cpu().numpy()[:, :cap2])
    # count only
    _, _, nacc3, fseen3 = Mg.generate(seed, first, n, fmax, LO, HI, CM, 0)
    assert nacc3 == nacc and fseen3 == fseen


def test_blocks_of_work_join_in_order():
    """more candidates than one internal block of work (2^21): the result equals the two halves generated separately, in order"""
    Mg = gpu_model(W.resonances(0), W.couplings(0))
    seed, n1, n2 = 99, 1 << 21, 70_000
    _, _, _, fs = Mg.generate(seed, 0, 1 << 18, 0.0, LO, HI, CM, 0)
    fmax = 1.2 * fs
    x, idx, nacc, fseen = Mg.generate(seed, 0, n1 + n2, fmax, LO, HI, CM, n1 + n2, with_index=True)
    xa, ia, na, fa = Mg.generate(seed, 0, n1, fmax, LO, HI, CM, n1, with_index=True)
    xb, ib, nb, fb = Mg.generate(seed, n1, n2, fmax, LO, HI, CM, n2, with_index=True)
    assert nacc == na + nb and fseen == max(fa, fb)
    assert torch.equal(idx[:na], ia[:na]) and torch.equal(idx[na:nacc], ib[:nb])
    assert torch.equal(x[:, :na], xa[:, :na]) and torch.equal(x[:, na:nacc], xb[:, :nb])
    got = idx[:nacc].cpu().numpy()
    assert np.all(np.diff(got) > 0)
    xo, _ = T.candidates(seed, 0, n1 + n2, LO, HI, CM)
    assert np.array_equal(x[:, :nacc].cpu().numpy(), xo[:, got])


def test_toy_follows_the_model_density():
    """distribution check at a size the oracle cannot reach event by event: for 2e5 toy events of the K* + Z model, the m_Kpi
    histogram agrees (chi2) with the expectation p_B q S integrated per bin by the ORACLE on an independent uniform sample"""
    cfg = 2
    res, c = W.resonances(cfg), W.couplings(cfg)
    Mg = gpu_model(res, c)
    n_ev = 200_000
    x, used, fmax, fseen = Mg.generate_toy(n_ev, 31337, LO, HI, CM, block=1 << 21)
    assert fseen <= fmax
    x = x.cpu().numpy()
    assert x.shape == (4, n_ev) and np.all(np.isfinite(x))
    Mo = O.Model(W.DECAY, res)
    xo, _ = T.candidates(777, 0, 400_000, LO, HI, CM)               # uniform in the four variables
    fo = T.weights(Mo, c, xo)
    edges = np.linspace(LO, HI, 31)
    num = np.histogram(xo[0], edges, weights=fo)[0]
    num2 = np.histogram(xo[0], edges, weights=fo * fo)[0]
    exp = num / num.sum() * n_ev
    var_exp = num2 / num.sum() ** 2 * n_ev ** 2                       # Monte-Carlo error of the expectation
    obs = np.histogram(x[0], edges)[0]
    chi2 = float(np.sum((obs - exp) ** 2 / (exp + var_exp)))
    assert chi2 < 30 + 6 * np.sqrt(60), chi2
    # and in phi, where the helicity-+-1 interference modulates the rate
    edges = np.linspace(-np.pi, np.pi, 21)
    num = np.histogram(xo[3], edges, weights=fo)[0]
    num2 = np.histogram(xo[3], edges, weights=fo * fo)[0]
    exp = num / num.sum() * n_ev
    var_exp = num2 / num.sum() ** 2 * n_ev ** 2
    obs = np.histogram(x[3], edges)[0]
    chi2 = float(np.sum((obs - exp) ** 2 / (exp + var_exp)))
    assert chi2 < 20 + 6 * np.sqrt(40), chi2
    assert np.max(obs) > 1.05 * np.min(obs)                           # there is a modulation to see


def test_generate_errors():
    from paper_2007_14931_b200 import binding as B
    res, c = W.resonances(1), W.couplings(1)
    Mg = B.Model(W.DECAY, res)
    with pytest.raises(B.AmpError):                                   # no parameters yet
        Mg.generate(1, 0, 100, 0.0, LO, HI, CM, 100)
    Mg.set_params(c)
    for bad in [dict(m_lo=W.DECAY[2] + W.DECAY[3]), dict(m_hi=W.DECAY[0] - W.DECAY[1]), dict(cos_max=1.5), dict(cos_max=0.0), dict(f_max=-1.0), dict(f_max=float("nan"))]:
        kw = dict(f_max=0.0, m_lo=LO, m_hi=HI, cos_max=CM)
        kw.update(bad)
        with pytest.raises(B.AmpError):
            Mg.generate(1, 0, 100, kw["f_max"], kw["m_lo"], kw["m_hi"], kw["cos_max"], 100)
    x, _, nacc, _ = Mg.generate(1, 0, 0, 0.0, LO, HI, CM, 10)        # no candidates: nothing accepted
    assert nacc == 0
    Mg.set_params(np.stack([c, c * 1.01]))                            # two points: not a generator state
    with pytest.raises(B.AmpError):
        Mg.generate(1, 0, 100, 0.0, LO, HI, CM, 100)
