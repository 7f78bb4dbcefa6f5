"""Host logic of the fit loop (paper_2007_14931_b200/fit.py) on CPU: a stand-in model whose NLL and gradient come from the
oracle takes the place of the CUDA library, so the parameter packing, the fixed slots (Eq. 6), the ties (Eq. 11) and their
chain rule are exercised without a GPU."""
import numpy as np

from oracle import oracle as O
from paper_2007_14931_b200 import fit as F
from paper_2007_14931_b200 import workloads as W


class OracleBackedModel:
    """the two calls fit_couplings makes, answered by the oracle"""

    def __init__(self, cfg, n, m):
        self.res = W.resonances(cfg)
        self.Mo = O.Model(W.DECAY, self.res)
        self.K, self.R = self.Mo.K, self.Mo.R
        self.c_true = W.couplings(cfg)
        self.xn, self.wn = W.norm_events(cfg, m)
        self.x, self.eff = W.data_events(cfg, lambda xx, ee: self.Mo.eval_events(self.c_true, xx, ee), n=n)
        self.c = None

    def set_params(self, c, mass_width=None):
        assert mass_width is None
        self.c = np.asarray(c, dtype=np.complex128).reshape(self.K)

    def nll_grad(self):
        return self.Mo.nll_gradient(self.c, self.x, self.eff, self.xn, self.wn)


def test_fit_loop_fixed_slots_and_ties():
    cfg = 2
    M = OracleBackedModel(cfg, 3000, 12000)
    slots = W.slot_table(M.res)
    fixed = [k for k, (r, lam) in enumerate(slots) if r == 1 and lam == 0]
    ties = [(k, k - 2) for k, (r, lam) in enumerate(slots) if M.res[r][0] == W.ZRES and lam == +1]
    rng = np.random.default_rng(2)
    start = M.c_true * (1 + 0.2 * rng.uniform(-1, 1, M.K)) * np.exp(0.2j * rng.uniform(-1, 1, M.K))
    start[fixed[0]] = M.c_true[fixed[0]]
    M.set_params(M.c_true)
    nll_true = M.nll_grad()[0]
    r = F.fit_couplings(M, start, fixed=fixed, ties=ties, maxiter=400, gtol=1e-2)
    assert r.nll < nll_true                                     # 3000 events: the fit goes below the generating point
    assert r.couplings[fixed[0]] == M.c_true[fixed[0]]           # Eq. 6 slot untouched
    d, s = ties[0]
    assert r.couplings[d] == r.couplings[s]                      # Eq. 11 tie holds
    # stationary in the constrained parameters: free slots' gradient ~ 0, tied pair's SUM ~ 0 (chain rule), fixed slot free to be non-zero
    M.set_params(r.couplings)
    _nll, g = M.nll_grad()
    gsum = g.copy()
    gsum[s] += gsum[d]
    free = [k for k in range(M.K) if k not in fixed and k != d]
    assert np.max(np.abs(gsum[free] * np.abs(start[free])[:, None])) < 0.5
