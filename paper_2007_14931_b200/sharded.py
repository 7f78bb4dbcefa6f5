"""Event-sharded NLL over several processes (one per GPU): the multi-GPU extension point of DESIGN.md "Multi-GPU".

Events are independent (one PDF evaluation per event), so a data set and its normalisation sample can be
cut into one shard per rank.  Every rank runs the same kernels on its own shard; the only exchange per call is ONE
all-reduce of 2 P doubles (sum_i log S_i(p) and sum_j w_j S_j(p)), plus one all-reduce of four constants at load time:

    NLL(p) = -( SUM_ranks sum_log[p] + SUM_ranks sum_log_eff ) + N_total * log( SUM_ranks sum_wS[p] / SUM_ranks sum_w )

The message is <= 4 KB: latency-bound over NVLink 5 / NVSwitch (NCCL) — there is no tile-by-tile overlap to gain from a
fused compute+collective kernel here.  This module holds only the host logic (it needs no GPU and is covered by a
world_size-2 gloo test); `ShardedModel` plugs the C-ABI model in.
"""
import numpy as np


def shard_bounds(n, rank, world):
    """[lo, hi) of the contiguous shard of `n` events owned by `rank`: sizes differ by at most one event."""
    return n * rank // world, n * (rank + 1) // world


def combine_constants(n_data, sum_log_eff, n_norm, sum_w, group=None, device="cpu"):
    """all-reduce (sum) of the per-shard constants -> (N_total, sum_log_eff_total, M_total, sum_w_total).
    The counts travel as float64 (exact below 2^53 events)."""
    import torch
    import torch.distributed as dist
    t = torch.tensor([float(n_data), float(sum_log_eff), float(n_norm), float(sum_w)], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.SUM, group=group)
    t = t.cpu()
    return int(round(t[0].item())), t[1].item(), int(round(t[2].item())), t[3].item()


def combine_terms(sum_log, sum_wS, totals, group=None, device="cpu"):
    """One all-reduce of the 2 P per-shard sums, then the NLL of every point on every rank.

    sum_log, sum_wS: this rank's [P] arrays (amp_nll_terms); totals: the tuple returned by `combine_constants`.
    Returns (nll [P], integral [P]) as numpy arrays, identical on all ranks (all-reduce results are identical by
    construction on every rank of NCCL and gloo)."""
    import torch
    import torch.distributed as dist
    sum_log, sum_wS = np.asarray(sum_log, dtype=np.float64), np.asarray(sum_wS, dtype=np.float64)
    P = sum_log.shape[0]
    t = torch.from_numpy(np.concatenate([sum_log, sum_wS])).to(device)
    dist.all_reduce(t, op=dist.ReduceOp.SUM, group=group)
    t = t.cpu().numpy()
    n_total, sle_total, _m_total, sw_total = totals
    integral = t[P:] / sw_total
    with np.errstate(divide="ignore", invalid="ignore"):
        nll = -(t[:P] + sle_total) + n_total * np.log(integral)
    nll = np.where(np.isfinite(nll) & (integral > 0), nll, np.inf)
    return nll, integral


class ShardedModel:
    """One rank's view of an event-sharded fit: wraps a `binding.Model` that holds this rank's shard.

    load_events / load_norm take the FULL host arrays (SoA [4][n]) and upload only this rank's slice; `nll()` returns the
    global NLL of every parameter point on every rank."""

    def __init__(self, decay, resonances, group=None):
        import torch.distributed as dist
        from . import binding as B
        self.model = B.Model(decay, resonances)
        self.group = group
        self.rank, self.world = dist.get_rank(group), dist.get_world_size(group)
        self.totals = None
        self.K, self.R = self.model.K, self.model.R

    def _slice(self, x, w):
        import torch
        lo, hi = shard_bounds(x.shape[1], self.rank, self.world)
        dev = lambda a: torch.as_tensor(np.ascontiguousarray(a), dtype=torch.float64, device="cuda")
        return dev(x[:, lo:hi]), (None if w is None else dev(w[lo:hi]))

    def load_events(self, x, eff=None):
        self.model.load_events(*self._slice(x, eff))
        self.totals = None

    def load_norm(self, x, w=None):
        self.model.load_norm(*self._slice(x, w))
        self.totals = None

    def set_params(self, couplings, mass_width=None):
        self.model.set_params(couplings, mass_width)

    def nll(self):
        import torch
        dev = torch.device("cuda", torch.cuda.current_device())
        if self.totals is None:
            self.totals = combine_constants(*self.model.dataset_sums(), group=self.group, device=dev)
        sl, sw = self.model.nll_terms()
        return combine_terms(sl, sw, self.totals, group=self.group, device=dev)[0]
