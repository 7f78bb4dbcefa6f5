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


class TorchReducer:
    """sum-all-reduce of a small float64 vector over a torch.distributed process group (NCCL over NVLink 5 / NVSwitch on GPUs,
    gloo on CPU): the one exchange step of the event-sharded path"""

    def __init__(self, group=None, device="cpu"):
        import torch.distributed as dist
        self.group, self.device = group, device
        self.rank, self.world = dist.get_rank(group), dist.get_world_size(group)

    def __call__(self, values):
        import torch
        import torch.distributed as dist
        t = torch.from_numpy(np.ascontiguousarray(values, dtype=np.float64)).to(self.device)
        dist.all_reduce(t, op=dist.ReduceOp.SUM, group=self.group)
        return t.cpu().numpy()


class ThreadReducer:
    """The same exchange between `world` host threads of ONE process (one virtual rank per thread, each with its own model):
    every rank deposits its vector, all wait, every rank adds the vectors in rank order (bitwise identical results on all
    ranks).  Lets the sharded path run complete on a single GPU — and is how one process would drive several GPUs."""

    def __init__(self, world):
        import threading
        self.world = world
        self.slots = [None] * world
        self.barrier = threading.Barrier(world)

    def port(self, rank):
        red = self

        class Port:
            world = red.world

            def __init__(self):
                self.rank = rank

            def __call__(self, values):
                red.slots[rank] = np.array(values, dtype=np.float64)
                red.barrier.wait()
                total = np.zeros_like(red.slots[0])
                for r in range(red.world):
                    total = total + red.slots[r]
                red.barrier.wait()
                return total
        return Port()


def nll_from_sums(sum_log_total, sum_wS_total, totals):
    """NLL(p) = -(sum_log + sum_log_eff) + N log(sum_wS / sum_w) from the sums over ALL shards; +inf where the integral is not positive"""
    n_total, sle_total, _m_total, sw_total = totals
    integral = np.asarray(sum_wS_total, dtype=np.float64) / sw_total
    with np.errstate(divide="ignore", invalid="ignore"):
        nll = -(np.asarray(sum_log_total, dtype=np.float64) + sle_total) + n_total * np.log(integral)
    return np.where(np.isfinite(nll) & (integral > 0), nll, np.inf), integral


def combine_constants(n_data, sum_log_eff, n_norm, sum_w, group=None, device="cpu", reduce=None):
    """all-reduce (sum) of the per-shard constants -> (N_total, sum_log_eff_total, M_total, sum_w_total).
    The counts travel as float64 (exact below 2^53 events)."""
    reduce = reduce or TorchReducer(group, device)
    t = reduce(np.array([float(n_data), float(sum_log_eff), float(n_norm), float(sum_w)]))
    return int(round(t[0])), float(t[1]), int(round(t[2])), float(t[3])


def combine_terms(sum_log, sum_wS, totals, group=None, device="cpu", reduce=None):
    """One all-reduce of the 2 P per-shard sums, then the NLL of every point on every rank.

    sum_log, sum_wS: this rank's [P] arrays (amp_nll_terms); totals: the tuple returned by `combine_constants`.
    Returns (nll [P], integral [P]) as numpy arrays, identical on all ranks (all-reduce results are identical by
    construction on every rank of NCCL and gloo)."""
    reduce = reduce or TorchReducer(group, device)
    sum_log, sum_wS = np.asarray(sum_log, dtype=np.float64), np.asarray(sum_wS, dtype=np.float64)
    P = sum_log.shape[0]
    t = reduce(np.concatenate([sum_log, sum_wS]))
    return nll_from_sums(t[:P], t[P:], totals)


class ShardedModel:
    """One rank's view of an event-sharded fit: wraps a `binding.Model` that holds this rank's shard.

    load_events / load_norm take the FULL host arrays (SoA [4][n]) and upload only this rank's slice; `nll()` returns the
    global NLL of every parameter point on every rank.  `reduce`: the exchange step — default a TorchReducer on `group`
    (NCCL when the process group is NCCL); a ThreadReducer port runs several virtual ranks inside one process."""

    def __init__(self, decay, resonances, group=None, reduce=None, device=None):
        import torch
        from . import binding as B
        self.device = torch.device("cuda", torch.cuda.current_device()) if device is None else torch.device(device)
        with torch.cuda.device(self.device):
            self.model = B.Model(decay, resonances)
        self.reduce = reduce or TorchReducer(group, self.device)
        self.rank, self.world = self.reduce.rank, self.reduce.world
        self.totals = None
        self.K, self.R = self.model.K, self.model.R

    def _slice(self, x, w):
        import torch
        lo, hi = shard_bounds(x.shape[1], self.rank, self.world)
        dev = lambda a: torch.as_tensor(np.ascontiguousarray(a), dtype=torch.float64, device=self.device)
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
        if self.totals is None:
            self.totals = combine_constants(*self.model.dataset_sums(), reduce=self.reduce)
        sl, sw = self.model.nll_terms()
        return combine_terms(sl, sw, self.totals, reduce=self.reduce)[0]
