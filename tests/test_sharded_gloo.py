"""Multi-process host logic of the event-sharded NLL (paper_2007_14931_b200/sharded.py) on CPU: world_size 2, gloo.

Each rank owns a contiguous shard of the data and normalisation events, forms its two per-shard sums (here with the
oracle, standing in for amp_nll_terms of the CUDA library — the sharding logic under test is the same), and the ranks
combine them with one all-reduce.  The result must equal the oracle's NLL of the unsharded sample on every rank.
"""
import os
import socket
import sys

import numpy as np
import pytest

torch = pytest.importorskip("torch")
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, out_dir):
    sys.path.insert(0, ROOT)
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        from oracle import oracle as O
        from paper_2007_14931_b200 import sharded as S
        from paper_2007_14931_b200 import workloads as W
        O.set_num_threads(2)
        cfg = 2
        Mo = O.Model(W.DECAY, W.resonances(cfg))
        c = W.couplings(cfg)
        xn, wn = W.norm_events(cfg, 5003)                       # odd sizes: the two shards differ by one event
        x, eff = W.data_events(cfg, lambda xx, ee: Mo.eval_events(c, xx, ee), n=1501)
        cs = np.stack([c, c * np.exp(0.2j * np.arange(len(c))), 0.7 * c])
        mws = np.stack([W.step_mass_width(3, s) for s in range(3)])
        # this rank's shard and its per-shard sums (what amp_nll_terms / amp_dataset_sums return on a GPU rank)
        lo, hi = S.shard_bounds(x.shape[1], rank, world)
        ln, hn = S.shard_bounds(xn.shape[1], rank, world)
        xs, es, xns, wns = x[:, lo:hi], eff[lo:hi], xn[:, ln:hn], wn[ln:hn]
        sum_log, sum_wS = np.zeros(3), np.zeros(3)
        for p in range(3):
            res = [(r[0], r[1], mws[p, i, 0], mws[p, i, 1], r[4]) for i, r in enumerate(W.resonances(cfg))]
            Mp = O.Model(W.DECAY, res)
            sum_log[p] = np.sum(np.log(Mp.eval_events(cs[p], xs, None)))          # eps = 1: sum log S
            sum_wS[p] = np.sum(Mp.eval_events(cs[p], xns, wns))                    # sum w S
        totals = S.combine_constants(xs.shape[1], float(np.sum(np.log(es))), xns.shape[1], float(np.sum(wns)))
        assert totals[0] == x.shape[1] and totals[2] == xn.shape[1]
        nll, integral = S.combine_terms(sum_log, sum_wS, totals)
        ref_nll, ref_I = Mo.nll(cs, x, eff, xn, wn, mass_width=mws)
        assert np.max(np.abs(nll - ref_nll) / np.abs(ref_nll)) < 1e-12, (nll, ref_nll)
        assert np.max(np.abs(integral - ref_I) / ref_I) < 1e-12
        # every rank holds the same bits
        t = torch.from_numpy(nll.copy())
        gathered = [torch.zeros_like(t) for _ in range(world)]
        dist.all_gather(gathered, t)
        assert all(torch.equal(g, gathered[0]) for g in gathered)
        # a point whose integral is not positive gives +inf, not NaN
        bad_nll, _ = S.combine_terms(sum_log, np.zeros(3), totals)
        assert np.all(np.isinf(bad_nll))
        open(os.path.join(out_dir, f"ok{rank}"), "w").write("ok")
    finally:
        dist.destroy_process_group()


def test_shard_bounds_cover_everything():
    sys.path.insert(0, ROOT)
    from paper_2007_14931_b200 import sharded as S
    for n in (0, 1, 7, 1000, 2_000_003):
        for world in (1, 2, 3, 8):
            b = [S.shard_bounds(n, r, world) for r in range(world)]
            assert b[0][0] == 0 and b[-1][1] == n
            assert all(b[r][1] == b[r + 1][0] for r in range(world - 1))
            sizes = [hi - lo for lo, hi in b]
            assert max(sizes) - min(sizes) <= 1


def test_sharded_nll_two_ranks_gloo(tmp_path):
    world = 2
    mp.spawn(_worker, args=(world, _free_port(), str(tmp_path)), nprocs=world, join=True)
    assert all((tmp_path / f"ok{r}").exists() for r in range(world))


def test_thread_reducer_two_virtual_ranks():
    """sharded.ThreadReducer (the exchange step between virtual ranks of one process): two threads form the per-shard sums with
    the oracle and must both get the oracle's NLL of the whole sample, bit for bit the same"""
    import threading
    sys.path.insert(0, ROOT)
    from oracle import oracle as O
    from paper_2007_14931_b200 import sharded as S
    from paper_2007_14931_b200 import workloads as W
    cfg = 1
    Mo = O.Model(W.DECAY, W.resonances(cfg))
    c = W.couplings(cfg)
    xn, wn = W.norm_events(cfg, 3001)
    x, eff = W.data_events(cfg, lambda xx, ee: Mo.eval_events(c, xx, ee), n=801)
    red = S.ThreadReducer(2)
    out = [None, None]

    def rank_main(r):
        port = red.port(r)
        lo, hi = S.shard_bounds(x.shape[1], port.rank, port.world)
        ln, hn = S.shard_bounds(xn.shape[1], port.rank, port.world)
        totals = S.combine_constants(hi - lo, float(np.sum(np.log(eff[lo:hi]))), hn - ln, float(np.sum(wn[ln:hn])), reduce=port)
        sl = np.array([np.sum(np.log(Mo.eval_events(c, x[:, lo:hi], None)))])
        sw = np.array([np.sum(Mo.eval_events(c, xn[:, ln:hn], wn[ln:hn]))])
        out[r] = S.combine_terms(sl, sw, totals, reduce=port)

    th = [threading.Thread(target=rank_main, args=(r,)) for r in range(2)]
    [t.start() for t in th]
    [t.join() for t in th]
    ref, ref_I = Mo.nll(c, x, eff, xn, wn)
    assert np.array_equal(out[0][0], out[1][0]) and np.array_equal(out[0][1], out[1][1])
    assert abs(out[0][0][0] - ref[0]) < 1e-12 * abs(ref[0]) and abs(out[0][1][0] - ref_I[0]) < 1e-12 * ref_I[0]
