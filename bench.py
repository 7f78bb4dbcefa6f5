#!/usr/bin/env python
"""bench.py — NLL evaluations per second of the 4D amplitude model on B200 (BASELINE.json metric).

Workload (config.workload): BASELINE.json configs[3] at its headline point — the full K* + Z model
(11 resonances, K = 27 couplings), 2M data events and 10M normalisation events, FP64 structure-of-arrays,
every lineshape floating: each timed step is one `amp_set_params` (new masses and widths for all 11
resonances, new couplings) + one `amp_nll` through the C ABI, i.e. one pass of the whole hot path
(lineshapes -> combine -> normalisation -> -log L reduction) over the data and the normalisation sample.
The kinematics cache is built once per dataset (step a1, outside the per-step metric, reported separately).

One JSON line on stdout (rank 0).  `--impl reference` times the CPU oracle instead (rank 0 only).
"""
import argparse
import json
import os
import subprocess
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

from paper_2007_14931_b200 import workloads as W  # noqa: E402

METRIC = "4D amplitude NLL evals/sec at 2M events (FP64)"
UNIT = "NLL evals/s"

# Algorithmic work per event of the fused streaming kernel with all lineshapes evaluated in registers
# (DESIGN.md "Rooflines"): 22 cached FP64 values read per event (+ the weight on the normalisation side);
# flops: + - x once, FMA twice, / sqrt log once each.
BYTES_PER_EVENT_DATA = 22 * 8
BYTES_PER_EVENT_NORM = 23 * 8
FLOP_PER_EVENT = 730.0
FP64_PEAK_NOMINAL = 148 * 64 * 2 * 1.965e9   # 148 SMs x 64 DFMA/clk x 2 flop x 1965 MHz
# dram__bytes_read.sum + dram__bytes_write.sum of the dominant kernel from the committed `ncu --set full` capture
# (profiles/): per launch, at the default sizes; None until a capture of the current kernel exists
TRAFFIC_NCU_BYTES = 2.192250e9 + 3.63e6       # profiles/r01g_ncu_full_stream_fused_cfg3.csv (2M + 10M events)
TRAFFIC_NCU_BYTES_CFG4 = 2.195064e9 + 9.09e6  # profiles/r01g_ncu_full_delta_cfg4.csv
# Algorithmic flop per event of the gradient batch of configs[4] in its sparse form: point 0 (730) + 31 slots
# (Breit-Wigner of point 0 from the saved barrier factors ~20, angular factor ~8, two complex products 12, and the expansion
# coefficients T2 = 2 sum conj(A(0)) SLOT, n = sum |SLOT|^2: 25) + 100 coupling points (S(0) + Re(coef T2) + |coef|^2 n: 6, guard 1,
# accumulate 1) + 20 mass/width points (perturbed Breit-Wigner ~22, difference to point 0 and |coef|^2: 5, expansion 6)
DELTA_FLOP_PER_EVENT = 730.0 + 31 * 65.0 + 100 * 8.0 + 20 * 33.0
# normalisation events: the 100 coupling points cost nothing per point there — three weighted sums per group of four on one slot
# (25 groups x 3 FMA), the points are formed from them once per launch
DELTA_FLOP_PER_NORM_EVENT = 730.0 + 31 * 65.0 + 25 * 6.0 + 20 * 33.0
# analytic gradient: the point (730) + per coupling slot: angular factor ~8, T = sum_xi conj(g) A 16, conj(BW) T 8, weight 2
GRAD_FLOP_PER_EVENT = 730.0 + 27 * 34.0
# its shape-specialised form (gradf.cu): the point (730) + the three W_lambda and three Y_lambda' (u A, conj(g) A:
# ~110) + one real scaling of them per spin (~30) + per coupling slot conj(BW) X into its register pair (4 FMA = 8)
GRADF_FLOP_PER_EVENT = 730.0 + 140.0 + 27 * 8.0


LASS = False   # --lass: the paper's LASS variant of the model (Eq. 9) instead of kappa(800) + K0*(1430)


def model_def(cfg):
    """(resonance list, seeded couplings) of the benchmarked model"""
    if LASS:
        return W.resonances_lass(True), W.couplings_lass(True)
    return W.resonances(cfg), W.couplings(cfg)


def measured_peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        d = json.load(open(p))
        return float(d["hbm_gbs"]), "measured"
    return 6650.0, "fallback"


class ClockSampler:
    """SM clock and throttle reasons sampled through NVML (pynvml) in a thread DURING the timed region."""

    def __init__(self, index):
        self.index, self.rows, self.stop_flag, self.thread = index, [], False, None

    def start(self):
        try:
            import pynvml as nv
            nv.nvmlInit()
            self.nv = nv
            self.h = nv.nvmlDeviceGetHandleByIndex(self.index)
            self.smax = nv.nvmlDeviceGetMaxClockInfo(self.h, nv.NVML_CLOCK_SM)
        except Exception as e:   # noqa: BLE001
            self.nv = None
            self.err = repr(e)
            return
        self.thread = threading.Thread(target=self._poll, daemon=True)
        self.thread.start()

    def _poll(self):
        nv = self.nv
        while not self.stop_flag:
            try:
                sm = nv.nvmlDeviceGetClockInfo(self.h, nv.NVML_CLOCK_SM)
                rs = nv.nvmlDeviceGetCurrentClocksEventReasons(self.h)
                pw = nv.nvmlDeviceGetPowerUsage(self.h) / 1e3
                self.rows.append((time.perf_counter(), sm, rs, pw))
            except Exception:   # noqa: BLE001
                pass
            time.sleep(0.002)

    def stop(self, t0=None, t1=None):
        if not getattr(self, "nv", None):
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvml unavailable: " + getattr(self, "err", "")]}
        self.stop_flag = True
        self.thread.join(timeout=2)
        nv = self.nv
        rows = [r for r in self.rows if (t0 is None or r[0] >= t0) and (t1 is None or r[0] <= t1)] or self.rows[-3:]
        names = {"hw_slowdown": nv.nvmlClocksEventReasonHwSlowdown, "hw_thermal_slowdown": nv.nvmlClocksEventReasonHwThermalSlowdown,
                 "sw_thermal_slowdown": nv.nvmlClocksEventReasonSwThermalSlowdown, "sw_power_cap": nv.nvmlClocksEventReasonSwPowerCap}
        reasons = sorted(k for k, bit in names.items() if any(r[2] & bit for r in rows))
        return {"sm_mhz": float(np.median([r[1] for r in rows])) if rows else None, "sm_max_mhz": float(self.smax), "reasons": reasons,
                "power_w_max": max(r[3] for r in rows) if rows else None, "samples": len(rows)}


def build_workload(args, device):
    """events on the device, model with data + norm loaded.  Data events: accept-reject driven by the product's
    own amp_eval_events (toy generation with the fitter itself)."""
    import torch
    from paper_2007_14931_b200 import binding as B

    cfg = args.cfg
    res, c = model_def(cfg)
    dev = lambda a: torch.as_tensor(np.ascontiguousarray(a), dtype=torch.float64, device=device)
    gen = B.Model(W.DECAY, res)

    def density(xx, ee):
        gen.load_events(dev(xx), dev(ee))
        gen.set_params(c)
        return gen.eval_events(0).cpu().numpy()

    t0 = time.time()
    x, eff = W.data_events(cfg, density, n=args.n_data)
    gen.close()
    xn, wn = W.norm_events(cfg, args.n_norm)
    t_gen = time.time() - t0
    model = B.Model(W.DECAY, res)
    # cold start, once: the events as HOST buffers (pinned) -> device -> kinematics cache -> first NLL, by the wall clock
    pin = lambda a: torch.from_numpy(np.ascontiguousarray(a, dtype=np.float64)).pin_memory()
    h_x, h_e, h_xn, h_wn = pin(x), pin(eff), pin(xn), pin(wn)
    torch.cuda.synchronize()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    t0 = time.perf_counter()
    d_x, d_e, d_xn, d_wn = (t.to(device, non_blocking=True) for t in (h_x, h_e, h_xn, h_wn))
    e0.record()
    model.load_events(d_x, d_e)
    model.load_norm(d_xn, d_wn)
    e1.record()
    cs, mws = step_params(cfg, c, 0)
    model.set_params(cs, mws)
    model.nll()
    torch.cuda.synchronize()
    cold_ms = (time.perf_counter() - t0) * 1e3
    load_ms = e0.elapsed_time(e1)
    h2d = sum(t.numel() * 8 for t in (h_x, h_e, h_xn, h_wn))
    del d_x, d_e, d_xn, d_wn, h_x, h_e, h_xn, h_wn
    return model, c, {"gen_s": t_gen, "load_ms": load_ms,
                      "cold_start": {"ms": cold_ms, "h2d_bytes": int(h2d),
                                     "what": "pinned host events -> H2D -> kinematics cache (k_kinematics) -> amp_set_params + first amp_nll, wall clock"}}


def step_params(cfg, c, step):
    """parameters of timed call `step`: every mass and width moved by a seeded 1e-4 step (cfg 3 call pattern) and
    the couplings rotated by a small seeded amount, so that successive calls genuinely differ."""
    if cfg == 4:
        return W.fit_points(cfg, step)
    if LASS:
        mw = np.array([[r[2], r[3]] for r in W.resonances_lass(True)], dtype=np.float64)
        mw *= 1.0 + 1e-4 * np.random.default_rng(np.random.SeedSequence([W.SEED, 98, int(step)])).uniform(-1, 1, mw.shape)
    else:
        mw = W.step_mass_width(cfg, step)
    rng = np.random.default_rng(np.random.SeedSequence([W.SEED, 99, int(step)]))
    cc = c * (1.0 + 1e-3 * rng.uniform(-1, 1, c.size)) * np.exp(1e-3j * rng.uniform(-1, 1, c.size))
    return cc[None], mw[None]


def run_own(args):
    import torch
    import torch.distributed as dist

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    torch.cuda.set_device(local)
    device = torch.device("cuda", local)
    if world > 1:
        dist.init_process_group("nccl", device_id=device)
    from paper_2007_14931_b200 import binding as B

    model, c, info = build_workload(args, device)
    P = 121 if args.cfg == 4 else 1
    params = [step_params(args.cfg, c, s) for s in range(args.warmup + args.steps)]
    h2d = sum(a.nbytes for a in (np.zeros((P, model.K, 2)), np.zeros((P, model.R, 2))))
    d2h = 8 * P

    if args.dense:
        model.set_batch_mode(2)   # configs[4] as the dense DMMA contraction + extended-basis normalisation matrix

    def one_step(s):
        cs, mws = params[s]
        model.set_params(cs, mws)
        if args.grad:
            return np.array([model.nll_grad()[0]])   # NLL + its analytic gradient in all K couplings, one launch
        return model.nll()

    for s in range(args.warmup):
        one_step(s)
    if world > 1:
        dist.barrier()
    torch.cuda.synchronize()
    sampler = ClockSampler(local)
    if rank == 0:
        sampler.start()
        time.sleep(0.02)
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    nll_last = None
    t_wall0 = time.perf_counter()
    ev0.record()
    for s in range(args.warmup, args.warmup + args.steps):
        nll_last = one_step(s)          # nothing else in the timed region: amp_set_params + amp_nll through the C ABI
    ev1.record()
    torch.cuda.synchronize()
    t_wall = time.perf_counter() - t_wall0
    if world > 1:
        dist.barrier()
    clocks = sampler.stop(t_wall0, t_wall0 + t_wall) if rank == 0 else None
    dev_ms = ev0.elapsed_time(ev1)
    # per-step launch counts, path and kernel times, read AFTER the timed region: every step of a run takes the same path;
    # the kernel times come from the library's ring of CUDA event pairs recorded around each launch on its stream
    st = model.last_call_stats()
    launches, paths = st["launches"] * args.steps, {st["norm_path"]}
    if st["norm_path"] in (4, 5, 7, 8):
        ring = model.recent_launch_ms(min(args.steps, 256))
        t_data, t_norm, t_line = [float(v) for v in ring], [0.0], [0.0]
    else:
        tm = model.last_call_timing()
        t_data, t_norm, t_line = [tm["data_ms"]], [tm["norm_ms"]], [tm["lineshape_ms"]]
    if world > 1:
        t = torch.tensor([dev_ms, t_wall * 1e3], dtype=torch.float64, device=device)
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        dev_ms, t_wall = float(t[0]), float(t[1]) / 1e3
    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return
    evals = P * args.steps * world          # replicas: every rank evaluates its own data set
    value = evals / (dev_ms * 1e-3)
    e2e = evals / t_wall
    hbm_peak, peak_kind = measured_peaks()
    norm_ms = float(np.mean(t_norm))
    if args.cfg == 4 and paths == {5}:
        # gradient batch: one fused k_delta launch per step, bound by the plain FP64 ALUs (DESIGN.md 5.6 / 6)
        k_ms = float(np.mean(t_data))
        flop = DELTA_FLOP_PER_EVENT * args.n_data + DELTA_FLOP_PER_NORM_EVENT * args.n_norm
        ach = flop / (k_ms * 1e-3) / 1e12
        roof = {"bound": "alu", "kernel": "k_delta (gradient batch: point 0 + 120 sparse points, data then norm tiles, one launch)",
                "achieved": ach, "peak": FP64_PEAK_NOMINAL / 1e12,
                "peak_source": "148 SMs x 64 DFMA/clk x 2 flop x 1.965 GHz (DESIGN.md 6; the DFMA probe below measures it)", "unit": "TFLOP/s",
                "frac": ach / (FP64_PEAK_NOMINAL / 1e12), "traffic": TRAFFIC_NCU_BYTES_CFG4 if (args.n_data, args.n_norm) == (2_000_000, 10_000_000) else None, "kernel_ms": k_ms,
                "flop_per_event": [DELTA_FLOP_PER_EVENT, DELTA_FLOP_PER_NORM_EVENT], "flop_per_launch": flop,
                "hbm_frac": (BYTES_PER_EVENT_DATA * args.n_data + BYTES_PER_EVENT_NORM * args.n_norm) / (k_ms * 1e-3) / 1e9 / hbm_peak}
    elif paths == {7} or paths == {8}:
        # --grad: NLL and analytic gradient in one k_gradf (the paper's resonance lists) or k_grad launch per step; plain FP64 ALUs
        k_ms = float(np.mean(t_data))
        fpe = GRADF_FLOP_PER_EVENT if paths == {8} else GRAD_FLOP_PER_EVENT
        flop = fpe * (args.n_data + args.n_norm)
        ach = flop / (k_ms * 1e-3) / 1e12
        roof = {"bound": "alu", "kernel": ("k_gradf (shape-specialised, gradient components in registers" if paths == {8} else "k_grad (generic") +
                ": NLL + dNLL/dH_k for all K = 27 couplings, data then norm tiles, one launch)",
                "achieved": ach, "peak": FP64_PEAK_NOMINAL / 1e12, "peak_source": "148 SMs x 64 DFMA/clk x 2 flop x 1.965 GHz", "unit": "TFLOP/s",
                "frac": ach / (FP64_PEAK_NOMINAL / 1e12), "traffic": None, "kernel_ms": k_ms, "flop_per_event": fpe,
                "hbm_frac": (BYTES_PER_EVENT_DATA * args.n_data + BYTES_PER_EVENT_NORM * args.n_norm) / (k_ms * 1e-3) / 1e9 / hbm_peak}
    elif args.cfg == 4:
        # dense form (--dense): k_batch (data, DMMA contraction) + k_herk (normalisation matrix, DMMA) + k_lineshape
        tm = model.last_call_timing()
        flop = 2 * 27 * 8 * 121 * args.n_data     # two helicities x 27 complex multiply-adds x 121 points per data event
        ach = flop / (tm["data_ms"] * 1e-3) / 1e12
        roof = {"bound": "tensor", "kernel": "k_batch<14, MODE_DATA> (dense FP64 DMMA contraction points x events, mma.sync.m8n8k4.f64)",
                "achieved": ach, "peak": FP64_PEAK_NOMINAL / 1e12, "peak_source": "FP64 tensor peak = FP64 FMA peak on B200, 148 x 64 x 2 x 1.965 GHz "
                "(the DMMA probe below measures it)", "unit": "TFLOP/s", "frac": ach / (FP64_PEAK_NOMINAL / 1e12), "traffic": None,
                "kernel_ms": tm["data_ms"], "flop_per_launch": flop, "norm_matrix_ms": tm["norm_ms"], "lineshape_ms": tm["lineshape_ms"]}
    elif paths == {4}:
        # one fused launch per step: lineshapes + combine + both reductions over the data tiles then the norm tiles
        k_ms = float(np.mean(t_data))
        nbytes = BYTES_PER_EVENT_DATA * args.n_data + BYTES_PER_EVENT_NORM * args.n_norm
        ach = nbytes / (k_ms * 1e-3) / 1e9
        roof = {"bound": "hbm", "kernel": "k_stream<MODE_FUSED> (the whole step: lineshapes + combine + -log L / normalisation reductions, data then norm tiles)",
                "achieved": ach, "peak": hbm_peak, "peak_source": f"MEASURED_PEAKS.json hbm_gbs ({peak_kind})", "unit": "GB/s",
                "frac": ach / hbm_peak, "traffic": TRAFFIC_NCU_BYTES if (args.n_data, args.n_norm) == (2_000_000, 10_000_000) else None,
                "alu_frac_nominal": FLOP_PER_EVENT * (args.n_data + args.n_norm) / (k_ms * 1e-3) / FP64_PEAK_NOMINAL,
                "kernel_ms": k_ms, "bytes_per_launch": nbytes, "bytes_per_event": [BYTES_PER_EVENT_DATA, BYTES_PER_EVENT_NORM],
                "flop_per_event": FLOP_PER_EVENT}
    else:
        ach = BYTES_PER_EVENT_NORM * args.n_norm / (norm_ms * 1e-3) / 1e9
        roof = {"bound": "hbm", "kernel": "k_stream<MODE_NORM> (fused lineshape + combine + reduce over the norm sample)",
                "achieved": ach, "peak": hbm_peak, "peak_source": f"MEASURED_PEAKS.json hbm_gbs ({peak_kind})", "unit": "GB/s",
                "frac": ach / hbm_peak, "traffic": None,
                "alu_frac_nominal": FLOP_PER_EVENT * args.n_norm / (norm_ms * 1e-3) / FP64_PEAK_NOMINAL,
                "kernel_ms": norm_ms, "bytes_per_event": BYTES_PER_EVENT_NORM, "flop_per_event": FLOP_PER_EVENT}
    fp64 = {"dfma_tflops_measured": B.probe_fp64(0, 4000) / 1e12, "dmma_tflops_measured": B.probe_fp64(1, 4000) / 1e12,
            "nominal_tflops": FP64_PEAK_NOMINAL / 1e12}
    if roof["bound"] == "hbm":
        # the streaming kernels' own TMA tile pipeline with the model arithmetic taken out (amp_probe_hbm_read, after the timed
        # region): how fast this access pattern reads HBM on this box, next to the copy figure `peak` is
        roof["read_probe_gbs"] = B.probe_hbm_read(BYTES_PER_EVENT_NORM * 12_000_000)
        roof["frac_of_read_probe"] = roof["achieved"] / roof["read_probe_gbs"]
    line = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
        "ms_per_step": dev_ms / args.steps, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "f64", "data": "synthetic",
        "config": {"workload": ("LASS variant (Eq. 9: LASS S-wave + 8 K* + Z, R=10, K=26) of " if LASS else "") + f"configs[{args.cfg}]: full K*+Z model (R=11, K=27), {args.n_data} data / {args.n_norm} norm events per GPU, "
                               f"P={P}, all lineshapes floating" + (", each step returns the NLL AND its analytic gradient in the 27 couplings" if args.grad else ""), "n_data": args.n_data, "n_norm": args.n_norm, "P": P,
                   "l2": "inputs (2.1 GB kinematics cache) larger than L2; no flush needed", "parallelism": f"replicas x{world}"},
        "e2e": {"value": e2e, "unit": UNIT, "h2d_bytes_per_step": int(h2d), "d2h_bytes_per_step": int(d2h),
                "note": "host wall clock around amp_set_params (host parameter arrays in) + amp_nll (host NLL out) per step; the events are "
                        "resident as in a fit (PAPER.md:45) - the one-off upload of the events from host buffers is setup.cold_start",
                # the other reading of "host buffers": EVERY evaluation uploads the events again (pinned host -> device -> kinematics
                # cache -> parameters -> NLL): P evaluations per cold start
                "value_if_events_uploaded_every_step": P * world / (info["cold_start"]["ms"] * 1e-3),
                "h2d_bytes_per_step_if_events_uploaded": int(info["cold_start"]["h2d_bytes"] + h2d)},
        "gpu_launches": int(launches),
        "event_evals_per_s": value * (args.n_data + args.n_norm),
        "phase_ms": {"lineshape": float(np.mean(t_line)), "data": float(np.mean(t_data)), "norm": norm_ms},
        "roofline": roof, "fp64_probe": fp64, "clocks": clocks,
        "setup": info, "nll_last": [float(v) for v in np.atleast_1d(nll_last)[:3]],
    }
    if not args.no_cpu_baseline:
        line["cpu_baseline"] = cpu_baseline(args)
    print(json.dumps(line))
    if world > 1:
        dist.destroy_process_group()


def cpu_baseline(args, target_evals=None):
    """The oracle, as it stands, timed on this box's host cores on a bounded sample of the same workload (about 10-30 s
    of CPU work): same model and call pattern, data and norm sizes scaled down by one factor (1 = the full workload) and
    the evaluation repeated so that about `target_evals` event-evaluations are timed; data events drawn by
    oracle-driven accept-reject (no oracle input comes from the CUDA path)."""
    from oracle import oracle as O
    cfg = args.cfg
    P = 121 if cfg == 4 else 1
    if target_evals is None:   # ~10-20 s on 16 cores: the oracle shares an event's angles between the points of a batch
        target_evals = 180_000_000 if P > 1 else 36_000_000
    total = args.n_data + args.n_norm
    frac = min(1.0, target_evals / (P * total))
    n = max(int(args.n_data * frac), 1000)
    m = max(int(args.n_norm * frac), 5000)
    reps = max(1, int(round(target_evals / (P * (n + m)))))
    res, c = model_def(cfg)
    Mo = O.Model(W.DECAY, res)
    xn, wn = W.norm_events(cfg, m)
    x, eff = W.data_events(cfg, lambda xx, ee: Mo.eval_events(c, xx, ee), n=n)
    dt = 0.0
    for r in range(reps):
        cs, mws = step_params(cfg, c, r)
        t0 = time.perf_counter()
        Mo.nll(cs, x, eff, xn, wn, mass_width=mws)
        dt += time.perf_counter() - t0
    full = dt / reps * total / (n + m)            # time of one full-size call (scaled linearly if the sample is smaller)
    return {"value": P / full, "unit": UNIT, "cores": O.num_threads(), "kind": "oracle",
            "sample": f"{reps} x ({n} data + {m} norm events, same model, P={P}), {dt:.2f} s measured"
                      + ("" if n + m == total else f", scaled linearly to {args.n_data}+{args.n_norm}"),
            "event_evals_per_s": P * (n + m) * reps / dt}


def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    from oracle import oracle as O
    cfg = args.cfg
    P = 121 if cfg == 4 else 1
    # bounded sample per step so that steps+warmup finish in a few minutes
    per_step = max(30_000_000 // (P * max(args.steps + args.warmup, 1)), 4000)
    per_step = min(per_step, args.n_data + args.n_norm)
    n = max(int(per_step * args.n_data / (args.n_data + args.n_norm)), 500)
    m = max(per_step - n, 2000)
    res, c = model_def(cfg)
    Mo = O.Model(W.DECAY, res)
    xn, wn = W.norm_events(cfg, m)
    x, eff = W.data_events(cfg, lambda xx, ee: Mo.eval_events(c, xx, ee), n=n)
    times = []
    for s in range(args.warmup + args.steps):
        cs, mws = step_params(cfg, c, s)
        t0 = time.perf_counter()
        Mo.nll(cs, x, eff, xn, wn, mass_width=mws)
        if s >= args.warmup:
            times.append(time.perf_counter() - t0)
    dt = float(np.sum(times))
    scale = (args.n_data + args.n_norm) / (n + m)
    value = P * args.steps / (dt * scale)
    sample = f"{n} data + {m} norm events per step (same model, P={P}), scaled linearly to {args.n_data}+{args.n_norm}"
    line = {"impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": int(os.environ.get("WORLD_SIZE", "1")),
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": dt * scale / args.steps * 1e3, "higher_is_better": True,
            "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": f"configs[{cfg}]: full K*+Z model (R=11, K=27), {args.n_data} data / {args.n_norm} norm events, P={P}, "
                                   "all lineshapes floating", "n_data": args.n_data, "n_norm": args.n_norm, "P": P},
            "cpu_baseline": {"value": value, "unit": UNIT, "cores": O.num_threads(), "kind": "oracle", "sample": sample},
            "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}, "gpu_launches": 0}
    print(json.dumps(line))


def run_pseudo(args):
    """Context only (not the headline metric): the workload of the paper's one performance figure (Fig. 2, PAPER.md:201,
    207-209: pseudo-experiments of 10,000 events generated and fitted with models of an increasing number of K*s; the figure's
    values are not in the text).  Per model: --steps pseudo-experiments are generated on the device (amp_generate), fitted
    from a perturbed start on the analytic gradient (amp_nll_grad) and given Hessian errors; wall clock around all of it."""
    import torch
    from paper_2007_14931_b200 import binding as B
    from paper_2007_14931_b200 import fit as F
    torch.cuda.set_device(0)
    ks = W.KSTARS
    models = {"3 K*": (1, 3, 4), "6 K*": (1, 2, 3, 4, 5, 6), "10 K*": tuple(range(10))}
    lo, hi, cm = W.DECAY[2] + W.DECAY[3] + W.M_LO_MARGIN, W.M_HI, W.COS_MAX
    xn = torch.as_tensor(W.phase_space_events(np.random.default_rng(77), args.n_norm)).cuda()
    per_model, total_t, total_n = {}, 0.0, 0
    for name, idx in models.items():
        res = [(ks[i][1], ks[i][2], ks[i][3], ks[i][4], W.RADIUS) for i in idx]
        slots = W.slot_table(res)
        rng = np.random.default_rng(len(idx))
        c = rng.uniform(0.6, 1.4, len(slots)) * np.exp(1j * rng.uniform(-np.pi, np.pi, len(slots)))
        fixed = [k for k, (r, lam) in enumerate(slots) if r == 0 and lam == 0]
        c[fixed[0]] = 1.0
        M = B.Model(W.DECAY, res)
        M.load_norm(xn)
        F.pull_study(M, c, 2, args.pseudo, 1, lo, hi, cm, fixed=fixed)            # warm-up (first launches, the matrix M)
        torch.cuda.synchronize()
        t0 = time.perf_counter()
        out = F.pull_study(M, c, args.steps, args.pseudo, 1000, lo, hi, cm, fixed=fixed)
        torch.cuda.synchronize()
        dt = time.perf_counter() - t0
        per_model[name] = {"free_parameters": 2 * (len(slots) - 1), "ms_per_pseudo_experiment": dt / args.steps * 1e3,
                           "likelihood_calls": float(out["n_calls"].mean()), "converged": float(out["converged"].mean())}
        total_t += dt
        total_n += args.steps
    print(json.dumps({"metric": "pseudo-experiments generated and fitted per second (context: workload of the paper's Fig. 2)", "value": total_n / total_t,
                      "unit": "pseudo-experiments/s", "n_gpus": 1, "steps": args.steps, "warmup": 2, "higher_is_better": True, "vs_baseline": None,
                      "dtype": "f64", "data": "synthetic",
                      "config": {"workload": f"{args.pseudo} events per pseudo-experiment, {args.n_norm} normalisation points, masses and widths fixed, "
                                             "generate (amp_generate) + BFGS fit on amp_nll_grad + Hessian errors", "models": per_model}}))


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=200)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="own", choices=["own", "reference"])
    ap.add_argument("--cfg", type=int, default=3, choices=[3, 4], help="3: P=1 all lineshapes floating (headline); 4: P=121 fit-loop pattern")
    ap.add_argument("--n-data", type=int, default=2_000_000)
    ap.add_argument("--n-norm", type=int, default=10_000_000)
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--dense", action="store_true", help="--cfg 4 through the dense DMMA contraction instead of the gradient-batch kernel")
    ap.add_argument("--grad", action="store_true", help="--cfg 3 steps that also return the analytic gradient in all couplings (amp_nll_grad)")
    ap.add_argument("--lass", action="store_true", help="configs[3] call pattern on the LASS variant of the model (Eqs. 7-9; SURVEY.md 8(f)-1)")
    ap.add_argument("--pseudo", type=int, default=0, metavar="N_EVENTS",
                    help="context mode: generate and fit --steps pseudo-experiments of N_EVENTS each for models of 3, 6 and 10 K*s (the paper's Fig. 2 workload)")
    args = ap.parse_args()
    if args.pseudo:
        args.steps = min(args.steps, 50)
        args.n_norm = min(args.n_norm, 1_000_000)
        return run_pseudo(args)
    global LASS
    LASS = bool(args.lass)
    if LASS and args.cfg != 3:
        ap.error("--lass goes with --cfg 3")
    args.warmup = max(args.warmup, 3) if args.impl == "own" else args.warmup
    if args.impl == "reference":
        run_reference(args)
    else:
        run_own(args)


if __name__ == "__main__":
    main()
