#!/usr/bin/env python
"""bench.py — NLL evaluations per second of the 4D amplitude model on B200 (BASELINE.json metric).

Workload (config.workload): BASELINE.json configs[3] at its headline point — the full K* + Z model
(11 resonances, K = 27 couplings), 2M data events and 10M normalisation events, FP64 structure-of-arrays,
every lineshape floating: each timed step is one `amp_set_params` (new masses and widths for all 11
resonances, new couplings) + one `amp_nll` through the C ABI, i.e. one pass of the whole hot path
(lineshapes -> combine -> normalisation -> -log L reduction) over the data and the normalisation sample.
The kinematics cache is built once per dataset (step a1, outside the per-step metric, reported separately).

The default run then times configs[4] (P = 121: the MINUIT-style gradient batch of the fit loop) on the same
loaded events and prints it inside the same JSON line as "cfg4".

One JSON line on stdout (rank 0).  `--impl reference` times the CPU oracle instead (rank 0 only).
Multi-GPU: `--gpus N` under torchrun (or alone: bench.py starts the N ranks itself) runs N independent replicas (weak
scaling, no data-path collective: the paper's validation is hundreds of independent toy fits); `--shard`
cuts ONE data set N ways (strong scaling) with the 2 P-double all-reduce on NCCL inside every timed step.
"""
import argparse
import csv
import hashlib
import json
import os
import socket
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
# Algorithmic flop per event of the gradient batch of configs[4] in its sparse form: point 0 (730) + 31 slots
# (Breit-Wigner of point 0 from the saved barrier factors ~20, angular factor ~8, two complex products 12, and the expansion
# coefficients T2 = 2 sum conj(A(0)) SLOT, n = sum |SLOT|^2: 25) + 100 coupling points (S(0) + Re(coef T2) + |coef|^2 n: 6, guard 1,
# accumulate 1) + 20 mass/width points (perturbed Breit-Wigner ~22, difference to point 0 and |coef|^2: 5, expansion 6)
DELTA_FLOP_PER_EVENT = 730.0 + 31 * 65.0 + 100 * 8.0 + 20 * 33.0
# normalisation events: the 100 coupling points cost nothing per point there — three weighted sums per group of four on one slot
# (25 groups x 3 FMA), the points are formed from them once per launch
DELTA_FLOP_PER_NORM_EVENT = 730.0 + 31 * 65.0 + 25 * 6.0 + 20 * 33.0
# The shape-specialised gradient-batch kernel (deltaf.cu), per event: point 0 (730) + the W / Y sums and the per-spin
# scalings (140 + 50) + the eleven lineshapes evaluated again from the saved barrier factors (11 x 14) + per coupling position in use
# (25): L = conj(BW) X (6), n (2), data: four points x (3 FMA + the product through the exchange) = 28 + guard 4, normalisation: three
# sums (3) + per floating lineshape (5): Q (22), G and n_R (44), four points x (BW(p) 12, Delta 4, |Delta|^2 3, x 6, exchange 1)
DELTAF_FLOP_PER_EVENT = 730.0 + 190.0 + 154.0 + 25 * 40.0 + 5 * 170.0
DELTAF_FLOP_PER_NORM_EVENT = 730.0 + 190.0 + 154.0 + 25 * 11.0 + 5 * 170.0
# The same batch as three launches (batch mode 0: deltan.cu pass 0 and pass 1 over the normalisation events, then deltaf.cu over the
# data events; DESIGN.md 5.6a/5.6b): FP64 operations EXECUTED per event (DFMA = 2, DMUL / DADD / MUFU = 1), read off the instruction
# counts of the ncu source page of profiles/r02_ncu_full_deltaf3.csv's report — both passes carry the forward pass of point 0.
DELTAN0_FLOP_PER_NORM_EVENT = 1019.0
DELTAN1_FLOP_PER_NORM_EVENT = 1705.0
DELTAF_DATA_FLOP_PER_EVENT = 3086.0
# analytic gradient: the point (730) + per coupling slot: angular factor ~8, T = sum_xi conj(g) A 16, conj(BW) T 8, weight 2
GRAD_FLOP_PER_EVENT = 730.0 + 27 * 34.0
# its shape-specialised form (gradf.cu): the point (730) + the three W_lambda and three Y_lambda' (u A, conj(g) A:
# ~110) + one real scaling of them per spin (~30) + per coupling slot conj(BW) X into its register pair (4 FMA = 8)
GRADF_FLOP_PER_EVENT = 730.0 + 140.0 + 27 * 8.0

# `ncu --set full` captures whose DRAM traffic the roofline object quotes: profiles/captures.json lists, per kernel, the CSV
# (plain `ncu -i <rep> --page raw --csv --metrics ...` output), the sizes it was taken at and the SHA-256 of the kernel's source
# files at capture time.  `traffic` is null when the sources have changed since (a stale capture is not evidence).
CAPTURES = os.path.join(ROOT, "profiles", "captures.json")

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


def source_hash(files):
    h = hashlib.sha256()
    for f in files:
        h.update(open(os.path.join(ROOT, f), "rb").read())
    return h.hexdigest()


def traffic_from_profiles(key, n_data, n_norm):
    """(dram bytes read + written per launch, source) of the committed `ncu --set full` capture of kernel `key`, or (None, why)"""
    try:
        cap = json.load(open(CAPTURES))[key]
    except Exception as e:   # noqa: BLE001
        return None, f"no capture listed for {key} in profiles/captures.json ({type(e).__name__})"
    if (cap["n_data"], cap["n_norm"]) != (n_data, n_norm):
        return None, f"capture {cap['csv']} was taken at {cap['n_data']}/{cap['n_norm']} events"
    if source_hash(cap["sources"]) != cap["sha256"]:
        return None, f"kernel sources changed since capture {cap['csv']}"
    rows = list(csv.reader(open(os.path.join(ROOT, "profiles", cap["csv"]))))
    hdr, units, data = rows[0], rows[1], [r for r in rows[2:] if r]
    if cap.get("kernel"):   # a capture of several kernels: the rows of this one
        data = [r for r in data if cap["kernel"] in r[hdr.index("Kernel Name")]]
        if not data:
            return None, f"no row of {cap['kernel']} in {cap['csv']}"
    mult = {"byte": 1.0, "Kbyte": 1e3, "Mbyte": 1e6, "Gbyte": 1e9}
    tot = []
    for r in data:
        t = 0.0
        for name in ("dram__bytes_read.sum", "dram__bytes_write.sum"):
            j = hdr.index(name)
            t += float(r[j]) * mult[units[j]]
        tot.append(t)
    return float(np.mean(tot)), f"profiles/{cap['csv']} ({len(tot)} launches, mean)"


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
            time.sleep(0.0005)

    def window(self, t0, t1):
        """clocks over [t0, t1] of the perf_counter clock (the sampler keeps running)"""
        if not getattr(self, "nv", None):
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvml unavailable: " + getattr(self, "err", "")]}
        nv = self.nv
        rows = [r for r in list(self.rows) if t0 <= r[0] <= t1] or list(self.rows)[-3:]
        names = {"hw_slowdown": nv.nvmlClocksEventReasonHwSlowdown, "hw_thermal_slowdown": nv.nvmlClocksEventReasonHwThermalSlowdown,
                 "sw_thermal_slowdown": nv.nvmlClocksEventReasonSwThermalSlowdown, "sw_power_cap": nv.nvmlClocksEventReasonSwPowerCap}
        reasons = sorted(k for k, bit in names.items() if any(r[2] & bit for r in rows))
        return {"sm_mhz": float(np.median([r[1] for r in rows])) if rows else None, "sm_max_mhz": float(self.smax), "reasons": reasons,
                "power_w_max": max(r[3] for r in rows) if rows else None, "samples": len(rows)}

    def stop(self):
        self.stop_flag = True
        if self.thread:
            self.thread.join(timeout=2)


def generate_events(args, device):
    """seeded synthetic events of the workload on the HOST.  Data events: accept-reject driven by the product's own
    amp_eval_events (toy generation with the fitter itself)."""
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
    return x, eff, xn, wn, time.time() - t0


def build_workload(args, device):
    """events on the device, model with data + norm loaded; the cold start (pinned host events -> device -> kinematics cache ->
    first NLL) is timed once by the wall clock"""
    import torch
    from paper_2007_14931_b200 import binding as B
    res, c = model_def(args.cfg)
    x, eff, xn, wn, t_gen = generate_events(args, device)
    model = B.Model(W.DECAY, res)
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
    cs, mws = step_params(args.cfg, c, 0)
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


def timed_steps(step_fn, steps, warmup, world, device, sampler=None):
    """`warmup` untimed steps, then EXACTLY `steps` timed ones between a barrier + synchronize on both sides: total device
    time from CUDA events on the launching stream (max over ranks), per-step device and wall times."""
    import torch
    import torch.distributed as dist
    for s in range(warmup):
        step_fn(s)
    if world > 1:
        dist.barrier()
    torch.cuda.synchronize()
    ev = [torch.cuda.Event(enable_timing=True) for _ in range(steps + 1)]
    walls, last = [], None
    t_wall0 = time.perf_counter()
    ev[0].record()
    for k in range(steps):
        t0 = time.perf_counter()
        last = step_fn(warmup + k)      # nothing else in the timed region: amp_set_params + amp_nll through the C ABI
        walls.append(time.perf_counter() - t0)
        ev[k + 1].record()
    torch.cuda.synchronize()
    t_wall = time.perf_counter() - t_wall0
    if world > 1:
        dist.barrier()
    clocks = sampler.window(t_wall0, t_wall0 + t_wall) if sampler is not None else None
    dev_ms = ev[0].elapsed_time(ev[steps])
    per_step = [ev[k].elapsed_time(ev[k + 1]) for k in range(steps)]
    if world > 1:
        t = torch.tensor([dev_ms, t_wall * 1e3], dtype=torch.float64, device=device)
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        dev_ms, t_wall = float(t[0]), float(t[1]) / 1e3
    return {"dev_ms": dev_ms, "wall_s": t_wall, "per_step_ms": per_step, "per_step_wall_ms": [w * 1e3 for w in walls], "last": last, "clocks": clocks}


def roofline(model, args, cfg, n_data, n_norm, hbm_peak, peak_kind, steps):
    """the roofline object of the dominant kernel of the steps just timed (kernel durations: the library's CUDA event pairs)"""
    st = model.last_call_stats()
    path = st["norm_path"]
    if path in (4, 5, 7, 8, 9):
        t_k = [float(v) for v in model.recent_launch_ms(min(steps, 256))]   # the launches of the `steps` calls just timed
        phase = {"lineshape": 0.0, "data": float(np.mean(t_k)), "norm": 0.0}
    else:
        tm = model.last_call_timing()
        t_k = [tm["data_ms"]]
        phase = {"lineshape": tm["lineshape_ms"], "data": tm["data_ms"], "norm": tm["norm_ms"]}
    k_ms, k_med = float(np.mean(t_k)), float(np.median(t_k))
    nbytes = BYTES_PER_EVENT_DATA * n_data + BYTES_PER_EVENT_NORM * n_norm
    if cfg == 4 and path == 9 and st["launches"] == 3:
        # gradient batch of the paper's resonance lists: k_deltan pass 0, pass 1 (normalisation events), k_deltaf (data events) per step,
        # all bound by the plain FP64 ALUs (DESIGN.md 5.6a/b).  The ring times the three together; the last step's event split gives the shares.
        tm = model.last_call_timing()
        parts = [("k_deltan<pass 0> (normalisation events: sum w S0 and the 54 sums of L', registers)", tm["norm_ms"], DELTAN0_FLOP_PER_NORM_EVENT, n_norm, "k_deltan0_cfg4"),
                 ("k_deltan<pass 1> (normalisation events: sums of n' and the lineshape sums, registers; scatters the totals)", tm["final_ms"], DELTAN1_FLOP_PER_NORM_EVENT, n_norm, "k_deltan1_cfg4"),
                 ("k_deltaf (data events: r = S(p)/S(0) of 120 points through the shared-memory value tile; forms NLL(p), I(p))", tm["data_ms"], DELTAF_DATA_FLOP_PER_EVENT, n_data, "k_deltaf_cfg4")]
        tsum = sum(p[1] for p in parts)
        peak = FP64_PEAK_NOMINAL / 1e12
        launches = []
        for name, ms, fpe, nev, key in parts:
            ms_avg = ms / tsum * k_ms                      # this launch's share of the last step x the mean over the timed steps
            traffic, tsrc = traffic_from_profiles(key, n_data, n_norm)
            launches.append({"kernel": name, "kernel_ms": ms_avg, "flop_per_event": fpe, "events": nev, "achieved": fpe * nev / (ms_avg * 1e-3) / 1e12,
                             "frac": fpe * nev / (ms_avg * 1e-3) / 1e12 / peak, "traffic": traffic, "traffic_source": tsrc})
        dom = max(launches, key=lambda l: l["kernel_ms"])
        flop = sum(l["flop_per_event"] * l["events"] for l in launches)
        flop1 = DELTAF_FLOP_PER_EVENT * n_data + DELTAF_FLOP_PER_NORM_EVENT * n_norm
        roof = {"bound": "alu", "kernel": dom["kernel"], "achieved": dom["achieved"], "peak": peak,
                "peak_source": "148 SMs x 64 DFMA/clk x 2 flop x 1.965 GHz (DESIGN.md 6; the DFMA probe below measures it)", "unit": "TFLOP/s",
                "frac": dom["frac"], "traffic": dom["traffic"], "traffic_source": dom["traffic_source"], "kernel_ms": dom["kernel_ms"],
                "flop_per_event": dom["flop_per_event"], "flop_per_launch": dom["flop_per_event"] * dom["events"],
                "flop_note": "FP64 operations executed per event (DFMA = 2), from the ncu source page; the longest of the step's three launches",
                "step": {"kernel_ms": k_ms, "kernel_ms_median": k_med, "launches": launches, "flop": flop, "achieved": flop / (k_ms * 1e-3) / 1e12,
                         "frac": flop / (k_ms * 1e-3) / 1e12 / peak,
                         "frac_at_one_launch_flop": flop1 / (k_ms * 1e-3) / 1e12 / peak,
                         "note": "frac: the three launches' executed flop (both normalisation passes carry the forward pass of point 0) over their total time; "
                                 "frac_at_one_launch_flop: the algorithmic flop of the one-launch form (batch mode 4) over the same time",
                         "hbm_frac": (nbytes + BYTES_PER_EVENT_NORM * n_norm) / (k_ms * 1e-3) / 1e9 / hbm_peak}}
    elif cfg == 4 and path == 9:
        # ... as ONE k_deltaf launch over both samples (batch mode 4)
        flop = DELTAF_FLOP_PER_EVENT * n_data + DELTAF_FLOP_PER_NORM_EVENT * n_norm
        ach = flop / (k_ms * 1e-3) / 1e12
        traffic, tsrc = traffic_from_profiles("k_deltaf1_cfg4", n_data, n_norm)
        roof = {"bound": "alu", "kernel": "k_deltaf (shape-specialised gradient batch: point 0 + 100 coupling points + 20 mass/width points, data then norm units, one launch)",
                "achieved": ach, "peak": FP64_PEAK_NOMINAL / 1e12,
                "peak_source": "148 SMs x 64 DFMA/clk x 2 flop x 1.965 GHz (DESIGN.md 6; the DFMA probe below measures it)", "unit": "TFLOP/s",
                "frac": ach / (FP64_PEAK_NOMINAL / 1e12), "traffic": traffic, "traffic_source": tsrc, "kernel_ms": k_ms, "kernel_ms_median": k_med,
                "flop_per_event": [DELTAF_FLOP_PER_EVENT, DELTAF_FLOP_PER_NORM_EVENT], "flop_per_launch": flop,
                "flop_note": "algorithmic flop of THIS design; the general kernel (k_delta, --general) needs 4205 / 3555 flop per event for the same batch",
                "hbm_frac": nbytes / (k_ms * 1e-3) / 1e9 / hbm_peak}
    elif cfg == 4 and path == 5:
        # gradient batch: one fused k_delta launch per step, bound by the plain FP64 ALUs (DESIGN.md 5.6 / 6)
        flop = DELTA_FLOP_PER_EVENT * n_data + DELTA_FLOP_PER_NORM_EVENT * n_norm
        ach = flop / (k_ms * 1e-3) / 1e12
        traffic, tsrc = traffic_from_profiles("k_delta_cfg4", n_data, n_norm)
        roof = {"bound": "alu", "kernel": "k_delta (gradient batch: point 0 + 120 sparse points, data then norm tiles, one launch)",
                "achieved": ach, "peak": FP64_PEAK_NOMINAL / 1e12,
                "peak_source": "148 SMs x 64 DFMA/clk x 2 flop x 1.965 GHz (DESIGN.md 6; the DFMA probe below measures it)", "unit": "TFLOP/s",
                "frac": ach / (FP64_PEAK_NOMINAL / 1e12), "traffic": traffic, "traffic_source": tsrc, "kernel_ms": k_ms, "kernel_ms_median": k_med,
                "flop_per_event": [DELTA_FLOP_PER_EVENT, DELTA_FLOP_PER_NORM_EVENT], "flop_per_launch": flop,
                "hbm_frac": nbytes / (k_ms * 1e-3) / 1e9 / hbm_peak}
    elif path in (7, 8):
        # --grad: NLL and analytic gradient in one k_gradf (the paper's resonance lists) or k_grad launch per step; plain FP64 ALUs
        fpe = GRADF_FLOP_PER_EVENT if path == 8 else GRAD_FLOP_PER_EVENT
        flop = fpe * (n_data + n_norm)
        ach = flop / (k_ms * 1e-3) / 1e12
        traffic, tsrc = traffic_from_profiles("k_gradf_cfg3" if path == 8 else "k_grad_cfg3", n_data, n_norm)
        roof = {"bound": "alu", "kernel": ("k_gradf (shape-specialised, gradient components in registers" if path == 8 else "k_grad (generic") +
                ": NLL + dNLL/dH_k for all K = 27 couplings, data then norm tiles, one launch)",
                "achieved": ach, "peak": FP64_PEAK_NOMINAL / 1e12, "peak_source": "148 SMs x 64 DFMA/clk x 2 flop x 1.965 GHz", "unit": "TFLOP/s",
                "frac": ach / (FP64_PEAK_NOMINAL / 1e12), "traffic": traffic, "traffic_source": tsrc, "kernel_ms": k_ms, "kernel_ms_median": k_med,
                "flop_per_event": fpe, "hbm_frac": nbytes / (k_ms * 1e-3) / 1e9 / hbm_peak}
    elif cfg == 4:
        # dense form (--dense): k_batch (data, DMMA contraction) + k_herk (normalisation matrix, DMMA) + k_lineshape
        tm = model.last_call_timing()
        flop = 2 * 27 * 8 * 121 * n_data     # two helicities x 27 complex multiply-adds x 121 points per data event
        ach = flop / (tm["data_ms"] * 1e-3) / 1e12
        roof = {"bound": "tensor", "kernel": "k_batch<14, MODE_DATA> (dense FP64 DMMA contraction points x events, mma.sync.m8n8k4.f64)",
                "achieved": ach, "peak": FP64_PEAK_NOMINAL / 1e12, "peak_source": "FP64 tensor peak = FP64 FMA peak on B200, 148 x 64 x 2 x 1.965 GHz "
                "(the DMMA probe below measures it)", "unit": "TFLOP/s", "frac": ach / (FP64_PEAK_NOMINAL / 1e12), "traffic": None,
                "kernel_ms": tm["data_ms"], "flop_per_launch": flop, "norm_matrix_ms": tm["norm_ms"], "lineshape_ms": tm["lineshape_ms"]}
    elif path == 4:
        # one fused launch per step: lineshapes + combine + both reductions over the data tiles then the norm tiles
        ach = nbytes / (k_ms * 1e-3) / 1e9
        traffic, tsrc = traffic_from_profiles("k_stream_fused_cfg3", n_data, n_norm)
        roof = {"bound": "hbm", "kernel": "k_stream<MODE_FUSED> (the whole step: lineshapes + combine + -log L / normalisation reductions, data then norm tiles)",
                "achieved": ach, "peak": hbm_peak, "peak_source": f"MEASURED_PEAKS.json hbm_gbs ({peak_kind})", "unit": "GB/s",
                "frac": ach / hbm_peak, "traffic": traffic, "traffic_source": tsrc,
                "alu_frac_nominal": FLOP_PER_EVENT * (n_data + n_norm) / (k_ms * 1e-3) / FP64_PEAK_NOMINAL,
                "kernel_ms": k_ms, "kernel_ms_median": k_med, "bytes_per_launch": nbytes, "bytes_per_event": [BYTES_PER_EVENT_DATA, BYTES_PER_EVENT_NORM],
                "flop_per_event": FLOP_PER_EVENT}
    else:
        norm_ms = phase["norm"]
        ach = BYTES_PER_EVENT_NORM * n_norm / (norm_ms * 1e-3) / 1e9
        roof = {"bound": "hbm", "kernel": "k_stream<MODE_NORM> (fused lineshape + combine + reduce over the norm sample)",
                "achieved": ach, "peak": hbm_peak, "peak_source": f"MEASURED_PEAKS.json hbm_gbs ({peak_kind})", "unit": "GB/s",
                "frac": ach / hbm_peak, "traffic": None,
                "alu_frac_nominal": FLOP_PER_EVENT * n_norm / (norm_ms * 1e-3) / FP64_PEAK_NOMINAL,
                "kernel_ms": norm_ms, "bytes_per_event": BYTES_PER_EVENT_NORM, "flop_per_event": FLOP_PER_EVENT}
    return roof, phase, st


def measure(model, args, cfg, c, steps, warmup, world, device, sampler, n_data, n_norm, hbm):
    """time `steps` steps of configuration `cfg` on the loaded model -> the fields of a bench line"""
    P = 121 if cfg == 4 else 1
    params = [step_params(cfg, c, s) for s in range(warmup + steps)]

    def one_step(s):
        cs, mws = params[s]
        model.set_params(cs, mws)
        if args.grad:
            return np.array([model.nll_grad()[0]])   # NLL + its analytic gradient in all K couplings, one launch
        return model.nll()

    t = timed_steps(one_step, steps, warmup, world, device, sampler)
    roof, phase, st = roofline(model, args, cfg, n_data, n_norm, *hbm, steps)
    evals = P * steps * world          # replicas: every rank evaluates its own data set
    h2d = 8 * (P * model.K * 2 + P * model.R * 2)
    return {"value": evals / (t["dev_ms"] * 1e-3), "ms_per_step": t["dev_ms"] / steps, "ms_per_step_median": float(np.median(t["per_step_ms"])),
            "steps": steps, "P": P,
            "e2e": {"value": evals / t["wall_s"], "unit": UNIT, "h2d_bytes_per_step": int(h2d), "d2h_bytes_per_step": int(8 * P),
                    "ms_per_step_median": float(np.median(t["per_step_wall_ms"]))},
            "gpu_launches": int(st["launches"] * steps), "phase_ms": phase, "roofline": roof, "clocks": t["clocks"],
            "nll_last": [float(v) for v in np.atleast_1d(t["last"])[:3]]}


def workload_text(cfg, n_data, n_norm, P, grad=False):
    return (("LASS variant (Eq. 9: LASS S-wave + 8 K* + Z, R=10, K=26) of " if LASS else "") +
            f"configs[{cfg}]: full K*+Z model (R=11, K=27), {n_data} data / {n_norm} norm events per GPU, P={P}, " +
            ("all lineshapes floating" if cfg == 3 else "gradient batch of a fit step: 60 free parameters (46 K* moduli/phases, 4 Z, Z mass/width, 4 K* masses/widths) x +-h around a moving central point") +
            (", each step returns the NLL AND its analytic gradient in the 27 couplings" if grad else ""))


def run_own(args):
    import torch
    import torch.distributed as dist

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if local >= torch.cuda.device_count():
        raise SystemExit(f"bench.py: local rank {local} has no GPU (this box has {torch.cuda.device_count()}): --gpus N needs N devices")
    torch.cuda.set_device(local)
    device = torch.device("cuda", local)
    if world > 1:
        dist.init_process_group("nccl", device_id=device)
    from paper_2007_14931_b200 import binding as B

    if args.shard:
        return run_shard(args, world, rank, device)
    model, c, info = build_workload(args, device)
    if args.dense:
        model.set_batch_mode(2)   # configs[4] as the dense DMMA contraction + extended-basis normalisation matrix
    if args.one_launch:
        model.set_batch_mode(4)   # configs[4] as ONE k_deltaf launch over both samples (the cross-check form of the three-launch default)
    if args.general:
        model.set_batch_mode(3)   # configs[4] through the general gradient-batch kernel (k_delta) instead of the shape-specialised one
    sampler = ClockSampler(local)
    if rank == 0:
        sampler.start()
        time.sleep(0.01)
    hbm = measured_peaks()
    main = measure(model, args, args.cfg, c, args.steps, args.warmup, world, device, sampler if rank == 0 else None, args.n_data, args.n_norm, hbm)
    # the default run: configs[4] (P = 121) on the same loaded events, in the same line
    cfg4 = None
    if args.cfg == 3 and not (args.grad or args.lass or args.dense or args.general or args.one_launch or args.no_cfg4):
        steps4 = max(20, min(args.steps, 50))
        cfg4 = measure(model, args, 4, W.couplings(4), steps4, 3, world, device, sampler if rank == 0 else None, args.n_data, args.n_norm, hbm)
    sweep = None
    if args.sweep and rank == 0:
        sweep = run_sweep(args, device, sampler, hbm)
    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return
    sampler.stop()
    fp64 = {"dfma_tflops_measured": B.probe_fp64(0, 4000) / 1e12, "dmma_tflops_measured": B.probe_fp64(1, 4000) / 1e12,
            "nominal_tflops": FP64_PEAK_NOMINAL / 1e12}
    roof = main["roofline"]
    if roof["bound"] == "hbm":
        # the streaming kernels' own TMA tile pipeline with the model arithmetic taken out (amp_probe_hbm_read, after the timed
        # region): how fast this access pattern reads HBM on this box, next to the copy figure `peak` is
        roof["read_probe_gbs"] = B.probe_hbm_read(BYTES_PER_EVENT_NORM * 12_000_000)
        roof["frac_of_read_probe"] = roof["achieved"] / roof["read_probe_gbs"]
    P = main["P"]
    e2e = dict(main["e2e"])
    e2e.update({"note": "host wall clock around amp_set_params (host parameter arrays in) + amp_nll (host NLL out) per step; the events are "
                        "resident as in a fit (PAPER.md:45) - the one-off upload of the events from host buffers is setup.cold_start",
                # the other reading of "host buffers": EVERY evaluation uploads the events again (pinned host -> device -> kinematics
                # cache -> parameters -> NLL): P evaluations per cold start
                "value_if_events_uploaded_every_step": P * world / (info["cold_start"]["ms"] * 1e-3),
                "h2d_bytes_per_step_if_events_uploaded": int(info["cold_start"]["h2d_bytes"] + e2e["h2d_bytes_per_step"])})
    line = {
        "metric": METRIC, "value": main["value"], "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
        "ms_per_step": main["ms_per_step"], "ms_per_step_median": main["ms_per_step_median"], "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "f64", "data": "synthetic",
        "config": {"workload": workload_text(args.cfg, args.n_data, args.n_norm, P, args.grad), "n_data": args.n_data, "n_norm": args.n_norm, "P": P,
                   "l2": "inputs (2.1 GB kinematics cache) larger than L2; no flush needed", "parallelism": f"replicas x{world}"},
        "e2e": e2e, "gpu_launches": main["gpu_launches"],
        "event_evals_per_s": main["value"] * (args.n_data + args.n_norm),
        "phase_ms": main["phase_ms"], "roofline": roof, "fp64_probe": fp64, "clocks": main["clocks"],
        "setup": info, "nll_last": main["nll_last"],
    }
    if cfg4 is not None:
        line["cfg4"] = {"metric": METRIC, "unit": UNIT, "value": cfg4["value"], "ms_per_step": cfg4["ms_per_step"], "ms_per_step_median": cfg4["ms_per_step_median"],
                        "steps": cfg4["steps"], "warmup": 3, "workload": workload_text(4, args.n_data, args.n_norm, 121),
                        "e2e": cfg4["e2e"], "gpu_launches": cfg4["gpu_launches"], "roofline": cfg4["roofline"], "clocks": cfg4["clocks"],
                        "nll_last": cfg4["nll_last"]}
        line["gpu_launches"] += cfg4["gpu_launches"]
    if sweep is not None:
        line["sweep"] = sweep
    if not args.no_cpu_baseline:
        line["cpu_baseline"] = cpu_baseline(args)
    print(json.dumps(line))
    if world > 1:
        dist.destroy_process_group()


def run_sweep(args, device, sampler, hbm):
    """the six points of BASELINE.json configs[3]: data in {1M, 2M, 8M} x normalisation in {2M, 10M}, each its own loaded model"""
    out = []
    for n_norm in (2_000_000, 10_000_000):
        for n_data in (1_000_000, 2_000_000, 8_000_000):
            a = argparse.Namespace(**vars(args))
            a.n_data, a.n_norm = n_data, n_norm
            model, c, _info = build_workload(a, device)
            m = measure(model, a, 3, c, a.steps, a.warmup, 1, device, sampler, n_data, n_norm, hbm)
            out.append({"n_data": n_data, "n_norm": n_norm, "value": m["value"], "ms_per_step": m["ms_per_step"], "ms_per_step_median": m["ms_per_step_median"],
                        "kernel_ms": m["roofline"]["kernel_ms"], "hbm_gbs": m["roofline"]["achieved"], "frac": m["roofline"]["frac"],
                        "e2e_value": m["e2e"]["value"], "nll_last": m["nll_last"][0]})
            model.close()
    return out


def run_shard(args, world, rank, device):
    """Strong scaling: ONE data set of n_data / n_norm events cut into `world` contiguous shards (ShardedModel); every timed step
    is amp_set_params + amp_nll_terms on each rank's shard and ONE all-reduce of 2 P doubles on the process group (NCCL over
    NVLink 5 / NVSwitch), after which every rank holds the NLL of the whole sample."""
    import torch
    import torch.distributed as dist
    from paper_2007_14931_b200 import sharded as S
    single = world == 1 and not dist.is_initialized()
    if single:   # one GPU: a one-rank NCCL group, so the same code path (collective included) runs
        with socket.socket() as sk:
            sk.bind(("127.0.0.1", 0))
            port = sk.getsockname()[1]
        os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
        os.environ.setdefault("MASTER_PORT", str(port))
        dist.init_process_group("nccl", rank=0, world_size=1, device_id=device)
    cfg = args.cfg
    res, c = model_def(cfg)
    # every rank generates the same seeded events on the host and keeps its own slice (no data-path exchange at load)
    x, eff, xn, wn, t_gen = generate_events(args, device)
    sm = S.ShardedModel(W.DECAY, res)
    sm.load_events(x, eff)
    sm.load_norm(xn, wn)
    P = 121 if cfg == 4 else 1
    params = [step_params(cfg, c, s) for s in range(args.warmup + args.steps)]

    def one_step(s):
        cs, mws = params[s]
        sm.set_params(cs, mws)
        return sm.nll()

    sampler = ClockSampler(device.index)
    if rank == 0:
        sampler.start()
        time.sleep(0.01)
    t = timed_steps(one_step, args.steps, args.warmup, world, device, sampler if rank == 0 else None)
    st = sm.model.last_call_stats()
    k_ms = [float(v) for v in sm.model.recent_launch_ms(min(args.steps, 256))] if st["norm_path"] in (4, 5) else [float("nan")]
    if rank == 0:
        sampler.stop()
        hbm_peak, peak_kind = measured_peaks()
        lo, hi = S.shard_bounds(args.n_data, 0, world)
        ln, hn = S.shard_bounds(args.n_norm, 0, world)
        nbytes = BYTES_PER_EVENT_DATA * (hi - lo) + BYTES_PER_EVENT_NORM * (hn - ln)
        evals = P * args.steps                       # strong scaling: the ranks share ONE evaluation per point
        kern = float(np.mean(k_ms))
        line = {"metric": METRIC, "value": evals / (t["dev_ms"] * 1e-3), "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
                "ms_per_step": t["dev_ms"] / args.steps, "ms_per_step_median": float(np.median(t["per_step_ms"])), "higher_is_better": True,
                "scaling": "strong", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
                "config": {"workload": workload_text(cfg, args.n_data, args.n_norm, P).replace(" per GPU", " in total"), "n_data": args.n_data, "n_norm": args.n_norm, "P": P,
                           "l2": "inputs larger than L2 per rank down to 16 shards; no flush", "parallelism": f"event shards x{world}",
                           "collective": "one all-reduce (sum) of 2 P float64 per step on the NCCL process group + one of 4 constants at load"},
                "e2e": {"value": evals / t["wall_s"], "unit": UNIT, "h2d_bytes_per_step": int(8 * (P * sm.K * 2 + P * sm.R * 2) + 16 * P), "d2h_bytes_per_step": int(16 * P + 16 * P),
                        "ms_per_step_median": float(np.median(t["per_step_wall_ms"])),
                        "note": "per step and rank: parameters host -> library, the two per-shard sums library -> host -> device tensor, NCCL all-reduce, result -> host"},
                "gpu_launches": int(st["launches"] * args.steps) * world,
                "roofline": {"bound": "hbm", "kernel": "k_stream<MODE_FUSED> on one rank's shard", "achieved": nbytes / (kern * 1e-3) / 1e9, "peak": hbm_peak,
                             "peak_source": f"MEASURED_PEAKS.json hbm_gbs ({peak_kind})", "unit": "GB/s", "frac": nbytes / (kern * 1e-3) / 1e9 / hbm_peak,
                             "traffic": None, "kernel_ms": kern, "kernel_ms_median": float(np.median(k_ms)),
                             "exchange_ms_per_step": t["dev_ms"] / args.steps - kern},
                "clocks": t["clocks"], "setup": {"gen_s": t_gen}, "nll_last": [float(v) for v in np.atleast_1d(t["last"])[:3]]}
        print(json.dumps(line))
    if dist.is_initialized():
        dist.destroy_process_group()


def cpu_baseline(args, target_evals=None):
    """The oracle, as it stands, timed on this box's host cores on a bounded sample of the same workload (about 10-30 s
    of CPU work): same model and call pattern, data and norm sizes scaled down by one factor (1 = the full workload) and
    the evaluation repeated so that about `target_evals` event-evaluations are timed; data events drawn by
    oracle-driven accept-reject (no oracle input comes from the CUDA path).  `value_1thread`: the same call with ONE thread on
    1/8 of that sample's events, scaled linearly to the full sizes."""
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
    cores = O.num_threads()
    n1, m1 = max(n // 8, 500), max(m // 8, 2000)
    O.set_num_threads(1)
    cs, mws = step_params(cfg, c, 0)
    t0 = time.perf_counter()
    Mo.nll(cs, x[:, :n1], eff[:n1], xn[:, :m1], wn[:m1], mass_width=mws)
    dt1 = time.perf_counter() - t0
    O.set_num_threads(cores)
    full1 = dt1 * total / (n1 + m1)
    return {"value": P / full, "unit": UNIT, "cores": cores, "kind": "oracle",
            "sample": f"{reps} x ({n} data + {m} norm events, same model, P={P}), {dt:.2f} s measured"
                      + ("" if n + m == total else f", scaled linearly to {args.n_data}+{args.n_norm}"),
            "event_evals_per_s": P * (n + m) * reps / dt,
            "value_1thread": P / full1, "sample_1thread": f"1 x ({n1} data + {m1} norm events), 1 thread, {dt1:.2f} s measured, scaled linearly to {args.n_data}+{args.n_norm}"}


def run_reference(args):
    """The reference arm = the oracle on the host cores.  Every step is the FULL workload (same config as the own arm) unless
    the first warm-up step shows that steps + warm-up would not end within ~5 minutes; then the sample is cut by a stated factor."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    from oracle import oracle as O
    cfg = args.cfg
    P = 121 if cfg == 4 else 1
    res, c = model_def(cfg)
    Mo = O.Model(W.DECAY, res)
    n, m = args.n_data, args.n_norm
    t0 = time.perf_counter()
    xn, wn = W.norm_events(cfg, m)
    x, eff = W.data_events(cfg, lambda xx, ee: Mo.eval_events(c, xx, ee), n=n)
    t_gen = time.perf_counter() - t0
    # probe: one evaluation of 1/16 of the events decides whether the full workload fits the budget
    cs, mws = step_params(cfg, c, 0)
    t0 = time.perf_counter()
    Mo.nll(cs, x[:, :n // 16], eff[:n // 16], xn[:, :m // 16], wn[:m // 16], mass_width=mws)
    est_full = (time.perf_counter() - t0) * 16
    budget = 300.0
    cut = 1
    while est_full / cut * (args.steps + args.warmup) > budget and cut < 64:
        cut *= 2
    ns, ms = n // cut, m // cut
    times = []
    for s in range(args.warmup + args.steps):
        cs, mws = step_params(cfg, c, s)
        t0 = time.perf_counter()
        Mo.nll(cs, x[:, :ns], eff[:ns], xn[:, :ms], wn[:ms], mass_width=mws)
        if s >= args.warmup:
            times.append(time.perf_counter() - t0)
    dt = float(np.sum(times))
    scale = (n + m) / (ns + ms)
    value = P * args.steps / (dt * scale)
    sample = (f"every step the full workload: {n} data + {m} norm events (same model, P={P})" if cut == 1 else
              f"{ns} data + {ms} norm events per step (same model, P={P}; 1/{cut} of the workload: the full one would not end within {budget:.0f} s on "
              f"{O.num_threads()} cores), scaled linearly to {n}+{m}")
    line = {"impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": int(os.environ.get("WORLD_SIZE", "1")),
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": dt * scale / args.steps * 1e3, "ms_per_step_median": float(np.median(times)) * scale * 1e3,
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": workload_text(cfg, n, m, P), "n_data": n, "n_norm": m, "P": P, "full_workload_every_step": cut == 1},
            "cpu_baseline": {"value": value, "unit": UNIT, "cores": O.num_threads(), "kind": "oracle", "sample": sample},
            "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}, "gpu_launches": 0,
            "setup": {"gen_s": t_gen}}
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


def spawn_ranks(args):
    """`--gpus N` without a launcher: start the N ranks the way the driver does (torch.distributed.run, 127.0.0.1)"""
    with socket.socket() as sk:
        sk.bind(("127.0.0.1", 0))
        port = sk.getsockname()[1]
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", f"--nproc-per-node={args.gpus}", "--master-addr", "127.0.0.1",
           "--master-port", str(port), os.path.abspath(__file__)] + sys.argv[1:]
    return subprocess.call(cmd)


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=200)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="own", choices=["own", "reference"])
    ap.add_argument("--cfg", type=int, default=3, choices=[3, 4], help="3: P=1 all lineshapes floating (headline; the default run adds the cfg 4 timing as \"cfg4\"); 4: P=121 fit-loop pattern only")
    ap.add_argument("--n-data", type=int, default=2_000_000)
    ap.add_argument("--n-norm", type=int, default=10_000_000)
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-cfg4", action="store_true", help="skip the configs[4] timing of the default run")
    ap.add_argument("--sweep", action="store_true", help="also time the six configs[3] points {1M, 2M, 8M} data x {2M, 10M} normalisation events (\"sweep\" in the line)")
    ap.add_argument("--shard", action="store_true", help="strong scaling: ONE data set cut over the ranks (ShardedModel), the all-reduce on NCCL inside the timed step")
    ap.add_argument("--dense", action="store_true", help="--cfg 4 through the dense DMMA contraction instead of the gradient-batch kernel")
    ap.add_argument("--one-launch", action="store_true", help="configs[4] as one k_deltaf launch over both samples instead of k_deltan x 2 + k_deltaf")
    ap.add_argument("--general", action="store_true", help="configs[4] through the general gradient-batch kernel (k_delta) instead of the shape-specialised k_deltaf")
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
    if args.impl == "reference":
        return run_reference(args)
    world = int(os.environ.get("WORLD_SIZE", "0"))
    if world == 0 and args.gpus > 1:
        return sys.exit(spawn_ranks(args))
    if world and world != args.gpus:
        ap.error(f"--gpus {args.gpus} but the launcher started {world} ranks")
    args.warmup = max(args.warmup, 3)
    run_own(args)


if __name__ == "__main__":
    main()
