#!/usr/bin/env python
"""bench.py -- throughput of the oscillation-reweighting hot path on B200 (contract: see DESIGN.md "Measurement").

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--events n]
    python -m torch.distributed.run --nnodes=1 --nproc-per-node N --master-addr 127.0.0.1 --master-port P \
        bench.py --gpus N --steps K --warmup W

Workload (BASELINE.json configs[2], the one the metric "oscillation-reweighted events/s" is quoted on): per GPU
1e7 synthetic events (E_true, E_reco, w0 fp64 + channel int8, 250 MB > L2) in 4 channels, Table 1 parameters; one
STEP = osc_set_params (row a1) followed by osc_reweight_bin (rows a2a-a3c fused) for each of the three energy-scale
values {0.97, 1.00, 1.03}, i.e. three full reweight-and-histogram passes over the events.  value = event
reweightings per second = N_gpus * n * 3 * K / time.  With N > 1 every rank holds its own n events (weak scaling) and
the partial histograms are summed with one NCCL all-reduce per step.

rank 0 prints ONE JSON line.  --impl reference times the CPU oracle (test infrastructure) on a bounded sample of the
same workload; it is a deliberately slow program and its number is a reported baseline, not a target.
"""
from __future__ import annotations

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

from paper_1311_7579_b200 import workloads as wl  # noqa: E402  (no method arithmetic in there)

METRIC = "fp64 oscillation-reweighted events/sec"
UNIT = "events/s"
N_EVENTS = 10_000_000
SCALES = wl.ENERGY_SCALES
BYTES_PER_EVENT = 25          # E_true + E_reco + w0 (fp64) + channel (int8): SURVEY.md 8(d), DESIGN.md "k2"
# fp64 operations k2 executes per event (DFMA = 2, DMUL/DADD = 1), counted by ncu
# (smsp__sass_thread_inst_executed_op_{dfma,dmul,dadd}_pred_on.sum / events): DESIGN.md 5.1, profiles/r1_k2_full_a.md.
FLOP_PER_EVENT = 199.1        # 75.0 DFMA + 42.0 DMUL + 7.1 DADD per event (profiles/r1_launches_d.md)
# dram__bytes_read.sum + dram__bytes_write.sum of one k2 launch over 1e7 events (same capture); algorithmic: 250.0e6
NCU_TRAFFIC_BYTES_1E7 = 253.20e6
NCU_TRAFFIC_SOURCE = "profiles/r1_launches_d.md"
FP64_LANES_PER_SM_CLK = 64    # B200 (sm_100): 4 sub-partitions x 16 fp64 lanes; DESIGN.md "fp64 roofline"


def parse():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=5)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--events", type=int, default=None, help="events per GPU (default: the size the config names)")
    ap.add_argument("--no-cpu-baseline", action="store_true", help="skip the oracle timing leg")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--workload", default="config2", choices=["config0", "config1", "config2", "config3", "config3-k5",
                                                               "config4"],
                    help="config2 (default) is the bench line; the others time the remaining BASELINE.json configs "
                         "for BASELINE.md section 4 and give ncu a committed command for k1 / k1b / k4 / k5 "
                         "(config3-k5 forces the unfactorised batched kernel; config4 is the size sweep)")
    return ap.parse_args()


def peaks():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(path):
        with open(path) as f:
            d = json.load(f)
        return float(d["hbm_gbs"]), "measured (MEASURED_PEAKS.json)"
    return 6650.0, "fallback (B200_PROFILING.md)"


class ClockSampler:
    """nvidia-smi clocks/throttle reasons during the timed region (B200_PROFILING.md 'clocks line')."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.rows = []
        self.proc = None
        try:
            self.proc = subprocess.Popen(["nvidia-smi", f"--id={index}", f"--query-gpu={self.Q}",
                                          "--format=csv,noheader,nounits", "-lms", "20"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.t = threading.Thread(target=self._read, daemon=True)
            self.t.start()
        except OSError:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append((time.time(), line.strip()))

    def stop(self, t0: float, t1: float):
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.15)
        self.proc.terminate()
        try:
            self.proc.wait(timeout=5)
        except subprocess.TimeoutExpired:
            self.proc.kill()
        sm, smax, reasons, power = [], [], set(), []
        names = ("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap")
        rows = [r for (t, r) in self.rows if t0 - 0.05 <= t <= t1 + 0.15] or [r for (_, r) in self.rows]
        for r in rows:
            f = [x.strip() for x in r.split(",")]
            if len(f) < 7:
                continue
            try:
                sm.append(float(f[0]))
                smax.append(float(f[1]))
                power.append(float(f[2]))
            except ValueError:
                continue
            for name, v in zip(names, f[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(name)
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": max(smax) if smax else None,
                "power_w_max": max(power) if power else None, "samples": len(sm), "reasons": sorted(reasons)}


def oracle_rate(n_target_seconds: float = 15.0):
    """Oracle (as it stands) on a bounded sample of the configs[2] workload; events/s over all host cores."""
    import oracle

    oracle.build()
    par = oracle.Params(**wl.table1())
    edges = wl.bin_edges()
    cores = oracle.threads()
    probe_n = 20_000
    ev = wl.events(probe_n, seed=2)
    t = time.perf_counter()
    oracle.reweight_bin(par, *ev, 1.0, edges)
    rate = probe_n / max(time.perf_counter() - t, 1e-9)
    n = int(min(max(rate * n_target_seconds / len(SCALES), 10_000), 2_000_000))
    ev = wl.events(n, seed=2)
    t = time.perf_counter()
    for s in SCALES:
        oracle.reweight_bin(par, *ev, s, edges)
    dt = time.perf_counter() - t
    return {"value": n * len(SCALES) / dt, "unit": UNIT, "cores": cores, "kind": "oracle",
            "sample": f"first {n} events of the configs[2] arrays (seed 2) x {len(SCALES)} energy scales, "
                      f"long-double Jacobi oracle, OpenMP over events, {dt:.1f} s"}, n, dt


def run_reference(args):
    """The oracle timed on the host cores: K steps, each a bounded sample of the workload."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    import oracle

    oracle.build()
    par = oracle.Params(**wl.table1())
    edges = wl.bin_edges()
    cores = oracle.threads()
    ev = wl.events(20_000, seed=2)
    t = time.perf_counter()
    oracle.reweight_bin(par, *ev, 1.0, edges)
    rate = 20_000 / max(time.perf_counter() - t, 1e-9)
    total_steps = max(args.steps + args.warmup, 1)
    n = int(min(max(rate * 60.0 / (len(SCALES) * total_steps), 2_000), 1_000_000))   # whole run ~1 minute
    ev = wl.events(n, seed=2)
    for _ in range(args.warmup):
        for s in SCALES:
            oracle.reweight_bin(par, *ev, s, edges)
    t = time.perf_counter()
    for _ in range(args.steps):
        for s in SCALES:
            oracle.reweight_bin(par, *ev, s, edges)
    dt = time.perf_counter() - t
    value = n * len(SCALES) * args.steps / dt
    sample = (f"each step = first {n} events of the configs[2] arrays (seed 2) x {len(SCALES)} energy scales; "
              f"long-double Jacobi oracle with OpenMP over events")
    print(json.dumps({
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": 1e3 * dt / max(args.steps, 1), "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None, "dtype": "f64 (long double inside the oracle)", "data": "synthetic",
        "config": {"workload": "configs[2] bounded sample: 4 channels, 50 bins, 3 energy scales, Table 1 parameters",
                   "events_per_step": n, "passes_per_step": len(SCALES)},
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }))


K5_FLOP_PER_UNIT = 175.6      # all kernels of one k5 call, ncu (profiles/r1_k5.md)
K4_FLOP_PER_UNIT = 17.4       # all kernels of one factorised call, ncu (profiles/r1_launches_k4.md)
# Per-config description of the secondary workloads: (events, units per event per step, bytes per unit, flop per unit)
#   flop per unit: ncu-counted fp64 operations of the kernel that runs, bytes: algorithmic.
OTHER = {
    "config0": dict(n=100_000, kernel="prob_kernel (k1)", bytes_per_unit=16.0, flop_per_unit=178.0,
                    what="configs[0]: 1e5 events, Table 1, P(numu->numu) and P(numu->nue) (2 osc_prob calls)"),
    "config1": dict(n=10_000_000, kernel="prob_all_kernel (k1b)", bytes_per_unit=80.0, flop_per_unit=241.0,
                    what="configs[1]: 1e7 events, all 9 transitions for nu and nubar (2 osc_prob_all calls = "
                         "18 output arrays), delta_cp drawn per step, both hierarchies alternate"),
    # k4: fp64 operations the factorised path executes per (event, point), all its kernels together, counted by ncu
    # (profiles/r1_k4_ops.md): the eigen-solve is shared by the 32 points of a dm2_32 group
    "config3": dict(n=1_000_000, kernel="scan_main_kernel + sort/merge kernels (k4, factorised)",
                    bytes_per_unit=25.0 / 1024, flop_per_unit=K4_FLOP_PER_UNIT,
                    what="configs[3]: 1e6 events x 1024 oscillation points (32x32 grid of sin2_th23 x dm2_32, "
                         "delta_cp per point) in ONE osc_reweight_bin_batch call (factorised path k4)"),
    "config3-k5": dict(n=1_000_000, kernel="scan_full_kernel + sort/merge kernels (k5)", bytes_per_unit=25.0 / 1024,
                       flop_per_unit=K5_FLOP_PER_UNIT,
                       what="configs[3] with OSC_BATCH_PATH=k5: every (event, point) pair gets the full closed form, on "
                            "events sorted by histogram cell (the path of point lists without scan structure)"),
}


def run_other(args):
    """Secondary workloads (one GPU): same JSON schema, unit = event (x point) evaluations per second."""
    import torch

    import paper_1311_7579_b200 as osc
    from paper_1311_7579_b200 import build as _build

    _build.build_library()
    assert torch.cuda.is_available(), "bench.py needs a CUDA device (no CPU fallback)"
    torch.cuda.set_device(0)
    osc.osc_set_device(0)
    dev = torch.device("cuda", 0)
    cfg = OTHER[args.workload]
    n = args.events or cfg["n"]
    stream = torch.cuda.current_stream()
    flush = torch.empty(256 * 1024 * 1024, dtype=torch.uint8, device=dev)       # > L2 (126 MB)
    if args.workload == "config0":
        d_et = torch.from_numpy(wl.e_true(n, seed=0)).to(dev)
        out = torch.empty((2, n), dtype=torch.float64, device=dev)
        units = 2 * n

        def step(i):
            flush.fill_(i & 1)                                                  # inputs fit L2: flush between steps
            osc.osc_set_params(**wl.table1())
            osc.osc_prob(d_et, 1, 1, 0, P_out=out[0])
            osc.osc_prob(d_et, 1, 0, 0, P_out=out[1])
    elif args.workload == "config1":
        d_et = torch.from_numpy(wl.e_true(n, seed=1)).to(dev)
        out = torch.empty((2, 9, n), dtype=torch.float64, device=dev)
        runs = wl.config1_runs()
        units = 2 * n                                                           # (event, nu/nubar) solves; 9 outputs each

        def step(i):
            osc.osc_set_params(**runs[i % len(runs)])
            osc.osc_prob_all(d_et, 0, P_out=out[0])
            osc.osc_prob_all(d_et, 1, P_out=out[1])
    else:
        et, er, w0, ch = wl.events(n, seed=2)
        d_et, d_er, d_w0, d_ch = (torch.from_numpy(a).to(dev) for a in (et, er, w0, ch))
        d_edges = torch.from_numpy(wl.bin_edges()).to(dev)
        if args.workload == "config3-k5":
            os.environ["OSC_BATCH_PATH"] = "k5"
        pts = osc.pack_params(wl.scan_points())                                 # marshalled once (binding only)
        out = torch.empty((len(pts), osc.N_CHANNELS, wl.N_BINS), dtype=torch.float64, device=dev)
        units = n * len(pts)

        def step(i):
            osc.osc_reweight_bin_batch(pts, d_et, d_er, d_w0, d_ch, 1.0, d_edges, hist_out=out)

    warm = max(args.warmup, 3)
    for i in range(warm):
        step(i)
    torch.cuda.synchronize()
    sampler = ClockSampler(0)
    # per-step CUDA events so that the L2 flush of config0 stays outside the timed intervals
    evs = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(args.steps)]
    l0 = osc.osc_launch_count()
    t0 = time.time()
    for i, (a, b) in enumerate(evs):
        if args.workload == "config0":
            flush.fill_(i & 1)
            a.record(stream)
            osc.osc_set_params(**wl.table1())
            osc.osc_prob(d_et, 1, 1, 0, P_out=out[0])
            osc.osc_prob(d_et, 1, 0, 0, P_out=out[1])
        else:
            a.record(stream)
            step(i)
        b.record(stream)
    torch.cuda.synchronize()
    t1 = time.time()
    launches = osc.osc_launch_count() - l0
    ms = sum(a.elapsed_time(b) for a, b in evs)
    clocks = sampler.stop(t0, t1)
    value = units * args.steps / (ms * 1e-3)
    hbm_peak, peak_src = peaks()
    sm_count = torch.cuda.get_device_properties(dev).multi_processor_count
    sm_max = (clocks or {}).get("sm_max_mhz") or 1965.0
    nominal = sm_count * FP64_LANES_PER_SM_CLK * 2 * sm_max * 1e6 / 1e12
    tf = value * cfg["flop_per_unit"] / 1e12
    gbs = value * cfg["bytes_per_unit"] / 1e9
    hbm_bound = args.workload == "config1"
    roof = ({"bound": "hbm", "achieved": gbs, "peak": hbm_peak, "unit": "GB/s", "frac": gbs / hbm_peak,
             "peak_source": peak_src} if hbm_bound else
            {"bound": "alu", "achieved": tf, "peak": nominal, "unit": "TFLOP/s", "frac": tf / nominal,
             "peak_source": "unit counts and clocks.max.sm (DESIGN.md section 6)"})
    roof.update({"traffic": None, "kernel": cfg["kernel"], "flop_per_unit": cfg["flop_per_unit"],
                 "bytes_per_unit": cfg["bytes_per_unit"], "alu_tflops": tf, "hbm_gbs": gbs,
                 "note": "whole-step average (all launches of the step are this kernel)"
                         + ("; launch-latency bound at this size, fractions are not kernel quality" if n < 1_000_000 else "")})
    print(json.dumps({
        "metric": METRIC, "value": value, "unit": "event evaluations/s", "n_gpus": 1, "steps": args.steps, "warmup": warm,
        "ms_per_step": ms / args.steps, "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64",
        "data": "synthetic", "config": {"workload": cfg["what"], "events": n, "units_per_step": units,
                                        "l2": "flushed between steps" if args.workload == "config0" else "working set > L2"},
        "clocks": clocks, "e2e": None, "gpu_launches": int(launches), "roofline": roof, "cpu_baseline": None}))


def run_sweep(args):
    """configs[4]: size sweep N = 1e3 .. 1e9 on the configs[2] path (k2, one energy scale per launch, Table 1), plus
    the 12 (rho, L, hierarchy) settings at N = 1e7.  One JSON line; `value` is the rate at the largest N."""
    import torch

    import paper_1311_7579_b200 as osc
    from paper_1311_7579_b200 import build as _build

    _build.build_library()
    assert torch.cuda.is_available(), "bench.py needs a CUDA device (no CPU fallback)"
    torch.cuda.set_device(0)
    osc.osc_set_device(0)
    dev = torch.device("cuda", 0)
    stream = torch.cuda.current_stream()
    d_edges = torch.from_numpy(wl.bin_edges()).to(dev)
    hist = torch.zeros((osc.N_CHANNELS, wl.N_BINS), dtype=torch.float64, device=dev)
    flush = torch.empty(256 * 1024 * 1024, dtype=torch.uint8, device=dev)       # > L2 (126 MB)
    hbm_peak, peak_src = peaks()
    sm_count = torch.cuda.get_device_properties(dev).multi_processor_count
    n_max = args.events or 1_000_000_000
    sizes = [10 ** k for k in range(3, 10) if 10 ** k <= n_max]
    sampler = ClockSampler(0)
    t0 = time.time()
    launches0 = osc.osc_launch_count()

    def time_k2(ev, par, reps):
        """Mean duration of one k2 launch (ms).  Inputs below the L2 size are evicted before every launch."""
        osc.osc_set_params(**par)
        small = ev[0].numel() * BYTES_PER_EVENT < 200e6
        for _ in range(3):
            osc.osc_reweight_bin(*ev, 1.0, d_edges, hist_out=hist)
        total = 0.0
        a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        if small:
            for i in range(reps):
                flush.fill_(i & 1)
                a.record(stream)
                osc.osc_reweight_bin(*ev, 1.0, d_edges, hist_out=hist)
                b.record(stream)
                torch.cuda.synchronize()
                total += a.elapsed_time(b)
            return total / reps
        a.record(stream)
        for _ in range(reps):
            osc.osc_reweight_bin(*ev, 1.0, d_edges, hist_out=hist)
        b.record(stream)
        torch.cuda.synchronize()
        return a.elapsed_time(b) / reps

    rows = []
    ev = None
    for n in sizes:
        ev = wl.events_device(n, seed=4, device=dev)
        ms = time_k2(ev, wl.table1(), max(3, min(args.steps, 20)))
        rows.append({"N": n, "ms_per_launch": ms, "events_per_s": n / (ms * 1e-3)})
        if n == 10_000_000:
            settings = []
            for par in wl.sweep_settings():
                ms_s = time_k2(ev, par, 5)
                settings.append({"rho": par["rho_g_cm3"], "L": par["L_km"], "hierarchy": par["hierarchy"],
                                 "events_per_s": n / (ms_s * 1e-3)})
            rows[-1]["settings"] = settings
    torch.cuda.synchronize()
    clocks = sampler.stop(t0, time.time())
    sm_max = (clocks or {}).get("sm_max_mhz") or 1965.0
    nominal = sm_count * FP64_LANES_PER_SM_CLK * 2 * sm_max * 1e6 / 1e12
    for r in rows:
        r["frac_fp64"] = r["events_per_s"] * FLOP_PER_EVENT / 1e12 / nominal
        r["frac_hbm"] = r["events_per_s"] * BYTES_PER_EVENT / 1e9 / hbm_peak
    last = rows[-1]
    print(json.dumps({
        "metric": METRIC, "value": last["events_per_s"], "unit": UNIT, "n_gpus": 1, "steps": args.steps,
        "warmup": 3, "ms_per_step": last["ms_per_launch"], "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f64", "data": "synthetic (drawn on the device with torch's generator, seed 4)",
        "config": {"workload": "configs[4]: size sweep on the configs[2] path (k2, one launch per row), Table 1; "
                               "rho x L x hierarchy settings at N = 1e7",
                   "sizes": sizes, "l2": "inputs smaller than L2 are evicted (256 MB fill) before every timed launch"},
        "clocks": clocks, "e2e": None, "gpu_launches": int(osc.osc_launch_count() - launches0),
        "roofline": {"bound": "alu", "achieved": last["events_per_s"] * FLOP_PER_EVENT / 1e12, "peak": nominal,
                     "unit": "TFLOP/s", "frac": last["frac_fp64"], "traffic": None, "kernel": "reweight_bin_kernel (k2)",
                     "peak_source": "unit counts and clocks.max.sm (DESIGN.md section 6)",
                     "hbm_peak": hbm_peak, "hbm_peak_source": peak_src},
        "sweep": rows, "cpu_baseline": None}))


def main():
    args = parse()
    if args.impl == "reference":
        run_reference(args)
        return
    if args.workload == "config4":
        run_sweep(args)
        return
    if args.workload != "config2":
        run_other(args)
        return

    import torch
    import torch.distributed as dist

    import paper_1311_7579_b200 as osc   # raises if libosc_b200.so is missing: no fallback
    from paper_1311_7579_b200 import build as _build
    from paper_1311_7579_b200 import sharding

    _build.build_library()
    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if world != args.gpus:
        if world == 1 and args.gpus > 1:
            raise SystemExit("launch with torch.distributed.run --nproc-per-node N for --gpus N")
    assert torch.cuda.is_available(), "bench.py needs a CUDA device (no CPU fallback)"
    torch.cuda.set_device(local)
    osc.osc_set_device(local)
    device = torch.device("cuda", local)
    if world > 1:
        dist.init_process_group("nccl", device_id=device)

    n = args.events or N_EVENTS
    par = wl.table1()
    et, er, w0, ch = wl.events(n, seed=2 + 1000 * rank)          # each rank its own shard (weak scaling)
    edges = wl.bin_edges()
    # pinned host copies (e2e leg) and device-resident copies (value leg)
    h_et, h_er, h_w0, h_ch = (torch.from_numpy(a).pin_memory() for a in (et, er, w0, ch))
    d_et, d_er, d_w0, d_ch = (t.to(device) for t in (h_et, h_er, h_w0, h_ch))
    d_edges = torch.from_numpy(edges).to(device)
    hist = torch.zeros((len(SCALES), osc.N_CHANNELS, wl.N_BINS), dtype=torch.float64, device=device)
    stream = torch.cuda.current_stream()

    def step():
        osc.osc_set_params(**par)                                                           # a1
        for k, s in enumerate(SCALES):
            osc.osc_reweight_bin(d_et, d_er, d_w0, d_ch, s, d_edges, hist_out=hist[k])      # a2a-a3c
        sharding.allreduce_hist(hist)                                                       # 8(e): no-op at N = 1

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    for _ in range(max(args.warmup, 3)):
        step()
    barrier()

    # ---- timed region: device-resident inputs -----------------------------------------------------------------
    sampler = ClockSampler(local) if rank == 0 else None
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    launches0 = osc.osc_launch_count()
    barrier()
    t_wall0 = time.time()
    ev0.record(stream)
    for _ in range(args.steps):
        step()
    ev1.record(stream)
    barrier()
    t_wall1 = time.time()
    launches = osc.osc_launch_count() - launches0
    ms = ev0.elapsed_time(ev1)
    # the clock sampler keeps running through the legs below (the same kernels on the same data, back to back): the
    # timed region of `value` alone is a few milliseconds, too short for more than a sample or two
    t_ms = torch.tensor([ms], dtype=torch.float64, device=device)
    if world > 1:
        dist.all_reduce(t_ms, op=dist.ReduceOp.MAX)
    ms = float(t_ms.item())
    value = world * n * len(SCALES) * args.steps / (ms * 1e-3)

    # ---- dominant kernel alone (k2), CUDA events per launch, for the roofline ----------------------------------
    osc.osc_set_params(**par)
    reps = 30
    ks, ke = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    torch.cuda.synchronize()
    ks.record(stream)
    for i in range(reps):
        osc.osc_reweight_bin(d_et, d_er, d_w0, d_ch, SCALES[i % 3], d_edges, hist_out=hist[i % 3])
    ke.record(stream)
    torch.cuda.synchronize()
    k_ms = ks.elapsed_time(ke) / reps

    # ---- the same step through the one-pass call (osc_reweight_bin_scales, NEXT-3): reported beside `value` --------
    def step_fused():
        osc.osc_set_params(**par)
        osc.osc_reweight_bin_scales(d_et, d_er, d_w0, d_ch, SCALES, d_edges, hist_out=hist)
        sharding.allreduce_hist(hist)

    for _ in range(3):
        step_fused()
    barrier()
    fs, fe = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    fs.record(stream)
    for _ in range(args.steps):
        step_fused()
    fe.record(stream)
    barrier()
    f_ms = torch.tensor([fs.elapsed_time(fe)], dtype=torch.float64, device=device)
    if world > 1:
        dist.all_reduce(f_ms, op=dist.ReduceOp.MAX)
    fused = {"value": world * n * len(SCALES) * args.steps / (float(f_ms.item()) * 1e-3), "unit": UNIT,
             "ms_per_step": float(f_ms.item()) / args.steps,
             "api": "osc_reweight_bin_scales: the three energy scales in one pass, closed form once per event; "
                    "same three histograms as the step behind `value`"}

    # ---- the same three histograms from plans (osc_plan_*): events sorted by cell once per (sample, scale), outside
    # the timed region; a step is osc_set_params + one osc_plan_reweight_bin per scale.  This is the Markov-chain use
    # of the paper (same events, new parameters every step), reported beside `value`, not instead of it. ------------
    plans = [osc.osc_plan_create(d_et, d_er, d_w0, d_ch, s, d_edges) for s in SCALES]

    def step_plan():
        osc.osc_set_params(**par)
        for k, pl in enumerate(plans):
            osc.osc_plan_reweight_bin(pl, hist_out=hist[k])
        sharding.allreduce_hist(hist)

    for _ in range(3):
        step_plan()
    barrier()
    qs, qe = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    qs.record(stream)
    for _ in range(args.steps):
        step_plan()
    qe.record(stream)
    barrier()
    p_ms = torch.tensor([qs.elapsed_time(qe)], dtype=torch.float64, device=device)
    if world > 1:
        dist.all_reduce(p_ms, op=dist.ReduceOp.MAX)
    planned = {"value": world * n * len(SCALES) * args.steps / (float(p_ms.item()) * 1e-3), "unit": UNIT,
               "ms_per_step": float(p_ms.item()) / args.steps,
               "api": "osc_plan_reweight_bin on three plans (one per energy scale) built before the timed region: "
                      "events pre-sorted by histogram cell, kernel k5 for one parameter set"}
    for pl in plans:
        osc.osc_plan_destroy(pl)
    clocks = sampler.stop(t_wall0, time.time()) if sampler else None
    if clocks is not None:
        clocks["window"] = "timed region of `value` and the kernel-alone, fused_scales and planned legs that follow it"

    # ---- fp64 peak probe in the same run (DFMA-only, register resident) ----------------------------------------
    probe_flops = osc.osc_fp64_peak_probe(1 << 14, 4)
    torch.cuda.synchronize()
    ps, pe = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    ps.record(stream)
    for _ in range(5):
        osc.osc_fp64_peak_probe(1 << 14, 4)
    pe.record(stream)
    torch.cuda.synchronize()
    fp64_peak_tflops = 5 * probe_flops / (ps.elapsed_time(pe) * 1e-3) / 1e12

    # ---- e2e: same step through the C ABI with HOST buffers (H2D and D2H inside the timed region) ---------------
    e2e = None
    if not args.no_e2e:
        np_in = [t.numpy() for t in (h_et, h_er, h_w0, h_ch)]
        h_hist = torch.zeros((len(SCALES), osc.N_CHANNELS, wl.N_BINS), dtype=torch.float64).pin_memory()
        np_hist = h_hist.numpy()

        def step_host():                                  # the call a user makes for the step: all scales at once
            osc.osc_set_params(**par)
            osc.osc_reweight_bin_scales_host(*np_in, SCALES, edges, hist_out=np_hist)

        def step_host_per_scale():                         # the same step as three single-scale host calls
            osc.osc_set_params(**par)
            for k, s in enumerate(SCALES):
                osc.osc_reweight_bin_host(*np_in, s, edges, hist_out=np_hist[k])

        def time_host(fn):
            for _ in range(2):
                fn()
            barrier()
            t0 = time.perf_counter()
            for _ in range(e_steps):
                fn()
            barrier()
            dt = torch.tensor([time.perf_counter() - t0], dtype=torch.float64, device=device)
            if world > 1:
                dist.all_reduce(dt, op=dist.ReduceOp.MAX)
            return world * n * len(SCALES) * e_steps / float(dt.item())

        e_steps = max(2, min(args.steps, 5))
        v_one = time_host(step_host)
        v_three = time_host(step_host_per_scale)
        d2h = len(SCALES) * osc.N_CHANNELS * wl.N_BINS * 8
        e2e = {"value": v_one, "unit": UNIT,
               "h2d_bytes_per_step": n * BYTES_PER_EVENT + edges.nbytes, "d2h_bytes_per_step": d2h, "steps": e_steps,
               "api": "osc_reweight_bin_scales_host (pinned host buffers; the events cross PCIe once per step, the "
                      "three energy scales share the pass)",
               "per_scale_calls": {"value": v_three, "h2d_bytes_per_step": len(SCALES) * (n * BYTES_PER_EVENT + edges.nbytes),
                                   "api": "osc_reweight_bin_host, one call per energy scale"}}

    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return

    hbm_peak, peak_src = peaks()
    sm_count = torch.cuda.get_device_properties(device).multi_processor_count
    sm_max = (clocks or {}).get("sm_max_mhz") or 1965.0
    nominal_tflops = sm_count * FP64_LANES_PER_SM_CLK * 2 * sm_max * 1e6 / 1e12
    achieved_tflops = n * FLOP_PER_EVENT / (k_ms * 1e-3) / 1e12
    roofline = {"bound": "alu", "achieved": achieved_tflops, "peak": nominal_tflops, "unit": "TFLOP/s",
                "frac": achieved_tflops / nominal_tflops,
                "traffic": NCU_TRAFFIC_BYTES_1E7 if n == N_EVENTS else None,
                "traffic_unit": f"DRAM bytes per launch, ncu ({NCU_TRAFFIC_SOURCE}); algorithmic {n * BYTES_PER_EVENT}",
                "kernel": "reweight_bin_kernel (k2)", "kernel_ms": k_ms,
                "flop_per_event": FLOP_PER_EVENT,
                "peak_source": f"{sm_count} SMs x {FP64_LANES_PER_SM_CLK} fp64 lanes x 2 flop x {sm_max:.0f} MHz "
                               "(unit counts and clocks.max.sm; DESIGN.md section 6)",
                "peak_probe": fp64_peak_tflops, "frac_of_probe": achieved_tflops / fp64_peak_tflops,
                "peak_probe_source": "DFMA-only probe kernel measured in this run (osc_fp64_peak_probe)",
                "hbm": {"achieved": n * BYTES_PER_EVENT / (k_ms * 1e-3) / 1e9, "peak": hbm_peak, "unit": "GB/s",
                        "frac": n * BYTES_PER_EVENT / (k_ms * 1e-3) / 1e9 / hbm_peak, "peak_source": peak_src}}

    cpu = None
    if not args.no_cpu_baseline and world == 1:
        cpu, _, _ = oracle_rate()

    out = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": max(args.warmup, 3),
        "ms_per_step": ms / args.steps, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "f64", "data": "synthetic",
        "config": {"workload": "configs[2]: 1e7 events/GPU x 4 channels, 50-bin E_reco histograms over 0-5 GeV, "
                               "energy scales {0.97,1.00,1.03}, Table 1 parameters (normal hierarchy)",
                   "events_per_gpu": n, "passes_per_step": len(SCALES), "n_bins": wl.N_BINS,
                   "l2": "inputs (250 MB per pass) larger than L2 (126 MB); no explicit flush",
                   "parallelism": f"events sharded over {world} GPU(s); histogram all-reduce" if world > 1 else "1 GPU"},
        "clocks": clocks, "e2e": e2e, "gpu_launches": int(launches), "roofline": roofline, "cpu_baseline": cpu,
        "fused_scales": fused, "planned": planned,
    }
    print(json.dumps(out))
    if world > 1:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
