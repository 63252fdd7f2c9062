#!/usr/bin/env python
"""bench.py -- throughput of the oscillation-reweighting hot path on B200 (contract: see DESIGN.md "Measurement").

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--events n] [--scaling weak|strong]
    python -m torch.distributed.run --nnodes=1 --nproc-per-node N --master-addr 127.0.0.1 --master-port P \
        bench.py --gpus N --steps K --warmup W

Workload of `value` (BASELINE.json configs[2], the one the metric "oscillation-reweighted events/s" is quoted on): per
GPU 1e7 synthetic events (E_true, E_reco, w0 fp64 + channel int8, 250 MB > L2) in 4 channels, Table 1 parameters; one
STEP = osc_set_params (row a1) followed by osc_reweight_bin (rows a2a-a3c fused) for each of the three energy-scale
values {0.97, 1.00, 1.03}, i.e. three full reweight-and-histogram passes over the events.  value = event
reweightings per second = events of all GPUs * 3 * K / time.  With N > 1 the partial histograms are summed with one NCCL
all-reduce per step; --scaling weak (default): every rank holds its own 1e7 events; --scaling strong:
ONE seeded sample of --events (default 1e7) events is cut into contiguous per-rank slices (the paper's use: one Monte
Carlo sample).

The same line carries, under "configs", the other four BASELINE.json configs measured in the same process
(configs[0] k1, configs[1] k1b, configs[3] k4, configs[4] the size sweep 1e3 .. 1e9 of k2), each with its own roofline
object and clock sample; `--workload configN` prints one of them as a line of its own (the commands the ncu captures
under profiles/ use).  The fp64 operation counts behind every roofline fraction come from profiles/opcounts.json
(paper_1311_7579_b200/opcounts.py), never from constants in this file.

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

from paper_1311_7579_b200 import opcounts  # noqa: E402  (reads profiles/opcounts.json; no method arithmetic)
from paper_1311_7579_b200 import workloads as wl  # noqa: E402  (no method arithmetic in there)

METRIC = "fp64 oscillation-reweighted events/sec"
UNIT = "events/s"
N_EVENTS = 10_000_000
SCALES = wl.ENERGY_SCALES
BYTES_PER_EVENT = 25          # E_true + E_reco + w0 (fp64) + channel (int8): SURVEY.md 8(d), DESIGN.md "k2"
FP64_LANES_PER_SM_CLK = 64    # B200 (sm_100): 4 sub-partitions x 16 fp64 lanes; DESIGN.md "fp64 roofline"


def parse():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=5)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--events", type=int, default=None, help="events per GPU (--scaling strong: of the whole sample)")
    ap.add_argument("--scaling", default="weak", choices=["weak", "strong"])
    ap.add_argument("--no-cpu-baseline", action="store_true", help="skip the oracle timing leg")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-configs", action="store_true", help="skip the legs of configs[0], [1], [3], [4]")
    ap.add_argument("--sweep-max", type=int, default=1_000_000_000, help="largest N of the configs[4] sweep")
    ap.add_argument("--workload", default="config2", choices=["config0", "config1", "config2", "config3", "config3-k5",
                                                               "config4"],
                    help="config2 (default) is the bench line; the others print the leg of one other BASELINE.json "
                         "config as a line of its own (config3-k5 forces the unfactorised batched kernel)")
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
        self.t_start = time.time()
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

    def wait_first_row(self, timeout: float = 3.0):
        t = time.time()
        while self.proc is not None and not self.rows and time.time() - t < timeout:
            time.sleep(0.01)

    def stop(self, t0: float = None, t1: float = None):
        t0 = self.t_start if t0 is None else t0
        t1 = time.time() if t1 is None else t1
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


# ---------------------------------------------------------------------------------------------------------------
# the oracle on the host cores (cpu_baseline, --impl reference)
# ---------------------------------------------------------------------------------------------------------------
def _oracle_time(oracle, par, edges, n, seconds, fp64_build, threads):
    """events/s of oracle.reweight_bin over the three energy scales on the first n events; n is grown from a probe so
    that the timing takes about `seconds`."""
    oracle.set_threads(threads)
    probe_n = 4_000 * max(threads, 1)
    ev = wl.events(probe_n, seed=2)
    oracle.reweight_bin(par, *ev, 1.0, edges, fp64_build=fp64_build)         # first call: page in, OpenMP team start
    t = time.perf_counter()
    oracle.reweight_bin(par, *ev, 1.0, edges, fp64_build=fp64_build)
    rate = probe_n / max(time.perf_counter() - t, 1e-9)
    n = int(min(max(rate * seconds / len(SCALES), 5_000), n))
    ev = wl.events(n, seed=2)
    t = time.perf_counter()
    for s in SCALES:
        oracle.reweight_bin(par, *ev, s, edges, fp64_build=fp64_build)
    dt = time.perf_counter() - t
    return n * len(SCALES) / dt, n, dt


def oracle_rate():
    """cpu_baseline: the oracle as it stands (long double, all host cores) on a bounded sample of the configs[2]
    workload, plus the same on ONE core and the timing-only fp64 build of the same source on all cores and on one
    (SURVEY.md 8(d) "Oracle timing"; the paper's comparator is a single CPU core)."""
    import oracle

    oracle.build()
    par = oracle.Params(**wl.table1())
    edges = wl.bin_edges()
    cores = oracle.threads()
    v_all, n_all, dt_all = _oracle_time(oracle, par, edges, 2_000_000, 10.0, False, cores)
    v_one, n_one, dt_one = _oracle_time(oracle, par, edges, 400_000, 4.0, False, 1)
    # the fp64 build is a mechanical double-precision copy of the same source; make sure it computes the same thing
    ev = wl.events(20_000, seed=2)
    a = oracle.reweight_bin(par, *ev, 1.0, edges)
    b = oracle.reweight_bin(par, *ev, 1.0, edges, fp64_build=True)
    agree = float(np.max(np.abs(a - b) / np.maximum(np.abs(a), 1e-300) * (a > 0)))
    v64_all, n64_all, dt64_all = _oracle_time(oracle, par, edges, 2_000_000, 4.0, True, cores)
    v64_one, n64_one, dt64_one = _oracle_time(oracle, par, edges, 400_000, 3.0, True, 1)
    oracle.set_threads(cores)
    return {"value": v_all, "unit": UNIT, "cores": cores, "kind": "oracle",
            "sample": f"first {n_all} events of the configs[2] arrays (seed 2) x {len(SCALES)} energy scales, "
                      f"long-double Jacobi oracle, OpenMP over events, {dt_all:.1f} s",
            "one_core": {"value": v_one, "cores": 1, "sample": f"first {n_one} events x {len(SCALES)} scales, {dt_one:.1f} s"},
            "fp64_build": {"value": v64_all, "cores": cores, "one_core": v64_one,
                           "sample": f"first {n64_all} ({n64_one} on one core) events x {len(SCALES)} scales, "
                                     f"{dt64_all:.1f} s ({dt64_one:.1f} s)",
                           "what": "timing only: oracle/osc_oracle.c with long double mechanically replaced by double "
                                   "(oracle.build_fp64); parity always uses the long-double build",
                           "max_rel_bin_diff_vs_long_double": agree}}


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
        "scaling": args.scaling, "vs_baseline": None, "dtype": "f64 (long double inside the oracle)", "data": "synthetic",
        "config": {"workload": "configs[2] bounded sample: 4 channels, 50 bins, 3 energy scales, Table 1 parameters",
                   "events_per_step": n, "passes_per_step": len(SCALES)},
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }))


# ---------------------------------------------------------------------------------------------------------------
# roofline objects (counts from profiles/opcounts.json)
# ---------------------------------------------------------------------------------------------------------------
class Ctx:
    """What every leg needs: the binding, torch, the device and the peaks."""

    def __init__(self, local: int = 0):
        import torch

        import paper_1311_7579_b200 as osc   # raises if libosc_b200.so is missing: no fallback
        from paper_1311_7579_b200 import build as _build

        _build.build_library()
        assert torch.cuda.is_available(), "bench.py needs a CUDA device (no CPU fallback)"
        torch.cuda.set_device(local)
        osc.osc_set_device(local)
        self.torch, self.osc, self.local = torch, osc, local
        self.dev = torch.device("cuda", local)
        self.stream = torch.cuda.current_stream()
        self.hbm_peak, self.hbm_src = peaks()
        self.sm_count = torch.cuda.get_device_properties(self.dev).multi_processor_count
        self.counts = opcounts.load()
        self._flush = None

    def flush(self, i: int):
        if self._flush is None:
            self._flush = self.torch.empty(256 * 1024 * 1024, dtype=self.torch.uint8, device=self.dev)   # > L2 (126 MB)
        self._flush.fill_(i & 1)

    def nominal_tflops(self, clocks) -> float:
        sm_max = (clocks or {}).get("sm_max_mhz") or 1965.0
        return self.sm_count * FP64_LANES_PER_SM_CLK * 2 * sm_max * 1e6 / 1e12, sm_max

    def roofline(self, key: str, units_per_s: float, bytes_per_unit: float, clocks, bound: str = "alu", note: str = None):
        """`achieved` = counted flop (or algorithmic bytes) per unit x units/s; null fraction if the counts are stale."""
        c = opcounts.counts(key, self.counts)
        nominal, sm_max = self.nominal_tflops(clocks)
        tf = units_per_s * c["flop_per_unit"] / 1e12
        gbs = units_per_s * bytes_per_unit / 1e9
        stale = bool(c["stale"])
        if bound == "hbm":
            r = {"bound": "hbm", "achieved": gbs, "peak": self.hbm_peak, "unit": "GB/s",
                 "frac": None if stale else gbs / self.hbm_peak, "peak_source": self.hbm_src}
        else:
            r = {"bound": "alu", "achieved": None if stale else tf, "peak": nominal, "unit": "TFLOP/s",
                 "frac": None if stale else tf / nominal,
                 "peak_source": f"{self.sm_count} SMs x {FP64_LANES_PER_SM_CLK} fp64 lanes x 2 flop x {sm_max:.0f} MHz "
                                "(unit counts and clocks.max.sm; DESIGN.md section 6)"}
        r.update({"traffic": None, "kernel": "; ".join(c["kernels"]), "flop_per_unit": c["flop_per_unit"],
                  "fp64_inst_per_unit": c["fp64_inst_per_unit"], "inst_per_unit": c["inst_per_unit"],
                  "bytes_per_unit": bytes_per_unit, "alu_tflops": None if stale else tf, "alu_frac": None if stale else tf / nominal,
                  "hbm_gbs": gbs, "hbm_frac": gbs / self.hbm_peak,
                  "counts_source": c["source"], "counts_commit": c["commit"], "counts_stale": c["stale"]})
        if note:
            r["note"] = note
        return r


def _time_steps(ctx: Ctx, step, steps: int, warm: int, flush: bool = False):
    """Per-step CUDA events on the launching stream (an L2 flush, if any, stays outside the timed intervals)."""
    torch = ctx.torch
    sampler = ClockSampler(ctx.local)
    for i in range(warm):
        step(i)
    sampler.wait_first_row()
    step(warm)
    torch.cuda.synchronize()
    evs = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(steps)]
    l0 = ctx.osc.osc_launch_count()
    for i, (a, b) in enumerate(evs):
        if flush:
            ctx.flush(i)
        a.record(ctx.stream)
        step(i)
        b.record(ctx.stream)
    torch.cuda.synchronize()
    launches = ctx.osc.osc_launch_count() - l0
    ms = sum(a.elapsed_time(b) for a, b in evs)
    return ms / steps, int(launches), sampler.stop()


def leg_config0(ctx: Ctx, steps: int, warm: int, n: int = None):
    torch, osc = ctx.torch, ctx.osc
    n = n or 100_000
    d_et = torch.from_numpy(wl.e_true(n, seed=0)).to(ctx.dev)
    out = torch.empty((2, n), dtype=torch.float64, device=ctx.dev)

    def step(i):
        osc.osc_set_params(**wl.table1())
        osc.osc_prob(d_et, 1, 1, 0, P_out=out[0])
        osc.osc_prob(d_et, 1, 0, 0, P_out=out[1])

    ms, launches, clocks = _time_steps(ctx, step, steps, warm, flush=True)
    ups = 2 * n / (ms * 1e-3)
    return {"workload": "configs[0]: 1e5 events, Table 1, P(numu->numu) and P(numu->nue) (2 osc_prob calls per step)",
            "events": n, "units_per_step": 2 * n, "unit": "event evaluations/s", "units_per_s": ups, "ms_per_step": ms,
            "gpu_launches": launches, "l2": "flushed between steps (inputs fit L2)", "clocks": clocks,
            "roofline": ctx.roofline("k1", ups, 16.0, clocks,
                                     note="launch-latency bound at this size: the fractions are not kernel quality"
                                     if n < 1_000_000 else None)}


def leg_config1(ctx: Ctx, steps: int, warm: int, n: int = None):
    torch, osc = ctx.torch, ctx.osc
    n = n or 10_000_000
    d_et = torch.from_numpy(wl.e_true(n, seed=1)).to(ctx.dev)
    out = torch.empty((2, 9, n), dtype=torch.float64, device=ctx.dev)
    runs = wl.config1_runs()

    def step(i):
        osc.osc_set_params(**runs[i % len(runs)])
        osc.osc_prob_all(d_et, 0, P_out=out[0])
        osc.osc_prob_all(d_et, 1, P_out=out[1])

    ms, launches, clocks = _time_steps(ctx, step, steps, warm)
    ups = 2 * n / (ms * 1e-3)
    return {"workload": "configs[1]: 1e7 events, all 9 transitions for nu and nubar (2 osc_prob_all calls = 18 output "
                        "arrays per step), delta_cp drawn per run, both hierarchies alternate",
            "events": n, "units_per_step": 2 * n, "unit": "(event, nu/nubar) solves/s", "units_per_s": ups, "ms_per_step": ms,
            "gpu_launches": launches, "l2": "working set > L2", "clocks": clocks,
            "roofline": ctx.roofline("k1b", ups, 80.0, clocks, bound="hbm",
                                     note="80 B per unit (8 in + 72 out): below the fp64/HBM ridge, so HBM is the formal "
                                          "bound; alu_frac is the fp64 fraction of the same launch")}


def leg_config3(ctx: Ctx, steps: int, warm: int, n: int = None, k5: bool = False):
    torch, osc = ctx.torch, ctx.osc
    n = n or 1_000_000
    et, er, w0, ch = wl.events(n, seed=2)
    d_et, d_er, d_w0, d_ch = (torch.from_numpy(a).to(ctx.dev) for a in (et, er, w0, ch))
    d_edges = torch.from_numpy(wl.bin_edges()).to(ctx.dev)
    pts = osc.pack_params(wl.scan_points())                                 # marshalled once (binding only)
    out = torch.empty((len(pts), osc.N_CHANNELS, wl.N_BINS), dtype=torch.float64, device=ctx.dev)
    if k5:
        osc.osc_set_batch_path("k5")

    def step(i):
        osc.osc_reweight_bin_batch(pts, d_et, d_er, d_w0, d_ch, 1.0, d_edges, hist_out=out)

    try:
        ms, launches, clocks = _time_steps(ctx, step, steps, warm)
    finally:
        if k5:
            osc.osc_set_batch_path("auto")
    units = n * len(pts)
    ups = units / (ms * 1e-3)
    return {"workload": "configs[3]: 1e6 events x 1024 oscillation points (32x32 grid of sin2_th23 x dm2_32, delta_cp per "
                        "point) in ONE osc_reweight_bin_batch call"
                        + (" forced through k5 (every (event, point) pair gets the full closed form)" if k5
                           else " (factorised path k4)"),
            "events": n, "points": len(pts), "units_per_step": units, "unit": "(event, point) evaluations/s",
            "units_per_s": ups, "ms_per_step": ms, "gpu_launches": launches, "l2": "25 MB of events, reused by 1024 points",
            "clocks": clocks,
            "roofline": ctx.roofline("k5" if k5 else "k4", ups, 25.0 / len(pts), clocks,
                                     note="whole call (sort, main kernel, merge); counts are of all its kernels")}


def leg_config4(ctx: Ctx, steps: int, n_max: int):
    """configs[4]: size sweep N = 1e3 .. n_max on the configs[2] path (k2, one energy scale per launch, Table 1), plus
    the 12 (rho, L, hierarchy) settings at N = 1e7.  The sizes are prefixes of one device-drawn sample."""
    torch, osc = ctx.torch, ctx.osc
    d_edges = torch.from_numpy(wl.bin_edges()).to(ctx.dev)
    hist = torch.zeros((osc.N_CHANNELS, wl.N_BINS), dtype=torch.float64, device=ctx.dev)
    sizes = [10 ** k for k in range(3, 10) if 10 ** k <= n_max]
    big = wl.events_device(sizes[-1], seed=4, device=ctx.dev)
    torch.cuda.synchronize()
    sampler = ClockSampler(ctx.local)
    launches0 = osc.osc_launch_count()

    def time_k2(ev, par, reps):
        """Mean duration of one k2 launch (ms).  Inputs below the L2 size are evicted before every launch."""
        osc.osc_set_params(**par)
        small = ev[0].numel() * BYTES_PER_EVENT < 200e6
        for _ in range(3):
            osc.osc_reweight_bin(*ev, 1.0, d_edges, hist_out=hist)
        a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        if small:
            total = 0.0
            for i in range(reps):
                ctx.flush(i)
                a.record(ctx.stream)
                osc.osc_reweight_bin(*ev, 1.0, d_edges, hist_out=hist)
                b.record(ctx.stream)
                torch.cuda.synchronize()
                total += a.elapsed_time(b)
            return total / reps
        a.record(ctx.stream)
        for _ in range(reps):
            osc.osc_reweight_bin(*ev, 1.0, d_edges, hist_out=hist)
        b.record(ctx.stream)
        torch.cuda.synchronize()
        return a.elapsed_time(b) / reps

    rows = []
    for n in sizes:
        ev = [t[:n] for t in big]
        ms = time_k2(ev, wl.table1(), max(3, min(steps, 20)))
        rows.append({"N": n, "ms_per_launch": ms, "events_per_s": n / (ms * 1e-3)})
        if n == 10_000_000:
            rows[-1]["settings"] = [{"rho": par["rho_g_cm3"], "L": par["L_km"], "hierarchy": par["hierarchy"],
                                     "events_per_s": n / (time_k2(ev, par, 5) * 1e-3)} for par in wl.sweep_settings()]
    torch.cuda.synchronize()
    clocks = sampler.stop()
    launches = int(osc.osc_launch_count() - launches0)
    del big
    torch.cuda.empty_cache()
    c = opcounts.counts("k2", ctx.counts)
    nominal, _ = ctx.nominal_tflops(clocks)
    for r in rows:
        r["frac_fp64"] = None if c["stale"] else r["events_per_s"] * c["flop_per_unit"] / 1e12 / nominal
        r["frac_hbm"] = r["events_per_s"] * BYTES_PER_EVENT / 1e9 / ctx.hbm_peak
    last = rows[-1]
    return {"workload": "configs[4]: size sweep on the configs[2] path (k2, one launch per row), Table 1; rho x L x "
                        "hierarchy settings at N = 1e7; sizes are prefixes of one sample drawn on the device (seed 4)",
            "sizes": sizes, "unit": UNIT, "units_per_s": last["events_per_s"], "ms_per_step": last["ms_per_launch"],
            "gpu_launches": launches, "l2": "inputs smaller than L2 are evicted (256 MB fill) before every timed launch",
            "clocks": clocks, "roofline": ctx.roofline("k2", last["events_per_s"], BYTES_PER_EVENT, clocks,
                                                       note=f"at the largest N ({last['N']}); per-N fractions under `sweep`"),
            "sweep": rows}


def print_leg(args, leg):
    """One secondary config as a JSON line of its own (same schema as the bench line)."""
    print(json.dumps({
        "metric": METRIC, "value": leg["units_per_s"], "unit": leg["unit"], "n_gpus": 1, "steps": args.steps,
        "warmup": max(args.warmup, 3), "ms_per_step": leg["ms_per_step"], "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {k: leg[k] for k in ("workload", "events", "points", "units_per_step", "sizes", "l2") if k in leg},
        "clocks": leg["clocks"], "e2e": None, "gpu_launches": leg["gpu_launches"], "roofline": leg["roofline"],
        "cpu_baseline": None, **({"sweep": leg["sweep"]} if "sweep" in leg else {})}))


def main():
    args = parse()
    if args.impl == "reference":
        run_reference(args)
        return
    warm = max(args.warmup, 3)
    if args.workload != "config2":
        ctx = Ctx(0)
        leg = {"config0": lambda: leg_config0(ctx, args.steps, warm, args.events),
               "config1": lambda: leg_config1(ctx, args.steps, warm, args.events),
               "config3": lambda: leg_config3(ctx, args.steps, warm, args.events),
               "config3-k5": lambda: leg_config3(ctx, args.steps, warm, args.events, k5=True),
               "config4": lambda: leg_config4(ctx, args.steps, args.events or args.sweep_max)}[args.workload]()
        print_leg(args, leg)
        return

    import torch.distributed as dist

    from paper_1311_7579_b200 import sharding

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if world != args.gpus:
        if world == 1 and args.gpus > 1:
            raise SystemExit("launch with torch.distributed.run --nproc-per-node N for --gpus N")
    ctx = Ctx(local)
    torch, osc, device, stream = ctx.torch, ctx.osc, ctx.dev, ctx.stream
    distributed = "RANK" in os.environ and "MASTER_ADDR" in os.environ      # under torchrun, also at world size 1
    if distributed:
        dist.init_process_group("nccl", device_id=device)

    par = wl.table1()
    if args.scaling == "strong":
        n_total = args.events or N_EVENTS
        b, e = sharding.shard_bounds(n_total, rank, world)
        et, er, w0, ch = (a[b:e].copy() for a in wl.events(n_total, seed=2))     # one seeded sample, contiguous slices
        n = e - b
    else:
        n = args.events or N_EVENTS
        n_total = n * world
        et, er, w0, ch = wl.events(n, seed=2 + 1000 * rank)                      # each rank its own 1e7 events
    edges = wl.bin_edges()
    # pinned host copies (e2e leg) and device-resident copies (value leg)
    h_et, h_er, h_w0, h_ch = (torch.from_numpy(a).pin_memory() for a in (et, er, w0, ch))
    d_et, d_er, d_w0, d_ch = (t.to(device) for t in (h_et, h_er, h_w0, h_ch))
    d_edges = torch.from_numpy(edges).to(device)
    hist = torch.zeros((len(SCALES), osc.N_CHANNELS, wl.N_BINS), dtype=torch.float64, device=device)

    def step():
        osc.osc_set_params(**par)                                                           # a1
        for k, s in enumerate(SCALES):
            osc.osc_reweight_bin(d_et, d_er, d_w0, d_ch, s, d_edges, hist_out=hist[k])      # a2a-a3c
        sharding.allreduce_hist(hist)                                                       # 8(e): no-op at N = 1

    def barrier():
        if distributed and world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    def max_over_ranks(ms: float) -> float:
        t = torch.tensor([ms], dtype=torch.float64, device=device)
        if distributed:
            dist.all_reduce(t, op=dist.ReduceOp.MAX)
        return float(t.item())

    def timed(fn, steps):
        a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        barrier()
        a.record(stream)
        for _ in range(steps):
            fn()
        b.record(stream)
        barrier()
        return max_over_ranks(a.elapsed_time(b))

    # the clock sampler starts BEFORE the warm-up and the timed region waits for its first row: the start-up of nvidia-smi
    # (~0.2 s of driver queries) otherwise falls into the few milliseconds that are timed and costs 0.7 % of `value`
    sampler = ClockSampler(local) if rank == 0 else None
    for _ in range(warm):
        step()
    if sampler is not None:
        sampler.wait_first_row()
    for _ in range(2):
        step()
    barrier()

    # ---- timed region: device-resident inputs -----------------------------------------------------------------
    launches0 = osc.osc_launch_count()
    t_wall0 = time.time()
    ms = timed(step, args.steps)
    launches = osc.osc_launch_count() - launches0
    # the clock sampler keeps running through the legs below (the same kernels on the same data, back to back): the
    # timed region of `value` alone is a few milliseconds, too short for more than a sample or two
    value = n_total * len(SCALES) * args.steps / (ms * 1e-3)

    # ---- dominant kernel alone (k2), CUDA events around back-to-back launches, for the roofline ----------------
    osc.osc_set_params(**par)
    reps = 30
    it = iter(range(10 ** 9))

    def one_k2():
        i = next(it)
        osc.osc_reweight_bin(d_et, d_er, d_w0, d_ch, SCALES[i % 3], d_edges, hist_out=hist[i % 3])

    torch.cuda.synchronize()
    ks, ke = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    for _ in range(3):             # the device has just idled through a host round trip: three untimed launches first
        one_k2()
    ks.record(stream)
    for _ in range(reps):
        one_k2()
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
    f_ms = timed(step_fused, args.steps)
    fused = {"value": n_total * len(SCALES) * args.steps / (f_ms * 1e-3), "unit": UNIT, "ms_per_step": f_ms / args.steps,
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
    p_ms = timed(step_plan, args.steps)
    planned = {"value": n_total * len(SCALES) * args.steps / (p_ms * 1e-3), "unit": UNIT, "ms_per_step": p_ms / args.steps,
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
            dt = max_over_ranks(time.perf_counter() - t0)
            return n_total * len(SCALES) * e_steps / dt

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
        if distributed:
            dist.destroy_process_group()
        return

    # ---- the two legs reported beside `value`: their own roofline objects (whole step of this rank: one launch of k2s;
    # three launches of the plan kernel plus their merges) -----------------------------------------------------------
    fused["roofline"] = ctx.roofline("k2s", n / (fused["ms_per_step"] * 1e-3), BYTES_PER_EVENT, clocks,
                                     note="whole step = one launch; a unit is an event weighted once and binned at three "
                                          "energy scales")
    planned["roofline"] = ctx.roofline("plan", n * len(SCALES) / (planned["ms_per_step"] * 1e-3), 16.0, clocks,
                                       note="whole step = three launches of the plan kernel and three merges; counts are of "
                                            "the main kernel; 16 B per event (sorted E_true, w0)")

    # ---- roofline of the dominant kernel ------------------------------------------------------------------------
    roofline = ctx.roofline("k2", n / (k_ms * 1e-3), BYTES_PER_EVENT, clocks)
    c2 = opcounts.counts("k2", ctx.counts)
    roofline.update({"kernel_ms": k_ms, "flop_per_event": c2["flop_per_unit"],
                     "traffic": c2["dram_bytes_per_call"] if (n == c2["units_per_call"] and not c2["stale"]) else None,
                     "traffic_unit": f"DRAM bytes per launch, ncu ({c2['source']}); algorithmic {n * BYTES_PER_EVENT}",
                     "peak_probe": fp64_peak_tflops,
                     "frac_of_probe": None if roofline["achieved"] is None else roofline["achieved"] / fp64_peak_tflops,
                     "peak_probe_source": "DFMA-only probe kernel measured in this run (osc_fp64_peak_probe)",
                     "hbm": {"achieved": roofline["hbm_gbs"], "peak": ctx.hbm_peak, "unit": "GB/s",
                             "frac": roofline["hbm_frac"], "peak_source": ctx.hbm_src}})

    # ---- the other four configs, same process, each with its own clock sample (N = 1 only) ---------------------
    configs = None
    if world == 1 and not args.no_configs:
        del d_et, d_er, d_w0, d_ch
        torch.cuda.empty_cache()
        k = max(5, min(args.steps, 20))
        configs = {"config0": leg_config0(ctx, k, warm), "config1": leg_config1(ctx, k, warm),
                   "config3": leg_config3(ctx, k, warm), "config4": leg_config4(ctx, k, args.sweep_max)}

    cpu = None
    if not args.no_cpu_baseline and world == 1:
        cpu = oracle_rate()

    out = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": warm,
        "ms_per_step": ms / args.steps, "higher_is_better": True, "scaling": args.scaling, "vs_baseline": None,
        "dtype": "f64", "data": "synthetic",
        "config": {"workload": "configs[2]: 1e7 events/GPU x 4 channels, 50-bin E_reco histograms over 0-5 GeV, "
                               "energy scales {0.97,1.00,1.03}, Table 1 parameters (normal hierarchy)",
                   "events_per_gpu": n, "events_total": n_total, "passes_per_step": len(SCALES), "n_bins": wl.N_BINS,
                   "l2": "inputs (250 MB per pass) larger than L2 (126 MB); no explicit flush",
                   "parallelism": (f"events sharded over {world} GPU(s) ({args.scaling} scaling); histogram all-reduce"
                                   if world > 1 else "1 GPU")},
        "clocks": clocks, "e2e": e2e, "gpu_launches": int(launches), "roofline": roofline, "cpu_baseline": cpu,
        "fused_scales": fused, "planned": planned, "configs": configs,
    }
    print(json.dumps(out))
    if distributed:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
