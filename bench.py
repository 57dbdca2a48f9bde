#!/usr/bin/env python
"""bench.py -- particle-turns/s of the longitudinal tracking hot path on B200.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl reference] [--only LEG]

Workload (config.workload): BASELINE.json:configs[1], the paper's profiled run shape
(10^5 macro-particles x 7*10^4 turns, leap-frog), as a seeded synthetic hollow
bunch.  One STEP = one pass of the whole hot path over that bunch: entry load, 70 000 turns
register-resident (fused mode), exit store, then the bucket-membership count of the final
state.  `value` is device-timed with the bunch already in HBM; `e2e` goes through the C ABI
with HOST buffers (lt_track_fused_host: H2D, track, count, D2H inside the timed region).

Everything else the measurement contract asks for sits INSIDE `roofline`.  The driver's record
keeps the SCALAR keys of that object and drops nested ones, so every leg's fraction is repeated
as a flat key (`per_turn_frac`, `per_turn_gbs`, `cfg2_frac`, `cfg4_*_frac`, `f2_*_frac`, `f3_*`,
`f4_*`, `f1_us_per_launch_1turn_*`, `traffic_source`; flat_summary()) and the scalars are printed
last.  The nested legs: `per_turn` (configs[3], the HBM-bound half of the metric), `configs`
(configs[0], [2] and the six configs[4] variants), `f1_chunk_sweep` (turns per launch 1 ..
2^14 at a fixed total: the B200 redo of the paper's Fig. 5), `size_sweep`
(n = 2^10 .. 2^24: the analogue of its Table 2), `next` (the
SURVEY.md sec. 8(f) rows) and `pipe_probe` (what the FP64 pipe issues).  Every leg carries the
NVML clock record sampled while it ran.  `traffic` values come from profiles/ncu_traffic.json.

N > 1 (torchrun): particles are independent, so every rank tracks its own
seeded bunch of the same size -- weak scaling, no data-path collective; the only collectives
are the barrier, the MAX over ranks of the device time, and one SUM all-reduce of the raw
per-turn sums in the sharded per-turn leg.

`--impl reference` times the CPU oracle (oracle/, as it stands) on the host cores on a
bounded sample of the same workload; it neither builds nor loads the CUDA library.
"""
from __future__ import annotations

import argparse
import json
import os
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "particle-turns/sec (fp64 leap-frog)"
UNIT = "particle-turns/s"
# Declared algorithmic pipe instructions per particle-turn, fixed before
# tuning: a smaller count makes the reported fraction smaller.  fp64: 1 merged drift + 3 exact
# range reduction + 1 square + 7 Horner + 1 kick FMA = 13; the cosine of the double harmonic adds
# 8 Horner + 2 = 23; Ruth4 = three kicks and drifts.  fp32 (degree-4 / degree-5 polynomials):
# 10, 17 and three times that.
FP64_INSTR = {("leapfrog", 0.0): 13, ("euler_cromer", 0.0): 13, ("ruth4", 0.0): 39,
              ("leapfrog", 0.5): 23, ("euler_cromer", 0.5): 23, ("ruth4", 0.5): 69}
FP32_INSTR = {("leapfrog", 0.0): 10, ("euler_cromer", 0.0): 10, ("ruth4", 0.0): 30,
              ("leapfrog", 0.5): 17, ("euler_cromer", 0.5): 17, ("ruth4", 0.5): 51}
FP64_INSTR_PER_PT = FP64_INSTR[("leapfrog", 0.0)]
INSTR_F2_PROGRAMME = 15                   # 13 + f*a_t + the phase-offset add
INSTR_F2_RAMP = 15                        # 13 + (G y + C) + the phase-offset add (scaled layout; 16 with f*(g amp) in the plain one)
BYTES_PER_PT_PER_TURN_MODE = 32           # 16 B read + 16 B write per particle-turn
SMS, FP64_LANES_PER_SM, FP32_LANES_PER_SM = 148, 64, 128
CPU_SAMPLE_TURNS = 10_000                 # all-cores oracle leg: 1e9 particle-turns
CPU_SAMPLE_TURNS_1T = 1_000               # one-thread oracle leg: 1e8 particle-turns


def measured_peaks() -> dict:
    try:
        return json.load(open(os.path.join(ROOT, "MEASURED_PEAKS.json")))
    except Exception:
        return {}


def ncu_traffic() -> dict:
    """DRAM bytes per launch (dram__bytes_read.sum + dram__bytes_write.sum, ncu --set full) of
    the kernels the rooflines are quoted on: profiles/ncu_traffic.json, written from the
    committed captures (each entry names its ncu command and the commit it was taken at)."""
    try:
        raw = json.load(open(os.path.join(ROOT, "profiles", "ncu_traffic.json")))
        out = {k: int(v["dram_bytes_read"]) + int(v["dram_bytes_write"])
               for k, v in raw.get("kernels", {}).items()}
        out.update({k + "_ncu_us": float(v["duration_us"]) for k, v in raw.get("kernels", {}).items()
                    if "duration_us" in v})
        out.update({k + "_source": "profiles/ncu_traffic.json, captured at %s" % v.get("captured_at_commit", "?")
                    for k, v in raw.get("kernels", {}).items()})
        return out
    except Exception:
        return {}


class ClockSampler:
    """Samples SM clock and throttle reasons through NVML while a timed region runs."""
    REASONS = {0x4: "sw_power_cap", 0x8: "hw_slowdown", 0x20: "sw_thermal_slowdown",
               0x40: "hw_thermal_slowdown", 0x80: "hw_power_brake_slowdown",
               0x2: "applications_clocks_setting", 0x10: "sync_boost"}

    def __init__(self, index: int, period_s: float = 0.005):
        self.samples, self.reasons, self.max_mhz = [], set(), None
        self.period, self._stop, self._thr, self._h = period_s, threading.Event(), None, None
        try:
            import pynvml
            pynvml.nvmlInit()
            self._nv = pynvml
            self._h = pynvml.nvmlDeviceGetHandleByIndex(index)
            self.max_mhz = int(pynvml.nvmlDeviceGetMaxClockInfo(self._h, pynvml.NVML_CLOCK_SM))
        except Exception:
            self._h = None

    def _sample(self):
        nv = self._nv
        try:
            self.samples.append(int(nv.nvmlDeviceGetClockInfo(self._h, nv.NVML_CLOCK_SM)))
            try:
                mask = int(nv.nvmlDeviceGetCurrentClocksEventReasons(self._h))
            except Exception:
                mask = int(nv.nvmlDeviceGetCurrentClocksThrottleReasons(self._h))
            for bit, name in self.REASONS.items():
                if mask & bit:
                    self.reasons.add(name)
        except Exception:
            pass

    def _run(self):
        while not self._stop.is_set():
            self._sample()
            self._stop.wait(self.period)

    def __enter__(self):
        if self._h is not None:
            self._thr = threading.Thread(target=self._run, daemon=True)
            self._thr.start()
        return self

    def __exit__(self, *a):
        self._stop.set()
        if self._thr:
            self._thr.join()

    def summary(self, short: bool = False) -> dict:
        s = sorted(self.samples)
        out = {"sm_mhz": s[len(s) // 2] if s else None, "sm_max_mhz": self.max_mhz,
               "reasons": sorted(self.reasons), "samples": len(s)}
        if short:
            out = {"sm_mhz": out["sm_mhz"], "reasons": out["reasons"], "samples": out["samples"]}
        return out


def physical_gpu_index(local: int) -> int:
    vis = os.environ.get("CUDA_VISIBLE_DEVICES")
    if vis:
        try:
            return int(vis.split(",")[local])
        except Exception:
            return local
    return local


def cpu_model() -> str:
    try:
        for line in open("/proc/cpuinfo"):
            if line.startswith("model name"):
                return line.split(":", 1)[1].strip()
    except Exception:
        pass
    return "unknown"


# ----------------------------------------------------------------------------- oracle legs
def oracle_rate(n: int, turns: int, seed: int, threads: int | None = None):
    """Times the CPU oracle as it stands: n particles of the cfg1 bunch x `turns` turns."""
    import oracle
    from paper_1610_05801_b200 import workloads as wl
    cores = len(os.sched_getaffinity(0))
    use = threads or cores
    oracle.set_num_threads(use)
    z0, d0 = wl.hollow_bunch(n, seed)
    p = oracle.make_params(wl.RING, "leapfrog")
    oracle.track(p, z0[:1000], d0[:1000], 10)          # load the library, touch the pages
    t0 = time.perf_counter()
    oracle.track(p, z0, d0, turns)
    dt = time.perf_counter() - t0
    oracle.set_num_threads(cores)
    return n * turns / dt, dt, use


def run_reference(args) -> None:
    """--impl reference: the oracle on the host cores, same metric/config, bounded sample.
    Builds and loads oracle/ only -- nothing of the CUDA product is compiled or mapped."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    import oracle
    oracle.build()
    from paper_1610_05801_b200 import workloads as wl      # input recipe only (numpy)
    cfg = wl.CONFIGS[1]
    n, turns_sample = cfg["n"], 1000
    for _ in range(args.warmup):
        oracle_rate(n, 100, cfg["seed"])
    t_total, pts = 0.0, 0
    cores = None
    for _ in range(args.steps):
        rate, dt, cores = oracle_rate(n, turns_sample, cfg["seed"])
        t_total += dt
        pts += n * turns_sample
    value = pts / t_total
    sample = "%d particles x %d turns per step (of %d turns), %d steps" % (
        n, turns_sample, cfg["turns"], args.steps)
    print(json.dumps({
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * t_total / args.steps,
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64",
        "data": "synthetic",
        "config": {"workload": "configs[1] hollow bunch 1e5 particles x 7e4 turns, leap-frog, "
                               "single harmonic (bounded sample: first %d turns per step)" % turns_sample,
                   "particles": n, "turns": cfg["turns"]},
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": cores, "kind": "oracle",
                         "sample": sample, "cpu": cpu_model()},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }))


# ----------------------------------------------------------------------------- CUDA arm helpers
class Ctx:
    """What every leg needs: the binding, streams, peaks, timers with a clock record per leg."""

    def __init__(self, lt, wl, torch, dist, world, rank, local):
        self.lt, self.wl, self.torch, self.dist = lt, wl, torch, dist
        self.world, self.rank, self.local = world, rank, local
        self.stream = torch.cuda.current_stream()
        self.sp = self.stream.cuda_stream
        self.peaks = measured_peaks()
        self.traffic = ncu_traffic()
        self.sm_max_mhz = float(self.peaks.get("sm_max_mhz", 1965.0))
        self.peak_fp64 = SMS * FP64_LANES_PER_SM * self.sm_max_mhz * 1e-3      # G lane-instr/s
        self.peak_fp32 = SMS * FP32_LANES_PER_SM * self.sm_max_mhz * 1e-3
        self.hbm_peak = float(self.peaks.get("hbm_gbs", 6650.0))
        self.hbm_source = ("MEASURED_PEAKS.json hbm_gbs" if "hbm_gbs" in self.peaks
                           else "fallback 6650 GB/s (B200_PROFILING.md)")
        self.flush = torch.empty(256 << 20, dtype=torch.uint8, device="cuda")   # > 126 MB L2
        self.gpu_index = physical_gpu_index(local)

    def barrier(self):
        if self.world > 1:
            self.dist.barrier()

    def max_over_ranks(self, x: float) -> float:
        if self.world == 1:
            return x
        t = self.torch.tensor([x], dtype=self.torch.float64, device="cuda")
        self.dist.all_reduce(t, op=self.dist.ReduceOp.MAX)
        return float(t.item())

    def clock(self):
        return ClockSampler(self.gpu_index)

    def timed(self, fn, reps, restore=None, flush=True):
        """Mean device time of fn over `reps` repetitions after one warm-up repetition, CUDA
        events on the launching stream, L2 flushed (256 MB fill) before each; max over ranks."""
        torch = self.torch
        t = 0.0
        for r in range(reps + 1):
            if restore:
                restore()
            if flush:
                self.flush.fill_(r)
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record(self.stream)
            fn()
            e1.record(self.stream)
            torch.cuda.synchronize()
            if r:
                t += e0.elapsed_time(e1) * 1e-3
        return self.max_over_ranks(t) / reps

    def alu(self, instr, pts, sec, traffic=None, fp32=False):
        peak = self.peak_fp32 if fp32 else self.peak_fp64
        g = instr * pts / sec / 1e9
        return {"bound": "alu", "achieved": g, "peak": peak,
                "unit": "G FP32 instr/s" if fp32 else "G FP64 instr/s", "frac": g / peak,
                "instr_per_particle_turn": instr, "traffic": self.traffic.get(traffic)}

    def hbm(self, bytes_per_pt, pts, sec, traffic=None):
        g = bytes_per_pt * pts / sec / 1e9
        return {"bound": "hbm", "achieved": g, "peak": self.hbm_peak, "unit": "GB/s",
                "frac": g / self.hbm_peak, "bytes_per_particle_turn": bytes_per_pt,
                "traffic": self.traffic.get(traffic)}

    def dev(self, a, dtype=None):
        import numpy as np
        return self.torch.from_numpy(np.ascontiguousarray(a, dtype=dtype)).cuda()

    def shape(self, tr):
        lt = self.lt
        return {"mode": tr.get_stat(lt.STAT_LAST_MODE), "grid": tr.get_stat(lt.STAT_LAST_GRID),
                "block": tr.get_stat(lt.STAT_LAST_BLOCK), "ilp": tr.get_stat(lt.STAT_LAST_ILP),
                "item_turns": tr.get_stat(lt.STAT_LAST_ITEM_TURNS)}


# ----------------------------------------------------------------------------- configs[0], [2], [4]
def bench_configs(cx: Ctx) -> dict:
    """BASELINE.json:configs[0], configs[2] (full length) and the six configs[4] variants in fused
    mode (configs[1] is the headline, configs[3] the per-turn leg).  The particle-count axis is
    the analogue of the paper's Table 2."""
    lt, wl, np = cx.lt, cx.wl, __import__("numpy")
    out = {}
    with cx.clock() as clk:
        for idx, reps in ((0, 20), (2, 3)):
            cfg = wl.CONFIGS[idx]
            n, turns = cfg["n"], cfg["turns"]
            z0, d0 = wl.make_bunch(cfg, seed=cfg["seed"] + cx.rank)
            z, d = cx.dev(z0), cx.dev(d0)
            zi, di = z.clone(), d.clone()
            tr = lt.Tracker(wl.RING, "leapfrog")
            sec = cx.timed(lambda: tr.track_fused(z, d, n, turns, cx.sp), reps,
                           lambda: (z.copy_(zi), d.copy_(di)))
            out["configs[%d]" % idx] = {
                "n": n, "turns": turns, "variant": "leapfrog fp64", "ms": 1e3 * sec,
                "value": cx.world * n * turns / sec,
                "roofline": cx.alu(FP64_INSTR_PER_PT, n * turns, sec), "shape": cx.shape(tr)}
            del z, d, zi, di, tr
        cfg = wl.CONFIGS[4]
        n, turns, r = cfg["n"], cfg["turns"], cfg["ratio2"]
        z0, d0 = wl.gaussian_bunch(n, cfg["sigma_z"], cfg["seed"] + cx.rank, ratio2=r)
        for integ in cfg["integrators"]:
            for f32 in (False, True):
                dt = np.float32 if f32 else np.float64
                z, d = cx.dev(z0, dt), cx.dev(d0, dt)
                zi, di = z.clone(), d.clone()
                tr = lt.Tracker(wl.RING, integ, r)
                run = tr.track_fused_f32 if f32 else tr.track_fused
                sec = cx.timed(lambda: run(z, d, n, turns, cx.sp), 3,
                               lambda: (z.copy_(zi), d.copy_(di)))
                instr = (FP32_INSTR if f32 else FP64_INSTR)[(integ, r)]
                out["configs[4] %s %s" % (integ, "fp32" if f32 else "fp64")] = {
                    "n": n, "turns": turns, "ratio2": r, "ms": 1e3 * sec,
                    "value": cx.world * n * turns / sec,
                    "roofline": cx.alu(instr, n * turns, sec, fp32=f32), "shape": cx.shape(tr)}
                del z, d, zi, di, tr
    out["clocks"] = clk.summary(short=True)
    return out


# ----------------------------------------------------------------------------- particle-count sweep
def bench_sizes(cx: Ctx) -> dict:
    """The analogue of the paper's Table 2 (kernel time against the number of
    macro-particles, flat from 512 to 4096 on 14 SMs): 10^4 leap-frog turns in fused mode for
    n = 2^10 .. 2^24."""
    lt, wl = cx.lt, cx.wl
    turns = 10_000
    rows = []
    with cx.clock() as clk:
        for e in range(10, 25, 2):
            n = 1 << e
            z0, d0 = wl.make_bunch(wl.CONFIGS[0], n=n, seed=1000 + e + cx.rank)
            z, d = cx.dev(z0), cx.dev(d0)
            tr = lt.Tracker(wl.RING, "leapfrog")
            sec = cx.timed(lambda: tr.track_fused(z, d, n, turns, cx.sp), 2)
            rows.append({"n": "2^%d" % e, "ms": round(1e3 * sec, 4), "value": cx.world * n * turns / sec,
                         "frac": round(FP64_INSTR_PER_PT * n * turns / sec / 1e9 / cx.peak_fp64, 4),
                         "mode": tr.get_stat(lt.STAT_LAST_MODE), "block": tr.get_stat(lt.STAT_LAST_BLOCK),
                         "ilp": tr.get_stat(lt.STAT_LAST_ILP)})
            del z, d, tr
    return {"turns": turns, "rows": rows, "clocks": clk.summary(short=True)}


# ----------------------------------------------------------------------------- f1: chunk-size sweep
def bench_f1(cx: Ctx) -> dict:
    """SURVEY.md sec. 8(f) row f1, the B200 redo of the paper's Fig. 5 (PAPER.md:167-179,
    "Tracking execution times for different number of turns per inner kernel loops"): 2^14 turns
    of the configs[2] bunch (10^6 particles) with 1 .. 2^14 turns per kernel launch
    (LT_OPT_CHUNK_TURNS; the state goes through HBM between launches), plus the per-turn kernel
    (one turn per launch, no moments) with and without CUDA-graph replay."""
    lt, wl = cx.lt, cx.wl
    cfg = wl.CONFIGS[2]
    n, total = cfg["n"], 1 << 14
    z0, d0 = wl.make_bunch(cfg, seed=cfg["seed"] + cx.rank)
    z, d = cx.dev(z0), cx.dev(d0)
    rows = []
    with cx.clock() as clk:
        for chunk in (1, 4, 16, 64, 256, 1024, 4096, 16384):
            tr = lt.Tracker(wl.RING, "leapfrog")
            tr.set_option(lt.OPT_CHUNK_TURNS, chunk)
            l0 = tr.get_stat(lt.STAT_KERNEL_LAUNCHES)
            reps = 2 if chunk < 16 else 3
            sec = cx.timed(lambda: tr.track_fused(z, d, n, total, cx.sp), reps)
            rows.append({"turns_per_launch": chunk, "kernel": "fused",
                         "launches": (tr.get_stat(lt.STAT_KERNEL_LAUNCHES) - l0) // (reps + 1),
                         "ms": 1e3 * sec, "value": cx.world * n * total / sec,
                         "us_per_launch": 1e6 * sec * chunk / total})
            del tr
        for graph in (0, 1):
            tr = lt.Tracker(wl.RING, "leapfrog")
            tr.set_option(lt.OPT_PER_TURN_GRAPH, graph)
            turns = 2048
            sec = cx.timed(lambda: tr.track_per_turn(z, d, n, turns, None, None, cx.sp), 2)
            rows.append({"turns_per_launch": 1, "kernel": "per_turn graph=%d" % graph,
                         "launches": turns, "ms": 1e3 * sec * total / turns,
                         "value": cx.world * n * turns / sec, "us_per_launch": 1e6 * sec / turns,
                         "note": "2048 turns timed, ms scaled to 2^14"})
            del tr
    return {"n": n, "total_turns": total, "rows": rows, "clocks": clk.summary(short=True)}


# ----------------------------------------------------------------------------- FP64 pipe probe
def bench_probe(cx: Ctx, table: bool = False) -> dict:
    """What the FP64 pipe of this device issues (lt_probe_pipe, clock64-based): FP64
    warp-instructions per cycle and sub-partition; the nominal peak behind roofline.peak is 0.5
    (16 FP64 lanes per sub-partition, 64 per SM).  table=True (`--only probe`) adds the rate of
    the turn loop for every (particles per lane, warps per sub-partition, sign-flip place): the
    planner's loop_rate table in csrc/longtrack.cu."""
    from paper_1610_05801_b200 import probe           # liblongtrack_probe.so: measurement tooling only
    out = {}
    with cx.clock() as clk:
        for name, kind, threads, chains in (("dadd", 2, 1024, 4), ("dmul", 3, 1024, 4),
                                            ("dfma_2reg_1uniform", 1, 1024, 4),
                                            ("dfma_3reg", 0, 1024, 4),
                                            ("turn_no_sign_flip_ilp2_w4", 12, 512, 2),
                                            ("turn_flip_on_f_ilp2_w2", 11, 256, 2),
                                            ("turn_flip_on_f_ilp2_w4", 11, 512, 2),
                                            ("turn_flip_on_q_ilp1_w5", 10, 640, 1),
                                            ("turn_flip_on_q_ilp1_w8", 10, 1024, 1)):
            rate, mhz = probe.probe_pipe(kind, SMS, threads, chains, 20000 // chains)
            out[name] = round(rate, 4)
            out["sm_mhz_under_fp64_load"] = round(mhz)
        if table:
            tab = {}
            for kind, name in ((11, "flip_on_f"), (10, "flip_on_q"), (12, "no_flip")):
                for chains in (1, 2, 4):
                    tab["%s ilp%d W=1..8" % (name, chains)] = [
                        round(probe.probe_pipe(kind, SMS, 128 * w, chains, 8000 // chains)[0], 4)
                        for w in range(1, 9)]
            out["turn_loop_table"] = tab
    out["unit"] = "FP64 warp-instr/cycle/sub-partition (nominal peak 0.5)"
    out["clocks"] = clk.summary(short=True)
    return out


# ----------------------------------------------------------------------------- launch-shape sweep
def bench_shapes(cx: Ctx) -> dict:
    """`--only shapes`: the planner against forced launch shapes of the fused kernel (particles per
    lane, warps per sub-partition, sign-flip place, item length) at the configs[1] size and at
    10^6 particles x 10^4 turns -- what profiles/r2_fused_shapes.md tabulates."""
    lt, wl = cx.lt, cx.wl
    out = {}
    with cx.clock() as clk:
        for n, turns, cfg in ((100_000, 70_000, wl.CONFIGS[1]), (1_000_000, 10_000, wl.CONFIGS[2])):
            z0, d0 = wl.make_bunch(cfg, n=n)
            z, d = cx.dev(z0), cx.dev(d0)
            cases = [("planner", {})]
            for ilp, w, fq in ((2, 1, 0), (2, 2, 0), (2, 2, 1), (2, 3, 0), (2, 4, 0), (2, 4, 1),
                               (1, 4, 1), (1, 5, 0), (1, 5, 1), (1, 6, 1), (1, 8, 0), (1, 8, 1)):
                for item in ((512, 2048, 8192) if (ilp, w, fq) in ((2, 2, 0), (2, 4, 0), (1, 5, 1)) else (2048,)):
                    cases.append(("ilp%d W%d %s item%d" % (ilp, w, "q" if fq else "f", item),
                                  {lt.OPT_FUSED_MODE: 3, lt.OPT_FUSED_ILP: ilp, lt.OPT_WARPS_PER_SMSP: w,
                                   lt.OPT_FLIP_ON_Q: fq, lt.OPT_ITEM_TURNS: item}))
            for ilp, w, fq in ((2, 2, 0), (2, 3, 0), (2, 4, 0), (1, 5, 1), (1, 8, 1)):
                cases.append(("wrap ilp%d W%d %s" % (ilp, w, "q" if fq else "f"),
                              {lt.OPT_FUSED_MODE: 4, lt.OPT_FUSED_ILP: ilp, lt.OPT_WARPS_PER_SMSP: w,
                               lt.OPT_FLIP_ON_Q: fq}))
            for w in (4, 8):
                cases.append(("static ilp2 W%d" % w, {lt.OPT_FUSED_MODE: 2, lt.OPT_FUSED_ILP: 2,
                                                        lt.OPT_WARPS_PER_SMSP: min(w, 4)}))
                cases.append(("static ilp1 W%d" % w, {lt.OPT_FUSED_MODE: 2, lt.OPT_FUSED_ILP: 1,
                                                        lt.OPT_WARPS_PER_SMSP: w}))
            cases.append(("plain kernel block64 ilp2", {lt.OPT_FUSED_MODE: 1, lt.OPT_FUSED_ILP: 2,
                                                        lt.OPT_FUSED_BLOCK: 64}))
            rows = {}
            for label, opts in cases:
                tr = lt.Tracker(wl.RING, "leapfrog")
                for k, v in opts.items():
                    tr.set_option(k, v)
                sec = cx.timed(lambda: tr.track_fused(z, d, n, turns, cx.sp), 3, flush=False)
                rows[label] = {"ms": round(1e3 * sec, 3), "mode": tr.get_stat(lt.STAT_LAST_MODE),
                               "frac": round(FP64_INSTR_PER_PT * n * turns / sec / 1e9 / cx.peak_fp64, 4),
                               "block": tr.get_stat(lt.STAT_LAST_BLOCK), "ilp": tr.get_stat(lt.STAT_LAST_ILP),
                               "item": tr.get_stat(lt.STAT_LAST_ITEM_TURNS)}
                del tr
            out["n=%d turns=%d" % (n, turns)] = rows
            del z, d
    out["clocks"] = clk.summary(short=True)
    return out


# ----------------------------------------------------------------------------- next rows (f2-f4)
def bench_next(cx: Ctx) -> dict:
    """SURVEY.md sec. 8(f) rows f2 (RF programme and energy ramp, fused and per-turn), f4 (per-turn
    + slicing histogram) and f3 (transverse maps, fused and per-turn) at their NEXT_CONFIGS sizes,
    each against the roofline that bounds it."""
    lt, wl, torch = cx.lt, cx.wl, cx.torch
    sp = cx.sp
    W = cx.world
    out = {}
    with cx.clock() as clk:
        # f2: programme, fused mode
        c = wl.NEXT_CONFIGS["f2_programme"]
        n, turns = c["n"], c["turns"]
        z0, d0 = wl.gaussian_bunch(n, c["sigma_z"], c["seed"] + cx.rank)
        a, psi = wl.rf_programme(turns, c["programme_seed"])
        z, d = cx.dev(z0), cx.dev(d0)
        zi, di = z.clone(), d.clone()
        at, pt = cx.dev(a), cx.dev(psi)
        tr = lt.Tracker(wl.RING, "leapfrog")
        sec = cx.timed(lambda: tr.track_programme(z, d, n, turns, at, pt, sp), 5,
                       lambda: (z.copy_(zi), d.copy_(di)))
        out["f2_programme_fused"] = {"n": n, "turns": turns, "value": W * n * turns / sec, "ms": 1e3 * sec,
                                     "roofline": cx.alu(INSTR_F2_PROGRAMME, n * turns, sec, "f2_programme_fused"),
                                     "shape": cx.shape(tr)}
        del z, d, zi, di, tr

        # f2 with acceleration: energy ramp 26 -> 60 GeV/c
        c = wl.NEXT_CONFIGS["f2_ramp"]
        n, turns = c["n"], c["turns"]
        z0, d0 = wl.gaussian_bunch(n, c["sigma_z"], c["seed"] + cx.rank)
        p0c, a, psi = wl.energy_ramp(turns, c["p_start"], c["p_end"])
        z, d = cx.dev(z0), cx.dev(d0)
        zi, di = z.clone(), d.clone()
        pc, at, pt = cx.dev(p0c), cx.dev(a), cx.dev(psi)
        tr = lt.Tracker(wl.RING, "leapfrog")
        sec = cx.timed(lambda: tr.track_ramp(z, d, n, turns, pc, at, pt, sp), 5,
                       lambda: (z.copy_(zi), d.copy_(di)))
        out["f2_ramp_fused"] = {"n": n, "turns": turns, "value": W * n * turns / sec, "ms": 1e3 * sec,
                                "roofline": cx.alu(INSTR_F2_RAMP, n * turns, sec, "f2_ramp_fused"),
                                "shape": cx.shape(tr)}
        del z, d, zi, di, tr
        n, turns = wl.CONFIGS[3]["n"], 256
        z0, d0 = wl.gaussian_bunch(n, 0.08, c["seed"] + 1 + cx.rank)
        z, d = cx.dev(z0), cx.dev(d0)
        mom = torch.zeros(turns * lt.MOMENTS_DTYPE.itemsize, dtype=torch.uint8, device="cuda")
        tr = lt.Tracker(wl.RING, "leapfrog")
        sec = cx.timed(lambda: tr.track_ramp_per_turn(z, d, n, turns, pc, at, pt, mom, None, sp), 2)
        out["f2_ramp_per_turn"] = {"n": n, "turns": turns, "moments": True, "value": W * n * turns / sec,
                                   "us_per_turn": 1e6 * sec / turns,
                                   "roofline": cx.hbm(32, n * turns, sec, "f2_ramp_per_turn")}
        del z, d, mom, tr, pc, at, pt

        # f4: per-turn mode + 64-slice histogram of z every turn (still 32 B per particle-turn)
        c = wl.NEXT_CONFIGS["f4_slices"]
        n, turns = c["n"], c["turns"]
        z0, d0 = wl.gaussian_bunch(n, c["sigma_z"], c["seed"] + cx.rank)
        z_lo, z_hi, S = wl.slice_grid(c)
        z, d = cx.dev(z0), cx.dev(d0)
        hist = torch.zeros(turns * (S + 2), dtype=torch.int64, device="cuda")
        mom = torch.zeros(turns * lt.MOMENTS_DTYPE.itemsize, dtype=torch.uint8, device="cuda")
        tr = lt.Tracker(wl.RING, "leapfrog")
        sec = cx.timed(lambda: tr.track_slices(z, d, n, turns, z_lo, z_hi, S, hist, None, None, sp), 2)
        out["f4_track_slices"] = {"n": n, "turns": turns, "slices": S, "value": W * n * turns / sec,
                                  "us_per_turn": 1e6 * sec / turns,
                                  "roofline": cx.hbm(32, n * turns, sec, "f4_track_slices")}
        sec = cx.timed(lambda: tr.track_slices(z, d, n, turns, z_lo, z_hi, S, hist, mom, None, sp), 2)
        out["f4_track_slices_with_moments"] = {"n": n, "turns": turns, "value": W * n * turns / sec,
                                               "us_per_turn": 1e6 * sec / turns,
                                               "roofline": cx.hbm(32, n * turns, sec)}
        zs = z.clone()
        h1 = torch.zeros(S + 2, dtype=torch.int64, device="cuda")
        sec = cx.timed(lambda: tr.slice_histogram(zs, n, z_lo, z_hi, S, h1, sp), 8)
        # context for a 12 us operation: the same 80 MB summed by the library reduction, same timer
        ref = cx.timed(lambda: zs.sum(), 8)
        # the 256 MB fill leaves the L2 full of DIRTY lines, which a read-only 80 MB pass then has to
        # evict: the same call over five rotating inputs (400 MB > L2, clean lines), back to back
        rot = [zs] + [zs.clone() for _ in range(4)]
        for zz in rot:
            tr.slice_histogram(zz, n, z_lo, z_hi, S, h1, sp)
        torch.cuda.synchronize()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record(cx.stream)
        for r in range(50):
            tr.slice_histogram(rot[r % 5], n, z_lo, z_hi, S, h1, sp)
        e1.record(cx.stream)
        torch.cuda.synchronize()
        clean = cx.max_over_ranks(e0.elapsed_time(e1) * 1e-3) / 50
        del rot
        # the row's roofline is the rotating-inputs time (inputs larger than L2, every line clean);
        # the time behind the 256 MB fill every other leg uses is reported beside it
        out["f4_slice_histogram"] = {"n": n, "slices": S, "value": W * n / clean, "unit": "particles/s",
                                     "us_per_call": 1e6 * clean,
                                     "l2": "5 rotating 80 MB inputs (400 MB > L2), 50 calls back to back",
                                     "us_per_call_after_256MB_fill": 1e6 * sec,
                                     "frac_after_256MB_fill": 8 * n / sec / 1e9 / cx.hbm_peak,
                                     "us_torch_sum_same_array_after_fill": 1e6 * ref,
                                     "us_in_kernel_ncu": cx.traffic.get("f4_slice_histogram_ncu_us"),
                                     "roofline": cx.hbm(8, n, clean, "f4_slice_histogram")}
        del z, d, zs, hist, mom, tr

        # f3: transverse maps, fused (16 per segment + 13 longitudinal FP64 instructions) and per-turn
        c = wl.NEXT_CONFIGS["f3_transverse"]
        mats, twiss = wl.transverse_lattice(c["n_seg"], c["lattice_seed"])
        tr = lt.Tracker(wl.RING, "leapfrog")
        tr.set_transverse(mats)
        n, turns = c["n"], c["turns"]
        co = [cx.dev(v) for v in wl.transverse_bunch(n, c["seed"] + cx.rank, twiss)]
        z0, d0 = wl.gaussian_bunch(n, c["sigma_z"], c["seed"] + 1 + cx.rank)
        z, d = cx.dev(z0), cx.dev(d0)
        sec = cx.timed(lambda: tr.track_transverse_fused(co[0], co[1], co[2], co[3], z, d, n, turns, sp), 3)
        instr = 16 * c["n_seg"] + FP64_INSTR_PER_PT
        out["f3_transverse_fused"] = {"n": n, "turns": turns, "segments": c["n_seg"],
                                      "value": W * n * turns / sec, "ms": 1e3 * sec,
                                      "roofline": cx.alu(instr, n * turns, sec, "f3_transverse_fused")}
        sec = cx.timed(lambda: tr.track_transverse_fused(co[0], co[1], co[2], co[3], None, None, n, turns, sp), 3)
        out["f3_transverse_fused_4d_only"] = {"n": n, "turns": turns, "value": W * n * turns / sec,
                                              "ms": 1e3 * sec,
                                              "roofline": cx.alu(16 * c["n_seg"], n * turns, sec)}
        del co, z, d
        n, turns = c["per_turn_n"], c["per_turn_turns"]
        co = [cx.dev(v) for v in wl.transverse_bunch(n, c["seed"] + 2 + cx.rank, twiss)]
        z0, d0 = wl.gaussian_bunch(n, c["sigma_z"], c["seed"] + 3 + cx.rank)
        z, d = cx.dev(z0), cx.dev(d0)
        sec = cx.timed(lambda: tr.track_transverse_per_turn(co[0], co[1], co[2], co[3], z, d, n, turns, sp), 2)
        out["f3_transverse_per_turn"] = {"n": n, "turns": turns, "value": W * n * turns / sec,
                                         "us_per_turn": 1e6 * sec / turns,
                                         "roofline": cx.hbm(96, n * turns, sec, "f3_transverse_per_turn")}
        del co, z, d
    out["clocks"] = clk.summary(short=True)
    return out


# ----------------------------------------------------------------------------- per-turn mode (configs[3])
def bench_per_turn(cx: Ctx) -> dict:
    """configs[3]: 10^7 particles x 1000 launches with moments + membership count fused into every
    launch; 32 B per particle-turn against the measured copy bandwidth.  Consecutive launches sweep
    a 160 MB working set (> 126 MB L2) in alternating directions."""
    lt, wl, torch = cx.lt, cx.wl, cx.torch
    c3 = wl.CONFIGS[3]
    n3, t3 = c3["n"], c3["turns"]
    z3, d3 = wl.make_bunch(c3, seed=c3["seed"] + cx.rank)
    z3, d3 = cx.dev(z3), cx.dev(d3)
    mom = torch.zeros(t3 * lt.MOMENTS_DTYPE.itemsize, dtype=torch.uint8, device="cuda")
    tr3 = lt.Tracker(wl.RING, "leapfrog")
    tr3.track_per_turn(z3, d3, n3, 128, mom, None, cx.sp)
    torch.cuda.synchronize()
    reps = 3
    e0 = [torch.cuda.Event(enable_timing=True) for _ in range(reps)]
    e1 = [torch.cuda.Event(enable_timing=True) for _ in range(reps)]
    l0 = tr3.get_stat(lt.STAT_KERNEL_LAUNCHES)
    cx.barrier()
    with cx.clock() as clk3:
        for r in range(reps):
            e0[r].record(cx.stream)
            tr3.track_per_turn(z3, d3, n3, t3, mom, None, cx.sp)
            e1[r].record(cx.stream)
        torch.cuda.synchronize()
    t_pt = cx.max_over_ranks(sum(a.elapsed_time(b) for a, b in zip(e0, e1)) * 1e-3)
    gbs = BYTES_PER_PT_PER_TURN_MODE * n3 * t3 * reps / t_pt / 1e9
    # The same kernel where the L2 cannot help: the configs[3] bunch tiled to 2e7 .. 8e7 particles
    # (0.32 .. 1.28 GB of state against 126 MB of L2).  configs[3]'s own 160 MB working set is only
    # 1.3x the L2, and the alternating sweep direction keeps part of it there, which is how its
    # algorithmic rate exceeds the copy peak; these rows are the plain HBM-bound rate.
    import numpy as np
    zh, dh = z3.cpu().numpy(), d3.cpu().numpy()
    del z3, d3
    beyond = []
    with cx.clock() as clkb:
        for mult in (2, 4, 8):
            nb, tb = mult * n3, 128
            zb, db = cx.dev(np.tile(zh, mult)), cx.dev(np.tile(dh, mult))
            trb = lt.Tracker(wl.RING, "leapfrog")
            sec = cx.timed(lambda: trb.track_per_turn(zb, db, nb, tb, mom, None, cx.sp), 2, flush=False)
            gb = BYTES_PER_PT_PER_TURN_MODE * nb * tb / sec / 1e9
            beyond.append({"n": nb, "turns": tb, "us_per_turn": round(1e6 * sec / tb, 2),
                           "value": cx.world * nb * tb / sec, "achieved": round(gb, 1),
                           "frac": round(gb / cx.hbm_peak, 4)})
            del zb, db, trb
    return {"workload": "configs[3] 1e7 particles x 1000 turns, one launch per turn, moments + count",
            "beyond_l2": {"rows": beyond, "clocks": clkb.summary(short=True),
                          "note": "same kernel, configs[3] bunch tiled; inputs larger than L2, no flush"},
            "value": cx.world * n3 * t3 * reps / t_pt, "unit": UNIT,
            "ms_per_turn": 1e3 * t_pt / (t3 * reps),
            "gpu_launches": tr3.get_stat(lt.STAT_KERNEL_LAUNCHES) - l0,
            "bound": "hbm", "achieved": gbs, "peak": cx.hbm_peak, "unit_roofline": "GB/s",
            "frac": gbs / cx.hbm_peak, "traffic": cx.traffic.get("per_turn"),
            "algorithmic_bytes": BYTES_PER_PT_PER_TURN_MODE * n3, "peak_source": cx.hbm_source,
            "frac_of_nominal_8TBs": gbs / 8000.0, "clocks": clk3.summary(short=True)}


def bench_per_turn_sharded(cx: Ctx) -> dict:
    """ONE configs[3]-shaped bunch split into contiguous particle ranges
    (workloads.shard_range), one per rank; every rank runs lt_track_per_turn with raw sums on its
    shard, ONE SUM all-reduce of lt_sums[turns] at the end, lt_moments_from_sums on every rank.
    At world size 1 the two shards run on two streams of the one GPU (no collective)."""
    import numpy as np
    lt, wl, torch = cx.lt, cx.wl, cx.torch
    c3 = wl.CONFIGS[3]
    n, turns = 1_000_001, 256                      # odd first shard: the second starts 8-byte aligned
    z0, d0 = wl.make_bunch(c3, n=n)
    nshard = cx.world if cx.world > 1 else 2
    mine = [cx.rank] if cx.world > 1 else [0, 1]
    zfull, dfull = cx.dev(z0), cx.dev(d0)
    streams = [torch.cuda.Stream() for _ in mine]
    trackers = [lt.Tracker(wl.RING, "leapfrog") for _ in mine]
    sums = [torch.zeros(turns * lt.SUMS_DTYPE.itemsize, dtype=torch.uint8, device="cuda") for _ in mine]
    torch.cuda.synchronize()
    cx.barrier()
    t0 = time.perf_counter()
    for k, s in enumerate(mine):
        lo, hi = wl.shard_range(n, s, nshard)
        trackers[k].track_per_turn(zfull[lo:hi], dfull[lo:hi], hi - lo, turns, None, sums[k],
                                   streams[k].cuda_stream)
    torch.cuda.synchronize()
    total = torch.zeros(turns * 8, dtype=torch.float64, device="cuda")
    for sbuf in sums:
        total += sbuf.view(torch.float64)
    if cx.world > 1:
        cx.dist.all_reduce(total, op=cx.dist.ReduceOp.SUM)     # the path's only data collective
    torch.cuda.synchronize()
    dt = cx.max_over_ranks(time.perf_counter() - t0)
    mom = lt.moments_from_sums(total.cpu().numpy().view(lt.SUMS_DTYPE))
    ok = bool(int(round(float(total.cpu().numpy().view(lt.SUMS_DTYPE)["n"][0]))) == n)
    return {"n": n, "turns": turns, "shards": nshard, "all_reduce_bytes": turns * 64,
            "value": n * turns / dt, "unit": UNIT, "particle_count_reduced_ok": ok,
            "rms_z_last_turn": float(mom["rms_z"][-1]), "timing": "wall clock incl. launch overhead"}


# ----------------------------------------------------------------------------- CUDA arm
def flat_summary(roofline: dict, cx: Ctx) -> dict:
    """Both halves of BASELINE.json's metric ("% of FP64 / HBM roofline") and one fraction per
    config / sec. 8(f) row as FLAT SCALAR keys of `roofline`: the driver's record keeps the
    scalars of that object and drops nested ones.  Values are copied from the legs above, nothing
    is measured here; a leg that did not run (or failed) leaves its keys out."""
    out = {"traffic_source": cx.traffic.get("fused_source")}

    def leg(*path):
        node = roofline
        for k in path:
            if not isinstance(node, dict) or k not in node:
                return None
            node = node[k]
        return node

    def put(key, value, digits=4):
        if isinstance(value, (int, float)):
            out[key] = round(float(value), digits)

    pt = leg("per_turn")
    if isinstance(pt, dict) and "frac" in pt:
        put("per_turn_frac", pt["frac"])                       # algorithmic bytes / time / copy peak
        put("per_turn_gbs", pt["achieved"], 1)
        put("per_turn_us", 1e3 * pt["ms_per_turn"], 2)
        put("per_turn_frac_of_8TBs", pt["frac_of_nominal_8TBs"])
        put("per_turn_value", pt["value"], 0)
        if pt.get("traffic"):                                  # ncu DRAM bytes (committed capture) / this run's time
            put("per_turn_dram_frac", pt["traffic"] / (pt["ms_per_turn"] * 1e-3) / 1e9 / pt["peak"])
        rows = leg("per_turn", "beyond_l2", "rows") or []
        if rows:
            put("per_turn_beyond_l2_frac_min", min(r["frac"] for r in rows))
            put("per_turn_beyond_l2_frac_max", max(r["frac"] for r in rows))
    for key, name in (("cfg0_frac", "configs[0]"), ("cfg2_frac", "configs[2]"),
                      ("cfg4_ec_f64_frac", "configs[4] euler_cromer fp64"),
                      ("cfg4_lf_f64_frac", "configs[4] leapfrog fp64"),
                      ("cfg4_ruth4_f64_frac", "configs[4] ruth4 fp64"),
                      ("cfg4_ec_f32_frac", "configs[4] euler_cromer fp32"),
                      ("cfg4_lf_f32_frac", "configs[4] leapfrog fp32"),
                      ("cfg4_ruth4_f32_frac", "configs[4] ruth4 fp32")):
        cfgs = leg("configs") or {}
        hit = [v for k, v in cfgs.items() if k.startswith(name) and isinstance(v, dict)]
        if hit:
            put(key, (hit[0].get("roofline") or {}).get("frac"))
    for key, name in (("f2_programme_frac", "f2_programme_fused"), ("f2_ramp_frac", "f2_ramp_fused"),
                      ("f2_programme_per_turn_frac", "f2_programme_per_turn"),
                      ("f2_ramp_per_turn_frac", "f2_ramp_per_turn"),
                      ("f3_fused_frac", "f3_transverse_fused"), ("f3_per_turn_frac", "f3_transverse_per_turn"),
                      ("f4_hist_frac", "f4_slice_histogram"), ("f4_track_slices_frac", "f4_track_slices"),
                      ("f4_track_slices_moments_frac", "f4_track_slices_with_moments")):
        put(key, leg("next", name, "roofline", "frac"))
    put("f4_hist_us", leg("next", "f4_slice_histogram", "us_per_call"), 2)
    for r in leg("f1_chunk_sweep", "rows") or []:
        if r.get("turns_per_launch") == 1:
            tag = {"fused": "f1_us_per_launch_1turn_fused", "per_turn graph=0": "f1_us_per_launch_1turn_per_turn_stream",
                   "per_turn graph=1": "f1_us_per_launch_1turn_per_turn_graph"}.get(r.get("kernel"))
            if tag:
                put(tag, r["us_per_launch"], 2)
    return out


def run_cuda(args) -> None:
    import numpy as np
    import torch
    import torch.distributed as dist

    from paper_1610_05801_b200 import longtrack as lt        # fails loudly if the .so is missing
    from paper_1610_05801_b200 import workloads as wl

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device -- the hot path has no CPU fallback")
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    cx = Ctx(lt, wl, torch, dist, world, rank, local)

    if args.only:                                        # profiling aid: one leg, printed alone
        leg = {"per_turn": bench_per_turn, "configs": bench_configs, "f1": bench_f1,
               "next": bench_next, "probe": lambda c: bench_probe(c, table=True), "shapes": bench_shapes,
               "sizes": bench_sizes,
               "sharded": bench_per_turn_sharded}.get(args.only)
        if leg is not None:
            res = leg(cx)
            if rank == 0:
                print(json.dumps({args.only: res}))
            if world > 1:
                dist.destroy_process_group()
            return

    cfg = wl.CONFIGS[1]
    n, turns = cfg["n"], cfg["turns"]
    z0, d0 = wl.make_bunch(cfg, seed=cfg["seed"] + rank)     # weak scaling: one bunch per rank
    z, d = cx.dev(z0), cx.dev(d0)
    count = torch.zeros(1, dtype=torch.int64, device="cuda")
    tr = lt.Tracker(wl.RING, "leapfrog")
    stream, sp = cx.stream, cx.sp

    def step():
        tr.track_fused(z, d, n, turns, sp)
        tr.bucket_count(z, d, n, count, sp)

    warmup = max(args.warmup, 3)
    for _ in range(warmup):
        step()
    torch.cuda.synchronize()

    ev = [[torch.cuda.Event(enable_timing=True) for _ in range(3)] for _ in range(args.steps)]
    cx.barrier()
    torch.cuda.synchronize()
    launches0 = tr.get_stat(lt.STAT_KERNEL_LAUNCHES)
    with cx.clock() as clk:
        wall0 = time.perf_counter()
        for k in range(args.steps):
            cx.flush.fill_(k & 0xFF)                    # L2 flush between timed iterations
            ev[k][0].record(stream)
            tr.track_fused(z, d, n, turns, sp)
            ev[k][1].record(stream)
            tr.bucket_count(z, d, n, count, sp)
            ev[k][2].record(stream)
        torch.cuda.synchronize()
        wall = time.perf_counter() - wall0
    cx.barrier()
    launches = tr.get_stat(lt.STAT_KERNEL_LAUNCHES) - launches0
    t_steps = sum(e[0].elapsed_time(e[2]) for e in ev) * 1e-3
    t_fused = sum(e[0].elapsed_time(e[1]) for e in ev) * 1e-3
    t_max = cx.max_over_ranks(t_steps)
    value = world * n * turns * args.steps / t_max
    fused_launch_s = t_fused / args.steps              # one fused kernel launch per step
    achieved_ginstr = n * turns * FP64_INSTR_PER_PT / fused_launch_s / 1e9
    mode = {1: "fused_kernel (plain)", 2: "fused_persistent_kernel (static slots)",
            3: "fused_persistent_kernel (ticket queue)",
            4: "fused_persistent_kernel (static wrap-around schedule)"}[tr.get_stat(lt.STAT_LAST_MODE)]
    roofline = {"bound": "alu", "kernel": mode + " <double, leap-frog, single harmonic, merged drifts>",
                "achieved": achieved_ginstr, "peak": cx.peak_fp64, "unit": "G FP64 instr/s",
                "frac": achieved_ginstr / cx.peak_fp64,
                "traffic": cx.traffic.get("fused"), "algorithmic_bytes": 32 * n,
                "instr_per_particle_turn": FP64_INSTR_PER_PT,
                "peak_source": "148 SMs x 64 FP64 lanes x sm_max_mhz; lt_probe_pipe measures DADD, DMUL and "
                               "two-register DFMA at exactly this rate (pipe_probe), MEASURED_PEAKS.json has no FP64 entry",
                "ms_per_launch": 1e3 * fused_launch_s}
    roofline.update(cx.shape(tr))
    clocks = clk.summary()
    if args.only == "headline":
        if rank == 0:
            print(json.dumps({"value": value, "roofline": roofline, "clocks": clocks}))
        if world > 1:
            dist.destroy_process_group()
        return

    # ---- e2e: host buffers through the C ABI (H2D + track + count + D2H per step)
    zh, dh = torch.from_numpy(z0.copy()).pin_memory(), torch.from_numpy(d0.copy()).pin_memory()
    tr.track_fused_host(zh, dh, n, 100, want_count=True)
    cx.barrier()
    torch.cuda.synchronize()
    e2e_steps = max(3, min(args.steps, 10))
    with cx.clock() as clk_e2e:
        t0 = time.perf_counter()
        for _ in range(e2e_steps):
            tr.track_fused_host(zh, dh, n, turns, want_count=True)
        t_e2e = cx.max_over_ranks(time.perf_counter() - t0)
    e2e = {"value": world * n * turns * e2e_steps / t_e2e, "unit": UNIT,
           "h2d_bytes_per_step": 2 * 8 * n, "d2h_bytes_per_step": 2 * 8 * n + 8,
           "steps": e2e_steps, "api": "lt_track_fused_host", "clocks": clk_e2e.summary(short=True)}

    def guarded(fn):
        try:
            return fn(cx)
        except Exception as e:                          # a failing side leg must not void the headline
            return {"error": "%s: %s" % (type(e).__name__, e)}

    if not args.skip_per_turn:
        roofline["per_turn"] = guarded(bench_per_turn)
        roofline["per_turn_sharded"] = guarded(bench_per_turn_sharded)
    if not args.skip_configs:
        roofline["configs"] = guarded(bench_configs)
        roofline["f1_chunk_sweep"] = guarded(bench_f1)
        roofline["size_sweep"] = guarded(bench_sizes)
    if not args.skip_next:
        roofline["next"] = guarded(bench_next)
    probe = guarded(bench_probe)
    roofline["pipe_probe"] = probe
    if isinstance(probe.get("dadd"), float):
        roofline["frac_of_measured_turn_loop_ceiling"] = (
            roofline["frac"] / (max(probe["turn_flip_on_f_ilp2_w4"], probe["turn_flip_on_q_ilp1_w8"]) / 0.5))

    roofline.update(flat_summary(roofline, cx))

    # ---- CPU oracle beside it (rank 0, N = 1 only): all cores, and one thread
    cpu_baseline = None
    if world == 1 and not args.skip_cpu:
        rate, dt, cores = oracle_rate(n, CPU_SAMPLE_TURNS, cfg["seed"])
        rate1, dt1, _ = oracle_rate(n, CPU_SAMPLE_TURNS_1T, cfg["seed"], threads=1)
        cpu_baseline = {"value": rate, "unit": UNIT, "cores": cores, "kind": "oracle",
                        "sample": "configs[1] bunch: %d particles x %d turns (of %d), %.1f s wall x %d threads"
                                  % (n, CPU_SAMPLE_TURNS, turns, dt, cores),
                        "one_thread": {"value": rate1, "cores": 1,
                                       "sample": "%d particles x %d turns, %.1f s wall" % (n, CPU_SAMPLE_TURNS_1T, dt1)},
                        "cpu": cpu_model()}

    if rank == 0:
        print(json.dumps({
            "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
            "warmup": warmup, "ms_per_step": 1e3 * t_max / args.steps,
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64",
            "data": "synthetic",
            "config": {"workload": "configs[1] hollow bunch: 1e5 particles x 7e4 turns, leap-frog, "
                                   "single harmonic, fused mode + membership count",
                       "particles_per_gpu": n, "turns": turns, "seed": cfg["seed"],
                       "l2": "flushed between timed iterations (256 MB fill)",
                       "parallelism": "particles sharded, no collective (weak)"},
            "clocks": clocks, "e2e": e2e, "gpu_launches": launches,
            "cpu_baseline": cpu_baseline, "wall_s_timed_region": wall,
            # last, and inside it the nested legs before the scalars: the tail of the line -- what a
            # truncated log keeps -- is the compact summary (frac, per_turn_frac, cfg*_frac, f*_frac)
            "roofline": {**{k: v for k, v in roofline.items() if isinstance(v, (dict, list))},
                         **{k: v for k, v in roofline.items() if not isinstance(v, (dict, list))}},
        }))
    if world > 1:
        dist.destroy_process_group()


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=50)
    ap.add_argument("--warmup", type=int, default=5)
    ap.add_argument("--impl", default="cuda", choices=["cuda", "reference"])
    ap.add_argument("--skip-per-turn", action="store_true")
    ap.add_argument("--skip-configs", action="store_true")
    ap.add_argument("--skip-cpu", action="store_true")
    ap.add_argument("--skip-next", action="store_true")
    ap.add_argument("--only", default=None,
                    choices=["headline", "per_turn", "sharded", "configs", "f1", "sizes", "next", "probe", "shapes"],
                    help="run one leg alone (for ncu captures and sweeps)")
    args = ap.parse_args()
    if args.impl == "reference":
        run_reference(args)                              # builds and maps oracle/ only
        return
    if int(os.environ.get("LOCAL_RANK", "0")) == 0:
        import __graft_entry__ as entry
        entry.build()
    else:                                               # torchrun: local rank 0 builds, the others wait
        from paper_1610_05801_b200 import build as lt_build
        lt_build.wait_until_built()                     # the library appears by an atomic rename
    run_cuda(args)


if __name__ == "__main__":
    main()
