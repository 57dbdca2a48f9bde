#!/usr/bin/env python
"""bench.py -- particle-turns/s of the longitudinal tracking hot path on B200.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl reference]

Workload (config.workload): BASELINE.json:configs[1], the paper's profiled run shape
(10^5 macro-particles x 7*10^4 turns, leap-frog), as a seeded synthetic hollow
bunch.  One STEP = one pass of the whole hot path over that bunch: entry load, 70 000 turns
register-resident (fused mode), exit store, then the bucket-membership count of the final
state.  `value` is device-timed with the bunch already in HBM; `e2e` goes through the C ABI
with HOST buffers (lt_track_fused_host: H2D, track, count, D2H inside the timed region).
The HBM-bound per-turn mode (configs[3]: 10^7 particles x 1000 launches with fused moments)
is timed in the same run and reported under "per_turn" with its own HBM roofline.

N > 1 (torchrun): particles are independent, so every rank tracks its own
seeded bunch of the same size -- weak scaling, no data-path collective; the only collectives
are the barrier and the MAX over ranks of the device time.

`--impl reference` times the CPU oracle (oracle/, as it stands) on the host cores on a
bounded sample of the same workload.
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
# declared algorithmic FP64-pipe instructions per particle-turn:
# 1 merged drift + 3 exact range reduction + 1 square + 7 Horner + 1 kick FMA
FP64_INSTR_PER_PT = 13
BYTES_PER_PT_PER_TURN_MODE = 32           # 16 B read + 16 B write per particle-turn
SMS, FP64_LANES_PER_SM = 148, 64          # B200: 2 dies x 74 SMs, 64 FP64 lanes per SM
# DRAM bytes per launch of the two dominant kernels from the committed ncu captures (profiles/)
CPU_SAMPLE_TURNS = 10_000                 # oracle leg: 1e9 particle-turns, about 20-25 core-seconds
NCU_TRAFFIC_FUSED_BYTES = 1_625_344 + 570_112
NCU_TRAFFIC_PER_TURN_BYTES = 160_020_480 + 100_925_184
# the sec. 8(f) rows, per launch (profiles/r1_next_rows_ncu.md)
NCU_TRAFFIC_NEXT = {"f2_fused": 2_747_904 + 388_608, "f4_per_turn": 160_019_968 + 101_635_840,
                    "f4_histogram": 80_013_824 + 1_831_936, "f3_fused": 48_093_440 + 15_289_600,
                    "f3_per_turn": 480_020_736 + 421_614_080,
                    "f2_ramp_fused": 4_984_576 + 154_880, "f2_ramp_per_turn": 160_047_104 + 101_511_424}


def measured_peaks() -> dict:
    try:
        return json.load(open(os.path.join(ROOT, "MEASURED_PEAKS.json")))
    except Exception:
        return {}


class ClockSampler:
    """Samples SM clock and throttle reasons through NVML while the timed region runs."""
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

    def _run(self):
        nv = self._nv
        while not self._stop.is_set():
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

    def summary(self) -> dict:
        s = sorted(self.samples)
        return {"sm_mhz": s[len(s) // 2] if s else None, "sm_max_mhz": self.max_mhz,
                "reasons": sorted(self.reasons), "samples": len(s)}


def physical_gpu_index(local: int) -> int:
    vis = os.environ.get("CUDA_VISIBLE_DEVICES")
    if vis:
        try:
            return int(vis.split(",")[local])
        except Exception:
            return local
    return local


# ----------------------------------------------------------------------------- oracle legs
def oracle_rate(n: int, turns: int, seed: int, threads: int | None = None):
    """Times the CPU oracle as it stands: n particles of the cfg1 bunch x `turns` turns."""
    import oracle
    from paper_1610_05801_b200 import workloads as wl
    cores = len(os.sched_getaffinity(0))
    oracle.set_num_threads(threads or cores)
    z0, d0 = wl.hollow_bunch(n, seed)
    p = oracle.make_params(wl.RING, "leapfrog")
    oracle.track(p, z0[:1000], d0[:1000], 10)          # load the library, touch the pages
    t0 = time.perf_counter()
    oracle.track(p, z0, d0, turns)
    dt = time.perf_counter() - t0
    return n * turns / dt, dt, threads or cores


def run_reference(args) -> None:
    """--impl reference: the oracle on the host cores, same metric/config, bounded sample."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    from paper_1610_05801_b200 import workloads as wl
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
                         "sample": sample},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }))



# ----------------------------------------------------------------------------- next rows (f2-f4)
def bench_next(lt, wl, torch, stream, peaks, peak_ginstr, max_over_ranks, world, rank):
    """SURVEY.md sec. 8(f) rows f2 (RF programme, fused), f4 (per-turn + slicing histogram) and
    f3 (transverse maps, fused and per-turn) at their NEXT_CONFIGS sizes, each against the
    roofline that bounds it.  Device-timed with CUDA events."""
    import numpy as np
    sp = stream.cuda_stream
    hbm_peak = float(peaks.get("hbm_gbs", 6650.0))
    flush = torch.empty(256 << 20, dtype=torch.uint8, device="cuda")

    def timed(fn, reps, restore=None):
        t = 0.0
        for r in range(reps + 1):                        # first repetition is the warm-up
            if restore:
                restore()
            flush.fill_(r)
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record(stream)
            fn()
            e1.record(stream)
            torch.cuda.synchronize()
            if r:
                t += e0.elapsed_time(e1) * 1e-3
        return max_over_ranks(t) / reps

    def alu(instr, pts, sec, traffic=None):
        g = instr * pts / sec / 1e9
        return {"bound": "alu", "achieved": g, "peak": peak_ginstr, "unit": "G FP64 instr/s",
                "frac": g / peak_ginstr, "instr_per_particle_turn": instr,
                "traffic": NCU_TRAFFIC_NEXT.get(traffic)}

    def hbm(bytes_per_pt, pts, sec, traffic=None):
        g = bytes_per_pt * pts / sec / 1e9
        return {"bound": "hbm", "achieved": g, "peak": hbm_peak, "unit": "GB/s",
                "frac": g / hbm_peak, "bytes_per_particle_turn": bytes_per_pt,
                "traffic": NCU_TRAFFIC_NEXT.get(traffic)}

    out = {}
    # f2: programme, fused mode, 15 FP64 instructions per particle-turn (13 + a_t scale + psi_t add)
    c = wl.NEXT_CONFIGS["f2_programme"]
    n, turns = c["n"], c["turns"]
    z0, d0 = wl.gaussian_bunch(n, c["sigma_z"], c["seed"] + rank)
    a, psi = wl.rf_programme(turns, c["programme_seed"])
    z, d = torch.from_numpy(z0).cuda(), torch.from_numpy(d0).cuda()
    zi, di = z.clone(), d.clone()
    at, pt = torch.from_numpy(a).cuda(), torch.from_numpy(psi).cuda()
    tr = lt.Tracker(wl.RING, "leapfrog")
    sec = timed(lambda: tr.track_programme(z, d, n, turns, at, pt, sp), 5,
                lambda: (z.copy_(zi), d.copy_(di)))
    out["f2_programme_fused"] = {
        "workload": "1e5 particles x 7e4 turns, per-turn (V_t, psi_t) tables, fused mode",
        "value": world * n * turns / sec, "unit": UNIT, "ms": 1e3 * sec,
        "roofline": alu(15, n * turns, sec, "f2_fused")}
    del z, d, zi, di, tr

    # f2 with acceleration: energy ramp 26 -> 60 GeV/c, 17 FP64 instructions per particle-turn
    # (13 + psi_t add + amplitude scale + damping FMA + the drift coefficient from the table)
    c = wl.NEXT_CONFIGS["f2_ramp"]
    n, turns = c["n"], c["turns"]
    z0, d0 = wl.gaussian_bunch(n, c["sigma_z"], c["seed"] + rank)
    p0c, a, psi = wl.energy_ramp(turns, c["p_start"], c["p_end"])
    z, d = torch.from_numpy(z0).cuda(), torch.from_numpy(d0).cuda()
    zi, di = z.clone(), d.clone()
    pc, at, pt = (torch.from_numpy(v).cuda() for v in (p0c, a, psi))
    tr = lt.Tracker(wl.RING, "leapfrog")
    sec = timed(lambda: tr.track_ramp(z, d, n, turns, pc, at, pt, sp), 5,
                lambda: (z.copy_(zi), d.copy_(di)))
    out["f2_ramp_fused"] = {
        "workload": "1e5 particles x 7e4 turns, reference momentum 26 -> 60 GeV/c on the synchronous phase, fused mode",
        "value": world * n * turns / sec, "unit": UNIT, "ms": 1e3 * sec,
        "roofline": alu(17, n * turns, sec, "f2_ramp_fused")}
    del z, d, zi, di, tr
    c3 = wl.CONFIGS[3]
    n, turns = c3["n"], 256
    z0, d0 = wl.gaussian_bunch(n, 0.08, c["seed"] + 1 + rank)
    z, d = torch.from_numpy(z0).cuda(), torch.from_numpy(d0).cuda()
    mom = torch.zeros(turns * lt.MOMENTS_DTYPE.itemsize, dtype=torch.uint8, device="cuda")
    tr = lt.Tracker(wl.RING, "leapfrog")
    sec = timed(lambda: tr.track_ramp_per_turn(z, d, n, turns, pc, at, pt, mom, None, sp), 2)
    out["f2_ramp_per_turn"] = {
        "workload": "1e7 particles x 256 turns of the same ramp, one launch per turn, moments every turn",
        "value": world * n * turns / sec, "unit": UNIT, "ms_per_turn": 1e3 * sec / turns,
        "roofline": hbm(32, n * turns, sec, "f2_ramp_per_turn")}
    del z, d, mom, tr, pc, at, pt

    # f4: per-turn mode + 64-slice histogram of z every turn (still 32 B per particle-turn)
    c = wl.NEXT_CONFIGS["f4_slices"]
    n, turns = c["n"], c["turns"]
    z0, d0 = wl.gaussian_bunch(n, c["sigma_z"], c["seed"] + rank)
    z_lo, z_hi, S = wl.slice_grid(c)
    z, d = torch.from_numpy(z0).cuda(), torch.from_numpy(d0).cuda()
    hist = torch.zeros(turns * (S + 2), dtype=torch.int64, device="cuda")
    mom = torch.zeros(turns * lt.MOMENTS_DTYPE.itemsize, dtype=torch.uint8, device="cuda")
    tr = lt.Tracker(wl.RING, "leapfrog")
    sec = timed(lambda: tr.track_slices(z, d, n, turns, z_lo, z_hi, S, hist, None, None, sp), 2)
    out["f4_track_slices"] = {
        "workload": "1e7 particles x 1000 turns, one launch per turn, 64-slice histogram of z per turn",
        "value": world * n * turns / sec, "unit": UNIT, "ms_per_turn": 1e3 * sec / turns,
        "roofline": hbm(32, n * turns, sec, "f4_per_turn")}
    sec = timed(lambda: tr.track_slices(z, d, n, turns, z_lo, z_hi, S, hist, mom, None, sp), 2)
    out["f4_track_slices_with_moments"] = {
        "workload": "as f4_track_slices plus moments and membership count every turn",
        "value": world * n * turns / sec, "unit": UNIT, "ms_per_turn": 1e3 * sec / turns,
        "roofline": hbm(32, n * turns, sec)}
    zs = z.clone()
    h1 = torch.zeros(S + 2, dtype=torch.int64, device="cuda")
    sec = timed(lambda: tr.slice_histogram(zs, n, z_lo, z_hi, S, h1, sp), 5)
    out["f4_slice_histogram"] = {
        "workload": "histogram of one state, 1e7 particles, 64 slices (8 B read per particle)",
        "value": world * n / sec, "unit": "particles/s", "ms": 1e3 * sec,
        "roofline": hbm(8, n, sec, "f4_histogram")}
    del z, d, zs, hist, mom, tr

    # f3: transverse maps, fused (4 segments x 16 + 13 longitudinal FP64 instructions) and per-turn
    c = wl.NEXT_CONFIGS["f3_transverse"]
    mats, twiss = wl.transverse_lattice(c["n_seg"], c["lattice_seed"])
    tr = lt.Tracker(wl.RING, "leapfrog")
    tr.set_transverse(mats)
    n, turns = c["n"], c["turns"]
    co = [torch.from_numpy(v).cuda() for v in wl.transverse_bunch(n, c["seed"] + rank, twiss)]
    z0, d0 = wl.gaussian_bunch(n, c["sigma_z"], c["seed"] + 1 + rank)
    z, d = torch.from_numpy(z0).cuda(), torch.from_numpy(d0).cuda()
    sec = timed(lambda: tr.track_transverse_fused(co[0], co[1], co[2], co[3], z, d, n, turns, sp), 3)
    instr = 16 * c["n_seg"] + FP64_INSTR_PER_PT
    out["f3_transverse_fused"] = {
        "workload": "1e6 particles x 1e4 turns, 4 segment matrices + the leap-frog turn, fused",
        "value": world * n * turns / sec, "unit": UNIT, "ms": 1e3 * sec,
        "roofline": alu(instr, n * turns, sec, "f3_fused")}
    sec = timed(lambda: tr.track_transverse_fused(co[0], co[1], co[2], co[3], None, None, n, turns, sp), 3)
    out["f3_transverse_fused_4d_only"] = {
        "workload": "as above without the longitudinal plane",
        "value": world * n * turns / sec, "unit": UNIT, "ms": 1e3 * sec,
        "roofline": alu(16 * c["n_seg"], n * turns, sec)}
    del co, z, d
    n, turns = c["per_turn_n"], c["per_turn_turns"]
    co = [torch.from_numpy(v).cuda() for v in wl.transverse_bunch(n, c["seed"] + 2 + rank, twiss)]
    z0, d0 = wl.gaussian_bunch(n, c["sigma_z"], c["seed"] + 3 + rank)
    z, d = torch.from_numpy(z0).cuda(), torch.from_numpy(d0).cuda()
    sec = timed(lambda: tr.track_transverse_per_turn(co[0], co[1], co[2], co[3], z, d, n, turns, sp), 2)
    out["f3_transverse_per_turn"] = {
        "workload": "1e7 particles x 200 turns, one launch per turn, six arrays through HBM (480 MB)",
        "value": world * n * turns / sec, "unit": UNIT, "ms_per_turn": 1e3 * sec / turns,
        "roofline": hbm(96, n * turns, sec, "f3_per_turn")}
    del co, z, d, flush
    return out

# ----------------------------------------------------------------------------- CUDA arm
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

    def barrier():
        if world > 1:
            dist.barrier()

    def max_over_ranks(x: float) -> float:
        if world == 1:
            return x
        t = torch.tensor([x], dtype=torch.float64, device="cuda")
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        return float(t.item())

    peaks = measured_peaks()
    sm_max_mhz = float(peaks.get("sm_max_mhz", 1965.0))
    if args.only_next:                                   # profiling aid: just the sec. 8(f) rows
        nxt = bench_next(lt, wl, torch, torch.cuda.current_stream(), peaks,
                         SMS * FP64_LANES_PER_SM * sm_max_mhz * 1e-3, max_over_ranks, world, rank)
        if rank == 0:
            print(json.dumps({"next": nxt}))
        if world > 1:
            dist.destroy_process_group()
        return
    cfg = wl.CONFIGS[1]
    n, turns = cfg["n"], cfg["turns"]
    z0, d0 = wl.make_bunch(cfg, seed=cfg["seed"] + rank)     # weak scaling: one bunch per rank
    z, d = torch.from_numpy(z0).cuda(), torch.from_numpy(d0).cuda()
    count = torch.zeros(1, dtype=torch.int64, device="cuda")
    flush = torch.empty(256 << 20, dtype=torch.uint8, device="cuda")   # > 126 MB L2
    tr = lt.Tracker(wl.RING, "leapfrog")
    stream = torch.cuda.current_stream()
    sp = stream.cuda_stream

    def step():
        tr.track_fused(z, d, n, turns, sp)
        tr.bucket_count(z, d, n, count, sp)

    for _ in range(max(args.warmup, 3)):
        step()
    torch.cuda.synchronize()

    ev = [[torch.cuda.Event(enable_timing=True) for _ in range(3)] for _ in range(args.steps)]
    barrier()
    torch.cuda.synchronize()
    launches0 = tr.get_stat(lt.STAT_KERNEL_LAUNCHES)
    with ClockSampler(physical_gpu_index(local)) as clk:
        wall0 = time.perf_counter()
        for k in range(args.steps):
            flush.fill_(k & 0xFF)                       # L2 flush between timed iterations
            ev[k][0].record(stream)
            tr.track_fused(z, d, n, turns, sp)
            ev[k][1].record(stream)
            tr.bucket_count(z, d, n, count, sp)
            ev[k][2].record(stream)
        torch.cuda.synchronize()
        wall = time.perf_counter() - wall0
    barrier()
    launches = tr.get_stat(lt.STAT_KERNEL_LAUNCHES) - launches0
    t_steps = sum(e[0].elapsed_time(e[2]) for e in ev) * 1e-3
    t_fused = sum(e[0].elapsed_time(e[1]) for e in ev) * 1e-3
    t_max = max_over_ranks(t_steps)
    value = world * n * turns * args.steps / t_max
    fused_launch_s = t_fused / args.steps              # one fused kernel launch per step
    achieved_ginstr = n * turns * FP64_INSTR_PER_PT / fused_launch_s / 1e9
    peak_ginstr = SMS * FP64_LANES_PER_SM * sm_max_mhz * 1e6 / 1e9
    mode = {1: "fused_kernel (plain)", 2: "fused_persistent_kernel (static slots)",
            3: "fused_persistent_kernel (dynamic chunk scheduling)"}[tr.get_stat(lt.STAT_LAST_MODE)]
    roofline = {"bound": "alu", "kernel": mode + " <double, leap-frog, single harmonic, merged drifts>",
                "achieved": achieved_ginstr, "peak": peak_ginstr, "unit": "G FP64 instr/s",
                "frac": achieved_ginstr / peak_ginstr,
                # dram__bytes_read.sum + dram__bytes_write.sum per launch, ncu --set full
                # (profiles/r1_fused_ncu_details.txt); algorithmic: 32 B x n = 3.2 MB per launch
                "traffic": NCU_TRAFFIC_FUSED_BYTES, "algorithmic_bytes": 32 * n,
                "instr_per_particle_turn": FP64_INSTR_PER_PT,
                "peak_source": "148 SMs x 64 FP64 lanes x sm_max_mhz (DESIGN.md); "
                               "MEASURED_PEAKS.json has no FP64 entry",
                "ms_per_launch": 1e3 * fused_launch_s,
                "grid": tr.get_stat(lt.STAT_LAST_GRID), "block": tr.get_stat(lt.STAT_LAST_BLOCK),
                "item_turns": tr.get_stat(lt.STAT_LAST_ITEM_TURNS)}
    clocks = clk.summary()

    # ---- e2e: host buffers through the C ABI (H2D + track + count + D2H per step)
    zh, dh = torch.from_numpy(z0.copy()).pin_memory(), torch.from_numpy(d0.copy()).pin_memory()
    tr.track_fused_host(zh, dh, n, 100, want_count=True)
    barrier()
    torch.cuda.synchronize()
    e2e_steps = max(3, min(args.steps, 10))
    t0 = time.perf_counter()
    for _ in range(e2e_steps):
        tr.track_fused_host(zh, dh, n, turns, want_count=True)
    t_e2e = max_over_ranks(time.perf_counter() - t0)
    e2e = {"value": world * n * turns * e2e_steps / t_e2e, "unit": UNIT,
           "h2d_bytes_per_step": 2 * 8 * n, "d2h_bytes_per_step": 2 * 8 * n + 8,
           "steps": e2e_steps, "api": "lt_track_fused_host"}

    # ---- per-turn mode (configs[3]): HBM roofline
    per_turn = None
    if not args.skip_per_turn:
        c3 = wl.CONFIGS[3]
        n3, t3 = c3["n"], c3["turns"]
        z3, d3 = wl.make_bunch(c3, seed=c3["seed"] + rank)
        z3, d3 = torch.from_numpy(z3).cuda(), torch.from_numpy(d3).cuda()
        mom = torch.zeros(t3 * lt.MOMENTS_DTYPE.itemsize, dtype=torch.uint8, device="cuda")
        tr3 = lt.Tracker(wl.RING, "leapfrog")
        tr3.track_per_turn(z3, d3, n3, 128, mom, None, sp)
        torch.cuda.synchronize()
        reps = 3
        e0 = [torch.cuda.Event(enable_timing=True) for _ in range(reps)]
        e1 = [torch.cuda.Event(enable_timing=True) for _ in range(reps)]
        l0 = tr3.get_stat(lt.STAT_KERNEL_LAUNCHES)
        barrier()
        with ClockSampler(physical_gpu_index(local)) as clk3:
            for r in range(reps):
                e0[r].record(stream)
                tr3.track_per_turn(z3, d3, n3, t3, mom, None, sp)
                e1[r].record(stream)
            torch.cuda.synchronize()
        t_pt = max_over_ranks(sum(a.elapsed_time(b) for a, b in zip(e0, e1)) * 1e-3)
        hbm_peak = float(peaks.get("hbm_gbs", 6650.0))
        gbs = BYTES_PER_PT_PER_TURN_MODE * n3 * t3 * reps / t_pt / 1e9
        per_turn = {"workload": "configs[3] 1e7 particles x 1000 turns, one launch per turn, "
                                "moments + membership count every turn (working set 160 MB > L2)",
                    "value": world * n3 * t3 * reps / t_pt, "unit": UNIT,
                    "ms_per_turn": 1e3 * t_pt / (t3 * reps),
                    "gpu_launches": tr3.get_stat(lt.STAT_KERNEL_LAUNCHES) - l0,
                    "roofline": {"bound": "hbm", "achieved": gbs, "peak": hbm_peak, "unit": "GB/s",
                                 "frac": gbs / hbm_peak,
                                 # ncu --set full, cold cache (profiles/r1_per_turn_ncu_details.txt)
                                 "traffic": NCU_TRAFFIC_PER_TURN_BYTES,
                                 "algorithmic_bytes": BYTES_PER_PT_PER_TURN_MODE * n3,
                                 "peak_source": "MEASURED_PEAKS.json hbm_gbs" if "hbm_gbs" in peaks
                                 else "fallback 6650 GB/s (B200_PROFILING.md)",
                                 "frac_of_nominal_8TBs": gbs / 8000.0},
                    "clocks": clk3.summary()}
        del z3, d3

    # ---- rows SURVEY.md sec. 8(f) marks "next"
    nxt = None
    if not args.skip_next:
        nxt = bench_next(lt, wl, torch, stream, peaks, peak_ginstr, max_over_ranks, world, rank)

    # ---- FP64 probe (measured DFMA issue rate, context for the derived peak)
    probe = None
    try:
        probe = max(lt.probe_fp64(SMS, 1024, ch, 400000)[0] for ch in (2, 4)) / 1e9
    except Exception:
        pass
    roofline["peak_measured_dfma_probe"] = probe
    if probe:
        roofline["frac_of_probe"] = achieved_ginstr / probe

    # ---- CPU oracle beside it (rank 0, N = 1 only)
    cpu_baseline = None
    if world == 1 and not args.skip_cpu:
        rate, dt, cores = oracle_rate(n, CPU_SAMPLE_TURNS, cfg["seed"])
        cpu_baseline = {"value": rate, "unit": UNIT, "cores": cores, "kind": "oracle",
                        "sample": "configs[1] bunch: %d particles x %d turns (of %d), %.1f s wall x %d threads"
                                  % (n, CPU_SAMPLE_TURNS, turns, dt, cores)}

    if rank == 0:
        print(json.dumps({
            "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
            "warmup": max(args.warmup, 3), "ms_per_step": 1e3 * t_max / args.steps,
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64",
            "data": "synthetic",
            "config": {"workload": "configs[1] hollow bunch: 1e5 particles x 7e4 turns, leap-frog, "
                                   "single harmonic, fused mode + membership count",
                       "particles_per_gpu": n, "turns": turns, "seed": cfg["seed"],
                       "l2": "flushed between timed iterations (256 MB fill)",
                       "parallelism": "particles sharded, no collective (weak)"},
            "clocks": clocks, "e2e": e2e, "gpu_launches": launches,
            "roofline": roofline, "cpu_baseline": cpu_baseline, "per_turn": per_turn, "next": nxt,
            "wall_s_timed_region": wall,
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
    ap.add_argument("--skip-cpu", action="store_true")
    ap.add_argument("--skip-next", action="store_true")
    ap.add_argument("--only-next", action="store_true")
    args = ap.parse_args()
    import __graft_entry__ as entry
    if int(os.environ.get("LOCAL_RANK", "0")) == 0:
        entry.build()
    if args.impl == "reference":
        run_reference(args)
    else:
        run_cuda(args)


if __name__ == "__main__":
    main()
