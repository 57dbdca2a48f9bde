"""Launch-shape and size sweeps of liblongtrack on the local GPU (prints markdown tables).

    python -m paper_1610_05801_b200.tune shapes      # fused mode: planner vs forced launch shapes
    python -m paper_1610_05801_b200.tune sizes       # fused mode: n = 2^10 .. 2^24 (Table 2)
    python -m paper_1610_05801_b200.tune chunks      # turns per launch 1 .. 2^16 at fixed total (Fig. 5)
    python -m paper_1610_05801_b200.tune per_turn    # per-turn mode: CTAs per SM, sweep direction, graph
    python -m paper_1610_05801_b200.tune variants    # integrators x harmonics x precision (BASELINE.json:configs[4])

Everything goes through the C ABI (lt_set_option / lt_track_*); timing is CUDA events on the
launching stream, best of `--reps` after one warm-up call.  The tables under profiles/ were made
with these commands; the rate table in csrc/longtrack.cu (loop_rate) comes from `shapes`.
"""
from __future__ import annotations

import argparse
import sys

import numpy as np
import torch

from . import longtrack as lt
from . import workloads as wl

FP64_PEAK = 148 * 64 * 1.965e9           # lane-instructions/s, DESIGN.md sec. 5.2
INSTR = {("leapfrog", 0.0): 13, ("euler_cromer", 0.0): 13, ("ruth4", 0.0): 39,
         ("leapfrog", 0.5): 23, ("euler_cromer", 0.5): 23, ("ruth4", 0.5): 69}


def _stream():
    return torch.cuda.current_stream().cuda_stream


def _time(fn, reps):
    best = float("inf")
    for _ in range(reps):
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        fn()
        e1.record()
        torch.cuda.synchronize()
        best = min(best, e0.elapsed_time(e1))
    return best * 1e-3


def _fused_rate(z0, d0, turns, opts, reps, integrator="leapfrog", ratio2=0.0, f32=False):
    tr = lt.Tracker(wl.RING, integrator, ratio2)
    for k, v in opts.items():
        tr.set_option(k, v)
    dt = np.float32 if f32 else np.float64
    z, d = torch.from_numpy(z0.astype(dt)).cuda(), torch.from_numpy(d0.astype(dt)).cuda()
    n = z.numel()
    run = tr.track_fused_f32 if f32 else tr.track_fused
    run(z, d, n, min(turns, 200), _stream())
    torch.cuda.synchronize()
    s = _time(lambda: run(z, d, n, turns, _stream()), reps)
    return n * turns / s, s, tr


def shapes(args):
    print("| n | launch shape | mode | grid | block | item turns | ms | particle-turns/s | % of FP64 peak (13 instr) |")
    print("|---|---|---|---|---|---|---|---|---|")
    for n, turns, cfg in ((100_000, 70_000, wl.CONFIGS[1]), (1_000_000, 8_000, wl.CONFIGS[2])):
        z0, d0 = wl.make_bunch(cfg, n=n)
        cases = [("planner", {})]
        for w in (4, 5, 6, 8):
            for fq in (0, 1):
                cases.append(("dynamic W=%d flip_on_q=%d item=1024" % (w, fq),
                              {lt.OPT_FUSED_MODE: 3, lt.OPT_WARPS_PER_SMSP: w, lt.OPT_FLIP_ON_Q: fq,
                               lt.OPT_ITEM_TURNS: 1024}))
        for item in (64, 256, 4096):
            cases.append(("dynamic W=8 flip_on_q=1 item=%d" % item,
                          {lt.OPT_FUSED_MODE: 3, lt.OPT_WARPS_PER_SMSP: 8, lt.OPT_FLIP_ON_Q: 1,
                           lt.OPT_ITEM_TURNS: item}))
        for w in (6, 8):
            cases.append(("static W=%d flip_on_q=1" % w,
                          {lt.OPT_FUSED_MODE: 2, lt.OPT_WARPS_PER_SMSP: w, lt.OPT_FLIP_ON_Q: 1}))
        for ilp in (1, 2):
            cases.append(("plain block=64 ilp=%d" % ilp,
                          {lt.OPT_FUSED_MODE: 1, lt.OPT_FUSED_ILP: ilp, lt.OPT_FUSED_BLOCK: 64}))
        for label, opts in cases:
            rate, s, tr = _fused_rate(z0, d0, turns, opts, args.reps)
            print("| %d | %s | %d | %d | %d | %d | %.3f | %.3e | %.1f |" % (
                n, label, tr.get_stat(lt.STAT_LAST_MODE), tr.get_stat(lt.STAT_LAST_GRID),
                tr.get_stat(lt.STAT_LAST_BLOCK), tr.get_stat(lt.STAT_LAST_ITEM_TURNS), 1e3 * s, rate,
                100 * rate * 13 / FP64_PEAK), flush=True)


def sizes(args):
    """The analogue of the paper's Table 2: fixed turns, growing ensemble."""
    turns = 10_000
    print("| n | mode | grid x block | ms for %d turns | particle-turns/s | %% of FP64 peak |" % turns)
    print("|---|---|---|---|---|---|")
    for e in range(10, 25):
        n = 1 << e
        z0, d0 = wl.make_bunch(wl.CONFIGS[0], n=n, seed=1000 + e)
        rate, s, tr = _fused_rate(z0, d0, turns, {}, args.reps)
        print("| 2^%d | %d | %d x %d | %.3f | %.3e | %.1f |" % (
            e, tr.get_stat(lt.STAT_LAST_MODE), tr.get_stat(lt.STAT_LAST_GRID),
            tr.get_stat(lt.STAT_LAST_BLOCK), 1e3 * s, rate, 100 * rate * 13 / FP64_PEAK), flush=True)


def chunks(args):
    """The paper's Fig. 5 on B200: total turns fixed, turns per kernel launch varied, from the
    per-turn regime (1 turn per launch, state through HBM) to one launch for everything."""
    n, total = 1_000_000, 1 << 14
    z0, d0 = wl.make_bunch(wl.CONFIGS[2], n=n)
    print("| turns per launch | launches | ms total | particle-turns/s | note |")
    print("|---|---|---|---|---|")
    for e in range(0, 15, 2):
        chunk = 1 << e
        rate, s, tr = _fused_rate(z0, d0, total, {lt.OPT_CHUNK_TURNS: chunk}, args.reps)
        print("| %d | %d | %.2f | %.3e | fused kernel, LT_OPT_CHUNK_TURNS |" % (
            chunk, total // chunk, 1e3 * s, rate), flush=True)
    tr = lt.Tracker(wl.RING)
    z, d = torch.from_numpy(z0).cuda(), torch.from_numpy(d0).cuda()
    for graph in (0, 1):
        tr.set_option(lt.OPT_PER_TURN_GRAPH, graph)
        tr.track_per_turn(z, d, n, 256, None, None, _stream())
        torch.cuda.synchronize()
        s = _time(lambda: tr.track_per_turn(z, d, n, 2048, None, None, _stream()), args.reps)
        print("| 1 | 2048 (scaled) | %.2f | %.3e | per-turn kernel, no moments, graph=%d |" % (
            1e3 * s * total / 2048, n * 2048 / s, graph), flush=True)


def per_turn(args):
    c3 = wl.CONFIGS[3]
    n, turns = c3["n"], 512
    z0, d0 = wl.make_bunch(c3)
    z, d = torch.from_numpy(z0).cuda(), torch.from_numpy(d0).cuda()
    mom = torch.zeros(turns * lt.MOMENTS_DTYPE.itemsize, dtype=torch.uint8, device="cuda")
    print("| CTAs per SM | reverse | graph | moments | us per turn | algorithmic GB/s |")
    print("|---|---|---|---|---|---|")
    for moments in (1, 0):
        for ctas in (2, 3, 4, 5, 6, 8):
            for reverse in (1, 0):
                for graph in ((1, 0) if ctas == 4 else (1,)):
                    tr = lt.Tracker(wl.RING)
                    tr.set_option(lt.OPT_PER_TURN_CTAS_PER_SM, ctas)
                    tr.set_option(lt.OPT_PER_TURN_REVERSE, reverse)
                    tr.set_option(lt.OPT_PER_TURN_GRAPH, graph)
                    m = mom if moments else None
                    tr.track_per_turn(z, d, n, 128, m, None, _stream())
                    torch.cuda.synchronize()
                    s = _time(lambda: tr.track_per_turn(z, d, n, turns, m, None, _stream()), args.reps)
                    print("| %d | %d | %d | %d | %.2f | %.0f |" % (
                        ctas, reverse, graph, moments, 1e6 * s / turns, 32.0 * n * turns / s / 1e9),
                        flush=True)


def variants(args):
    cfg = wl.CONFIGS[4]
    n, turns = cfg["n"], 2_000
    print("| integrator | r | precision | ms | particle-turns/s | FP64 instr/turn | % of FP64 peak |")
    print("|---|---|---|---|---|---|---|")
    for integ in ("euler_cromer", "leapfrog", "ruth4"):
        for r in (0.0, 0.5):
            z0, d0 = wl.gaussian_bunch(n, cfg["sigma_z"], cfg["seed"], ratio2=r)
            for f32 in (False, True):
                rate, s, _ = _fused_rate(z0, d0, turns, {}, args.reps, integ, r, f32)
                k = INSTR[(integ, r)]
                frac = "-" if f32 else "%.1f" % (100 * rate * k / FP64_PEAK)
                print("| %s | %.1f | %s | %.3f | %.3e | %s | %s |" % (
                    integ, r, "fp32" if f32 else "fp64", 1e3 * s, rate, "-" if f32 else k, frac),
                    flush=True)


def main(argv=None):
    ap = argparse.ArgumentParser(description=__doc__, formatter_class=argparse.RawDescriptionHelpFormatter)
    ap.add_argument("what", choices=["shapes", "sizes", "chunks", "per_turn", "variants"])
    ap.add_argument("--reps", type=int, default=3)
    args = ap.parse_args(argv)
    if not torch.cuda.is_available():
        sys.exit("tune: no CUDA device (the hot path has no CPU fallback)")
    print("<!-- %s on %s -->" % (args.what, torch.cuda.get_device_name(0)))
    {"shapes": shapes, "sizes": sizes, "chunks": chunks, "per_turn": per_turn,
     "variants": variants}[args.what](args)


if __name__ == "__main__":
    main()
