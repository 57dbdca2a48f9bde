"""-m "not gpu": the C-ABI library loads here (no GPU), exports every symbol that
include/longtrack.h declares, and its host-only entry points behave as documented."""
import os
import re

import numpy as np
import pytest

import __graft_entry__ as entry

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lt():
    entry.build()
    from paper_1610_05801_b200 import longtrack
    return longtrack


def declared_functions(header="longtrack.h"):
    src = open(os.path.join(ROOT, "include", header)).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(lt_[a-z0-9_]+)\s*\(", src)))


def test_every_declared_symbol_is_exported_and_bound(lt):
    import ctypes
    names = declared_functions()
    assert len(names) >= 19
    lib = ctypes.CDLL(lt.LIB_PATH)
    for n in names:
        assert hasattr(lib, n), "missing export " + n
    assert sorted(lt.EXPORTS) == names      # the binding covers exactly the header


def test_probe_library_is_separate_and_complete(lt):
    """The FP64-pipe probes are bench tooling: their own header and library; liblongtrack.so
    exports the tracking calls only."""
    import ctypes
    from paper_1610_05801_b200 import probe
    names = declared_functions("longtrack_probe.h")
    assert names == ["lt_probe_fp64", "lt_probe_pipe"] == sorted(probe.EXPORTS)
    plib = ctypes.CDLL(probe.LIB_PATH)
    main = ctypes.CDLL(lt.LIB_PATH)
    for n in names:
        assert hasattr(plib, n), "missing export " + n
        assert not hasattr(main, n), n + " is still exported by liblongtrack.so"
    assert not any(n.startswith("lt_probe") for n in declared_functions())


def test_version_and_strerror(lt):
    assert lt.version() == 100
    assert lt.strerror(0) == "ok"
    for code in range(-6, 0):
        assert lt.strerror(code) not in ("ok", "unknown error code")


def test_derived_constants_against_40_digit_values(lt):
    from paper_1610_05801_b200 import workloads as wl
    gold = {}
    for line in open(os.path.join(ROOT, "tests", "golden", "derived_constants.txt")):
        if not line.startswith("#"):
            k, v = line.split()
            gold[k] = float(v)
    d = lt.Tracker(wl.RING).derived()
    for k in ("R", "beta", "eta", "A", "d", "kappa", "K", "z_max", "H_sep"):
        assert abs(d[k] - gold[k]) <= 4 * np.spacing(abs(gold[k])), k
    assert d["mu"] == pytest.approx(gold["mu"], rel=1e-10)


def test_parameter_validation(lt):
    from paper_1610_05801_b200 import workloads as wl

    def code(**over):
        ring = dict(wl.RING)
        integ = over.pop("integrator", "leapfrog")
        r = over.pop("ratio2", 0.0)
        ring.update(over)
        try:
            lt.Tracker(ring, integ, r)
        except lt.LongtrackError as e:
            return e.code
        return 0

    assert code() == 0
    assert code(gamma=1.0) == lt.E_PARAM
    assert code(circumference_m=0.0) == lt.E_PARAM
    assert code(harmonic=0) == lt.E_PARAM
    assert code(p0c_eV=-1.0) == lt.E_PARAM
    assert code(voltage_V=float("nan")) == lt.E_PARAM
    assert code(integrator=7) == lt.E_PARAM
    assert code(voltage_V=-2.0e6) == lt.E_UNSTABLE          # K < 0
    assert code(voltage_V=2.0e6 * 3000) == lt.E_UNSTABLE    # K >= 4
    assert code(ratio2=-0.5) == 0                           # K_eff == 0 is allowed (G10)
    assert code(ratio2=-0.6) == lt.E_UNSTABLE


def test_options_and_stats(lt):
    from paper_1610_05801_b200 import workloads as wl
    tr = lt.Tracker(wl.RING)
    assert tr.get_option(lt.OPT_CHUNK_TURNS) == 1 << 22
    tr.set_option(lt.OPT_CHUNK_TURNS, 1000)
    assert tr.get_option(lt.OPT_CHUNK_TURNS) == 1000
    for opt, bad in ((lt.OPT_CHUNK_TURNS, 0), (lt.OPT_FUSED_ILP, 3), (lt.OPT_FUSED_BLOCK, 100),
                     (lt.OPT_PER_TURN_CTAS_PER_SM, -1), (lt.OPT_PER_TURN_CTAS_PER_SM, 33), (lt.OPT_FUSED_MODE, 5),
                     (lt.OPT_WARPS_PER_SMSP, 9), (lt.OPT_FLIP_ON_Q, 2), (99, 1)):
        with pytest.raises(lt.LongtrackError) as e:
            tr.set_option(opt, bad)
        assert e.value.code == lt.E_PARAM
    # round-2 options: defaults, round trip, range checks
    assert tr.get_option(lt.OPT_RAMP_SCALED) == 1 and tr.get_option(lt.OPT_LATTICE_SOURCE) == 0
    assert tr.get_option(lt.OPT_PER_TURN_CTAS_PER_SM) == 0          # planner
    tr.set_option(lt.OPT_RAMP_SCALED, 0)
    tr.set_option(lt.OPT_LATTICE_SOURCE, 2)
    tr.set_option(lt.OPT_FUSED_ILP, 8)                              # fused transverse kernel only
    assert (tr.get_option(lt.OPT_RAMP_SCALED), tr.get_option(lt.OPT_LATTICE_SOURCE), tr.get_option(lt.OPT_FUSED_ILP)) == (0, 2, 8)
    for opt, bad in ((lt.OPT_LATTICE_SOURCE, 3), (lt.OPT_LATTICE_SOURCE, -1), (lt.OPT_FUSED_ILP, 16)):
        with pytest.raises(lt.LongtrackError):
            tr.set_option(opt, bad)
    assert tr.get_stat(lt.STAT_KERNEL_LAUNCHES) == 0


def test_no_cpu_fallback_device_calls_fail_loudly_without_a_gpu(lt):
    import torch
    if torch.cuda.is_available():
        pytest.skip("a GPU is present")
    from paper_1610_05801_b200 import workloads as wl
    tr = lt.Tracker(wl.RING)
    z, d = np.full(8, 0.1), np.zeros(8)
    with pytest.raises(lt.LongtrackError) as e:
        tr.track_fused_host(z, d, 8, 10)
    assert e.value.code == lt.E_CUDA and e.value.cuda_error != 0
    assert np.all(z == 0.1) and np.all(d == 0.0)            # nothing was computed on the CPU
    # n == 0 is a no-op and needs no device
    tr.track_fused_host(z, d, 0, 10)
    tr.track_fused(0, 0, 0, 10)


def test_next_rows_validate_arguments_before_touching_a_device(lt):
    """f2-f4 entry points: host-side checks (NULL, slicing grid, lattice) come first, so they
    are testable without a GPU; with valid arguments and no GPU the calls fail with E_CUDA."""
    import torch
    from paper_1610_05801_b200 import workloads as wl
    tr = lt.Tracker(wl.RING)

    def code(fn, *args):
        try:
            fn(*args)
        except lt.LongtrackError as e:
            return e.code
        return 0

    buf = np.zeros(16)
    # f4: slicing grid
    for z_lo, z_hi, S in ((1.0, 1.0, 8), (1.0, -1.0, 8), (-1.0, 1.0, 0), (-1.0, 1.0, (1 << 20) + 1),
                          (float("nan"), 1.0, 8), (-1.0, float("inf"), 8)):
        assert code(tr.slice_histogram, buf, 8, z_lo, z_hi, S, buf) == lt.E_PARAM
        assert code(tr.track_slices, buf, buf, 8, 4, z_lo, z_hi, S, buf) == lt.E_PARAM
    assert code(tr.slice_histogram, buf, 8, -1.0, 1.0, 8, None) == lt.E_NULL
    assert code(tr.track_slices, buf, buf, 8, 4, -1.0, 1.0, 8, None) == lt.E_NULL
    assert code(tr.track_slices, buf, buf, 8, 0, -1.0, 1.0, 8, None) == 0      # zero turns: no-op
    # f2: tables are required
    assert code(tr.track_programme, buf, buf, 8, 4, None, buf) == lt.E_NULL
    assert code(tr.track_programme_per_turn, buf, buf, 8, 4, buf, None) == lt.E_NULL
    assert code(tr.track_programme, buf, buf, 0, 4, None, None) == 0           # n == 0: no-op
    # f2 with the energy ramp: p0c is required, the other two tables are optional, phi_s must be 0
    assert code(tr.track_ramp, buf, buf, 8, 4, None) == lt.E_NULL
    assert code(tr.track_ramp_per_turn, buf, buf, 8, 4, None, buf, buf) == lt.E_NULL
    assert code(tr.track_ramp, buf, buf, 0, 4, None) == 0                      # n == 0: no-op
    assert code(tr.track_ramp, buf, buf, 8, 0, None) == 0                      # zero turns: no-op
    assert code(lt.Tracker(wl.RING, "leapfrog", 0.0, 0.3).track_ramp, buf, buf, 8, 4, buf) == lt.E_PARAM
    if not torch.cuda.is_available():
        assert code(tr.track_ramp, buf, buf, 8, 4, buf) == lt.E_CUDA
        assert code(tr.track_ramp_per_turn, buf, buf, 8, 4, buf) == lt.E_CUDA
    # f3: the lattice
    four = (buf, buf, buf, buf)
    assert code(tr.track_transverse_fused, *four, None, None, 8, 4) == lt.E_PARAM   # none set
    bad = np.zeros((1, 4, 4))
    bad[0, 2, 1] = np.inf
    assert code(tr.set_transverse, bad) == lt.E_PARAM
    assert code(tr.set_transverse, np.zeros((257, 4, 4))) == lt.E_PARAM
    assert code(tr.set_transverse, np.eye(4)[None]) == 0
    assert code(tr.track_transverse_fused, *four, buf, None, 8, 4) == lt.E_NULL     # z without delta
    assert code(tr.track_transverse_per_turn, None, buf, buf, buf, None, None, 8, 4) == lt.E_NULL
    assert code(tr.track_transverse_fused, *four, None, None, 0, 4) == 0
    if not torch.cuda.is_available():
        assert code(tr.track_transverse_fused, *four, None, None, 8, 4) == lt.E_CUDA
        assert code(tr.track_programme, buf, buf, 8, 4, buf, buf) == lt.E_CUDA
        assert code(tr.slice_histogram, buf, 8, -1.0, 1.0, 8, buf) == lt.E_CUDA
        assert np.all(buf == 0.0)
    assert code(tr.set_transverse, None) == 0
    assert code(tr.track_transverse_fused, *four, None, None, 8, 4) == lt.E_PARAM


def test_moments_from_sums_host_helper(lt):
    rng = np.random.default_rng(2)
    z, d = rng.normal(0.01, 0.2, 1000), rng.normal(0, 2e-3, 1000)
    s = np.zeros(1, dtype=lt.SUMS_DTYPE)
    s["n"], s["sum_z"], s["sum_zz"] = z.size, z.sum(), (z * z).sum()
    s["sum_d"], s["sum_dd"], s["sum_zd"], s["n_in_bucket"] = d.sum(), (d * d).sum(), (z * d).sum(), 17
    m = lt.moments_from_sums(s)[0]
    assert m["mean_z"] == pytest.approx(z.mean(), rel=1e-12)
    assert m["rms_z"] == pytest.approx(z.std(), rel=1e-12)
    assert m["rms_d"] == pytest.approx(d.std(), rel=1e-12)
    assert m["cov_zd"] == pytest.approx(np.mean((z - z.mean()) * (d - d.mean())), rel=1e-9)
    assert m["n_in_bucket"] == 17


def test_product_path_never_touches_the_oracle():
    """The package must not import, link or read anything under oracle/."""
    pkg = os.path.join(ROOT, "paper_1610_05801_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                text = open(os.path.join(dirpath, f)).read()
                assert not re.search(r"^\s*(import|from)\s+oracle\b", text, flags=re.M), f
                assert "longtrack_oracle" not in text and "lto_" not in text, f
    oracle_files = sorted(f for f in os.listdir(os.path.join(ROOT, "oracle"))
                          if f.endswith((".c", ".h", ".inc", ".py")))
    assert {"longtrack_oracle.c", "map.inc", "programme.inc", "ramp.inc", "next_oracle.c"} <= set(oracle_files)
    for f in oracle_files:
        text = open(os.path.join(ROOT, "oracle", f)).read()
        assert "paper_1610_05801_b200" not in text.replace(
            "paper_1610_05801_b200/csrc/, include/longtrack.h", "").replace(
            "from ``paper_1610_05801_b200``", "") or f == "__init__.py"
        assert "longtrack.h\"" not in text and "kernels.cuh" not in text


# ---------------------------------------------------------------- host logic: schedule and planner
@pytest.mark.parametrize("turns,item", [(1, 1), (63, 64), (64, 64), (65, 64), (777, 50), (777, 200), (777, 776),
                                         (70_000, 2048), (100_000, 2048), (2400, 1024), (2047, 1024), (4096, 1)])
def test_item_schedule_covers_every_turn_once(lt, turns, item):
    """The tapered work-item schedule: chunks are contiguous, cover
    [0, turns) exactly, full items come first, the tail halves down to <= 64 turns, and the
    plain schedule is ceil(turns / item) equal chunks."""
    sched = lt.item_schedule(turns, item, taper=True)
    pos = 0
    for start, length in sched:
        assert start == pos and length >= 1
        pos += length
    assert pos == turns
    lens = [l for _, l in sched]
    nfull = max(turns // item - 1, 0)
    assert lens[:nfull] == [item] * nfull
    tail = lens[nfull:]
    assert all(a >= b for a, b in zip(tail, tail[1:])) or len(tail) <= 1 or tail[-1] <= 64
    assert tail[-1] <= max(64, 1) or len(tail) == 1
    assert sum(tail) == turns - nfull * item and sum(tail) < 2 * item + (item if turns < item else 0) + 1
    plain = lt.item_schedule(turns, item, taper=False)
    assert len(plain) == -(-turns // item) and sum(l for _, l in plain) == turns
    assert all(l == item for _, l in plain[:-1])


def test_planner_picks_the_measured_launch_shapes(lt):
    """lt_plan_fused is the host logic behind lt_track_fused (no GPU): at the configs[1] size two
    particles per lane on 2 warps per sub-partition with every slot busy; at 10^6 particles 4
    warps; a bunch smaller than one wave gets static slots; options force a shape."""
    from paper_1610_05801_b200 import workloads as wl
    tr = lt.Tracker(wl.RING, "leapfrog")
    p = tr.plan_fused(100_000, 70_000)                     # 2 = static wrap-around schedule
    assert (p["dynamic"], p["particles_per_lane"], p["warps_per_smsp"], p["threads"]) == (2, 2, 2, 256)
    assert p["item_turns"] == 0 and p["flip_on_q"] == 0
    groups, slots = -(-100_000 // 64), 148 * 4 * p["warps_per_smsp"]
    assert groups >= slots                                 # only when every slot stays busy
    p = tr.plan_fused(1_000_000, 100_000)                  # many groups per slot: the ticket queue
    assert (p["dynamic"], p["particles_per_lane"], p["warps_per_smsp"], p["item_turns"]) == (1, 2, 4, 2048)
    tr.set_option(lt.OPT_FUSED_MODE, lt.FUSED_PERSISTENT_DYNAMIC)
    p = tr.plan_fused(100_000, 70_000)                     # the ticket queue when forced
    assert (p["dynamic"], p["particles_per_lane"], p["warps_per_smsp"], p["item_turns"]) == (1, 2, 2, 2048)
    tr.set_option(lt.OPT_FUSED_MODE, lt.FUSED_PERSISTENT_WRAP)
    assert tr.plan_fused(1_000, 1_000)["dynamic"] == 0     # fewer groups than slots: static slots
    tr.set_option(lt.OPT_FUSED_MODE, lt.FUSED_AUTO)
    p = tr.plan_fused(1_000, 1_000)
    assert p["dynamic"] == 0 and p["item_turns"] == 0
    p = tr.plan_fused(1_000_000, 10_000, fp32=True)
    assert p["particles_per_lane"] in (2, 4)               # packed pairs
    tr.set_option(lt.OPT_FUSED_ILP, 1)
    tr.set_option(lt.OPT_WARPS_PER_SMSP, 5)
    tr.set_option(lt.OPT_FLIP_ON_Q, 1)
    tr.set_option(lt.OPT_ITEM_TURNS, 300)
    tr.set_option(lt.OPT_FUSED_MODE, lt.FUSED_PERSISTENT_DYNAMIC)
    p = tr.plan_fused(100_000, 70_000)
    assert (p["particles_per_lane"], p["warps_per_smsp"], p["flip_on_q"], p["item_turns"]) == (1, 5, 1, 300)
    assert p["threads"] == 640
    with pytest.raises(lt.LongtrackError):
        tr.plan_fused(0, 10)


def test_planner_returns_for_every_combination_of_forced_options(lt):
    """Each option value is valid on its own; no combination may hang or crash the planner
    (FUSED_ILP = 2 with more than 4 warps per sub-partition used to recurse without end).  A
    combination that no launch shape honours gives up ILP 2 first and keeps the warp count."""
    from paper_1610_05801_b200 import workloads as wl
    tr = lt.Tracker(wl.RING, "leapfrog")
    warps = [0, 1, 2, 3, 4, 5, 6, 7, 8, 10, 12, 14, 16]
    for n in (1, 63, 1_000, 100_000, 1_000_003):
        for fp32 in (False, True):
            for ilp in (0, 1, 2):
                for w in warps:
                    for mode in (lt.FUSED_AUTO, lt.FUSED_PERSISTENT_STATIC,
                                 lt.FUSED_PERSISTENT_DYNAMIC, lt.FUSED_PERSISTENT_WRAP):
                        for fq in (-1, 0, 1):
                            tr.set_option(lt.OPT_FUSED_ILP, ilp)
                            tr.set_option(lt.OPT_WARPS_PER_SMSP, w)
                            tr.set_option(lt.OPT_FUSED_MODE, mode)
                            tr.set_option(lt.OPT_FLIP_ON_Q, fq)
                            p = tr.plan_fused(n, 1000, fp32=fp32)
                            pv = 2 if fp32 else 1
                            assert p["particles_per_lane"] in (pv, 2 * pv)
                            assert p["threads"] * p["ctas_per_sm"] == 128 * p["warps_per_smsp"]
                            assert 32 <= p["threads"] <= 1024 and p["ctas_per_sm"] in (1, 2)
                            if w:
                                assert p["warps_per_smsp"] == w
                            if w > 4:
                                assert p["particles_per_lane"] == pv     # ILP 2 given up, W kept
                            elif ilp:
                                assert p["particles_per_lane"] == ilp * pv
                            if fq >= 0:
                                assert p["flip_on_q"] == fq
                            if mode == lt.FUSED_PERSISTENT_STATIC:
                                assert p["dynamic"] == 0
                            if mode == lt.FUSED_PERSISTENT_DYNAMIC:
                                assert p["dynamic"] == 1
    tr.set_option(lt.OPT_FUSED_ILP, 2)
    tr.set_option(lt.OPT_WARPS_PER_SMSP, 8)
    tr.set_option(lt.OPT_FUSED_MODE, lt.FUSED_AUTO)
    p = tr.plan_fused(100_000, 70_000)                       # the advisor's reproducer
    assert (p["particles_per_lane"], p["warps_per_smsp"], p["threads"]) == (1, 8, 1024)
