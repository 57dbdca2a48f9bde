"""-m gpu: the optional fp32 mode (BASELINE.json:configs[4] "Run in fp64 and in an optional fp32
mode; fp32 is checked against the fp64 oracle on moments at relative error <= 1e-4"; integrators
of PAPER.md:43, sec. 1.1.2) in EVERY launch shape the library can take -- in particular the one
bench.py times at 10^6 particles (ticket queue, 4 warps per sub-partition, two packed pairs = 4
particles per lane) -- and the fp32 observables lt_bucket_count_f32 / lt_track_per_turn_f32.

Gates.  Shapes among themselves: same bits (include/longtrack.h, LT_OPT_FUSED_MODE).  Against the
fp64 oracle: 1e-4 on moments (north_star).  Per particle there is no gate in BASELINE.json for
fp32; the one used here, 1e-4 of z_max / sigma_delta after 100 turns outside the G17 layer, is
~100 fp32 roundings of a value of order one (6e-8 each) with a factor 10 for the shear of the
bucket, and exists to catch a wrong lane / wrong particle, not to certify fp32 accuracy.
Membership is decided by each side in its own precision (fp32 on the GPU, G15), so the
counts may differ by the particles that lie within fp32 rounding of the separatrix; that band is
counted by the oracle and bounds the difference.
"""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")
if not torch.cuda.is_available():                      # collected but skipped on the CPU box
    pytest.skip("needs a CUDA device", allow_module_level=True)

import oracle                                           # noqa: E402
from paper_1610_05801_b200 import longtrack as lt       # noqa: E402
from paper_1610_05801_b200 import workloads as wl       # noqa: E402
from gpu_util import gpu_track, stream_ptr              # noqa: E402

INTEGRATORS = ("euler_cromer", "leapfrog", "ruth4")
F32_BAND = 2e-5       # |1 - H/H_sep| or |1 - |z|/z_max| below this: fp32 rounding decides membership


def both(integrator="leapfrog", ratio2=0.0):
    return (lt.Tracker(wl.RING, integrator, ratio2, None),
            oracle.make_params(wl.RING, integrator, ratio2, None))


def same_bits(a, b):
    return np.array_equal(a[0], b[0]) and np.array_equal(a[1], b[1])


def near_separatrix(p, z, d, band=F32_BAND):
    g = oracle.derive(p)
    Hn = oracle.hamiltonian(p, z, d) / g["H_sep"]
    return (np.abs(Hn - 1) < band) | (np.abs(np.abs(z) / g["z_max"] - 1) < band)


# ------------------------------------------------------------------ every schedule, same bits
@pytest.mark.parametrize("integrator", INTEGRATORS)
@pytest.mark.parametrize("ratio2", [0.0, 0.5])
def test_fp32_every_schedule_and_lane_count_gives_the_same_bits(integrator, ratio2):
    """fp32 twin of test_dynamic_scheduling_is_bit_identical_to_the_plain_kernel: plain kernel,
    static slots, ticket queue (tapered items), wrap-around schedule; one and two packed pairs
    per lane; merged and split drifts; several launches per call.  150 001 particles: odd, so
    the last packed pair is half empty."""
    tr, _ = both(integrator, ratio2)
    z0, d0 = wl.make_bunch(wl.CONFIGS[4], n=150_001)
    for split in (0, 1):
        tr.set_option(lt.OPT_SPLIT_DRIFTS, split)
        tr.set_option(lt.OPT_FUSED_MODE, lt.FUSED_PLAIN)
        ref = gpu_track(tr, z0, d0, 777, f32=True)
        assert ref[0].dtype == np.float32 and np.isfinite(ref[0]).all()
        tr.set_option(lt.OPT_FUSED_MODE, lt.FUSED_PERSISTENT_STATIC)
        for ilp, w in ((1, 0), (2, 0), (1, 7), (2, 4), (0, 0)):
            tr.set_option(lt.OPT_FUSED_ILP, ilp)
            tr.set_option(lt.OPT_WARPS_PER_SMSP, w)
            assert same_bits(gpu_track(tr, z0, d0, 777, f32=True), ref), (split, "static", ilp, w)
            if ilp:
                assert tr.get_stat(lt.STAT_LAST_ILP) == 2 * ilp      # particles per lane: packed pairs
        tr.set_option(lt.OPT_WARPS_PER_SMSP, 0)
        tr.set_option(lt.OPT_FUSED_MODE, lt.FUSED_PERSISTENT_DYNAMIC)
        for ilp in (1, 2, 0):
            tr.set_option(lt.OPT_FUSED_ILP, ilp)
            for item in (0, 50, 200, 776):              # 200: full items + a tapered tail of 377
                tr.set_option(lt.OPT_ITEM_TURNS, item)
                assert same_bits(gpu_track(tr, z0, d0, 777, f32=True), ref), (split, "queue", ilp, item)
                assert tr.get_stat(lt.STAT_LAST_MODE) == lt.FUSED_PERSISTENT_DYNAMIC
        tr.set_option(lt.OPT_ITEM_TURNS, 0)
        tr.set_option(lt.OPT_FUSED_MODE, lt.FUSED_PERSISTENT_WRAP)
        for ilp, w in ((1, 1), (1, 3), (2, 1), (0, 0)):   # groups of 64 / 128 particles >= slots
            tr.set_option(lt.OPT_FUSED_ILP, ilp)
            tr.set_option(lt.OPT_WARPS_PER_SMSP, w)
            assert same_bits(gpu_track(tr, z0, d0, 777, f32=True), ref), (split, "wrap", ilp, w)
            if w:
                assert tr.get_stat(lt.STAT_LAST_MODE) == lt.FUSED_PERSISTENT_WRAP
        tr.set_option(lt.OPT_WARPS_PER_SMSP, 0)
        tr.set_option(lt.OPT_FUSED_ILP, 0)
        tr.set_option(lt.OPT_FUSED_MODE, lt.FUSED_PERSISTENT_DYNAMIC)
        tr.set_option(lt.OPT_CHUNK_TURNS, 300)          # several launches, each with its own items
        assert same_bits(gpu_track(tr, z0, d0, 777, f32=True), ref), (split, "chunks")
        tr.set_option(lt.OPT_CHUNK_TURNS, 1 << 22)
        # per-turn mode runs the unmerged map: same bits as the fused mode with split drifts
        if split:
            assert same_bits(gpu_track(tr, z0, d0, 777, "per_turn", f32=True), ref)


# ------------------------------------------------------------------ ragged sizes, alignment
@pytest.mark.parametrize("n", [1, 2, 3, 31, 33, 63, 65, 127, 129, 255, 1000, 4097, 100_003])
def test_fp32_ragged_sizes_and_4_byte_aligned_arrays(n):
    """Sizes below one packed group (64 particles), odd sizes (half-empty pair), and arrays that
    are only 4-byte aligned (the packed 8-byte loads cannot be used): every shape the same bits,
    and those bits within the fp32 per-particle gate of the fp64 oracle."""
    tr, p = both()
    cfg = wl.CONFIGS[0]
    z0, d0 = wl.make_bunch(cfg, n=n, seed=177 + n)
    turns = 100
    zo, do = oracle.track(p, z0, d0, turns)
    g = oracle.derive(p)
    ref = gpu_track(tr, z0, d0, turns, f32=True)             # planner's choice
    layer = np.abs(1.0 - oracle.hamiltonian(p, z0, d0) / g["H_sep"]) <= 1e-4
    ez = np.abs(ref[0].astype(np.float64) - zo) / g["z_max"]
    ed = np.abs(ref[1].astype(np.float64) - do) / wl.sigma_delta_for_gate(cfg)
    assert ez[~layer].max(initial=0.0) <= 1e-4 and ed[~layer].max(initial=0.0) <= 1e-4, (ez.max(), ed.max())
    assert ez.max() <= 1e-2 and ed.max() <= 1e-2
    shapes = [(lt.FUSED_PLAIN, 0, 0, 0), (lt.FUSED_PLAIN, 2, 0, 0), (lt.FUSED_PLAIN, 4, 0, 0),
              (lt.FUSED_PERSISTENT_STATIC, 1, 0, 0), (lt.FUSED_PERSISTENT_STATIC, 2, 0, 0),
              (lt.FUSED_PERSISTENT_STATIC, 1, 16, 0), (lt.FUSED_PERSISTENT_STATIC, 2, 4, 0),
              (lt.FUSED_PERSISTENT_DYNAMIC, 1, 0, 0), (lt.FUSED_PERSISTENT_DYNAMIC, 2, 0, 0),
              (lt.FUSED_PERSISTENT_DYNAMIC, 1, 5, 7), (lt.FUSED_PERSISTENT_DYNAMIC, 2, 3, 33),
              (lt.FUSED_PERSISTENT_DYNAMIC, 2, 4, 1), (lt.FUSED_PERSISTENT_WRAP, 1, 1, 0),
              (lt.FUSED_PERSISTENT_WRAP, 2, 2, 0), (lt.FUSED_PERSISTENT_WRAP, 0, 0, 0)]
    for mode, ilp, w, item in shapes:
        tr.set_option(lt.OPT_FUSED_MODE, mode)
        tr.set_option(lt.OPT_FUSED_ILP, ilp)
        tr.set_option(lt.OPT_WARPS_PER_SMSP, w)
        tr.set_option(lt.OPT_ITEM_TURNS, item)
        assert same_bits(gpu_track(tr, z0, d0, turns, f32=True), ref), (mode, ilp, w, item)
        # the same arrays one float further on: 4-byte aligned only
        zbuf = torch.full((n + 3,), -7.0, dtype=torch.float32, device="cuda")
        dbuf = torch.full((n + 3,), -7.0, dtype=torch.float32, device="cuda")
        zv, dv = zbuf[1:n + 1], dbuf[1:n + 1]
        assert zv.data_ptr() % 8 == 4
        zv.copy_(torch.from_numpy(z0.astype(np.float32)))
        dv.copy_(torch.from_numpy(d0.astype(np.float32)))
        tr.track_fused_f32(zv, dv, n, turns, stream_ptr())
        torch.cuda.synchronize()
        assert same_bits((zv.cpu().numpy(), dv.cpu().numpy()), ref), ("misaligned", mode, ilp, w, item)
        for buf in (zbuf, dbuf):                                # nothing written outside [1, n]
            assert buf[0].item() == -7.0 and (buf[n + 1:] == -7.0).all().item()


# ------------------------------------------------------------------ the benchmarked shape
@pytest.mark.parametrize("integrator,ratio2", [("euler_cromer", 0.5), ("leapfrog", 0.5),
                                               ("ruth4", 0.5), ("leapfrog", 0.0)])
def test_fp32_cfg4_full_size_in_the_benchmarked_launch_shape(integrator, ratio2):
    """configs[4] in fp32 at FULL size, planner defaults = what bench.py times
    (roofline.configs["configs[4] ... fp32"]): all 10^6 particles x 10^4 turns on the GPU, the
    fp64 oracle on the seeded 10^5 subsample, 1e-4 on the moments (north_star), taken over the
    particles both sides keep in the bucket (G14: the few escapers carry the all-particle rms z)."""
    cfg = wl.CONFIGS[4]
    tr, p = both(integrator, ratio2)
    z0, d0 = wl.make_bunch(cfg)
    idx = wl.subsample_indices(cfg["n"], cfg["subsample"], cfg["seed"])
    zo, do = oracle.track(p, z0[idx], d0[idx], cfg["turns"])
    zg, dg = gpu_track(tr, z0, d0, cfg["turns"], f32=True)
    # the shape lt_plan_fused(fp32) returns for 10^6 particles and the one that actually ran
    plan = tr.plan_fused(cfg["n"], cfg["turns"], sm_count=tr.get_stat(lt.STAT_SM_COUNT), fp32=True)
    assert (plan["dynamic"], plan["warps_per_smsp"], plan["particles_per_lane"]) == (1, 4, 4)
    assert tr.get_stat(lt.STAT_LAST_MODE) == lt.FUSED_PERSISTENT_DYNAMIC
    assert tr.get_stat(lt.STAT_LAST_ILP) == 4 and tr.get_stat(lt.STAT_LAST_BLOCK) == plan["threads"]
    zs, ds = zg[idx].astype(np.float64), dg[idx].astype(np.float64)
    m = oracle.bucket_mask(p, zs, ds) & oracle.bucket_mask(p, zo, do)
    assert m.mean() > 0.99
    a, b = oracle.moments_of(p, zs[m], ds[m]), oracle.moments_of(p, zo[m], do[m])
    err = dict(rms_z=abs(a["rms_z"] / b["rms_z"] - 1), rms_d=abs(a["rms_d"] / b["rms_d"] - 1),
               mean_z=abs(a["mean_z"] - b["mean_z"]) / b["rms_z"],
               mean_d=abs(a["mean_d"] - b["mean_d"]) / b["rms_d"])
    print("cfg4 fp32 %s r=%.1f: moment errors %s, in bucket on both sides %.5f"
          % (integrator, ratio2, {k: "%.1e" % v for k, v in err.items()}, m.mean()))
    assert max(err.values()) <= 1e-4, err
    # every one of the 10^6 results is a finite number inside the machine (no lane left unwritten)
    assert np.isfinite(zg).all() and np.isfinite(dg).all()
    # membership of the GPU's own final state, counted by the GPU in fp32 and by the oracle in fp64
    cnt = torch.zeros(1, dtype=torch.int64, device="cuda")
    zt, dt = torch.from_numpy(zg).cuda(), torch.from_numpy(dg).cuda()
    tr.bucket_count_f32(zt, dt, zt.numel(), cnt, stream_ptr())
    torch.cuda.synchronize()
    z64, d64 = zg.astype(np.float64), dg.astype(np.float64)
    band = int(near_separatrix(p, z64, d64).sum())
    assert abs(int(cnt.item()) - oracle.bucket_count(p, z64, d64)) <= band, band
    assert band < 200                                          # the band is a sliver, not a loophole


# ------------------------------------------------------------------ fp32 observables
@pytest.mark.parametrize("ratio2", [0.0, 0.5])
def test_fp32_bucket_count_against_the_oracle_on_the_same_state(ratio2):
    """lt_bucket_count_f32 on a hollow bunch (configs[1]: particles on both sides of the
    separatrix): the oracle evaluates the same fp32 state in fp64; the two counts differ at most
    by the particles within fp32 rounding of the boundary -- which the oracle counts."""
    tr, p = both("leapfrog", ratio2)
    for n in (1, 63, 100_003):
        z0, d0 = wl.make_bunch(wl.CONFIGS[1], n=n, seed=5 + n)
        z32, d32 = z0.astype(np.float32), d0.astype(np.float32)
        zt, dt = torch.from_numpy(z32).cuda(), torch.from_numpy(d32).cuda()
        cnt = torch.full((1,), -1, dtype=torch.int64, device="cuda")
        tr.bucket_count_f32(zt, dt, n, cnt, stream_ptr())
        torch.cuda.synchronize()
        z64, d64 = z32.astype(np.float64), d32.astype(np.float64)
        want = oracle.bucket_count(p, z64, d64)
        band = int(near_separatrix(p, z64, d64).sum())
        assert abs(int(cnt.item()) - want) <= band, (n, int(cnt.item()), want, band)
        if n > 1000:
            assert 0.2 * n < want < 0.9 * n and band < 50


@pytest.mark.parametrize("integrator", INTEGRATORS)
def test_fp32_per_turn_moments_every_turn(integrator):
    """The lt_moments written by lt_track_per_turn_f32 (sums accumulated in fp64 from the fp32
    state): (i) the last record against oracle moments of the GPU's own final state at 1e-6 --
    that is the reduction alone; (ii) every turn against the fp64 oracle's run at 1e-4 -- that is
    fp32 tracking.  The bunch is shrunk to 0.8 of configs[4]'s so that no particle starts in the
    layer where a rounding decides whether it leaves the bucket (G14, G17): one escaper at
    |z| ~ 10 m would alone move the all-particle rms z by 1e-2."""
    cfg = wl.CONFIGS[4]
    tr, p = both(integrator, cfg["ratio2"])
    z0, d0 = wl.make_bunch(cfg, n=200_001)
    z0, d0 = 0.8 * z0, 0.8 * d0
    turns = 1000
    zo, do, mo = oracle.track_moments(p, z0, d0, turns)
    zg, dg, mg = gpu_track(tr, z0, d0, turns, "per_turn", want_moments=True, f32=True)
    z64, d64 = zg.astype(np.float64), dg.astype(np.float64)
    own = oracle.moments_of(p, z64, d64)
    assert abs(mg["rms_z"][-1] / own["rms_z"] - 1) <= 1e-6 and abs(mg["rms_d"][-1] / own["rms_d"] - 1) <= 1e-6
    assert abs(mg["mean_z"][-1] - own["mean_z"]) <= 1e-6 * own["rms_z"]
    assert abs(mg["mean_d"][-1] - own["mean_d"]) <= 1e-6 * own["rms_d"]
    band = int(near_separatrix(p, z64, d64).sum())
    assert abs(int(mg["n_in_bucket"][-1]) - own["n_in_bucket"]) <= band
    worst = 0.0
    for t in range(turns):
        e = max(abs(mg["rms_z"][t] / mo["rms_z"][t] - 1), abs(mg["rms_d"][t] / mo["rms_d"][t] - 1),
                abs(mg["mean_z"][t] - mo["mean_z"][t]) / mo["rms_z"][t],
                abs(mg["mean_d"][t] - mo["mean_d"][t]) / mo["rms_d"][t])
        worst = max(worst, e)
    print("fp32 per-turn %s: worst moment error over %d turns %.2e" % (integrator, turns, worst))
    assert worst <= 1e-4
    assert np.array_equal(mg["n_in_bucket"], mo["n_in_bucket"])   # nobody near the boundary: exact
