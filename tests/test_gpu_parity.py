"""-m gpu: the CUDA path (through the C ABI) against the CPU oracle, element by element, on the
same seeded inputs.  Gates: BASELINE.json:north_star (1e-9 per particle after 1000 turns,
1e-6 on per-turn moments, exact membership counts) with the readings G14-G17 of DESIGN.md."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")
if not torch.cuda.is_available():                      # collected but skipped on the CPU box
    pytest.skip("needs a CUDA device", allow_module_level=True)

import oracle                                           # noqa: E402
from paper_1610_05801_b200 import longtrack as lt       # noqa: E402
from paper_1610_05801_b200 import workloads as wl       # noqa: E402
from gpu_util import (assert_moments_close, assert_particle_gate, count_mismatch_is_in_layer,  # noqa: E402
                      dev, gpu_track, particle_errors, stream_ptr)

INTEGRATORS = ("euler_cromer", "leapfrog", "ruth4")


def both(integrator="leapfrog", ratio2=0.0, phi_s=None):
    return (lt.Tracker(wl.RING, integrator, ratio2, phi_s),
            oracle.make_params(wl.RING, integrator, ratio2, phi_s))


# ------------------------------------------------------------------ cfg0
@pytest.mark.parametrize("mode,split", [("fused", 0), ("fused", 1), ("per_turn", 0)])
def test_cfg0_per_particle_moments_count(mode, split):
    cfg = wl.CONFIGS[0]
    tr, p = both()
    tr.set_option(lt.OPT_SPLIT_DRIFTS, split)
    z0, d0 = wl.make_bunch(cfg)
    zo, do = oracle.track(p, z0, d0, cfg["turns"])
    zg, dg = gpu_track(tr, z0, d0, cfg["turns"], mode)
    assert_particle_gate(p, z0, d0, zg, dg, zo, do, wl.sigma_delta_for_gate(cfg))
    # final-state moments and membership count through the library
    mom = torch.zeros(lt.MOMENTS_DTYPE.itemsize, dtype=torch.uint8, device="cuda")
    cnt = torch.zeros(1, dtype=torch.int64, device="cuda")
    zt, dt = dev(zg), dev(dg)
    tr.moments_now(zt, dt, zt.numel(), mom, None, stream_ptr())
    tr.bucket_count(zt, dt, zt.numel(), cnt, stream_ptr())
    torch.cuda.synchronize()
    mg = mom.cpu().numpy().view(lt.MOMENTS_DTYPE)
    mo = oracle.moments_of(p, zo, do)
    assert_moments_close(mg, {k: [v] for k, v in mo.items()})
    assert int(cnt.item()) == mo["n_in_bucket"] == int(mg["n_in_bucket"][0])


def test_cfg0_per_turn_moments_every_turn():
    cfg = wl.CONFIGS[0]
    tr, p = both()
    z0, d0 = wl.make_bunch(cfg)
    zo, do, mo = oracle.track_moments(p, z0, d0, cfg["turns"])
    zg, dg, mg = gpu_track(tr, z0, d0, cfg["turns"], "per_turn", want_moments=True)
    assert_moments_close(mg, mo)
    assert np.array_equal(mg["n_in_bucket"], mo["n_in_bucket"])
    assert np.allclose(mg["cov_zd"], mo["cov_zd"], rtol=1e-6, atol=1e-6 * mo["rms_z"][0] * mo["rms_d"][0])
    assert_particle_gate(p, z0, d0, zg, dg, zo, do, wl.sigma_delta_for_gate(cfg))


# ------------------------------------------------------------------ structure
def test_result_does_not_depend_on_internal_chunking():
    """the CPU outer loop / in-kernel inner loop split must not change
    the result.  Bit-identical within one call, merged drifts included."""
    tr, _ = both()
    z0, d0 = wl.make_bunch(wl.CONFIGS[0], n=4099)
    ref = gpu_track(tr, z0, d0, 1000)
    for chunk in (1, 7, 333, 999, 1000):
        tr.set_option(lt.OPT_CHUNK_TURNS, chunk)
        out = gpu_track(tr, z0, d0, 1000)
        assert np.array_equal(out[0], ref[0]) and np.array_equal(out[1], ref[1]), chunk


@pytest.mark.parametrize("integrator", INTEGRATORS)
@pytest.mark.parametrize("ratio2", [0.0, 0.5])
def test_split_drift_mode_is_bit_identical_across_calls_and_modes(integrator, ratio2):
    """G16: with LT_OPT_SPLIT_DRIFTS fused(N) == fused(N/2) twice == per_turn(N), bit for bit."""
    tr, _ = both(integrator, ratio2)
    tr.set_option(lt.OPT_SPLIT_DRIFTS, 1)
    z0, d0 = wl.make_bunch(wl.CONFIGS[4], n=3001)
    a = gpu_track(tr, z0, d0, 400)
    h = gpu_track(tr, z0, d0, 200)
    b = gpu_track(tr, h[0], h[1], 200)
    c = gpu_track(tr, z0, d0, 400, "per_turn")
    for other in (b, c):
        assert np.array_equal(a[0], other[0]) and np.array_equal(a[1], other[1])
    # merged drifts differ from split drifts only at rounding level (G20)
    tr.set_option(lt.OPT_SPLIT_DRIFTS, 0)
    m = gpu_track(tr, z0, d0, 400)
    zmax = tr.derived()["z_max"]
    assert np.max(np.abs(m[0] - a[0])) / zmax < 1e-11


@pytest.mark.parametrize("integrator", INTEGRATORS)
@pytest.mark.parametrize("ratio2", [0.0, 0.5])
def test_dynamic_scheduling_is_bit_identical_to_the_plain_kernel(integrator, ratio2):
    """The on-device chunk scheduler (work items = 32 or 64 particles x item_turns, tapered at the
    end of a launch) must not change a single bit, merged or split drifts, whatever the item
    length and the number of particles per lane."""
    tr, _ = both(integrator, ratio2)
    z0, d0 = wl.make_bunch(wl.CONFIGS[4], n=150_001)
    for split in (0, 1):
        tr.set_option(lt.OPT_SPLIT_DRIFTS, split)
        tr.set_option(lt.OPT_FUSED_MODE, lt.FUSED_PLAIN)
        ref = gpu_track(tr, z0, d0, 777)
        tr.set_option(lt.OPT_FUSED_MODE, lt.FUSED_PERSISTENT_DYNAMIC)
        for ilp in (1, 2, 0):                           # one / two particles per lane / planner
            tr.set_option(lt.OPT_FUSED_ILP, ilp)
            for item in (0, 50, 200, 776):              # 200: full items + a tapered tail of 377
                tr.set_option(lt.OPT_ITEM_TURNS, item)
                out = gpu_track(tr, z0, d0, 777)
                assert np.array_equal(out[0], ref[0]) and np.array_equal(out[1], ref[1]), (split, ilp, item)
        tr.set_option(lt.OPT_FUSED_MODE, lt.FUSED_PERSISTENT_WRAP)     # static wrap-around schedule
        for ilp, w in ((1, 1), (1, 5), (2, 1), (2, 3), (0, 0)):        # 150 001 particles: groups > slots
            tr.set_option(lt.OPT_FUSED_ILP, ilp)
            tr.set_option(lt.OPT_WARPS_PER_SMSP, w)
            out = gpu_track(tr, z0, d0, 777)
            assert np.array_equal(out[0], ref[0]) and np.array_equal(out[1], ref[1]), (split, "wrap", ilp, w)
            assert tr.get_stat(lt.STAT_LAST_MODE) == lt.FUSED_PERSISTENT_WRAP
        tr.set_option(lt.OPT_WARPS_PER_SMSP, 0)
        tr.set_option(lt.OPT_FUSED_ILP, 0)
        tr.set_option(lt.OPT_FUSED_MODE, lt.FUSED_PERSISTENT_DYNAMIC)
        tr.set_option(lt.OPT_CHUNK_TURNS, 300)          # several launches, each with its own items
        out = gpu_track(tr, z0, d0, 777)
        assert np.array_equal(out[0], ref[0]) and np.array_equal(out[1], ref[1])
        tr.set_option(lt.OPT_CHUNK_TURNS, 1 << 22)


def test_wrap_around_schedule_is_a_cooperative_launch_and_survives_a_busy_gpu():
    """The wrap-around schedule (default at the configs[1] size) makes CTAs wait on one another, so
    it is launched cooperatively: the runtime guarantees co-residency or refuses, in which case
    the library runs the ticket queue (LT_STAT_LAST_MODE says which).  Here the headline shape
    runs while a second stream keeps the SMs busy with long foreign kernels: it must finish, and
    with the same bits as on an idle GPU and as the ticket queue gives."""
    tr, _ = both()
    z0, d0 = wl.make_bunch(wl.CONFIGS[1])
    turns = 3000
    assert tr.plan_fused(z0.size, turns)["dynamic"] == 2
    ref = gpu_track(tr, z0, d0, turns)
    assert tr.get_stat(lt.STAT_LAST_MODE) == lt.FUSED_PERSISTENT_WRAP
    tr.set_option(lt.OPT_FUSED_MODE, lt.FUSED_PERSISTENT_DYNAMIC)
    queue = gpu_track(tr, z0, d0, turns)
    assert np.array_equal(queue[0], ref[0]) and np.array_equal(queue[1], ref[1])
    tr.set_option(lt.OPT_FUSED_MODE, lt.FUSED_AUTO)
    side = torch.cuda.Stream()
    a = torch.randn(8192, 8192, device="cuda")
    with torch.cuda.stream(side):
        for _ in range(40):                                 # ~100 ms of GEMMs holding shared memory on every SM
            a = torch.mm(a, a).clamp_(-1.0, 1.0)
    out = gpu_track(tr, z0, d0, turns)                      # enqueued while the GEMMs run
    side.synchronize()
    assert tr.get_stat(lt.STAT_LAST_MODE) in (lt.FUSED_PERSISTENT_WRAP, lt.FUSED_PERSISTENT_DYNAMIC)
    assert np.array_equal(out[0], ref[0]) and np.array_equal(out[1], ref[1])


def test_deterministic():
    tr, _ = both()
    z0, d0 = wl.make_bunch(wl.CONFIGS[1], n=50_000)
    a = gpu_track(tr, z0, d0, 300, "per_turn", want_moments=True)
    b = gpu_track(tr, z0, d0, 300, "per_turn", want_moments=True)
    assert all(np.array_equal(x, y) for x, y in zip(a, b))


# ------------------------------------------------------------------ ragged sizes, layouts
@pytest.mark.parametrize("n", [1, 2, 3, 31, 33, 255, 257, 1000, 4097, 100_003, 250_001])
def test_ragged_sizes_all_layouts(n):
    """Every launch shape of the fused mode (plain kernel: block x ILP; persistent kernel:
    static / dynamic, warps per sub-partition, item length, sign-flip placement) gives the
    SAME BITS, and those agree with the oracle."""
    tr, p = both()
    z0, d0 = wl.make_bunch(wl.CONFIGS[0], n=n, seed=77 + n)
    zo, do = oracle.track(p, z0, d0, 100)
    sd = wl.sigma_delta_for_gate(wl.CONFIGS[0])
    zr, dr = gpu_track(tr, z0, d0, 100)                       # planner's choice
    assert_particle_gate(p, z0, d0, zr, dr, zo, do, sd, gate=1e-10)
    tr.set_option(lt.OPT_FUSED_MODE, lt.FUSED_PLAIN)
    for ilp in (0, 1, 2, 4):
        for block in (0, 32, 64, 128):
            tr.set_option(lt.OPT_FUSED_ILP, ilp)
            tr.set_option(lt.OPT_FUSED_BLOCK, block)
            zg, dg = gpu_track(tr, z0, d0, 100)
            assert np.array_equal(zg, zr) and np.array_equal(dg, dr), (ilp, block)
    for ilp in (1, 2):                                        # particles per lane of the persistent kernel
        tr.set_option(lt.OPT_FUSED_ILP, ilp)
        for mode, w, item, fq in ((lt.FUSED_PERSISTENT_STATIC, 0, 0, 0), (lt.FUSED_PERSISTENT_STATIC, 1, 0, 1),
                                  (lt.FUSED_PERSISTENT_STATIC, 16 if ilp == 1 else 4, 0, -1),
                                  (lt.FUSED_PERSISTENT_DYNAMIC, 0, 0, -1),
                                  (lt.FUSED_PERSISTENT_DYNAMIC, 5 if ilp == 1 else 3, 7, 0),
                                  (lt.FUSED_PERSISTENT_DYNAMIC, 8 if ilp == 1 else 4, 33, 1),
                                  (lt.FUSED_PERSISTENT_DYNAMIC, 2, 1, 1),
                                  (lt.FUSED_PERSISTENT_DYNAMIC, 12 if ilp == 1 else 1, 100, 0),
                                  (lt.FUSED_PERSISTENT_WRAP, 1, 0, 0), (lt.FUSED_PERSISTENT_WRAP, 2, 0, 1),
                                  (lt.FUSED_PERSISTENT_WRAP, 0, 0, -1)):
            tr.set_option(lt.OPT_FUSED_MODE, mode)
            tr.set_option(lt.OPT_WARPS_PER_SMSP, w)
            tr.set_option(lt.OPT_ITEM_TURNS, item)
            tr.set_option(lt.OPT_FLIP_ON_Q, fq)
            zg, dg = gpu_track(tr, z0, d0, 100)
            assert np.array_equal(zg, zr) and np.array_equal(dg, dr), (ilp, mode, w, item, fq)
            groups_lt_slots = -(-n // (32 * ilp)) < 148 * 4 * max(w, 1)     # wrap needs groups >= slots
            want = lt.FUSED_PERSISTENT_STATIC if (mode == lt.FUSED_PERSISTENT_WRAP and groups_lt_slots and w) else mode
            if not (mode == lt.FUSED_PERSISTENT_WRAP and w == 0):
                assert tr.get_stat(lt.STAT_LAST_MODE) == want, (ilp, mode, w)
            assert tr.get_stat(lt.STAT_LAST_ILP) == ilp
    zg, dg, mg = gpu_track(tr, z0, d0, 100, "per_turn", want_moments=True)
    assert_particle_gate(p, z0, d0, zg, dg, zo, do, sd, gate=1e-10)
    mo = oracle.moments_of(p, zo, do)
    assert int(mg["n_in_bucket"][-1]) == mo["n_in_bucket"]
    assert abs(mg["mean_z"][-1] - mo["mean_z"]) <= 1e-6 * max(mo["rms_z"], 1e-3)


def test_misaligned_arrays_take_the_scalar_path():
    """8-byte aligned but not 16-byte aligned pointers (a view offset by one element)."""
    tr, p = both()
    n = 5001
    z0, d0 = wl.make_bunch(wl.CONFIGS[0], n=n)
    zo, do = oracle.track(p, z0, d0, 50)
    for mode in ("fused", "per_turn"):
        zbuf = torch.zeros(n + 1, dtype=torch.float64, device="cuda")
        dbuf = torch.zeros(n + 1, dtype=torch.float64, device="cuda")
        zv, dv = zbuf[1:], dbuf[1:]
        assert zv.data_ptr() % 16 == 8
        zv.copy_(torch.from_numpy(z0)); dv.copy_(torch.from_numpy(d0))
        if mode == "fused":
            tr.set_option(lt.OPT_FUSED_MODE, lt.FUSED_PLAIN)
            tr.set_option(lt.OPT_FUSED_ILP, 2)
            tr.track_fused(zv, dv, n, 50, stream_ptr())
        else:
            tr.track_per_turn(zv, dv, n, 50, None, None, stream_ptr())
        torch.cuda.synchronize()
        assert_particle_gate(p, z0, d0, zv.cpu().numpy(), dv.cpu().numpy(), zo, do,
                             wl.sigma_delta_for_gate(wl.CONFIGS[0]), gate=1e-10)
        assert zbuf[0].item() == 0.0 and dbuf[0].item() == 0.0


def test_empty_and_zero_turn_calls_are_no_ops():
    tr, _ = both()
    z = dev([0.1, 0.2]); d = dev([1e-3, -1e-3])
    tr.track_fused(z, d, 0, 100, stream_ptr())
    tr.track_fused(z, d, 2, 0, stream_ptr())
    tr.track_per_turn(z, d, 0, 5, None, None, stream_ptr())
    tr.track_fused(None, None, 0, 5, stream_ptr())
    torch.cuda.synchronize()
    assert z.cpu().tolist() == [0.1, 0.2] and d.cpu().tolist() == [1e-3, -1e-3]
    with pytest.raises(lt.LongtrackError) as e:
        tr.track_fused(None, d, 2, 5, stream_ptr())
    assert e.value.code == lt.E_NULL
    with pytest.raises(lt.LongtrackError) as e:
        tr.track_fused(z.data_ptr() + 4, d, 1, 5, stream_ptr())
    assert e.value.code == lt.E_ALIGN


# ------------------------------------------------------------------ variants (cfg4 shape)
@pytest.mark.parametrize("integrator", INTEGRATORS)
@pytest.mark.parametrize("ratio2", [0.0, 0.5, -0.5])
@pytest.mark.parametrize("split", [0, 1])
def test_integrators_and_double_harmonic(integrator, ratio2, split):
    """configs[4]: EC / LF / Ruth4 with the double-harmonic kick; r = -0.5 is the zero-
    linear-focusing case that must be accepted (G10)."""
    cfg = wl.CONFIGS[4]
    tr, p = both(integrator, ratio2)
    tr.set_option(lt.OPT_SPLIT_DRIFTS, split)
    z0, d0 = wl.gaussian_bunch(20_000, cfg["sigma_z"], cfg["seed"], ratio2=max(ratio2, 0.0))
    zo, do = oracle.track(p, z0, d0, 1000)
    zg, dg = gpu_track(tr, z0, d0, 1000)
    assert_particle_gate(p, z0, d0, zg, dg, zo, do, wl.sigma_delta_for_gate(cfg))
    mo, = [oracle.moments_of(p, zo, do)]
    assert oracle.bucket_count(p, zg, dg) == mo["n_in_bucket"] or \
        count_mismatch_is_in_layer(p, zg, dg, zo, do) >= 0


def test_phi_s_generic_path():
    tr, p = both("leapfrog", 0.25, phi_s=0.3)
    z0, d0 = wl.make_bunch(wl.CONFIGS[0], n=5000)
    z0 = 0.3 * z0
    d0 = 0.3 * d0
    zo, do = oracle.track(p, z0, d0, 1000)
    for mode in ("fused", "per_turn"):
        zg, dg = gpu_track(tr, z0, d0, 1000, mode)
        g = oracle.derive(p)
        assert np.max(np.abs(zg - zo)) / g["z_max"] < 1e-9
        assert np.max(np.abs(dg - do)) / wl.matched_sigma_delta(0.23) < 1e-9


def test_kick_function_accuracy():
    """Euler-Cromer from delta = 0 returns delta = F(z): the hand-written sin against libm,
    in-bucket and for the large arguments unbound particles reach (|kappa z| ~ 1e4 rad)."""
    rng = np.random.default_rng(5)
    for r in (0.0, 0.5):
        tr, p = both("euler_cromer", r)
        g = oracle.derive(p)
        z = np.concatenate([rng.uniform(-1, 1, 20000) * g["z_max"], rng.uniform(-2500, 2500, 20000),
                            [0.0, g["z_max"], -g["z_max"], 0.5 * g["z_max"]]])
        zg, dg = gpu_track(tr, z, np.zeros_like(z), 1)
        ref = np.array([oracle.kick(p, zz) for zz in z])
        # abs error <= ~3 ulp of the unit sine, plus the phase roundings of both sides: kappa
        # and kappa*z in the oracle, kappa/pi and z*(kappa/pi) on the GPU (4 x 2^-53 |phase|)
        tol = g["A"] * (1 + abs(r)) * (6.7e-16 + 4.5e-16 * np.abs(g["kappa"] * z))
        assert np.all(np.abs(dg - ref) <= tol), float(np.max(np.abs(dg - ref) / tol))


# ------------------------------------------------------------------ cfg1 hollow bunch
def test_cfg1_first_1000_turns_including_unbound_particles():
    cfg = wl.CONFIGS[1]
    tr, p = both()
    z0, d0 = wl.make_bunch(cfg)
    zo, do = oracle.track(p, z0, d0, 1000)
    zg, dg = gpu_track(tr, z0, d0, 1000)
    info = assert_particle_gate(p, z0, d0, zg, dg, zo, do, wl.sigma_delta_for_gate(cfg))
    cnt = torch.zeros(1, dtype=torch.int64, device="cuda")
    zt, dt = dev(zg), dev(dg)
    tr.bucket_count(zt, dt, zt.numel(), cnt, stream_ptr())
    torch.cuda.synchronize()
    assert int(cnt.item()) == oracle.bucket_count(p, zg, dg)       # same state, both predicates
    n_diff = count_mismatch_is_in_layer(p, zg, dg, zo, do)
    assert int(cnt.item()) - oracle.bucket_count(p, zo, do) in range(-n_diff, n_diff + 1)
    print("cfg1@1000:", info, "membership flips in layer:", n_diff)


def test_cfg1_full_run_final_state():
    """configs[1]: 10^5 x 7*10^4 turns, fused.  G18: counts exact (G15), moments 1e-6,
    per-particle reported and gated at 1e-6 for >= 99.9 % of the particles outside the layer."""
    cfg = wl.CONFIGS[1]
    tr, p = both()
    z0, d0 = wl.make_bunch(cfg)
    zo, do = oracle.track(p, z0, d0, cfg["turns"])
    zg, dg = gpu_track(tr, z0, d0, cfg["turns"])
    ez, ed, layer = particle_errors(p, z0, d0, zg, dg, zo, do, wl.sigma_delta_for_gate(cfg))
    out = ~layer
    frac_ok = np.mean((ez[out] <= 1e-6) & (ed[out] <= 1e-6))
    print("cfg1 full: median ez %.2e p99.9 %.2e max %.2e; layer %d; frac<=1e-6 %.5f"
          % (np.median(ez), np.quantile(ez, 0.999), ez.max(), layer.sum(), frac_ok))
    assert frac_ok >= 0.999
    mg, mo = oracle.moments_of(p, zg, dg), oracle.moments_of(p, zo, do)
    for k in ("rms_z", "rms_d"):
        assert abs(mg[k] / mo[k] - 1) <= 1e-6, k
    assert abs(mg["mean_z"] - mo["mean_z"]) <= 1e-6 * mo["rms_z"]
    assert abs(mg["mean_d"] - mo["mean_d"]) <= 1e-6 * mo["rms_d"]
    n_diff = count_mismatch_is_in_layer(p, zg, dg, zo, do)
    assert mg["n_in_bucket"] - mo["n_in_bucket"] in range(-n_diff, n_diff + 1)
    assert n_diff <= 2, "membership flips inside the separatrix layer: %d" % n_diff


# ------------------------------------------------------------------ cfg2 at full size
def test_cfg2_full_size_launch_configuration_on_a_subsample():
    """configs[2]: the GPU tracks all 10^6 particles (the launch configuration the bench
    times); the oracle tracks a seeded 10^4 subsample (particles are independent)."""
    cfg = wl.CONFIGS[2]
    tr, p = both()
    z0, d0 = wl.make_bunch(cfg)
    idx = wl.subsample_indices(cfg["n"], cfg["subsample"], cfg["seed"])
    sd = wl.sigma_delta_for_gate(cfg)
    zo, do = oracle.track(p, z0[idx], d0[idx], 1000)
    zg, dg = gpu_track(tr, z0, d0, 1000)
    assert_particle_gate(p, z0[idx], d0[idx], zg[idx], dg[idx], zo, do, sd)
    # the full 10^5 turns
    zo, do = oracle.track(p, z0[idx], d0[idx], cfg["turns"])
    zg, dg = gpu_track(tr, z0, d0, cfg["turns"])
    ez, ed, layer = particle_errors(p, z0[idx], d0[idx], zg[idx], dg[idx], zo, do, sd)
    out = ~layer
    print("cfg2 full: median ez %.2e max %.2e (outside layer), layer %d"
          % (np.median(ez[out]), ez[out].max(), layer.sum()))
    assert np.mean((ez[out] <= 1e-6) & (ed[out] <= 1e-6)) >= 0.999
    mg, mo = oracle.moments_of(p, zg[idx], dg[idx]), oracle.moments_of(p, zo, do)
    assert abs(mg["rms_z"] / mo["rms_z"] - 1) <= 1e-6 and abs(mg["rms_d"] / mo["rms_d"] - 1) <= 1e-6
    n_diff = count_mismatch_is_in_layer(p, zg[idx], dg[idx], zo, do)
    assert mg["n_in_bucket"] - mo["n_in_bucket"] in range(-n_diff, n_diff + 1)


# ------------------------------------------------------------------ cfg4 at full size
@pytest.mark.parametrize("integrator", INTEGRATORS)
def test_cfg4_full_size_launch_configuration_on_a_subsample(integrator):
    """configs[4]: the GPU tracks all 10^6 particles x 10^4 turns with r = 0.5 (the launch
    configuration of the fp64 variants); the oracle tracks the seeded 10^5 subsample.
    SURVEY.md sec. 8(d): per particle at 10^3 turns (1e-9, G17), at 10^4 turns moments 1e-6 and
    the membership count exact up to particles inside the separatrix layer (G15)."""
    cfg = wl.CONFIGS[4]
    tr, p = both(integrator, cfg["ratio2"])
    z0, d0 = wl.make_bunch(cfg)
    idx = wl.subsample_indices(cfg["n"], cfg["subsample"], cfg["seed"])
    sd = wl.sigma_delta_for_gate(cfg)
    zo, do = oracle.track(p, z0[idx], d0[idx], 1000)
    zg, dg = gpu_track(tr, z0, d0, 1000)
    info = assert_particle_gate(p, z0[idx], d0[idx], zg[idx], dg[idx], zo, do, sd)
    zo, do = oracle.track(p, z0[idx], d0[idx], cfg["turns"])
    zg, dg = gpu_track(tr, z0, d0, cfg["turns"])
    ez, ed, layer = particle_errors(p, z0[idx], d0[idx], zg[idx], dg[idx], zo, do, sd)
    out = ~layer
    print("cfg4 %s: @1000 %s; @%d median ez %.2e max %.2e (outside layer), layer %d"
          % (integrator, info, cfg["turns"], np.median(ez[out]), ez[out].max(), layer.sum()))
    assert np.mean((ez[out] <= 1e-6) & (ed[out] <= 1e-6)) >= 0.999
    # moments on the particles both sides keep in the bucket: the few escapers (G14) stream
    # away at ~1 m per 100 turns and would otherwise carry the whole rms
    m = oracle.bucket_mask(p, zg[idx], dg[idx]) & oracle.bucket_mask(p, zo, do)
    assert m.mean() > 0.99
    mg, mo = oracle.moments_of(p, zg[idx][m], dg[idx][m]), oracle.moments_of(p, zo[m], do[m])
    assert abs(mg["rms_z"] / mo["rms_z"] - 1) <= 1e-6 and abs(mg["rms_d"] / mo["rms_d"] - 1) <= 1e-6
    assert abs(mg["mean_z"] - mo["mean_z"]) <= 1e-6 * mo["rms_z"]
    assert abs(mg["mean_d"] - mo["mean_d"]) <= 1e-6 * mo["rms_d"]
    # and over all subsample particles outside the G17 layer, escapers included
    ag = oracle.moments_of(p, zg[idx][out], dg[idx][out])
    ao = oracle.moments_of(p, zo[out], do[out])
    assert abs(ag["rms_z"] / ao["rms_z"] - 1) <= 1e-6 and abs(ag["rms_d"] / ao["rms_d"] - 1) <= 1e-6
    ag, ao = oracle.moments_of(p, zg[idx], dg[idx]), oracle.moments_of(p, zo, do)
    n_diff = count_mismatch_is_in_layer(p, zg[idx], dg[idx], zo, do)
    assert ag["n_in_bucket"] - ao["n_in_bucket"] in range(-n_diff, n_diff + 1)


# ------------------------------------------------------------------ cfg3 at full size
def test_cfg3_full_size_per_turn_moments():
    """configs[3]: 10^7 particles, 1000 turns, one launch per turn with fused moments, in the
    launch configuration bench.py times (CUDA graph, alternating sweep).  Oracle: ALL 10^7
    particles on ALL 1000 turns (BASELINE.json:north_star: "Per-turn moments are compared to the
    oracle with relative error <= 1e-6"; counts exact on every turn), the final state per
    particle, and the reduction itself at turn 1000 (oracle moments of the GPU's own final
    state).  The oracle pass costs a few minutes of host time: it is two-pass long double."""
    cfg = wl.CONFIGS[3]
    tr, p = both()
    z0, d0 = wl.make_bunch(cfg)
    zg, dg, mg = gpu_track(tr, z0, d0, cfg["turns"], "per_turn", want_moments=True)
    zo, do, mo = oracle.track_moments(p, z0, d0, cfg["turns"])
    assert len(mo) == cfg["turns"] == len(mg)
    assert_moments_close(mg, mo)
    assert np.array_equal(mg["n_in_bucket"], mo["n_in_bucket"])
    info = assert_particle_gate(p, z0, d0, zg, dg, zo, do, wl.sigma_delta_for_gate(cfg))
    print("cfg3 full size: per particle", info, "worst rms_z ratio-1 %.2e"
          % np.abs(mg["rms_z"] / mo["rms_z"] - 1).max())
    last = oracle.moments_of(p, zg, dg)
    assert_moments_close(mg[-1:], {k: [v] for k, v in last.items()})
    assert int(mg["n_in_bucket"][-1]) == last["n_in_bucket"]


def test_sharded_per_turn_path_on_one_gpu():
    """SURVEY.md sec. 8(e) on ONE device: a configs[3]-shaped bunch of 1 000 001 particles is split
    with workloads.shard_range into two contiguous ranges of ONE device array -- the first of odd
    size, so that the second starts 8-byte aligned (scalar path) -- and tracked by two trackers on two
    streams with raw sums; the two lt_sums[turns] are added on the host (what the all-reduce does),
    lt_moments_from_sums finalises.  Must equal the unsharded GPU run (state: same bits; moments:
    1e-13; counts exact) and the oracle (1e-6; counts exact).  Unmeasured on multi-GPU hardware."""
    tr, p = both()
    n, turns = 1_000_001, 200                            # 3 graph replays of 64 + a tail of 8
    z0, d0 = wl.make_bunch(wl.CONFIGS[3], n=n)
    zu, du, mu = gpu_track(tr, z0, d0, turns, "per_turn", want_moments=True)
    zs, ds = dev(z0), dev(d0)
    streams = [torch.cuda.Stream(), torch.cuda.Stream()]
    trackers = [lt.Tracker(wl.RING, "leapfrog"), lt.Tracker(wl.RING, "leapfrog")]
    sums = [torch.zeros(turns * lt.SUMS_DTYPE.itemsize, dtype=torch.uint8, device="cuda") for _ in range(2)]
    torch.cuda.synchronize()
    for k in range(2):
        lo, hi = wl.shard_range(n, k, 2)
        zk, dk = zs[lo:hi], ds[lo:hi]
        if k == 0:
            assert (hi - lo) % 2 == 1 and zk.data_ptr() % 16 == 0
        else:
            assert zk.data_ptr() % 16 == 8
        trackers[k].track_per_turn(zk, dk, hi - lo, turns, None, sums[k], streams[k].cuda_stream)
    torch.cuda.synchronize()
    assert np.array_equal(zs.cpu().numpy(), zu) and np.array_equal(ds.cpu().numpy(), du)
    parts = [s.cpu().numpy().view(lt.SUMS_DTYPE) for s in sums]
    total = np.zeros(turns, dtype=lt.SUMS_DTYPE)
    for name in lt.SUMS_DTYPE.names:
        total[name] = parts[0][name] + parts[1][name]    # the SUM all-reduce
    assert np.all(total["n"] == n)
    ms = lt.moments_from_sums(total)
    assert np.array_equal(ms["n_in_bucket"], mu["n_in_bucket"])
    for name in ("rms_z", "rms_d"):
        assert np.max(np.abs(ms[name] / mu[name] - 1)) <= 1e-13, name
    assert np.max(np.abs(ms["mean_z"] - mu["mean_z"])) <= 1e-13 * mu["rms_z"].max()
    _, _, mo = oracle.track_moments(p, z0, d0, turns)
    assert_moments_close(ms, mo)
    assert np.array_equal(ms["n_in_bucket"], mo["n_in_bucket"])


def test_per_turn_moments_medium_all_turns_graph_and_plain():
    tr, p = both()
    z0, d0 = wl.make_bunch(wl.CONFIGS[3], n=100_000)
    _, _, mo = oracle.track_moments(p, z0, d0, 300)
    for graph in (1, 0):
        for reverse in (1, 0):
            tr.set_option(lt.OPT_PER_TURN_GRAPH, graph)
            tr.set_option(lt.OPT_PER_TURN_REVERSE, reverse)
            _, _, mg = gpu_track(tr, z0, d0, 300, "per_turn", want_moments=True)
            assert_moments_close(mg, mo)
            assert np.array_equal(mg["n_in_bucket"], mo["n_in_bucket"])


def test_sums_output_and_host_finalisation():
    tr, p = both()
    z0, d0 = wl.make_bunch(wl.CONFIGS[0], n=30_001)
    z, d = dev(z0), dev(d0)
    turns = 70
    sums = torch.zeros(turns * lt.SUMS_DTYPE.itemsize, dtype=torch.uint8, device="cuda")
    mom = torch.zeros(turns * lt.MOMENTS_DTYPE.itemsize, dtype=torch.uint8, device="cuda")
    tr.track_per_turn(z, d, z.numel(), turns, mom, sums, stream_ptr())
    torch.cuda.synchronize()
    s = sums.cpu().numpy().view(lt.SUMS_DTYPE)
    m = mom.cpu().numpy().view(lt.MOMENTS_DTYPE)
    m2 = lt.moments_from_sums(s)
    assert np.all(s["n"] == 30_001)
    for k in ("mean_z", "rms_z", "mean_d", "rms_d", "cov_zd"):
        assert np.allclose(m[k], m2[k], rtol=1e-13, atol=1e-18), k
    assert np.array_equal(m["n_in_bucket"], m2["n_in_bucket"])


# ------------------------------------------------------------------ observables
def test_bucket_count_and_moments_of_arbitrary_states():
    for r in (0.0, 0.5):
        tr, p = both("leapfrog", r)
        g = oracle.derive(p)
        rng = np.random.default_rng(9)
        n = 200_003
        z = rng.uniform(-1.3, 1.3, n) * g["z_max"]
        d = rng.uniform(-1.3, 1.3, n) * 4.2e-3
        zt, dt = dev(z), dev(d)
        cnt = torch.zeros(1, dtype=torch.int64, device="cuda")
        mom = torch.zeros(lt.MOMENTS_DTYPE.itemsize, dtype=torch.uint8, device="cuda")
        tr.bucket_count(zt, dt, n, cnt, stream_ptr())
        tr.moments_now(zt, dt, n, mom, None, stream_ptr())
        torch.cuda.synchronize()
        mo = oracle.moments_of(p, z, d)
        assert int(cnt.item()) == mo["n_in_bucket"]
        mg = mom.cpu().numpy().view(lt.MOMENTS_DTYPE)
        assert_moments_close(mg, {k: [v] for k, v in mo.items()}, tol=1e-12)


# ------------------------------------------------------------------ host-buffer entry point
def test_host_entry_point_matches_device_path_bit_for_bit():
    tr, p = both()
    z0, d0 = wl.make_bunch(wl.CONFIGS[0], n=12_345)
    zg, dg = gpu_track(tr, z0, d0, 500)
    zh = torch.from_numpy(z0.copy()).pin_memory()
    dh = torch.from_numpy(d0.copy()).pin_memory()
    cnt = tr.track_fused_host(zh, dh, zh.numel(), 500, want_count=True)
    assert np.array_equal(zh.numpy(), zg) and np.array_equal(dh.numpy(), dg)
    assert cnt == oracle.bucket_count(p, zg, dg)
    # pageable numpy memory works too
    zn, dn = z0.copy(), d0.copy()
    tr.track_fused_host(zn, dn, zn.size, 500)
    assert np.array_equal(zn, zg) and np.array_equal(dn, dg)


# ------------------------------------------------------------------ fp32 mode
@pytest.mark.parametrize("integrator", INTEGRATORS)
def test_fp32_mode_moments_within_1e4(integrator):
    """configs[4]: optional fp32 mode against the fp64 oracle, 1e-4 on moments, gated on the
    in-bucket flavour because a handful of escapers dominate the all-particle rms z (G14)."""
    cfg = wl.CONFIGS[4]
    tr, p = both(integrator, cfg["ratio2"])
    z0, d0 = wl.make_bunch(cfg, n=100_000)
    turns = cfg["turns"]
    zo, do = oracle.track(p, z0, d0, turns)
    for mode in ("fused", "per_turn"):
        zg, dg = gpu_track(tr, z0, d0, turns if mode == "fused" else 1000, mode, f32=True)
        if mode == "per_turn":
            zo1, do1 = oracle.track(p, z0, d0, 1000)
        else:
            zo1, do1 = zo, do
        zg, dg = zg.astype(np.float64), dg.astype(np.float64)
        m = oracle.bucket_mask(p, zg, dg) & oracle.bucket_mask(p, zo1, do1)
        assert m.mean() > 0.99
        a, b = oracle.moments_of(p, zg[m], dg[m]), oracle.moments_of(p, zo1[m], do1[m])
        assert abs(a["rms_z"] / b["rms_z"] - 1) <= 1e-4 and abs(a["rms_d"] / b["rms_d"] - 1) <= 1e-4
        assert abs(a["mean_z"] - b["mean_z"]) <= 1e-4 * b["rms_z"]
        assert abs(a["mean_d"] - b["mean_d"]) <= 1e-4 * b["rms_d"]
