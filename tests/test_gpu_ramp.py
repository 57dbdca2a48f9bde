"""-m gpu: the CUDA path of the energy ramp (lt_track_ramp, lt_track_ramp_per_turn; SURVEY.md
sec. 8(f) row f2 "gamma ramps per turn"; G32) against oracle/ramp.inc, through the C
ABI, on the same seeded inputs.  Gates: per particle 1e-9 after 1000 turns, moments 1e-6 (G14),
bit-identity across chunkings and between the split-drift fused and the per-turn kernel (G16);
the long run per DESIGN.md G31 (particles the oracle itself resolves)."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")
if not torch.cuda.is_available():                      # collected but skipped on the CPU box
    pytest.skip("needs a CUDA device", allow_module_level=True)

import oracle                                           # noqa: E402
from paper_1610_05801_b200 import longtrack as lt       # noqa: E402
from paper_1610_05801_b200 import workloads as wl       # noqa: E402
from gpu_util import assert_moments_close, dev, gpu_track, stream_ptr  # noqa: E402

INTEGRATORS = ("euler_cromer", "leapfrog", "ruth4")
RAMP = wl.NEXT_CONFIGS["f2_ramp"]
SD = wl.matched_sigma_delta(0.23)


def both(integrator="leapfrog", ratio2=0.0):
    return lt.Tracker(wl.RING, integrator, ratio2), oracle.make_params(wl.RING, integrator, ratio2)


def moments_buffer(turns):
    return torch.zeros(turns * lt.MOMENTS_DTYPE.itemsize, dtype=torch.uint8, device="cuda")


def gpu_ramp(tr, z0, d0, p0c, a=None, psi=None, mode="fused", want_moments=False, zd=None):
    z, d = zd if zd is not None else (dev(z0), dev(d0))
    pt = dev(p0c)
    at = dev(a) if a is not None else None
    st = dev(psi) if psi is not None else None
    turns = len(p0c) - 1
    mom = moments_buffer(turns) if want_moments else None
    if mode == "fused":
        tr.track_ramp(z, d, z.numel(), turns, pt, at, st, stream_ptr())
    else:
        tr.track_ramp_per_turn(z, d, z.numel(), turns, pt, at, st, mom, None, stream_ptr())
    torch.cuda.synchronize()
    out = (z.cpu().numpy(), d.cpu().numpy())
    if want_moments:
        out += (mom.cpu().numpy().view(lt.MOMENTS_DTYPE),)
    return out


def assert_close(p, zg, dg, zo, do, gate=1e-9):
    g = oracle.derive(p)
    ez, ed = np.abs(zg - zo).max() / g["z_max"], np.abs(dg - do).max() / SD
    assert ez <= gate and ed <= gate, (ez, ed)
    return ez, ed


def test_ramp_per_particle_1000_turns_all_variants():
    """All integrators x single/double harmonic x {fused, fused split drifts, per-turn}: a fast
    ramp (sin phi_s up to 0.3) with a voltage programme on top, 1e-9 per particle."""
    N = 1000
    p0c, a, psi = wl.energy_ramp(N, 26e9, 26.3e9)
    a = a * (1.0 + 0.2 * np.sin(np.arange(N) / 50.0))
    for integrator in INTEGRATORS:
        for r in (0.0, 0.5):
            tr, p = both(integrator, r)
            z0, d0 = wl.gaussian_bunch(3001, 0.1, 41, ratio2=r)
            zo, do = oracle.track_ramp(p, z0, d0, p0c, a, psi)
            assert np.abs(zo - oracle.track(p, z0, d0, N)[0]).max() > 1e-2      # the ramp matters
            for mode, split in (("fused", 0), ("fused", 1), ("per_turn", 0)):
                tr.set_option(lt.OPT_SPLIT_DRIFTS, split)
                zg, dg = gpu_ramp(tr, z0, d0, p0c, a, psi, mode)
                e = assert_close(p, zg, dg, zo, do)
                print("ramp", integrator, r, mode, split, "ez %.1e ed %.1e" % e)


@pytest.mark.parametrize("integrator", INTEGRATORS)
def test_ramp_split_drift_fused_equals_per_turn_bits_and_chunking_is_invisible(integrator):
    tr, _ = both(integrator, 0.5)
    z0, d0 = wl.gaussian_bunch(5000, 0.1, 42, ratio2=0.5)
    p0c, a, psi = wl.energy_ramp(333, 26e9, 26.1e9)
    ref = gpu_ramp(tr, z0, d0, p0c, a, psi)
    for chunk, item in ((50, 0), (1 << 22, 17), (128, 32)):
        tr.set_option(lt.OPT_CHUNK_TURNS, chunk)
        tr.set_option(lt.OPT_ITEM_TURNS, item)
        tr.set_option(lt.OPT_FUSED_MODE, lt.FUSED_PERSISTENT_DYNAMIC if item else lt.FUSED_AUTO)
        out = gpu_ramp(tr, z0, d0, p0c, a, psi)
        assert np.array_equal(out[0], ref[0]) and np.array_equal(out[1], ref[1]), (chunk, item)
    tr.set_option(lt.OPT_SPLIT_DRIFTS, 1)
    zs, ds = gpu_ramp(tr, z0, d0, p0c, a, psi)
    zt, dt = gpu_ramp(tr, z0, d0, p0c, a, psi, "per_turn")
    assert np.array_equal(zs, zt) and np.array_equal(ds, dt)
    tr.set_option(lt.OPT_CHUNK_TURNS, 100)            # split drifts: also identical ACROSS calls
    zc, dc = gpu_ramp(tr, z0, d0, p0c, a, psi)
    assert np.array_equal(zs, zc) and np.array_equal(ds, dc)


@pytest.mark.parametrize("integrator", INTEGRATORS)
def test_ramp_scaled_and_plain_fast_layouts(integrator):
    """Merged-drift fused mode has two layouts: delta divided by the running kick amplitude (15 FP64
    instructions per sub-step, the default) and the plain one (16).  Both must sit inside the 1e-9
    gate against the oracle, with and without a voltage table; a voltage table that contains a
    ZERO cannot be divided by: the device-side scan of the table then selects the plain layout
    for the whole call, whose bits the result must equal -- also when the call is chunked and
    the zero sits in a later chunk than the first."""
    N = 700
    p0c, a, psi = wl.energy_ramp(N, 26e9, 26.2e9)
    a = a * (1.0 + 0.3 * np.sin(np.arange(N) / 40.0))
    for r in (0.0, 0.5):
        tr, p = both(integrator, r)
        z0, d0 = wl.gaussian_bunch(4001, 0.1, 71, ratio2=r)
        for volt in (a, None):
            zo, do = oracle.track_ramp(p, z0, d0, p0c, volt, psi)
            out = {}
            for scaled in (0, 1):
                tr.set_option(lt.OPT_RAMP_SCALED, scaled)
                out[scaled] = gpu_ramp(tr, z0, d0, p0c, volt, psi)
                assert_close(p, out[scaled][0], out[scaled][1], zo, do)
            assert not np.array_equal(out[0][1], out[1][1])          # they really are two evaluation orders
        a0 = a.copy()
        a0[[450, 451, 699]] = 0.0                                    # the RF is off for three turns
        zo, do = oracle.track_ramp(p, z0, d0, p0c, a0, psi)
        tr.set_option(lt.OPT_RAMP_SCALED, 0)
        ref = gpu_ramp(tr, z0, d0, p0c, a0, psi)
        assert_close(p, ref[0], ref[1], zo, do)
        tr.set_option(lt.OPT_RAMP_SCALED, 1)
        for chunk in (1 << 22, 128):
            tr.set_option(lt.OPT_CHUNK_TURNS, chunk)
            got = gpu_ramp(tr, z0, d0, p0c, a0, psi)
            assert np.array_equal(got[0], ref[0]) and np.array_equal(got[1], ref[1]), chunk
        tr.set_option(lt.OPT_CHUNK_TURNS, 1 << 22)


@pytest.mark.parametrize("integrator", INTEGRATORS)
def test_flat_ramp_without_tables_is_the_plain_map(integrator):
    """p0c constant at the create value, NULL tables: the plain map up to the rounding of
    beta(p) vs beta(gamma) (not bits: A and d are recomputed from p)."""
    tr, p = both(integrator)
    z0, d0 = wl.gaussian_bunch(4097, 0.23, 43)
    flat = np.full(501, wl.RING["p0c_eV"])
    for mode in ("fused", "per_turn"):
        zp, dp = gpu_track(tr, z0, d0, 500, mode)
        zg, dg = gpu_ramp(tr, z0, d0, flat, None, None, mode)
        assert_close(p, zg, dg, zp, dp, gate=1e-11)


@pytest.mark.parametrize("turns", [1, 2, 10, 11, 31, 32, 33, 64, 65])
def test_ramp_call_lengths_around_the_staging_block(turns):
    """The fused kernel stages 32 sub-steps per block in a cp.async double buffer (Ruth4: 3 per
    turn, so 10/11 turns straddle a block): lengths around the block size, merged and split."""
    p0c, a, psi = wl.energy_ramp(turns, 26e9, 26e9 * (1 + 1e-5 * turns))
    for integrator in INTEGRATORS:
        tr, p = both(integrator, 0.5)
        z0, d0 = wl.gaussian_bunch(777, 0.1, 47, ratio2=0.5)
        zo, do = oracle.track_ramp(p, z0, d0, p0c, a, psi)
        for split in (0, 1):
            tr.set_option(lt.OPT_SPLIT_DRIFTS, split)
            zg, dg = gpu_ramp(tr, z0, d0, p0c, a, psi)
            assert_close(p, zg, dg, zo, do, gate=1e-11)


@pytest.mark.parametrize("integrator", ["leapfrog", "ruth4"])
def test_ramp_every_launch_shape_returns_the_same_bits(integrator):
    """Warps per sub-partition 1 .. 16 (two CTAs per SM above 8: 32 warps x 3072 B of staging in
    each), one and two particles per lane, static and dynamic scheduling: same bits as the
    planner's launch, merged and split drifts."""
    tr, _ = both(integrator)
    n, turns = 40_003, 333
    z0, d0 = wl.gaussian_bunch(n, 0.08, 91)
    p0c, a, psi = wl.energy_ramp(turns, 26e9, 26.08e9)
    for split in (0, 1):
        tr.set_option(lt.OPT_SPLIT_DRIFTS, split)
        for opt in (lt.OPT_FUSED_MODE, lt.OPT_FUSED_ILP, lt.OPT_WARPS_PER_SMSP, lt.OPT_ITEM_TURNS):
            tr.set_option(opt, 0)
        ref = gpu_ramp(tr, z0, d0, p0c, a, psi)
        for mode, ilp, w, item in ((lt.FUSED_PERSISTENT_DYNAMIC, 1, 14, 40), (lt.FUSED_PERSISTENT_DYNAMIC, 1, 16, 0),
                                   (lt.FUSED_PERSISTENT_STATIC, 1, 16, 0), (lt.FUSED_PERSISTENT_DYNAMIC, 1, 8, 100),
                                   (lt.FUSED_PERSISTENT_DYNAMIC, 2, 1, 64), (lt.FUSED_PERSISTENT_DYNAMIC, 2, 4, 0),
                                   (lt.FUSED_PERSISTENT_STATIC, 2, 3, 0), (lt.FUSED_PERSISTENT_DYNAMIC, 1, 3, 7),
                                   (lt.FUSED_PERSISTENT_WRAP, 1, 2, 0), (lt.FUSED_PERSISTENT_WRAP, 2, 1, 0)):
            tr.set_option(lt.OPT_FUSED_MODE, mode)
            tr.set_option(lt.OPT_FUSED_ILP, ilp)
            tr.set_option(lt.OPT_WARPS_PER_SMSP, w)
            tr.set_option(lt.OPT_ITEM_TURNS, item)
            out = gpu_ramp(tr, z0, d0, p0c, a, psi)
            assert np.array_equal(out[0], ref[0]) and np.array_equal(out[1], ref[1]), (split, mode, ilp, w, item)
            assert tr.get_stat(lt.STAT_LAST_ILP) == ilp


def test_ramp_per_turn_moments_every_turn_graph_and_plain():
    tr, p = both()
    z0, d0 = wl.gaussian_bunch(20_001, 0.1, 44)
    p0c, a, psi = wl.energy_ramp(300, 26e9, 26.08e9)
    zo, do, mo = oracle.track_ramp_moments(p, z0, d0, p0c, a, psi)
    for graph in (1, 0):
        tr.set_option(lt.OPT_PER_TURN_GRAPH, graph)
        zg, dg, mg = gpu_ramp(tr, z0, d0, p0c, a, psi, "per_turn", want_moments=True)
        assert_moments_close(mg, mo)
        assert np.array_equal(mg["n_in_bucket"], mo["n_in_bucket"])
        assert_close(p, zg, dg, zo, do)


@pytest.mark.parametrize("n", [1, 2, 33, 4097, 100_003])
def test_ramp_ragged_sizes_and_misaligned_arrays(n):
    tr, p = both("ruth4", 0.5)
    z0, d0 = wl.gaussian_bunch(n, 0.1, 45 + n, ratio2=0.5)
    p0c, a, psi = wl.energy_ramp(100, 26e9, 26.03e9)
    zo, do = oracle.track_ramp(p, z0, d0, p0c, a, psi)
    for mode in ("fused", "per_turn"):
        zg, dg = gpu_ramp(tr, z0, d0, p0c, a, psi, mode)
        assert_close(p, zg, dg, zo, do, gate=1e-10)
        s = (n + 2) | 1                                  # both views start on an odd element
        buf = torch.zeros(s + n + 1, dtype=torch.float64, device="cuda")
        zt, dt = buf[1:n + 1], buf[s:s + n]
        assert zt.data_ptr() % 16 == 8 and dt.data_ptr() % 16 == 8
        zt.copy_(torch.from_numpy(z0)); dt.copy_(torch.from_numpy(d0))
        zm, dm = gpu_ramp(tr, None, None, p0c, a, psi, mode, zd=(zt, dt))
        assert np.array_equal(zm, zg) and np.array_equal(dm, dg), mode


def test_ramp_empty_calls_and_errors():
    tr, _ = both()
    z = torch.zeros(8, dtype=torch.float64, device="cuda")
    pt = dev(np.full(65, 26e9))
    tr.track_ramp(z, z, 0, 64, pt, None, None, stream_ptr())
    tr.track_ramp(z, z, 8, 0, pt, None, None, stream_ptr())
    tr.track_ramp_per_turn(z, z, 0, 64, pt, None, None, None, None, stream_ptr())
    torch.cuda.synchronize()
    assert float(z.abs().sum()) == 0.0
    with pytest.raises(lt.LongtrackError) as e:
        tr.track_ramp(z, z, 8, 64, None, None, None, stream_ptr())
    assert e.value.code == lt.E_NULL
    with pytest.raises(lt.LongtrackError) as e:
        lt.Tracker(wl.RING, "leapfrog", 0.0, 0.2).track_ramp(z, z, 8, 64, pt, None, None, stream_ptr())
    assert e.value.code == lt.E_PARAM


def test_ramp_full_size_launch_configuration():
    """f2_ramp config: 10^5 particles x 7*10^4 turns (the paper's run shape), 26 ->
    60 GeV/c on the synchronous phase, fused mode, in the launch configuration bench.py times;
    oracle on a seeded 2000-particle subsample.  First 1000 turns: 1e-9 per particle.  Full run:
    particles near the moving bucket's separatrix are lost during the ramp and are chaotic there
    (G31), so the long-run gates (1e-6 per particle, moments 1e-6) apply to the
    particles the ORACLE itself resolves: |fp64 - 80-bit twin| <= 1e-10 z_max."""
    tr, p = both()
    n, turns = RAMP["n"], RAMP["turns"]
    z0, d0 = wl.gaussian_bunch(n, RAMP["sigma_z"], RAMP["seed"])
    idx = wl.subsample_indices(n, 2000, RAMP["seed"])
    p0c, a, psi = wl.energy_ramp(turns, RAMP["p_start"], RAMP["p_end"])
    g = oracle.derive(p)
    zo, do = oracle.track_ramp(p, z0[idx], d0[idx], p0c[:1001], a[:1000], psi[:1000])
    zg, dg = gpu_ramp(tr, z0, d0, p0c[:1001], a[:1000], psi[:1000])
    assert_close(p, zg[idx], dg[idx], zo, do)
    zo, do = oracle.track_ramp(p, z0[idx], d0[idx], p0c, a, psi)
    zl, _ = oracle.track_ramp_ld(p, z0[idx], d0[idx], p0c, a, psi)
    resolved = np.abs(zo - zl.astype(np.float64)) / g["z_max"] <= 1e-10
    zg, dg = gpu_ramp(tr, z0, d0, p0c, a, psi)
    zg, dg = zg[idx], dg[idx]
    ez, ed = np.abs(zg - zo) / g["z_max"], np.abs(dg - do) / SD
    print("ramp full: resolved %.4f; on them median ez %.2e max ez %.2e max ed %.2e; rms_z %.4f -> %.4f"
          % (resolved.mean(), np.median(ez[resolved]), ez[resolved].max(), ed[resolved].max(),
             np.std(z0[idx]), np.std(zo[resolved])))
    assert resolved.mean() >= 0.95
    assert ez[resolved].max() <= 1e-6 and ed[resolved].max() <= 1e-6
    mg = oracle.moments_of(p, zg[resolved], dg[resolved])
    mo = oracle.moments_of(p, zo[resolved], do[resolved])
    assert abs(mg["rms_z"] / mo["rms_z"] - 1) <= 1e-6 and abs(mg["rms_d"] / mo["rms_d"] - 1) <= 1e-6
    assert abs(mg["mean_z"] - mo["mean_z"]) <= 1e-6 * mo["rms_z"]
    assert tr.get_stat(lt.STAT_LAST_GRID) % 148 == 0
