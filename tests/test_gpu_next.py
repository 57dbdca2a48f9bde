"""-m gpu: the CUDA path for SURVEY.md sec. 8(f) rows f2 (RF programme), f3 (transverse maps) and
f4 (slicing) against oracle/next_oracle.c, through the C ABI, on the same seeded inputs.
Gates: per particle 1e-9 after 1000 turns (G17), moments 1e-6 (G14), integer work bit-exact
(histograms: G29; membership counts: G15); long chaotic runs per DESIGN.md G31."""
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
                      dev, gpu_track, stream_ptr)

INTEGRATORS = ("euler_cromer", "leapfrog", "ruth4")
F2, F3, F4 = (wl.NEXT_CONFIGS[k] for k in ("f2_programme", "f3_transverse", "f4_slices"))


def both(integrator="leapfrog", ratio2=0.0, phi_s=None):
    return (lt.Tracker(wl.RING, integrator, ratio2, phi_s),
            oracle.make_params(wl.RING, integrator, ratio2, phi_s))


def moments_buffer(turns):
    return torch.zeros(turns * lt.MOMENTS_DTYPE.itemsize, dtype=torch.uint8, device="cuda")


# ================================================================== f2: RF programme
def gpu_programme(tr, z0, d0, a, psi, mode="fused", want_moments=False):
    z, d, at, pt = dev(z0), dev(d0), dev(a), dev(psi)
    turns = len(a)
    mom = moments_buffer(turns) if want_moments else None
    if mode == "fused":
        tr.track_programme(z, d, z.numel(), turns, at, pt, stream_ptr())
    else:
        tr.track_programme_per_turn(z, d, z.numel(), turns, at, pt, mom, None, stream_ptr())
    torch.cuda.synchronize()
    out = (z.cpu().numpy(), d.cpu().numpy())
    if want_moments:
        out += (mom.cpu().numpy().view(lt.MOMENTS_DTYPE),)
    return out


def strong_programme(turns, seed=7):
    """1000-turn test programme: every feature of the f2 recipe at full strength within a few
    synchrotron periods (ramp to 1.5 V, 0.15 rad near-resonant modulation, 1e-3 rad noise)."""
    return wl.rf_programme(turns, seed, mod_amplitude=0.15)


@pytest.mark.parametrize("integrator", INTEGRATORS)
@pytest.mark.parametrize("ratio2", [0.0, 0.5])
@pytest.mark.parametrize("mode", ["fused", "per_turn"])
def test_programme_per_particle_1000_turns(integrator, ratio2, mode):
    tr, p = both(integrator, ratio2)
    z0, d0 = wl.gaussian_bunch(3001, 0.23, 21, ratio2=ratio2)
    a, psi = strong_programme(1000)
    zo, do = oracle.track_programme(p, z0, d0, a, psi)
    zg, dg = gpu_programme(tr, z0, d0, a, psi, mode)
    info = assert_particle_gate(p, z0, d0, zg, dg, zo, do, wl.matched_sigma_delta(0.23))
    assert np.abs(zo - oracle.track(p, z0, d0, 1000)[0]).max() > 1e-3     # the programme matters
    print("f2", integrator, ratio2, mode, info)


def test_programme_generic_phi_s_path():
    tr, p = both("leapfrog", 0.3, phi_s=0.35)
    z0, d0 = wl.gaussian_bunch(1500, 0.1, 22)
    a, psi = strong_programme(500)
    zo, do = oracle.track_programme(p, z0, d0, a, psi)
    for mode in ("fused", "per_turn"):
        zg, dg = gpu_programme(tr, z0, d0, a, psi, mode)
        g = oracle.derive(p)
        assert np.abs(zg - zo).max() / g["z_max"] <= 1e-9, mode
        assert np.abs(dg - do).max() / wl.matched_sigma_delta(0.23) <= 1e-9, mode


@pytest.mark.parametrize("integrator", INTEGRATORS)
def test_trivial_programme_is_bit_identical_to_the_plain_kernels(integrator):
    """a_t = 1, psi_t = 0: v + 0 and q * 1 are exact, so both modes return the plain map's bits."""
    tr, _ = both(integrator, 0.5)
    z0, d0 = wl.gaussian_bunch(4097, 0.3, 23, ratio2=0.5)
    one, zero = np.ones(300), np.zeros(300)
    for mode in ("fused", "per_turn"):
        zp, dp = gpu_track(tr, z0, d0, 300, mode)
        zg, dg = gpu_programme(tr, z0, d0, one, zero, mode)
        assert np.array_equal(zg, zp) and np.array_equal(dg, dp), mode


@pytest.mark.parametrize("integrator", INTEGRATORS)
def test_programme_split_drift_fused_equals_per_turn_bits_and_chunking_is_invisible(integrator):
    """G16 for f2: with LT_OPT_SPLIT_DRIFTS the fused kernel and the per-turn kernel run the same
    instruction sequence per particle; and the result of a call never depends on chunking."""
    tr, _ = both(integrator, 0.0)
    z0, d0 = wl.gaussian_bunch(5000, 0.23, 24)
    a, psi = strong_programme(333)
    ref = gpu_programme(tr, z0, d0, a, psi, "fused")
    for chunk, item in ((50, 0), (1 << 22, 17), (128, 32)):
        tr.set_option(lt.OPT_CHUNK_TURNS, chunk)
        tr.set_option(lt.OPT_ITEM_TURNS, item)
        tr.set_option(lt.OPT_FUSED_MODE, lt.FUSED_PERSISTENT_DYNAMIC if item else lt.FUSED_AUTO)
        out = gpu_programme(tr, z0, d0, a, psi, "fused")
        assert np.array_equal(out[0], ref[0]) and np.array_equal(out[1], ref[1]), (chunk, item)
    tr.set_option(lt.OPT_SPLIT_DRIFTS, 1)
    zs, ds = gpu_programme(tr, z0, d0, a, psi, "fused")
    zt, dt = gpu_programme(tr, z0, d0, a, psi, "per_turn")
    assert np.array_equal(zs, zt) and np.array_equal(ds, dt)


@pytest.mark.parametrize("integrator,ratio2", [("leapfrog", 0.0), ("ruth4", 0.5)])
def test_programme_every_schedule_and_lane_count_returns_the_same_bits(integrator, ratio2):
    """Static slots, ticket queue (tapered items) and the wrap-around schedule, one and two
    particles per lane, at a size with more groups than warp slots (80 003 particles): the fused
    RF-programme kernel returns the bits of the planner's launch, merged and split drifts, also
    when the call is cut into several launches."""
    tr, p = both(integrator, ratio2)
    z0, d0 = wl.gaussian_bunch(80_003, 0.23, 25, ratio2=ratio2)
    a, psi = strong_programme(211)
    zo, do = oracle.track_programme(p, z0, d0, a, psi)
    for split in (0, 1):
        tr.set_option(lt.OPT_SPLIT_DRIFTS, split)
        for opt in (lt.OPT_FUSED_MODE, lt.OPT_FUSED_ILP, lt.OPT_WARPS_PER_SMSP, lt.OPT_ITEM_TURNS):
            tr.set_option(opt, 0)
        tr.set_option(lt.OPT_CHUNK_TURNS, 1 << 22)
        ref = gpu_programme(tr, z0, d0, a, psi, "fused")
        assert np.abs(ref[0] - zo).max() / oracle.derive(p)["z_max"] <= 1e-10
        for mode, ilp, w, item, chunk in ((lt.FUSED_PERSISTENT_WRAP, 2, 2, 0, 1 << 22), (lt.FUSED_PERSISTENT_WRAP, 1, 3, 0, 1 << 22),
                                          (lt.FUSED_PERSISTENT_WRAP, 2, 1, 0, 100), (lt.FUSED_PERSISTENT_DYNAMIC, 2, 2, 40, 1 << 22),
                                          (lt.FUSED_PERSISTENT_DYNAMIC, 1, 4, 70, 150), (lt.FUSED_PERSISTENT_STATIC, 2, 4, 0, 1 << 22),
                                          (lt.FUSED_PERSISTENT_STATIC, 1, 8, 0, 64)):
            tr.set_option(lt.OPT_FUSED_MODE, mode)
            tr.set_option(lt.OPT_FUSED_ILP, ilp)
            tr.set_option(lt.OPT_WARPS_PER_SMSP, w)
            tr.set_option(lt.OPT_ITEM_TURNS, item)
            tr.set_option(lt.OPT_CHUNK_TURNS, chunk)
            out = gpu_programme(tr, z0, d0, a, psi, "fused")
            assert np.array_equal(out[0], ref[0]) and np.array_equal(out[1], ref[1]), (split, mode, ilp, w, item, chunk)
            assert tr.get_stat(lt.STAT_LAST_MODE) == mode and tr.get_stat(lt.STAT_LAST_ILP) == ilp


@pytest.mark.parametrize("turns", [1, 2, 31, 32, 33, 64, 65, 97])
def test_programme_call_lengths_around_the_staging_block(turns):
    """The fused kernel stages the table in blocks of 32 entries per warp and peels the call's
    last turn: lengths around the block size, merged and split drifts, all integrators."""
    a, psi = strong_programme(turns, seed=70 + turns)
    for integrator in INTEGRATORS:
        tr, p = both(integrator, 0.5)
        z0, d0 = wl.gaussian_bunch(777, 0.23, 27, ratio2=0.5)
        zo, do = oracle.track_programme(p, z0, d0, a, psi)
        for split in (0, 1):
            tr.set_option(lt.OPT_SPLIT_DRIFTS, split)
            zg, dg = gpu_programme(tr, z0, d0, a, psi, "fused")
            g = oracle.derive(p)
            assert np.abs(zg - zo).max() / g["z_max"] <= 1e-11, (integrator, split)
            assert np.abs(dg - do).max() / wl.matched_sigma_delta(0.23) <= 1e-11, (integrator, split)


def test_programme_per_turn_moments_every_turn_graph_and_plain():
    tr, p = both()
    z0, d0 = wl.gaussian_bunch(20_001, 0.23, 25)
    a, psi = strong_programme(300)
    zo, do, mo = oracle.track_programme_moments(p, z0, d0, a, psi)
    for graph in (1, 0):
        tr.set_option(lt.OPT_PER_TURN_GRAPH, graph)
        zg, dg, mg = gpu_programme(tr, z0, d0, a, psi, "per_turn", want_moments=True)
        assert_moments_close(mg, mo)
        n_diff = count_mismatch_is_in_layer(p, zg, dg, zo, do)
        assert np.max(np.abs(mg["n_in_bucket"].astype(np.int64) - mo["n_in_bucket"].astype(np.int64))) <= n_diff
        assert_particle_gate(p, z0, d0, zg, dg, zo, do, wl.matched_sigma_delta(0.23))


def test_programme_empty_and_misaligned():
    tr, p = both()
    a, psi = strong_programme(64)
    at, pt = dev(a), dev(psi)
    z = torch.zeros(8, dtype=torch.float64, device="cuda")
    tr.track_programme(z, z, 0, 64, at, pt, stream_ptr())
    tr.track_programme(z, z, 8, 0, at, pt, stream_ptr())
    tr.track_programme_per_turn(z, z, 0, 64, at, pt, None, None, stream_ptr())
    with pytest.raises(lt.LongtrackError):
        tr.track_programme(z, z, 8, 64, None, pt, stream_ptr())
    # arrays offset by one double: the per-turn kernel takes its scalar path
    z0, d0 = wl.gaussian_bunch(1001, 0.23, 26)
    zo, do = oracle.track_programme(p, z0, d0, a, psi)
    buf = torch.zeros(2 * 1002 + 2, dtype=torch.float64, device="cuda")
    zt, dt = buf[1:1002], buf[1003:2004]
    assert zt.data_ptr() % 16 == 8
    zt.copy_(torch.from_numpy(z0)); dt.copy_(torch.from_numpy(d0))
    tr.track_programme_per_turn(zt, dt, 1001, 64, at, pt, None, None, stream_ptr())
    torch.cuda.synchronize()
    assert_particle_gate(p, z0, d0, zt.cpu().numpy(), dt.cpu().numpy(), zo, do, wl.matched_sigma_delta(0.23))


def test_f2_full_size_launch_configuration():
    """f2 config: 10^5 particles x 7*10^4 turns with the recipe's programme, fused mode, in the
    launch configuration bench.py times; oracle on a seeded 2000-particle subsample.
    First 1000 turns: 1e-9 per particle.  Full run: the modulated pendulum has a chaotic layer
    (G31), so the per-particle gate (1e-6) and the moment / count comparison apply to
    the particles the ORACLE itself resolves: |fp64 - 80-bit twin| <= 1e-10 z_max."""
    tr, p = both()
    z0, d0 = wl.gaussian_bunch(F2["n"], F2["sigma_z"], F2["seed"])
    idx = wl.subsample_indices(F2["n"], 2000, F2["seed"])
    a, psi = wl.rf_programme(F2["turns"], F2["programme_seed"])
    sd = wl.matched_sigma_delta(F2["sigma_z"])
    g = oracle.derive(p)
    zo, do = oracle.track_programme(p, z0[idx], d0[idx], a[:1000], psi[:1000])
    zg, dg = gpu_programme(tr, z0, d0, a[:1000], psi[:1000])
    assert_particle_gate(p, z0[idx], d0[idx], zg[idx], dg[idx], zo, do, sd)
    zo, do = oracle.track_programme(p, z0[idx], d0[idx], a, psi)
    zl, _ = oracle.track_programme_ld(p, z0[idx], d0[idx], a, psi)
    resolved = np.abs(zo - zl.astype(np.float64)) / g["z_max"] <= 1e-10
    zg, dg = gpu_programme(tr, z0, d0, a, psi)
    zg, dg = zg[idx], dg[idx]
    ez, ed = np.abs(zg - zo) / g["z_max"], np.abs(dg - do) / sd
    print("f2 full: resolved %.4f; on them median ez %.2e max ez %.2e max ed %.2e"
          % (resolved.mean(), np.median(ez[resolved]), ez[resolved].max(), ed[resolved].max()))
    assert resolved.mean() >= 0.95
    assert ez[resolved].max() <= 1e-6 and ed[resolved].max() <= 1e-6
    mg = oracle.moments_of(p, zg[resolved], dg[resolved])
    mo = oracle.moments_of(p, zo[resolved], do[resolved])
    assert abs(mg["rms_z"] / mo["rms_z"] - 1) <= 1e-6 and abs(mg["rms_d"] / mo["rms_d"] - 1) <= 1e-6
    n_diff = count_mismatch_is_in_layer(p, zg[resolved], dg[resolved], zo[resolved], do[resolved])
    assert mg["n_in_bucket"] - mo["n_in_bucket"] in range(-n_diff, n_diff + 1)


# ================================================================== f4: slicing
def gpu_hist(tr, z, z_lo, z_hi, S):
    zt = dev(z)
    h = torch.full((S + 2,), -1, dtype=torch.int64, device="cuda")      # must be overwritten
    tr.slice_histogram(zt, zt.numel(), z_lo, z_hi, S, h, stream_ptr())
    torch.cuda.synchronize()
    return h.cpu().numpy().astype(np.uint64)


@pytest.mark.parametrize("S", [1, 7, 64, 1000, 8190, 8191, 50_000])
def test_slice_histogram_of_a_state_is_exact(S):
    """Same z on both sides -> identical integers, for every shared-memory replica count and for
    the global-atomics path (S > 8190)."""
    rng = np.random.default_rng(31 + S)
    z = rng.normal(0.0, 0.3, 200_003)
    z[:7] = [np.nan, np.inf, -np.inf, -0.7, 0.7, np.nextafter(0.7, 0), np.nextafter(-0.7, -1)]
    tr, _ = both()
    assert np.array_equal(gpu_hist(tr, z, -0.7, 0.7, S), oracle.slice_histogram(z, -0.7, 0.7, S))


@pytest.mark.parametrize("n", [1, 2, 2047, 2048, 2049, 4097, 1_000_001])
@pytest.mark.parametrize("offset", [0, 1])
def test_slice_histogram_sizes_around_a_tile_and_8_byte_alignment(n, offset):
    """The kernel walks tiles of 2048 particles with 16-byte loads: sizes around the tile, a
    ragged tail, and a z pointer that is only 8-byte aligned (view starting at element 1)."""
    rng = np.random.default_rng(77 + n)
    z = rng.normal(0.0, 0.3, n + offset)
    tr, _ = both()
    zt = dev(z)[offset:]
    assert zt.data_ptr() % 16 == 8 * offset
    h = torch.full((64 + 2,), -1, dtype=torch.int64, device="cuda")
    tr.slice_histogram(zt, n, -0.7, 0.7, 64, h, stream_ptr())
    torch.cuda.synchronize()
    assert np.array_equal(h.cpu().numpy().astype(np.uint64),
                          oracle.slice_histogram(z[offset:], -0.7, 0.7, 64))


def test_slice_index_is_branch_free_but_exact_on_special_values():
    """The slice index is computed without branches (floor through a magic-number add, selects
    for the two overflow bins): signed zeros at z_lo = 0, values whose scaled offset overflows
    32 bits in either direction, denormals, infinities and NaN must land where G29 puts them."""
    tr, _ = both()
    big = [1e300, -1e300, 3e9, -3e9, 2.0 ** 31, -2.0 ** 31, 2.0 ** 52, -2.0 ** 52, 5e-324, -5e-324,
           0.0, -0.0, np.inf, -np.inf, np.nan, 1.0, np.nextafter(1.0, 0), np.nextafter(0.0, 1)]
    z = np.array(big * 3 + [0.25, 0.5, 0.75], dtype=np.float64)
    for z_lo, z_hi, S in ((0.0, 1.0, 4), (-0.0, 1.0, 4), (-1.0, 0.0, 3), (0.0, 1e-300, 5), (-1e300, 1e300, 7),
                          (0.0, 1.0, 1 << 20)):
        assert np.array_equal(gpu_hist(tr, z, z_lo, z_hi, S), oracle.slice_histogram(z, z_lo, z_hi, S)), (z_lo, z_hi, S)


def test_slice_histogram_repeated_calls_on_one_tracker():
    """Every call zeroes the caller's histogram itself (CTA 0 publishes an epoch the other CTAs
    wait for): back-to-back calls of one tracker into different and into the same output, with
    sizes on both sides of one wave of CTAs, never see each other's counts."""
    tr, _ = both()
    rng = np.random.default_rng(5)
    outs = []
    for k, n in enumerate((3, 700_001, 5, 1_300_000, 1_300_000, 64)):
        z = rng.normal(0.0, 0.3, n)
        zt = dev(z)
        h = torch.full((64 + 2,), 12345, dtype=torch.int64, device="cuda")
        for _ in range(3 if k == 4 else 1):                # the same output three times in a row
            tr.slice_histogram(zt, n, -0.7, 0.7, 64, h, stream_ptr())
        outs.append((h, oracle.slice_histogram(z, -0.7, 0.7, 64), zt))
    torch.cuda.synchronize()
    for h, ho, _ in outs:
        assert np.array_equal(h.cpu().numpy().astype(np.uint64), ho)


def test_slice_edges_on_a_dyadic_grid_and_empty_input():
    tr, _ = both()
    S = 8
    edges = np.arange(S + 1) / 4.0 - 1.0                 # exactly representable, inv = 4 exactly
    z = np.concatenate([edges, np.nextafter(edges, -10), np.nextafter(edges, 10)])
    assert np.array_equal(gpu_hist(tr, z, -1.0, 1.0, S), oracle.slice_histogram(z, -1.0, 1.0, S))
    h = torch.full((S + 2,), 5, dtype=torch.int64, device="cuda")
    tr.slice_histogram(None, 0, -1.0, 1.0, S, h, stream_ptr())
    torch.cuda.synchronize()
    assert int(h.abs().sum()) == 0
    for bad in ((1.0, 1.0, 8), (1.0, -1.0, 8), (-1.0, 1.0, 0), (-1.0, float("nan"), 8)):
        with pytest.raises(lt.LongtrackError):
            tr.slice_histogram(h, 1, bad[0], bad[1], bad[2], h, stream_ptr())


def gpu_track_slices(tr, z0, d0, turns, grid, want_moments=False, zd=None):
    z_lo, z_hi, S = grid
    z, d = zd if zd is not None else (dev(z0), dev(d0))
    h = torch.full((turns, S + 2), -1, dtype=torch.int64, device="cuda")
    mom = moments_buffer(turns) if want_moments else None
    tr.track_slices(z, d, z.numel(), turns, z_lo, z_hi, S, h, mom, None, stream_ptr())
    torch.cuda.synchronize()
    out = (z.cpu().numpy(), d.cpu().numpy(), h.cpu().numpy().astype(np.uint64))
    if want_moments:
        out += (mom.cpu().numpy().view(lt.MOMENTS_DTYPE),)
    return out


def assert_histograms_match(p, z0, d0, hg, ho, grid, z_err):
    """Bit-exact (G29), except where a particle of the ORACLE's own state sits closer to a slice
    edge than the two sides' z differ.  `z_err` is this run's measured max |z_gpu - z_oracle| [m];
    the band is twice that (floored at a few ulp of the grid), nothing looser.  EVERY mismatching
    turn is re-tracked with the oracle and checked edge by edge: the cumulative sum of
    hg[t] - ho[t] up to bin b is the net number of particles that crossed the edge above bin b,
    and it may not exceed the number of oracle particles within the band of THAT edge."""
    z_lo, z_hi, S = grid
    assert hg.shape == ho.shape
    assert np.array_equal(hg.sum(axis=1), ho.sum(axis=1))
    bad = np.where((hg != ho).any(axis=1))[0]
    if bad.size == 0:
        return 0
    band = max(2.0 * z_err, 8.0 * np.finfo(np.float64).eps * max(abs(z_lo), abs(z_hi)))
    width = (z_hi - z_lo) / S
    zt, dt, done = np.array(z0, dtype=np.float64), np.array(d0, dtype=np.float64), 0
    for t in bad:                                        # every mismatching turn, in order
        zt, dt = oracle.track(p, zt, dt, int(t) + 1 - done)
        done = int(t) + 1
        crossed = np.cumsum(hg[t].astype(np.int64) - ho[t].astype(np.int64))[:-1]   # edges 0 .. S
        e = np.rint((zt - z_lo) / width)                 # nearest edge of every particle
        close = (np.abs(zt - (z_lo + e * width)) <= band) & (e >= 0) & (e <= S)
        allowed = np.bincount(e[close].astype(np.int64), minlength=S + 1)
        over = np.where(np.abs(crossed) > allowed)[0]
        assert over.size == 0, ("turn %d: edge %d crossed by %d, %d oracle particles within %.1e m"
                                % (t, over[0], crossed[over[0]], allowed[over[0]], band))
    return len(bad)


@pytest.mark.parametrize("S", [64, 1000, 20_000])
def test_track_slices_every_turn_graph_and_plain(S):
    tr, p = both()
    z0, d0 = wl.gaussian_bunch(20_001, 0.23, 32)
    grid = (-oracle.derive(p)["z_max"], oracle.derive(p)["z_max"], S)
    turns = 200                                          # 2 graph replays of 64 + a tail of 72
    zo, do, ho = oracle.track_slices(p, z0, d0, turns, *grid)
    _, _, mo = oracle.track_moments(p, z0, d0, turns)
    for graph in (1, 0):
        tr.set_option(lt.OPT_PER_TURN_GRAPH, graph)
        zg, dg, hg, mg = gpu_track_slices(tr, z0, d0, turns, grid, want_moments=True)
        assert_histograms_match(p, z0, d0, hg, ho, grid, np.abs(zg - zo).max())
        assert_moments_close(mg, mo)
        assert np.array_equal(mg["n_in_bucket"], mo["n_in_bucket"])
        assert_particle_gate(p, z0, d0, zg, dg, zo, do, wl.matched_sigma_delta(0.23))
    # without moments the state must be the same bits, and equal to the plain per-turn kernel's
    zh, dh, hh = gpu_track_slices(tr, z0, d0, turns, grid)
    zp, dp = gpu_track(tr, z0, d0, turns, "per_turn")
    assert np.array_equal(zh, zg) and np.array_equal(zh, zp) and np.array_equal(dh, dp)
    assert np.array_equal(hh, hg)


@pytest.mark.parametrize("integrator,ratio2", [("euler_cromer", 0.5), ("ruth4", 0.0)])
def test_track_slices_variants_and_misaligned_arrays(integrator, ratio2):
    tr, p = both(integrator, ratio2)
    n = 3001
    z0, d0 = wl.gaussian_bunch(n, 0.3, 33, ratio2=ratio2)
    grid = (-0.5, 0.6, 37)                               # particles fall below and above too
    zo, do, ho = oracle.track_slices(p, z0, d0, 70, *grid)
    assert ho[:, 0].sum() > 0 and ho[:, -1].sum() > 0
    buf = torch.zeros(2 * (n + 1) + 2, dtype=torch.float64, device="cuda")
    for off in (0, 1):                                   # 16-byte aligned, then offset by 8 bytes
        zt, dt = buf[off:off + n], buf[n + 2 + off:2 * n + 2 + off]
        zt.copy_(torch.from_numpy(z0)); dt.copy_(torch.from_numpy(d0))
        zg, dg, hg = gpu_track_slices(tr, None, None, 70, grid, zd=(zt, dt))
        assert_histograms_match(p, z0, d0, hg, ho, grid, np.abs(zg - zo).max())
        assert np.abs(zg - zo).max() / oracle.derive(p)["z_max"] <= 1e-9


def test_f4_full_size_launch_configuration():
    """f4 config: 10^7 particles x 1000 turns, 64 slices over the bucket, one launch per turn.
    Oracle: all 10^7 particles for the first 10 turns (histograms exact); at turn 1000 the
    oracle's histogram of the GPU's own final z (the reduction itself, exact) and a seeded 10^5
    subsample per particle; every turn's histogram must hold all n particles."""
    tr, p = both()
    n, turns = F4["n"], F4["turns"]
    z0, d0 = wl.gaussian_bunch(n, F4["sigma_z"], F4["seed"])
    grid = wl.slice_grid(F4)
    zo10, _, ho = oracle.track_slices(p, z0, d0, 10, *grid)
    zg10, _, hg10 = gpu_track_slices(tr, z0, d0, 10, grid)
    assert_histograms_match(p, z0, d0, hg10, ho, grid, np.abs(zg10 - zo10).max())
    zg, dg, hg = gpu_track_slices(tr, z0, d0, turns, grid)
    assert np.all(hg.sum(axis=1) == n)
    assert np.array_equal(hg[:10], hg10)                 # same bits whatever the call length
    assert np.array_equal(hg[-1], oracle.slice_histogram(zg, *grid))
    idx = wl.subsample_indices(n, 100_000, F4["seed"])
    zo, do = oracle.track(p, z0[idx], d0[idx], turns)
    assert_particle_gate(p, z0[idx], d0[idx], zg[idx], dg[idx], zo, do, wl.matched_sigma_delta(F4["sigma_z"]))


# ================================================================== f3: transverse plane
def gpu_transverse(tr, coords, z0, d0, turns, mode="fused", arrays=None):
    t = arrays if arrays is not None else [dev(c) for c in coords]
    z, d = (dev(z0), dev(d0)) if z0 is not None else (None, None)
    fn = tr.track_transverse_fused if mode == "fused" else tr.track_transverse_per_turn
    fn(t[0], t[1], t[2], t[3], z, d, t[0].numel(), turns, stream_ptr())
    torch.cuda.synchronize()
    out = tuple(c.cpu().numpy() for c in t)
    return out + ((z.cpu().numpy(), d.cpu().numpy()) if z is not None else (None, None))


def assert_transverse_gate(out, ref, coords, gate=1e-9):
    """|difference| <= gate * rms of the coordinate (the analogue of |dz|/z_max, |dd|/sigma_d)."""
    worst = 0.0
    for k in range(4):
        e = np.abs(out[k] - ref[k]).max() / coords[k].std()
        assert e <= gate, (k, e)
        worst = max(worst, e)
    return worst


@pytest.mark.parametrize("n_seg", [1, 2, 3, 4, 5, 9])
@pytest.mark.parametrize("mode", ["fused", "per_turn"])
def test_transverse_per_particle_1000_turns(n_seg, mode):
    """Every lattice length: constant-bank matrices (<= 4 segments) and the global-memory path."""
    tr, p = both()
    mats, twiss = wl.transverse_lattice(n_seg, 40 + n_seg)
    coords = wl.transverse_bunch(3001, 41, twiss)
    z0, d0 = wl.gaussian_bunch(3001, 0.23, 42)
    tr.set_transverse(mats)
    ref = oracle.track_transverse(p, mats, *coords, z0, d0, 1000)
    out = gpu_transverse(tr, coords, z0, d0, 1000, mode)
    worst = assert_transverse_gate(out, ref, coords)
    assert_particle_gate(p, z0, d0, out[4], out[5], ref[4], ref[5], wl.matched_sigma_delta(0.23))
    print("f3", n_seg, mode, "worst transverse error / rms: %.2e" % worst)


def test_transverse_small_integer_matrices_are_exact():
    """Integers stay exact under FMA and under separate roundings alike: equality, and a
    transposed or column-major reading of the matrix would fail."""
    tr, p = both()
    M0 = np.array([[1, 1, 0, 0], [0, 1, 0, 0], [0, 0, 1, 2], [3, 0, 0, 1]], dtype=float)
    M1 = np.array([[1, 0, 0, 1], [2, 1, 0, 0], [0, 0, 1, 0], [0, 1, 1, 1]], dtype=float)
    rng = np.random.default_rng(43)
    coords = tuple(rng.integers(-5, 6, 777).astype(float) for _ in range(4))
    tr.set_transverse([M0, M1])
    ref = oracle.track_transverse(p, [M0, M1], *coords, None, None, 6)
    for mode in ("fused", "per_turn"):
        out = gpu_transverse(tr, coords, None, None, 6, mode)
        assert all(np.array_equal(out[k], ref[k]) for k in range(4)), mode


@pytest.mark.parametrize("integrator,ratio2,split", [("leapfrog", 0.0, 0), ("leapfrog", 0.0, 1),
                                                     ("ruth4", 0.5, 0), ("euler_cromer", 0.0, 0)])
def test_transverse_modes_agree_bit_for_bit_and_longitudinal_variants(integrator, ratio2, split):
    """The transverse FMA sequence is the same in both modes; the longitudinal plane is the
    tracker's own map whether it rides in the transverse kernel or runs after it."""
    tr, p = both(integrator, ratio2)
    tr.set_option(lt.OPT_SPLIT_DRIFTS, split)
    mats, twiss = wl.transverse_lattice(3, 44)
    coords = wl.transverse_bunch(2049, 45, twiss)
    z0, d0 = wl.gaussian_bunch(2049, 0.23, 46, ratio2=ratio2)
    tr.set_transverse(mats)
    ref = oracle.track_transverse(p, mats, *coords, z0, d0, 150)
    a = gpu_transverse(tr, coords, z0, d0, 150, "fused")
    b = gpu_transverse(tr, coords, z0, d0, 150, "per_turn")
    assert all(np.array_equal(a[k], b[k]) for k in range(4))
    zf, df = gpu_track(tr, z0, d0, 150, "fused")
    zp, dp = gpu_track(tr, z0, d0, 150, "per_turn")
    assert np.array_equal(a[4], zf) and np.array_equal(a[5], df)
    assert np.array_equal(b[4], zp) and np.array_equal(b[5], dp)
    assert_transverse_gate(a, ref, coords)
    assert_particle_gate(p, z0, d0, a[4], a[5], ref[4], ref[5], wl.matched_sigma_delta(0.23))
    # transverse plane alone
    c = gpu_transverse(tr, coords, None, None, 150, "fused")
    assert all(np.array_equal(a[k], c[k]) for k in range(4))


def test_transverse_chunking_is_invisible_and_misaligned_arrays_work():
    tr, p = both()
    mats, twiss = wl.transverse_lattice(4, 47)
    n = 5001
    coords = wl.transverse_bunch(n, 48, twiss)
    z0, d0 = wl.gaussian_bunch(n, 0.23, 49)
    tr.set_transverse(mats)
    ref = gpu_transverse(tr, coords, z0, d0, 333, "fused")
    for chunk, item in ((50, 0), (1 << 22, 17), (128, 32)):
        tr.set_option(lt.OPT_CHUNK_TURNS, chunk)
        tr.set_option(lt.OPT_ITEM_TURNS, item)
        tr.set_option(lt.OPT_FUSED_MODE, lt.FUSED_PERSISTENT_DYNAMIC if item else lt.FUSED_AUTO)
        out = gpu_transverse(tr, coords, z0, d0, 333, "fused")
        assert all(np.array_equal(out[k], ref[k]) for k in range(6)), (chunk, item)
    buf = torch.zeros(4 * (n + 1) + 1, dtype=torch.float64, device="cuda")
    arrays = [buf[1 + k * (n + 1):1 + k * (n + 1) + n] for k in range(4)]
    assert arrays[0].data_ptr() % 16 == 8
    for a, c in zip(arrays, coords):
        a.copy_(torch.from_numpy(c))
    out = gpu_transverse(tr, coords, None, None, 333, "per_turn", arrays=arrays)
    assert all(np.array_equal(out[k], ref[k]) for k in range(4))
    # empty calls, and the lattice is required
    tr.track_transverse_fused(None, None, None, None, None, None, 0, 10, stream_ptr())
    tr.track_transverse_per_turn(arrays[0], arrays[1], arrays[2], arrays[3], None, None, n, 0, stream_ptr())
    tr.set_transverse(None)
    with pytest.raises(lt.LongtrackError):
        tr.track_transverse_fused(arrays[0], arrays[1], arrays[2], arrays[3], None, None, n, 1, stream_ptr())


@pytest.mark.parametrize("n_seg", [4, 6, 24, 25])
def test_transverse_every_ilp_shape_returns_the_same_bits(n_seg):
    """1, 2, 4 or 8 particles per lane (8: 256 threads and 220 registers per thread, the planner's
    choice from 3*10^5 particles on), static slots or the ticket queue, unrolled (<= 4 segments) or
    looped lattice, lattice in shared memory or in the kernel-parameter space (at most 24 segments;
    25 silently stays in shared memory): the arithmetic per particle is the same, so the six arrays
    must be bit-identical, on a ragged n that leaves the last group partly empty."""
    tr, p = both()
    mats, twiss = wl.transverse_lattice(n_seg, 60 + n_seg)
    n = 40_000 + 77
    coords = wl.transverse_bunch(n, 61, twiss)
    z0, d0 = wl.gaussian_bunch(n, 0.23, 62)
    tr.set_transverse(mats)
    ref = None
    for source in (1, 2):              # lattice in shared memory / in the kernel-parameter space (uniform registers)
        tr.set_option(lt.OPT_LATTICE_SOURCE, source)
        for ilp in (1, 2, 4, 8):
            for mode in (lt.FUSED_PERSISTENT_STATIC, lt.FUSED_PERSISTENT_DYNAMIC):
                tr.set_option(lt.OPT_FUSED_ILP, ilp)
                tr.set_option(lt.OPT_FUSED_MODE, mode)
                tr.set_option(lt.OPT_ITEM_TURNS, 37 if mode == lt.FUSED_PERSISTENT_DYNAMIC else 0)
                out = gpu_transverse(tr, coords, z0, d0, 211, "fused")
                assert tr.get_stat(lt.STAT_LAST_ILP) == ilp
                if ref is None:
                    ref = out
                assert all(np.array_equal(out[k], ref[k]) for k in range(6)), (source, ilp, mode)
    idx = np.arange(0, n, 7)
    o = oracle.track_transverse(p, mats, *(c[idx] for c in coords), z0[idx], d0[idx], 211)
    assert_transverse_gate(tuple(r[idx] for r in ref[:4]), o, tuple(c[idx] for c in coords))


def test_f3_full_size_launch_configuration():
    """f3 config: 10^6 particles x 10^4 turns x 4 segments + the longitudinal turn, fused, in the
    launch configuration bench.py times; oracle on a seeded 10^4 subsample.  The transverse map
    is linear (errors grow at most linearly in the 4*10^4 matrix applications): gate 1e-9 of the
    rms.  Longitudinal plane: 1e-6 on >= 99.9 % outside the layer, as configs[2] (G18)."""
    tr, p = both()
    mats, twiss = wl.transverse_lattice(F3["n_seg"], F3["lattice_seed"])
    n = F3["n"]
    coords = wl.transverse_bunch(n, F3["seed"], twiss)
    z0, d0 = wl.gaussian_bunch(n, F3["sigma_z"], F3["seed"] + 1)
    idx = wl.subsample_indices(n, 10_000, F3["seed"])
    tr.set_transverse(mats)
    sub = tuple(c[idx] for c in coords)
    ref = oracle.track_transverse(p, mats, *sub, z0[idx], d0[idx], F3["turns"])
    out = gpu_transverse(tr, coords, z0, d0, F3["turns"], "fused")
    worst = assert_transverse_gate(tuple(o[idx] for o in out[:4]), ref, sub)
    g = oracle.derive(p)
    ez = np.abs(out[4][idx] - ref[4]) / g["z_max"]
    ed = np.abs(out[5][idx] - ref[5]) / wl.matched_sigma_delta(F3["sigma_z"])
    print("f3 full: worst transverse %.2e; longitudinal median %.2e max %.2e" % (worst, np.median(ez), ez.max()))
    assert np.mean((ez <= 1e-6) & (ed <= 1e-6)) >= 0.999
    # per-turn mode at its bench size for a few turns (10^7 particles, all six arrays through HBM)
    n2 = F3["per_turn_n"]
    coords2 = wl.transverse_bunch(n2, F3["seed"] + 2, twiss)
    z2, d2 = wl.gaussian_bunch(n2, F3["sigma_z"], F3["seed"] + 3)
    idx2 = wl.subsample_indices(n2, 10_000, F3["seed"] + 2)
    out2 = gpu_transverse(tr, coords2, z2, d2, 20, "per_turn")
    sub2 = tuple(c[idx2] for c in coords2)
    ref2 = oracle.track_transverse(p, mats, *sub2, z2[idx2], d2[idx2], 20)
    assert_transverse_gate(tuple(o[idx2] for o in out2[:4]), ref2, sub2)
    assert np.abs(out2[4][idx2] - ref2[4]).max() / g["z_max"] <= 1e-9
