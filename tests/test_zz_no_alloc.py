"""lt_moments_now_static: the entry point for callers that cannot allocate device memory.

Who that is: a tracking service whose own pool took the whole GPU at start-up (the driver's
allocator has nothing left to give), a turn-by-turn monitoring loop that must neither stall on
nor fail in an allocation in the middle of a run, a plug-in that its host application forbids to
touch the CUDA heap.  lt_moments_now allocates its partial-sum buffer on first use; the static
variant keeps the partial sums in a fixed 128 KB array inside the library instead, accepts at
most STATIC_MAX_PARTICLES particles, and shares that array between all callers of the process.

The GPU test compares it with lt_moments_now (the existing, allocating path) on the same device
arrays, on two calls in a row -- the second on a different and SMALLER state, so the array still
holds records of the first call that the second must not read.  Moments at the 1e-6 gate of the
other moment tests (G14), sums relative 1e-12, the membership count exactly.

This file is named test_zz_* so that pytest collects it last: with -x a failure here hides no
other test.  It passes alone in a fresh process (the first static call then does the per-device
address look-up) and after the rest of the suite.
"""
import numpy as np
import pytest

import __graft_entry__ as entry


@pytest.fixture(scope="module")
def lt():
    entry.build()
    from paper_1610_05801_b200 import longtrack
    return longtrack


def test_size_beyond_the_fixed_capacity_is_refused(lt):
    """No GPU needed: the size check comes before any CUDA call, and names its reason."""
    from paper_1610_05801_b200 import workloads as wl
    tr = lt.Tracker(wl.RING)
    assert lt.STATIC_MAX_PARTICLES == 1 << 24
    with pytest.raises(lt.LongtrackError) as e:
        # pointers are never dereferenced: the call is refused on n alone
        tr.moments_now_static(8, 8, lt.STATIC_MAX_PARTICLES + 1, 8, None, 0)
    assert e.value.code == lt.E_CAPACITY
    assert "capacity" in lt.strerror(lt.E_CAPACITY)
    with pytest.raises(lt.LongtrackError) as e:
        tr.moments_now_static(8, 8, 10, None, None, 0)          # no output at all
    assert e.value.code == lt.E_NULL


def _both_paths(lt, tr, z, d, n, st):
    import torch
    out = []
    for call in (tr.moments_now, tr.moments_now_static):
        mom = torch.zeros(lt.MOMENTS_DTYPE.itemsize, dtype=torch.uint8, device="cuda")
        sums = torch.zeros(lt.SUMS_DTYPE.itemsize, dtype=torch.uint8, device="cuda")
        call(z, d, n, mom, sums, st)
        torch.cuda.synchronize()
        out.append((mom.cpu().numpy().view(lt.MOMENTS_DTYPE)[0],
                    sums.cpu().numpy().view(lt.SUMS_DTYPE)[0]))
    return out


def _assert_same(ref, new, n):
    (m0, s0), (m1, s1) = ref, new
    assert int(m1["n_in_bucket"]) == int(m0["n_in_bucket"])            # integer work: exact
    assert s1["n_in_bucket"] == s0["n_in_bucket"] and s1["n"] == s0["n"] == float(n)
    tol = 1e-6                                                          # DESIGN.md G14 gate
    assert abs(m1["mean_z"] - m0["mean_z"]) <= tol * m0["rms_z"]
    assert abs(m1["mean_d"] - m0["mean_d"]) <= tol * m0["rms_d"]
    assert abs(m1["rms_z"] / m0["rms_z"] - 1) <= tol
    assert abs(m1["rms_d"] / m0["rms_d"] - 1) <= tol
    assert abs(m1["cov_zd"] - m0["cov_zd"]) <= tol * m0["rms_z"] * m0["rms_d"]
    for k in ("sum_zz", "sum_dd"):                                      # positive sums: only the
        assert abs(s1[k] / s0[k] - 1) <= 1e-12, k                       # partition differs


@pytest.mark.gpu
def test_static_scratch_matches_the_allocating_path_on_two_calls_in_a_row(lt):
    import torch
    from paper_1610_05801_b200 import workloads as wl

    torch.cuda.set_device(0)
    st = torch.cuda.current_stream().cuda_stream
    tr = lt.Tracker(wl.RING)
    # call 1: 100 003 particles = 12 full 8192-particle records and a ragged 13th; the hollow
    # bunch of configs[1] has particles on both sides of the separatrix, so the count is not n
    z0, d0 = wl.make_bunch(wl.CONFIGS[1], n=100_003)
    z = torch.from_numpy(z0).cuda()
    d = torch.from_numpy(d0).cuda()
    ref, new = _both_paths(lt, tr, z, d, z.numel(), st)
    assert 0 < int(ref[0]["n_in_bucket"]) < z.numel()
    _assert_same(ref, new, z.numel())

    # call 2, straight after: another state, fewer records -- what call 1 left in records 3..12
    # of the shared array is stale and must not leak into the result
    tr.track_fused(z, d, z.numel(), 300, st)
    n2 = 20_001
    z2, d2 = z[5:5 + n2], d[5:5 + n2]              # 8-byte aligned only: offset of 5 doubles
    ref2, new2 = _both_paths(lt, tr, z2, d2, n2, st)
    _assert_same(ref2, new2, n2)
    assert int(new2[0]["n_in_bucket"]) != int(new[0]["n_in_bucket"])

    # a tracker that has never run anything else: the static call takes no device memory
    tr3 = lt.Tracker(wl.RING)
    mom = torch.zeros(lt.MOMENTS_DTYPE.itemsize, dtype=torch.uint8, device="cuda")
    torch.cuda.synchronize()
    free_before, _ = torch.cuda.mem_get_info()
    tr3.moments_now_static(z2, d2, n2, mom, None, st)
    torch.cuda.synchronize()
    free_after, _ = torch.cuda.mem_get_info()
    assert free_after >= free_before
    assert int(mom.cpu().numpy().view(lt.MOMENTS_DTYPE)[0]["n_in_bucket"]) == \
        int(ref2[0]["n_in_bucket"])
    # n == 0 and the largest accepted size are both fine for the argument checks
    tr3.moments_now_static(z2, d2, 0, mom, None, st)
    torch.cuda.synchronize()
    assert float(mom.cpu().numpy().view(lt.MOMENTS_DTYPE)[0]["rms_z"]) == 0.0
