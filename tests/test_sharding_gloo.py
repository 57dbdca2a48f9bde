"""N > 1 path on CPU: world_size-2 gloo processes.

The path shards by contiguous particle ranges with NO data-path collective (particles are
independent).  What the ranks do exchange is host logic, covered here
without a GPU:
  - workloads.shard_range partitions [0, n) exactly, for every ragged n;
  - per-turn moments of a sharded bunch = ONE SUM all-reduce of the raw, additive lt_sums
    records, then lt_moments_from_sums (the library's host finaliser) -- compared with the
    oracle's moments of the unsharded bunch;
  - bench.py's timing reduction (MAX over ranks) and whole-job value.
Each rank forms its raw sums with numpy on its shard (on a GPU box the per-turn kernel writes the
same lt_sums records; tests/test_gpu_parity.py::test_sums_output_and_host_finalisation).
"""
import os
import socket
import sys

import numpy as np
import pytest

torch = pytest.importorskip("torch")
import torch.distributed as dist  # noqa: E402
import torch.multiprocessing as mp  # noqa: E402

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
WORLD = 2
N, TURNS = 10_007, 12          # ragged: N % WORLD != 0


def _free_port() -> int:
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank: int, port: int, out_dir: str) -> None:
    sys.path.insert(0, ROOT)
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank),
                      WORLD_SIZE=str(WORLD))
    import oracle
    from paper_1610_05801_b200 import longtrack as lt
    from paper_1610_05801_b200 import workloads as wl
    dist.init_process_group("gloo", rank=rank, world_size=WORLD)
    try:
        cfg = wl.CONFIGS[3]
        z0, d0 = wl.make_bunch(cfg, n=N)                 # every rank generates the same bunch ...
        lo, hi = wl.shard_range(N, rank, WORLD)          # ... and keeps its own range
        p = oracle.make_params(wl.RING, "leapfrog")
        z, d = z0[lo:hi].copy(), d0[lo:hi].copy()
        sums = np.zeros(TURNS, dtype=lt.SUMS_DTYPE)
        for t in range(TURNS):                           # the shard's trajectory, turn by turn
            z, d = oracle.track(p, z, d, 1)
            sums["n"][t] = z.size
            sums["sum_z"][t], sums["sum_zz"][t] = z.sum(), (z * z).sum()
            sums["sum_d"][t], sums["sum_dd"][t] = d.sum(), (d * d).sum()
            sums["sum_zd"][t] = (z * d).sum()
            sums["n_in_bucket"][t] = oracle.bucket_count(p, z, d)
        flat = torch.from_numpy(sums.view(np.float64).copy())
        dist.all_reduce(flat, op=dist.ReduceOp.SUM)      # the ONE collective of the sharded run
        total = flat.numpy().view(lt.SUMS_DTYPE)
        mom = lt.moments_from_sums(total)
        # bench.py's reductions: device time = MAX over ranks, value = all ranks' units / that
        t_local = torch.tensor([1.0 + rank], dtype=torch.float64)
        dist.all_reduce(t_local, op=dist.ReduceOp.MAX)
        sizes = torch.tensor([hi - lo], dtype=torch.int64)
        dist.all_reduce(sizes, op=dist.ReduceOp.SUM)
        if rank == 0:
            np.save(os.path.join(out_dir, "mom.npy"), mom)
            np.save(os.path.join(out_dir, "misc.npy"),
                    np.array([float(t_local.item()), float(sizes.item())]))
    finally:
        dist.destroy_process_group()


def test_shard_range_partitions_exactly():
    sys.path.insert(0, ROOT)
    from paper_1610_05801_b200 import workloads as wl
    for n in (0, 1, 2, 7, 100_003):
        for world in (1, 2, 3, 8):
            edges = [wl.shard_range(n, r, world) for r in range(world)]
            assert edges[0][0] == 0 and edges[-1][1] == n
            assert all(a[1] == b[0] for a, b in zip(edges, edges[1:]))
            sizes = [hi - lo for lo, hi in edges]
            assert max(sizes) - min(sizes) <= 1


def test_two_rank_moments_equal_the_unsharded_oracle(tmp_path):
    sys.path.insert(0, ROOT)
    import oracle
    from paper_1610_05801_b200 import workloads as wl
    mp.spawn(_worker, args=(_free_port(), str(tmp_path)), nprocs=WORLD, join=True)
    mom = np.load(tmp_path / "mom.npy")
    t_max, n_total = np.load(tmp_path / "misc.npy")
    assert t_max == 2.0 and n_total == N
    p = oracle.make_params(wl.RING, "leapfrog")
    z0, d0 = wl.make_bunch(wl.CONFIGS[3], n=N)
    _, _, ref = oracle.track_moments(p, z0, d0, TURNS)
    for k in ("rms_z", "rms_d"):
        assert np.max(np.abs(mom[k] / ref[k] - 1)) <= 1e-9, k
    assert np.max(np.abs(mom["mean_z"] - ref["mean_z"])) <= 1e-9 * ref["rms_z"][0]
    assert np.max(np.abs(mom["mean_d"] - ref["mean_d"])) <= 1e-9 * ref["rms_d"][0]
    assert np.array_equal(mom["n_in_bucket"], ref["n_in_bucket"])
