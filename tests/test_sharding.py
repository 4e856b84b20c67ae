"""N > 1 path on CPU: two `gloo` ranks run the host logic bench.py uses under torchrun
(paper_2106_02504_b200/shard.py): contiguous stream ranges, per-rank seed offsets, max-over-ranks
timing.  Each rank produces its shard with the oracle (standing in for its GPU: the sharding is
what is under test) and the gathered shards must equal ONE generator over all streams -- streams
are independent and the seeding is position independent, so there is
no data-path collective to test, only that the ranges tile the job exactly."""
import os
import socket

import numpy as np
import pytest

from paper_2106_02504_b200 import inputs, shard


def test_stream_range_tiles_the_job_exactly():
    for n in (0, 1, 5, 128, 1000, 2**20 + 64):
        for world in (1, 2, 3, 8):
            got = [shard.stream_range(r, world, n) for r in range(world)]
            assert got[0][0] == 0 and sum(c for _, c in got) == n
            for (f0, c0), (f1, _) in zip(got, got[1:]):
                assert f0 + c0 == f1
            counts = [c for _, c in got]
            assert max(counts) - min(counts) <= 1
    with pytest.raises(ValueError):
        shard.stream_range(2, 2, 10)
    assert shard.rank_seed(2**64 - 1, 3) == 2  # the library adds stream indices modulo 2^64
    assert shard.max_over_ranks(1.5) == 1.5   # no process group: identity


def _worker(rank, world, port, n_total, per, p, seed, tmpdir):
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    import torch
    import torch.distributed as dist
    import oracle
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        first, count = shard.stream_range(rank, world, n_total)
        seeds = inputs.seeds(count, shard.rank_seed(seed, first))
        mine = oracle.streams(seeds, p, per, want=("doubles",), nthreads=1)["doubles"]
        # gather the shards on rank 0 (test plumbing; the product path has no such collective)
        sizes = [torch.zeros(1, dtype=torch.int64) for _ in range(world)]
        dist.all_gather(sizes, torch.tensor([count], dtype=torch.int64))
        pad = int(max(s.item() for s in sizes))
        buf = torch.zeros((pad, per), dtype=torch.float64)
        buf[:count] = torch.from_numpy(mine)
        parts = [torch.zeros((pad, per), dtype=torch.float64) for _ in range(world)]
        dist.all_gather(parts, buf)
        slowest = shard.max_over_ranks(10.0 + rank, dist)
        if rank == 0:
            whole = np.concatenate([parts[r][: int(sizes[r].item())].numpy() for r in range(world)])
            np.save(os.path.join(tmpdir, "whole.npy"), whole)
            np.save(os.path.join(tmpdir, "slowest.npy"), np.array([slowest]))
    finally:
        dist.destroy_process_group()


def test_two_gloo_ranks_reproduce_one_generator(tmp_path, oracle):
    import torch.multiprocessing as mp
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        port = s.getsockname()[1]
    world, n_total, per, p, seed = 2, 37, 60, 2048, 11  # odd split: 19 + 18 streams
    mp.spawn(_worker, args=(world, port, n_total, per, p, seed, str(tmp_path)), nprocs=world, join=True)
    whole = np.load(tmp_path / "whole.npy")
    ref = oracle.streams(inputs.seeds(n_total, seed), p, per, want=("doubles",), nthreads=2)["doubles"]
    assert whole.shape == ref.shape
    assert np.array_equal(whole.view(np.uint64), ref.view(np.uint64))
    assert float(np.load(tmp_path / "slowest.npy")[0]) == 11.0  # max over ranks of 10 + rank


def test_bench_rank_logic_for_eight_ranks():
    """bench.py --gpus 8 on the host side (the pool has one GPU per lease: no scaling curve is measured).  Weak scaling:
    every rank owns its own 2^20 streams, the ranges tile the 8 x 2^20-stream job, rank g's seed argument is the job's
    seed + its first stream, and `value` is all ranks' units over the slowest rank's time."""
    import bench
    world, per_gpu = 8, 1 << 20
    lay = [bench.job_layout(r, world, per_gpu) for r in range(world)]
    assert [f for f, _, _ in lay] == [r * per_gpu for r in range(world)]
    assert all(c == per_gpu for _, c, _ in lay)
    assert [s for _, _, s in lay] == [1 + r * per_gpu for r in range(world)]  # seeds 1 .. 8 x 2^20, no overlap, no gap
    assert bench.job_layout(3, 8, 1 << 20, seed=2**64 - 5)[2] == (2**64 - 5 + 3 * (1 << 20)) % 2**64
    units = per_gpu * 1536
    assert bench.whole_job_rate(units, world, 2.0) == 8 * units / 2e-3
    assert bench.whole_job_rate(units, 1, 2.0) * 8 == bench.whole_job_rate(units, 8, 2.0)  # 100 % weak scaling = 8 x
    sp = bench.spread([3.0, 1.0, 2.0, 10.0])
    assert (sp["min"], sp["median"], sp["max"], sp["n"]) == (1.0, 2.5, 10.0, 4)


def _max_worker(rank, world, port, tmpdir):
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    import torch.distributed as dist
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        slowest = shard.max_over_ranks(2.0 + 0.125 * ((rank * 5) % world), dist)
        if rank == world - 1:
            np.save(os.path.join(tmpdir, "slowest8.npy"), np.array([slowest]))
    finally:
        dist.destroy_process_group()


def test_eight_gloo_ranks_agree_on_the_slowest():
    """The only communication of the multi-GPU bench: the job's time is the MAX over ranks (here 8 gloo ranks)."""
    import tempfile
    import torch.multiprocessing as mp
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        port = s.getsockname()[1]
    with tempfile.TemporaryDirectory() as d:
        mp.spawn(_max_worker, args=(8, port, d), nprocs=8, join=True)
        assert float(np.load(os.path.join(d, "slowest8.npy"))[0]) == 2.0 + 0.125 * 7
