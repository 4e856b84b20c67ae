"""Multi-GPU sharding of the stream set ("one state per thread to
avoid synchronization").

Streams are independent and the seeding is position independent (stream i of a job is seeded with
`seed + i`, X = G^(seed + i), reading c-7), so a job of N streams is split into contiguous stream
ranges, one per rank; rank g creates its handle with `rlxpp_create(count_g, seed + first_g, p)` and
writes its own slab (stream-major) or column block (interleaved) of the output.  There is NO
data-path collective; the only communication is the timing reduction of bench.py (max over ranks).

Host logic only -- no RANLUX++ arithmetic here.
"""
from typing import Tuple


def stream_range(rank: int, world: int, n_streams: int) -> Tuple[int, int]:
    """(first, count) of the contiguous range of rank `rank` when `n_streams` streams are split over
    `world` ranks; the remainder goes to the lowest ranks, so counts differ by at most one."""
    if world < 1 or not 0 <= rank < world:
        raise ValueError(f"rank {rank} outside world {world}")
    if n_streams < 0:
        raise ValueError("n_streams < 0")
    base, extra = divmod(n_streams, world)
    first = rank * base + min(rank, extra)
    return first, base + (1 if rank < extra else 0)


def rank_seed(seed: int, first: int) -> int:
    """Seed argument of rlxpp_create for a rank whose range starts at stream `first` (64-bit wrap,
    as the library adds the stream index modulo 2^64)."""
    return (seed + first) & (2**64 - 1)


def max_over_ranks(value: float, dist=None, device=None) -> float:
    """The job's time is the slowest rank's: all-reduce MAX over the default process group (NCCL on
    GPUs, gloo in the CPU tests).  With no process group it is the value itself."""
    if dist is None or not dist.is_initialized() or dist.get_world_size() == 1:
        return float(value)
    import torch
    t = torch.tensor([float(value)], dtype=torch.float64, device=device if device is not None else "cpu")
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())
