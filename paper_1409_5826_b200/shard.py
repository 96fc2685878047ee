"""Zone sharding for more than one GPU: zones are independent
networks, so rank r integrates one contiguous range of the
global batch with its own replica of the network tables; there is no exchange
step and no collective on the data path.  The only collectives are the barrier
and the timing reduction around the timed region (bench.py)."""
from __future__ import annotations


def zone_shard(total_zones: int, rank: int, world: int) -> tuple[int, int]:
    """[lo, hi) of rank's zones: contiguous, sizes differ by at most one."""
    if not (0 <= rank < world):
        raise ValueError("rank out of range")
    base, extra = divmod(int(total_zones), int(world))
    lo = rank * base + min(rank, extra)
    return lo, lo + base + (1 if rank < extra else 0)


def reduce_job(times, counts, device=None):
    """Whole-job figures from per-rank ones: element-wise MAX over ranks of
    ``times`` (the job is as slow as its slowest rank) and SUM over ranks of
    ``counts`` (units processed).  Works on any initialised torch.distributed
    backend (nccl on the GPUs, gloo in the CPU tests); identity without one."""
    import torch
    import torch.distributed as dist

    t = torch.tensor([float(x) for x in times], dtype=torch.float64, device=device)
    c = torch.tensor([float(x) for x in counts], dtype=torch.float64, device=device)
    if dist.is_available() and dist.is_initialized() and dist.get_world_size() > 1:
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        dist.all_reduce(c, op=dist.ReduceOp.SUM)
    return t.tolist(), c.tolist()
