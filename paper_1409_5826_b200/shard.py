"""Zone sharding for more than one GPU: zones are independent
networks, so rank r integrates one contiguous range of the
global batch with its own replica of the network tables; there is no exchange
step and no collective on the data path.  The only collectives are the barrier
and the timing reduction around the timed region (bench.py).

Zones "may require varying numbers of integration steps" (fn. 1, which
leaves the load balance open): on a hydro grid whose hot zones are neighbours a
contiguous split gives one rank all the long zones.  zone_shard_balanced deals the
zones out by temperature instead (the proxy the launch order inside one GPU uses
too); it is host-side index arithmetic, still without a collective."""
from __future__ import annotations

import numpy as np


def zone_shard(total_zones: int, rank: int, world: int) -> tuple[int, int]:
    """[lo, hi) of rank's zones: contiguous, sizes differ by at most one."""
    if not (0 <= rank < world):
        raise ValueError("rank out of range")
    base, extra = divmod(int(total_zones), int(world))
    lo = rank * base + min(rank, extra)
    return lo, lo + base + (1 if rank < extra else 0)


def zone_shard_balanced(T9, rank: int, world: int) -> np.ndarray:
    """Indices (ascending, int64) of rank's zones when the batch is dealt out by falling
    T9: the zones are ranked hottest first (ties and NaN in caller order, NaN last) and
    handed round the ranks in a snake -- 0, 1, .., W-1, W-1, .., 1, 0, 0, 1, .. -- so that
    every rank gets one zone of each group of W neighbours in the ranking and the
    systematic "first pick is hotter" bias of a plain round robin cancels between
    consecutive rounds.  Every rank computes the same deal from the same T9; the shards
    partition range(len(T9)) and their sizes differ by at most one.  Gather the inputs
    with the returned indices and scatter the outputs back with them."""
    if not (0 <= rank < world):
        raise ValueError("rank out of range")
    T9 = np.asarray(T9, dtype=np.float64).reshape(-1)
    key = np.where(np.isnan(T9), -np.inf, T9)
    ranking = np.argsort(-key, kind="stable")
    pos = np.arange(T9.size)
    rnd, slot = pos // world, pos % world
    owner = np.where(rnd % 2 == 0, slot, world - 1 - slot)
    return np.sort(ranking[owner == rank]).astype(np.int64)


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
