"""Zone sharding for more than one GPU: zones are independent
networks, so rank r integrates one contiguous range of the
global batch with its own replica of the network tables; there is no exchange
step and no collective on the data path."""
from __future__ import annotations


def zone_shard(total_zones: int, rank: int, world: int) -> tuple[int, int]:
    """[lo, hi) of rank's zones: contiguous, sizes differ by at most one."""
    if not (0 <= rank < world):
        raise ValueError("rank out of range")
    base, extra = divmod(int(total_zones), int(world))
    lo = rank * base + min(rank, extra)
    return lo, lo + base + (1 if rank < extra else 0)
