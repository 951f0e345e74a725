"""Work sharding for N > 1 GPUs: maps are independent problems, no data-path collective."""
from __future__ import annotations


def shard_range(total: int, world: int, rank: int) -> range:
    """Contiguous, balanced split of ``total`` independent units over ``world`` ranks (first ranks get the remainder)."""
    if not (0 <= rank < world):
        raise ValueError("rank out of range")
    base, rem = divmod(total, world)
    lo = rank * base + min(rank, rem)
    return range(lo, lo + base + (1 if rank < rem else 0))
