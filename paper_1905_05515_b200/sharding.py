"""Work split for more than one GPU: independent time frames / sectors, no data-path collective."""
from __future__ import annotations


def shard_units(n_units: int, world_size: int, rank: int) -> list[int]:
    """Round-robin assignment of independent units (time frames, or the 36 sectors of one frame) to ranks."""
    if world_size < 1 or not (0 <= rank < world_size):
        raise ValueError("bad rank / world_size")
    return list(range(rank, n_units, world_size))
