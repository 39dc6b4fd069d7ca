"""Host-side sharding of the path over ranks (one process per GPU).  Output tiles are independent, so
the path shards over token rows (M) or weight columns (N) with no data-path collective and bit-identical
results; the only cross-rank traffic is the timing reduction (max over ranks) in bench.py.
"""
from __future__ import annotations


def shard_rows(M: int, world: int, rank: int) -> tuple[int, int]:
    """Contiguous [begin, end) row range of rank `rank`; sizes differ by at most one row."""
    base, rem = divmod(M, world)
    begin = rank * base + min(rank, rem)
    return begin, begin + base + (1 if rank < rem else 0)


def shard_cols(N: int, world: int, rank: int, align: int = 128) -> tuple[int, int]:
    """Contiguous [begin, end) column range, boundaries on multiples of `align` (the 128-column weight
    panel / 16-byte TMA pitch) except the last; later ranks may be empty for tiny N."""
    units = (N + align - 1) // align
    b, e = shard_rows(units, world, rank)
    return min(b * align, N), min(e * align, N)


def aggregate_throughput(units_per_rank: list[float], ms_per_rank: list[float]) -> float:
    """Whole-job throughput: all units processed / the slowest rank's time (units per second)."""
    return sum(units_per_rank) / (max(ms_per_rank) * 1e-3)
