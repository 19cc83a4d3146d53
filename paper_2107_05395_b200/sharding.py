"""Batch sharding across ranks: every system is independent, so a
batch is cut into contiguous ranges of system indices, one per rank; each rank holds its OWN
interleaved array with its local batch size (element i of local system j at ``i*local + j``) and its own
copy of the factor handle.  There is no data-path collective.  Pure index arithmetic: no CUDA, no torch.
"""
from __future__ import annotations


def shard_bounds(total: int, world: int, rank: int):
    """[j0, j1) of rank ``rank`` when ``total`` systems are split over ``world`` ranks (strong scaling):
    contiguous, sizes differ by at most one, earlier ranks take the remainder."""
    if world < 1 or not (0 <= rank < world) or total < 0:
        raise ValueError("bad shard request")
    base, rem = divmod(total, world)
    j0 = rank * base + min(rank, rem)
    return j0, j0 + base + (1 if rank < rem else 0)


def weak_shard(per_rank: int, rank: int):
    """[j0, j1) of rank ``rank`` when every rank owns ``per_rank`` systems (weak scaling, bench.py)."""
    if per_rank < 0 or rank < 0:
        raise ValueError("bad shard request")
    return rank * per_rank, (rank + 1) * per_rank


def max_over_ranks_ms(local_ms: float, world: int, all_reduce_max=None) -> float:
    """Job time = the slowest rank's device time; ``all_reduce_max(x) -> max over ranks`` (identity for world 1)."""
    if world <= 1 or all_reduce_max is None:
        return float(local_ms)
    return float(all_reduce_max(float(local_ms)))
