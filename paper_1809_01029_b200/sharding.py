"""Data-parallel sharding of a state set over ranks (one process per GPU).

States are independent (one state per work-item; no coupling in Eqs. 1-9), so the path shards
with no data-path collective: every rank owns a contiguous range of states whose start is a multiple of the
layout tile, creates its own mechanism handle (tables are < 2 MB) and writes its own outputs.  The only
collective is the MAX-reduction of the per-rank timings in bench.py.
"""
from __future__ import annotations


def shard_range(n_states: int, rank: int, world: int, tile: int = 1):
    """Contiguous [begin, end) of `rank`; begins are multiples of `tile`; the union covers [0, n_states)."""
    if world < 1 or not 0 <= rank < world or tile < 1 or n_states < 0:
        raise ValueError("bad shard arguments")
    n_tiles = (n_states + tile - 1) // tile
    per, extra = divmod(n_tiles, world)
    t0 = rank * per + min(rank, extra)
    t1 = t0 + per + (1 if rank < extra else 0)
    return min(t0 * tile, n_states), min(t1 * tile, n_states)


def weak_scaling_offset(n_per_rank: int, rank: int) -> int:
    """First global state index of `rank` when every rank owns `n_per_rank` states (bench.py, scaling = weak)."""
    return rank * n_per_rank
