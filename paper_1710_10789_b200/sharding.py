"""Host logic of the multi-GPU path: which cubes a rank owns.

Cubes are independent and the result is additive, so the grid is cut into contiguous z-slabs, one per
rank; a rank reads the k-planes z_lo .. z_hi (the last one is its halo, wrapping to plane 0)."""
from __future__ import annotations


def z_slab(rank: int, world: int, n3: int):
    """Cube planes [z_lo, z_hi) of `rank`: contiguous, disjoint, covering 0..n3, sizes differing by <= 1."""
    if not (0 <= rank < world) or n3 < 1:
        raise ValueError("bad rank/world/n3")
    return (n3 * rank) // world, (n3 * (rank + 1)) // world


def planes_read(rank: int, world: int, n3: int):
    """k-planes a rank reads: its slab plus one halo plane (periodic)."""
    lo, hi = z_slab(rank, world, n3)
    return [z % n3 for z in range(lo, hi + 1)] if hi > lo else []
