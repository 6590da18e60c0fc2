"""The N > 1 step of the hot path: every rank computes the additive fp64
share of its z-slab of cubes, ONE all-reduce sums the shares (the path's only exchange step), rank-local finalize.
bench.py and tests/test_multirank_gpu.py run exactly this function; only the `all_reduce` callable differs (NCCL on
the device in bench.py, a host round trip over gloo where a box has a single GPU)."""
from __future__ import annotations

from . import sharding


def sharded_step(plan, E, W, omega, nk3: int, rank: int, world: int, part, dos, nos, all_reduce, layout: int = 0,
                 stream=None, slab_local: bool = False):
    """One pass of the path on `world` ranks.  `part` is this rank's device tensor float64[3][norb][nE] (scratch),
    `all_reduce(part)` must sum it over the ranks in place (and order itself after the work enqueued on `stream`).
    slab_local: E and W hold only this rank's k-planes z_lo .. z_hi (sharding.planes_read: slab + halo plane) instead
    of the whole grid."""
    z_lo, z_hi = sharding.z_slab(rank, world, nk3)
    if slab_local and z_hi > z_lo:
        plan.tetra_dos_partial_slab(E, W, omega, z_lo, z_hi, part, layout=layout, stream=stream)
    else:
        plan.tetra_dos_partial(E, W, omega, z_lo, z_hi, part, layout=layout, stream=stream)
    all_reduce(part)
    plan.tetra_dos_finalize(part, int(omega.shape[0]), dos, nos, stream=stream)
