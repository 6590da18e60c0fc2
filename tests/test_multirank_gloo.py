"""Host logic of the N > 1 path on CPU: world_size-2 gloo processes.  Each rank takes its z-slab
(paper_1710_10789_b200.sharding), produces the additive share of its cubes -- here with the oracle's
cube_range, since no GPU exists on this box -- the shares are all-reduced exactly as bench.py does with
the fp64 partials, and the sum must equal the single-process result."""
import os
import socket

import numpy as np
import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from paper_1710_10789_b200 import sharding, workloads as wl


def test_z_slabs_partition_the_grid():
    for n3 in (1, 2, 5, 7, 128, 192):
        for world in (1, 2, 3, 4, 8):
            slabs = [sharding.z_slab(r, world, n3) for r in range(world)]
            assert slabs[0][0] == 0 and slabs[-1][1] == n3
            assert all(a[1] == b[0] for a, b in zip(slabs, slabs[1:]))
            sizes = [b - a for a, b in slabs]
            assert max(sizes) - min(sizes) <= 1
    assert sharding.planes_read(1, 2, 4) == [2, 3, 0]      # halo wraps
    with pytest.raises(ValueError):
        sharding.z_slab(2, 2, 4)


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, out):
    import oracle
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    nk, nb, norb, nE = (6, 5, 7), 2, 3, 150
    E, W = wl.random_bands(nk, nb, norb, seed=11)
    om = wl.omega_grid(-1.2, 1.3, nE)
    z_lo, z_hi = sharding.z_slab(rank, world, nk[2])
    plane = nk[0] * nk[1]
    share = oracle.tetra_dos(E, W, nk, om, cube_range=(z_lo * plane, z_hi * plane))
    part = torch.from_numpy(np.stack([share["dos"], share["nos"]]))
    cnt = torch.tensor([share["n_tb"], share["n_eval"]])
    dist.all_reduce(part)
    dist.all_reduce(cnt)
    ms = torch.tensor([float(rank + 1)], dtype=torch.float64)
    dist.all_reduce(ms, op=dist.ReduceOp.MAX)       # bench.py's max-over-ranks timing
    if rank == 0:
        full = oracle.tetra_dos(E, W, nk, om)
        ok = (np.allclose(part[0].numpy(), full["dos"], rtol=1e-12, atol=1e-15)
              and np.allclose(part[1].numpy(), full["nos"], rtol=1e-12, atol=1e-15)
              and int(cnt[0]) == full["n_tb"] and int(cnt[1]) == full["n_eval"] and float(ms) == world)
        out.put(bool(ok))
    dist.destroy_process_group()


def test_two_ranks_sum_of_slab_shares_equals_full_result():
    ctx = mp.get_context("spawn")
    out = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, 2, port, out)) for r in range(2)]
    for p in procs:
        p.start()
    for p in procs:
        p.join(120)
        assert p.exitcode == 0
    assert out.get(timeout=5) is True
