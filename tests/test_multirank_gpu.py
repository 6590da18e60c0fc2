"""The N > 1 PRODUCT path on the one GPU a box has: two ranks, both on cuda:0, each runs tetra_dos_partial on its own
z-slab through the C ABI, the fp64 shares are all-reduced (gloo, over the host -- NCCL needs one GPU per rank), every
rank finalizes and compares with the oracle at the north-star tolerances.  The step is paper_1710_10789_b200.multigpu.
sharded_step, the function bench.py runs under torchrun; the ranks do not wait on one another's kernels, only on the
all-reduce of finished shares."""
import os
import socket

import numpy as np
import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

pytestmark = pytest.mark.gpu


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, out):
    import oracle
    from paper_1710_10789_b200 import binding, multigpu, workloads as wl
    from gpu_util import errors, TOL_DOS, TOL_N
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    dev = torch.device("cuda:0")
    results = []
    for nk, nb, norb, nE, model in (((12, 12, 7), 8, 8, 600, "tb8"), ((6, 5, 9), 2, 3, 150, "random")):
        if model == "tb8":
            E, W = wl.tb8_bands(nk, threads=1)
            om = wl.omega_grid(-6.0, 4.0, nE)
        else:
            E, W = wl.random_bands(nk, nb, norb, seed=11)
            om = wl.omega_grid(-1.2, 1.3, nE)
        dE, dW, dOm = (torch.from_numpy(a).to(dev) for a in (E, W, om))
        part = torch.zeros((3, norb, nE), dtype=torch.float64, device=dev)
        dos = torch.full((norb, nE), float("nan"), device=dev)
        nos = torch.full((norb, nE), float("nan"), device=dev)

        def all_reduce(t):
            h = t.cpu()              # waits for this rank's share
            dist.all_reduce(h)
            t.copy_(h)

        # what SURVEY.md 8(e) describes: this rank's k-planes only (its slab plus the halo plane), nothing else on the device
        from paper_1710_10789_b200 import sharding
        plane = nk[0] * nk[1]
        idx = np.concatenate([np.arange(z * plane, (z + 1) * plane) for z in sharding.planes_read(rank, world, nk[2])])
        lE, lW = torch.from_numpy(np.ascontiguousarray(E[idx])).to(dev), torch.from_numpy(np.ascontiguousarray(W[idx])).to(dev)
        with binding.Plan(nk, nb, norb, nE) as plan:
            for _ in range(2):       # twice on one plan: the shares do not accumulate across calls
                multigpu.sharded_step(plan, dE, dW, dOm, nk[2], rank, world, part, dos, nos, all_reduce)
                torch.cuda.synchronize()
            full = (dos.clone(), nos.clone())
            dos.fill_(float("nan"))
            nos.fill_(float("nan"))
            multigpu.sharded_step(plan, lE, lW, dOm, nk[2], rank, world, part, dos, nos, all_reduce, slab_local=True)
            torch.cuda.synchronize()
            cnt = plan.last_counters()
            assert torch.allclose(dos, full[0], rtol=1e-5, atol=1e-7 * float(full[0].max()))
            assert torch.allclose(nos, full[1], rtol=1e-5, atol=1e-7 * float(full[1].max()))
        c = torch.tensor([cnt["n_tb"], cnt["n_eval"]])
        dist.all_reduce(c)
        ref = oracle.tetra_dos(E, W, nk, om)
        d, en, zero_ok = errors(ref, dos.cpu().numpy(), nos.cpu().numpy())
        results.append(bool(d <= TOL_DOS and en <= TOL_N and zero_ok and int(c[0]) == ref["n_tb"] and int(c[1]) == ref["n_eval"]))
    out.put((rank, results))
    dist.destroy_process_group()


def test_two_ranks_on_one_gpu_partial_allreduce_finalize():
    ctx = mp.get_context("spawn")
    out = ctx.Queue()
    port = _free_port()
    here = os.path.dirname(os.path.abspath(__file__))
    os.environ["PYTHONPATH"] = os.pathsep.join([here, os.path.dirname(here), os.environ.get("PYTHONPATH", "")])
    procs = [ctx.Process(target=_worker, args=(r, 2, port, out)) for r in range(2)]
    for p in procs:
        p.start()
    for p in procs:
        p.join(300)
        assert p.exitcode == 0
    got = dict(out.get(timeout=5) for _ in range(2))
    assert got[0] == [True, True] and got[1] == [True, True]
