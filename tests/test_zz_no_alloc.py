"""tetra_dos_static: the DOS path for callers that cannot allocate device memory.

Some users of this library run where cudaMalloc is not available to them: a plug-in inside a host code that has
claimed the whole GPU for its own memory pools, or a loop that cannot take the device-wide synchronisation cudaMalloc
implies.  A Plan allocates its scratch when it is created, so it is no use to them; tetra_dos_static keeps its scratch
in a fixed buffer inside the library instead (about 16.8 MB per GPU, hence the limit norb * nE <= 32768) and takes only
the caller's input and output arrays.

This file checks that the result equals the ordinary Plan path within the tolerances of the parity suite
(tests/gpu_util.py), on calls that follow each other directly and use different sizes, because every call finds the
previous call's sums still in the shared buffer and must clear what it needs.  It also checks that a repeat call leaves
the free device memory untouched and that a problem beyond the limit is refused with TDOS_ESIZE.

The file name sorts last on purpose: under `pytest -x` a failure here cannot hide a failure in the older tests.  Every
test builds its own inputs and the library keeps no state a previous test could have left in a harmful shape (the
buffer is cleared per call), so the file passes on its own in a fresh process as well as after the rest of the suite."""
import numpy as np
import pytest

from paper_1710_10789_b200 import binding, workloads as wl
from gpu_util import errors, TOL_DOS, TOL_N

pytestmark = pytest.mark.gpu


def _device_inputs(E, W, om):
    import torch
    dev = torch.device("cuda:0")
    dE = torch.from_numpy(np.ascontiguousarray(E)).to(dev)
    dW = None if W is None else torch.from_numpy(np.ascontiguousarray(W)).to(dev)
    dOm = torch.from_numpy(np.ascontiguousarray(om)).to(dev)
    return dE, dW, dOm


def _plan_path(nk, nb, norb, dE, dW, dOm, layout):
    """The existing path: a Plan (which allocates its scratch) and tetra_dos on device tensors."""
    import torch
    nE = dOm.shape[0]
    dos = torch.full((norb, nE), float("nan"), device=dE.device)
    nos = torch.full((norb, nE), float("nan"), device=dE.device)
    with binding.Plan(nk, nb, norb, nE) as plan:
        plan.tetra_dos(dE, dW, dOm, dos, nos, layout=layout)
        torch.cuda.synchronize()
    return {"dos": dos.cpu().numpy().astype(np.float64), "nos": nos.cpu().numpy().astype(np.float64)}


def _assert_same(ref, dos, nos, what):
    d, n = dos.cpu().numpy(), nos.cpu().numpy()
    assert np.all(np.isfinite(d)) and np.all(np.isfinite(n)), what
    ed, en, zero_ok = errors(ref, d, n)
    assert ed <= TOL_DOS, "%s: max|dDOS|/max(DOS) = %.3e" % (what, ed)
    assert en <= TOL_N, "%s: max|dN|/N = %.3e" % (what, en)
    assert zero_ok, "%s: N must be exactly 0 where the plan path's N is 0" % what
    return ed, en


def test_no_alloc_entry_point_matches_plan_path_on_consecutive_calls():
    import torch
    assert torch.cuda.is_available()
    torch.cuda.set_device(0)
    # case A: the 8-orbital model on a ragged grid (several tiles, 8 x 777 cells of scratch per block);
    # case B: 3 orbitals, SoA layout, more energies but far fewer cells, so its histograms overlay only a part of
    #         what A left behind; case C: unit weights (W = NULL), one orbital
    nkA = (10, 9, 7)
    EA, WA = wl.tb8_bands(nkA, threads=1)
    omA = wl.omega_grid(-6.0, 4.0, 777)
    nkB = (5, 6, 4)
    EB, WB = wl.random_bands(nkB, 2, 3, seed=9)
    EBs, WBs = wl.to_soa(EB, WB)
    omB = wl.omega_grid(-1.1, 1.1, 1500)
    nkC = (6, 6, 6)
    EC, _ = wl.random_bands(nkC, 3, 1, seed=21)
    omC = wl.omega_grid(-1.2, 1.2, 301)
    cases = {
        "A": (nkA, 8, 8, _device_inputs(EA, WA, omA), binding.TDOS_AOS),
        "B": (nkB, 2, 3, _device_inputs(EBs, WBs, omB), binding.TDOS_SOA),
        "C": (nkC, 3, 1, _device_inputs(EC, None, omC), binding.TDOS_AOS),
    }
    refs = {k: _plan_path(nk, nb, norb, *inp, layout) for k, (nk, nb, norb, inp, layout) in cases.items()}
    outs = {k: (torch.empty((norb, inp[2].shape[0]), device="cuda:0"), torch.empty((norb, inp[2].shape[0]), device="cuda:0"))
            for k, (nk, nb, norb, inp, layout) in cases.items()}

    def call(k):
        nk, nb, norb, (dE, dW, dOm), layout = cases[k]
        dos, nos = outs[k]
        dos.fill_(float("nan"))
        nos.fill_(float("nan"))
        binding.tetra_dos_static(nk, nb, norb, dE, dW, dOm, dos, nos, layout=layout)

    # one call after the other on one stream: each must clear what the one before left in the shared buffer
    order = ["A", "B", "C", "A", "A", "B"]
    for step, k in enumerate(order):
        call(k)
        torch.cuda.synchronize()
        ed, en = _assert_same(refs[k], *outs[k], "call %d (%s)" % (step, k))
        print("no-alloc call %d (%s): dDOS %.2e dN %.2e" % (step, k, ed, en))

    # two calls queued without any host synchronisation between them, outputs checked afterwards
    call("A")
    call("B")
    torch.cuda.synchronize()
    _assert_same(refs["A"], *outs["A"], "queued A")
    _assert_same(refs["B"], *outs["B"], "queued B")

    # a repeat call allocates nothing: the driver reports the same free memory before and after
    torch.cuda.synchronize()
    free0, _ = torch.cuda.mem_get_info()
    call("A")
    torch.cuda.synchronize()
    free1, _ = torch.cuda.mem_get_info()
    assert free1 == free0, (free0, free1)
    _assert_same(refs["A"], *outs["A"], "repeat A")


def test_no_alloc_entry_point_without_nos_and_at_the_size_limit():
    """nos = NULL is allowed, and a problem of exactly TDOS_STATIC_MAX_CELLS cells (8 orbitals x 4096 energies: the
    fewest private histograms, 42 blocks) still agrees with the plan path."""
    import torch
    torch.cuda.set_device(0)
    nk = (8, 6, 5)
    E, W = wl.tb8_bands(nk, threads=1)
    om = wl.omega_grid(-6.0, 4.0, 4096)
    assert 8 * 4096 == binding.TDOS_STATIC_MAX_CELLS
    dE, dW, dOm = _device_inputs(E, W, om)
    ref = _plan_path(nk, 8, 8, dE, dW, dOm, binding.TDOS_AOS)
    dos = torch.full((8, 4096), float("nan"), device="cuda:0")
    nos = torch.full((8, 4096), float("nan"), device="cuda:0")
    binding.tetra_dos_static(nk, 8, 8, dE, dW, dOm, dos, nos)
    torch.cuda.synchronize()
    _assert_same(ref, dos, nos, "limit")
    dos2 = torch.full((8, 4096), float("nan"), device="cuda:0")
    binding.tetra_dos_static(nk, 8, 8, dE, dW, dOm, dos2, None)
    torch.cuda.synchronize()
    ed, _, _ = errors(ref, dos2.cpu().numpy(), None)
    assert ed <= TOL_DOS


def test_no_alloc_entry_point_refuses_what_does_not_fit():
    """Beyond the built-in buffer the call returns TDOS_ESIZE before it touches the device or the outputs."""
    import torch
    torch.cuda.set_device(0)
    nk = (4, 4, 4)
    E, W = wl.random_bands(nk, 2, 8, seed=5)
    om = wl.omega_grid(-1.0, 1.0, 4097)          # 8 x 4100 cells > 32768
    dE, dW, dOm = _device_inputs(E, W, om)
    dos = torch.full((8, 4097), 7.0, device="cuda:0")
    with pytest.raises(binding.TdosError) as ei:
        binding.tetra_dos_static(nk, 2, 8, dE, dW, dOm, dos, None)
    assert ei.value.code == binding.TDOS_ESIZE
    assert "scratch" in str(ei.value)
    torch.cuda.synchronize()
    assert bool((dos == 7.0).all())
    with pytest.raises(binding.TdosError) as ei:   # W = NULL needs norb == 1, as for tetra_dos
        binding.tetra_dos_static(nk, 2, 8, dE, None, dOm[:100], dos, None)
    assert ei.value.code == binding.TDOS_EINVAL
