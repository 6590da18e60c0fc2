"""Helpers for the GPU parity tests: run the CUDA path through the C-ABI binding and compare
with the oracle at the north-star tolerances (BASELINE.json):
    max|dDOS| <= 1e-4 * max(DOS)      and      |dN|/N <= 1e-5
G17: |dN|/N is taken over bins with N_oracle > 0 (strict); bins where the oracle's N
is exactly 0 must be exactly 0 on the GPU."""
import numpy as np
import torch

from paper_1710_10789_b200 import binding

TOL_DOS = 1e-4
TOL_N = 1e-5


def run_gpu(E, W, nk, om, layout=binding.TDOS_AOS, memspace=binding.TDOS_DEVICE, want_nos=True, plan=None):
    nb = E.shape[1] if layout == binding.TDOS_AOS else E.shape[0]
    if W is None:
        norb = 1
    else:
        norb = W.shape[2] if layout == binding.TDOS_AOS else W.shape[1]
    nE = len(om)
    own = plan is None
    if own:
        plan = binding.Plan(nk, nb, norb, nE)
    try:
        if memspace == binding.TDOS_DEVICE:
            dev = torch.device("cuda:0")
            dE = torch.from_numpy(np.ascontiguousarray(E)).to(dev)
            dW = None if W is None else torch.from_numpy(np.ascontiguousarray(W)).to(dev)
            dOm = torch.from_numpy(np.ascontiguousarray(om)).to(dev)
            dos = torch.full((norb, nE), float("nan"), device=dev)
            nos = torch.full((norb, nE), float("nan"), device=dev) if want_nos else None
            plan.tetra_dos(dE, dW, dOm, dos, nos, layout=layout)
            torch.cuda.synchronize()
            return dos.cpu().numpy(), (nos.cpu().numpy() if want_nos else None)
        hE = torch.from_numpy(np.ascontiguousarray(E)).pin_memory()
        hW = None if W is None else torch.from_numpy(np.ascontiguousarray(W)).pin_memory()
        hOm = torch.from_numpy(np.ascontiguousarray(om)).pin_memory()
        dos = torch.full((norb, nE), float("nan")).pin_memory()
        nos = torch.full((norb, nE), float("nan")).pin_memory() if want_nos else None
        plan.tetra_dos(hE, hW, hOm, dos, nos, layout=layout, memspace=binding.TDOS_HOST)
        return dos.numpy().copy(), (nos.numpy().copy() if want_nos else None)
    finally:
        if own:
            plan.close()


def errors(ref, dos, nos):
    """(max|dDOS|/max(DOS), max|dN|/N over N_ref>0, exact-zero flag)"""
    d = np.abs(dos.astype(np.float64) - ref["dos"]).max() / max(ref["dos"].max(), 1e-300)
    en, zero_ok = 0.0, True
    if nos is not None:
        pos = ref["nos"] > 0
        if pos.any():
            en = (np.abs(nos.astype(np.float64) - ref["nos"])[pos] / ref["nos"][pos]).max()
        zero_ok = not nos[~pos].any()
    return d, en, zero_ok


def assert_parity(ref, dos, nos, what=""):
    assert np.all(np.isfinite(dos)), what
    d, en, zero_ok = errors(ref, dos, nos)
    assert d <= TOL_DOS, "%s: max|dDOS|/max(DOS) = %.3e > %.0e" % (what, d, TOL_DOS)
    if nos is not None:
        assert np.all(np.isfinite(nos)), what
        assert en <= TOL_N, "%s: max|dN|/N = %.3e > %.0e" % (what, en, TOL_N)
        assert zero_ok, "%s: N must be exactly 0 where the oracle's N is 0" % what
    return d, en
