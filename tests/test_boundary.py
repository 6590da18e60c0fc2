"""CPU-side checks of the boundary: the C-ABI library builds, loads and exports every symbol that
include/tetrados.h declares; host-side argument validation; no CPU fallback."""
import ctypes
import os
import re

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def binding():
    from paper_1710_10789_b200 import build, binding as b
    build.build()
    b.load()
    return b


def _declared_symbols():
    src = open(os.path.join(ROOT, "include", "tetrados.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(t(?:dos|etra)_[a-z0-9_]+)\s*\(", src)))


def test_header_symbols_are_exported(binding):
    names = _declared_symbols()
    assert {"tetra_dos", "tetra_dos_simple", "tdos_plan_create", "tdos_plan_destroy", "tdos_version",
            "tdos_strerror", "tetra_dos_partial", "tetra_dos_finalize"} <= set(names)
    assert sorted(binding.SYMBOLS) == names, (binding.SYMBOLS, names)
    lib = ctypes.CDLL(os.path.join(ROOT, "paper_1710_10789_b200", "libtetrados.so"))
    for n in names:
        assert getattr(lib, n) is not None


def test_version_and_strerror(binding):
    assert binding.tdos_version() >= 100
    for code in (0, -1, -2, -3, -4, -5, -99):
        assert isinstance(binding.tdos_strerror(code), str) and binding.tdos_strerror(code)


def test_null_and_bad_arguments_rejected_without_gpu(binding):
    lib = binding.load()
    h = ctypes.c_void_p()
    nk = (ctypes.c_int * 3)(4, 4, 4)
    assert lib.tdos_plan_create(None, 0, nk, 1, 1, 10) == binding.TDOS_EINVAL
    assert lib.tdos_plan_create(ctypes.byref(h), 0, None, 1, 1, 10) == binding.TDOS_EINVAL
    bad = (ctypes.c_int * 3)(4, 0, 4)
    assert lib.tdos_plan_create(ctypes.byref(h), 0, bad, 1, 1, 10) == binding.TDOS_EINVAL
    assert lib.tdos_plan_create(ctypes.byref(h), 0, nk, 0, 1, 10) == binding.TDOS_EINVAL
    assert lib.tdos_plan_create(ctypes.byref(h), 0, nk, 1, 1, binding.TDOS_MAX_NE + 1) == binding.TDOS_EINVAL
    assert lib.tdos_plan_destroy(None) == binding.TDOS_OK
    assert lib.tetra_dos(None, None, None, 0, None, 1, None, None, 0, None) == binding.TDOS_EINVAL
    e = np.zeros(8, dtype=np.float32)
    assert lib.tetra_dos_simple(None, None, 2, 1, 1, 0.0, 1.0, 4, e.ctypes.data, None) == binding.TDOS_EINVAL
    assert lib.tetra_dos_simple(e.ctypes.data, None, 2, 1, 1, 1.0, 0.0, 4, e.ctypes.data, None) == binding.TDOS_EINVAL


def test_no_cpu_fallback(binding):
    """Without a CUDA device the product path must fail loudly, never compute on the CPU."""
    import torch
    if torch.cuda.is_available():
        pytest.skip("a GPU is present")
    with pytest.raises(binding.TdosError) as ei:
        binding.Plan((4, 4, 4), 1, 1, 10)
    assert ei.value.code in (binding.TDOS_ECUDA, binding.TDOS_EARCH)
    E = np.zeros((8, 1), dtype=np.float32)
    out = np.zeros(4, dtype=np.float32)
    with pytest.raises(binding.TdosError):
        binding.tetra_dos_simple(E, None, 2, 1, 1, -1.0, 1.0, 4, out, None)


def test_product_does_not_import_oracle():
    """The product package and bench's product arm never touch oracle/ (parity would be void)."""
    pkg = os.path.join(ROOT, "paper_1710_10789_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                txt = open(os.path.join(dirpath, f)).read()
                assert not re.search(r"^\s*(import|from)\s+oracle\b", txt, flags=re.M), f
                assert "tetra_oracle" not in txt and "liboracle" not in txt, f
    otxt = open(os.path.join(ROOT, "oracle", "oracle.py")).read() + open(os.path.join(ROOT, "oracle", "tetra_oracle.c")).read()
    assert "paper_1710_10789_b200" not in otxt.replace("paper_1710_10789_b200/", "")
