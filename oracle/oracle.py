"""ctypes loader for oracle/tetra_oracle.c (TEST INFRASTRUCTURE ONLY; see the C header).

The arithmetic lives in the C file, written from PAPER.md Eq. 8-15; this module only
marshals numpy arrays.  `build()` compiles the C file with gcc -- building the checker
is not using it.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "tetra_oracle.c")
_LIB = os.path.join(_HERE, "liboracle.so")
AOS, SOA = 0, 1
_lib = None


def build(force: bool = False) -> str:
    """gcc -O2 -fopenmp -shared; rebuilt when the source is newer than the .so."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        cmd = ["gcc", "-O2", "-fopenmp", "-shared", "-fPIC", "-std=c99", "-o", _LIB, _SRC, "-lm"]
        subprocess.run(cmd, check=True)
    return _LIB


def _load():
    global _lib
    if _lib is None:
        build()
        lib = C.CDLL(_LIB)
        dp, ip, fp = C.POINTER(C.c_double), C.POINTER(C.c_int), C.POINTER(C.c_float)
        lib.oracle_corner_weights.argtypes = [dp, C.c_double, C.c_double, dp, dp]
        lib.oracle_corner_weights.restype = C.c_int
        lib.oracle_sort4.argtypes = [dp, dp, ip]
        lib.oracle_tetra_weights.argtypes = [fp, ip, C.c_int, C.c_int, fp, C.c_int, dp, dp]
        lib.oracle_tetra_weights.restype = C.c_int
        lib.oracle_table_I.argtypes = [ip]
        lib.oracle_corner_offset.argtypes = [C.c_int, ip]
        lib.oracle_tetra_dos.argtypes = [fp, fp, ip, C.c_int, C.c_int, C.c_int, fp, C.c_int,
                                         C.c_long, C.c_long, C.c_int, C.c_int, dp, dp,
                                         C.POINTER(C.c_longlong)]
        lib.oracle_tetra_dos.restype = C.c_int
        lib.oracle_max_threads.restype = C.c_int
        _lib = lib
    return _lib


def _dptr(a):
    return a.ctypes.data_as(C.POINTER(C.c_double))


def corner_weights(e_sorted, E: float, V: float):
    """(w[4], dw[4], case) for sorted corner energies -- PAPER.md Eq. 11-15."""
    lib = _load()
    e = np.ascontiguousarray(e_sorted, dtype=np.float64)
    assert e.shape == (4,)
    w = np.zeros(4)
    dw = np.zeros(4)
    k = lib.oracle_corner_weights(_dptr(e), float(E), float(V), _dptr(w), _dptr(dw))
    return w, dw, k


def sort4(e_in):
    lib = _load()
    e = np.ascontiguousarray(e_in, dtype=np.float64)
    out = np.zeros(4)
    perm = np.zeros(4, dtype=np.int32)
    lib.oracle_sort4(_dptr(e), _dptr(out), perm.ctypes.data_as(C.POINTER(C.c_int)))
    return out, perm


def table_I():
    lib = _load()
    t = np.zeros(24, dtype=np.int32)
    lib.oracle_table_I(t.ctypes.data_as(C.POINTER(C.c_int)))
    return t.reshape(6, 4)


def corner_offset(c: int):
    lib = _load()
    d = np.zeros(3, dtype=np.int32)
    lib.oracle_corner_offset(int(c), d.ctypes.data_as(C.POINTER(C.c_int)))
    return tuple(int(x) for x in d)


def max_threads() -> int:
    return int(_load().oracle_max_threads())


def tetra_dos(E, W, nk, omega, layout: int = AOS, windowed: bool = False, nthreads: int = 1,
              cube_range=None):
    """Run the oracle.  E, W fp32 arrays in `layout` (AOS: E[ik][n], W[ik][n][m];
    SOA: E[n][ik], W[n][m][ik]); W may be None (W == 1, norb = 1).
    Returns dict(dos[norb][nE], nos[norb][nE] (float64), n_tb, n_eval, n_case[3])."""
    lib = _load()
    nk = tuple(int(x) for x in nk)
    nkt = nk[0] * nk[1] * nk[2]
    E = np.ascontiguousarray(E, dtype=np.float32)
    if layout == AOS:
        assert E.ndim == 2 and E.shape[0] == nkt, E.shape
        nb = E.shape[1]
    else:
        assert E.ndim == 2 and E.shape[1] == nkt, E.shape
        nb = E.shape[0]
    if W is None:
        norb, Wp = 1, None
    else:
        W = np.ascontiguousarray(W, dtype=np.float32)
        if layout == AOS:
            assert W.shape[:2] == (nkt, nb), W.shape
            norb = W.shape[2]
        else:
            assert W.shape[0] == nb and W.shape[2] == nkt, W.shape
            norb = W.shape[1]
        Wp = W.ctypes.data_as(C.POINTER(C.c_float))
    omega = np.ascontiguousarray(omega, dtype=np.float32)
    nE = omega.shape[0]
    lo, hi = (0, nkt) if cube_range is None else cube_range
    dos = np.zeros((norb, nE))
    nos = np.zeros((norb, nE))
    cnt = np.zeros(5, dtype=np.int64)
    nk_arr = (C.c_int * 3)(*nk)
    rc = lib.oracle_tetra_dos(E.ctypes.data_as(C.POINTER(C.c_float)), Wp, nk_arr, nb, norb, layout,
                              omega.ctypes.data_as(C.POINTER(C.c_float)), nE, lo, hi,
                              1 if windowed else 0, int(nthreads), _dptr(dos), _dptr(nos),
                              cnt.ctypes.data_as(C.POINTER(C.c_longlong)))
    if rc != 0:
        raise ValueError("oracle_tetra_dos: bad arguments (rc=%d)" % rc)
    return {"dos": dos, "nos": nos, "n_tb": int(cnt[0]), "n_eval": int(cnt[1]),
            "n_case": [int(x) for x in cnt[2:5]]}


def tetra_weights(E, nk, energies, layout: int = AOS):
    """Per-k-point integration weights of PAPER.md Eq. 5-7: returns (wk, dwk), each [nW][nb][nk] float64."""
    lib = _load()
    nk = tuple(int(x) for x in nk)
    nkt = nk[0] * nk[1] * nk[2]
    E = np.ascontiguousarray(E, dtype=np.float32)
    nb = E.shape[1] if layout == AOS else E.shape[0]
    en = np.ascontiguousarray(energies, dtype=np.float32)
    wk = np.zeros((len(en), nb, nkt))
    dwk = np.zeros((len(en), nb, nkt))
    rc = lib.oracle_tetra_weights(E.ctypes.data_as(C.POINTER(C.c_float)), (C.c_int * 3)(*nk), nb, layout,
                                  en.ctypes.data_as(C.POINTER(C.c_float)), len(en), _dptr(wk), _dptr(dwk))
    if rc != 0:
        raise ValueError("oracle_tetra_weights: bad arguments")
    return wk, dwk


def eigh_bands(H):
    """PAPER.md Eq. 1 (:37-39): H(k) "is diagonalised to obtain band energies E_n(k) and eigenvector elements a_n^m(k)".
    H[ik][nb][nb] complex Hermitian -> (E[ik][nb] ascending, W[ik][n][m] = |a_n^m(k)|^2), both float64.  The
    diagonalisation itself is the library routine numpy.linalg.eigh (LAPACK zheevd) in complex128; nothing else is
    done here.  Pinned in tests/test_oracle_pins.py by a closed-form 2 x 2 case, the two sum rules of |a|^2 and, for the
    [n][m] orientation of W, by the Hellmann-Feynman derivative dE_n/dH_mm = |a_n^m|^2 of its own eigenvalues."""
    H = np.asarray(H).astype(np.complex128)
    w, U = np.linalg.eigh(H)                      # U[ik][m][n]: column n is eigenvector n
    W = (U.real ** 2 + U.imag ** 2).transpose(0, 2, 1)
    return w, np.ascontiguousarray(W)
