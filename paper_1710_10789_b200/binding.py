"""ctypes binding over libtetrados.so (include/tetrados.h): argument marshalling only.

PyTorch is used for device memory and streams; every step of the path runs in the CUDA kernels.
There is no CPU fallback: if the library is missing or the call fails, an exception is raised.
"""
from __future__ import annotations

import ctypes as C
import os

from . import build as _build

TDOS_OK, TDOS_EINVAL, TDOS_ENOMEM, TDOS_ECUDA, TDOS_EARCH, TDOS_ESIZE = 0, -1, -2, -3, -4, -5
TDOS_AOS, TDOS_SOA = 0, 1
TDOS_ACC_FP32, TDOS_ACC_FP64, TDOS_ACC_FP64_ALL = 0, 1, 2
TDOS_DEVICE, TDOS_HOST = 0, 1
TDOS_MAX_NE = 65534
TDOS_STATIC_MAX_CELLS = 32768   # tetra_dos_static: norb * (nE rounded up to 4) it accepts

# every symbol include/tetrados.h declares
SYMBOLS = ["tdos_version", "tdos_strerror", "tdos_last_cuda_error", "tdos_plan_create", "tdos_plan_destroy", "tdos_plan_set_accumulation",
           "tetra_dos", "tetra_dos_complex", "tetra_dos_select", "tetra_eigh", "tetra_weights", "tetra_dos_partial", "tetra_dos_partial_slab", "tetra_dos_finalize", "tetra_dos_simple", "tetra_dos_static", "tdos_plan_info",
           "tdos_last_counters", "tdos_kernel_ms", "tdos_last_kernel_ms", "tdos_fp32_fma_probe"]

_lib = None


class TdosError(RuntimeError):
    def __init__(self, code: int, where: str):
        lib = load()
        msg = lib.tdos_strerror(code).decode()
        cu = lib.tdos_last_cuda_error().decode()
        super().__init__("%s failed: %s (%d)%s" % (where, msg, code, (": " + cu) if cu and code == TDOS_ECUDA else ""))
        self.code = code


def load():
    """dlopen the in-tree library; raise loudly if it has not been built."""
    global _lib
    if _lib is not None:
        return _lib
    path = _build.LIB
    if not os.path.exists(path):
        raise ImportError("libtetrados.so is not built (%s); run __graft_entry__.build() or "
                          "python paper_1710_10789_b200/build.py -- there is no CPU fallback" % path)
    lib = C.CDLL(path)
    vp, fp, ip = C.c_void_p, C.c_void_p, C.POINTER(C.c_int)
    lib.tdos_version.restype = C.c_int
    lib.tdos_strerror.argtypes = [C.c_int]
    lib.tdos_strerror.restype = C.c_char_p
    lib.tdos_last_cuda_error.restype = C.c_char_p
    lib.tdos_plan_create.argtypes = [C.POINTER(vp), C.c_int, ip, C.c_int, C.c_int, C.c_int]
    lib.tdos_plan_destroy.argtypes = [vp]
    lib.tdos_plan_set_accumulation.argtypes = [vp, C.c_int]
    lib.tetra_dos.argtypes = [vp, fp, fp, C.c_int, fp, C.c_int, fp, fp, C.c_int, vp]
    lib.tetra_dos_complex.argtypes = [vp, fp, fp, C.c_int, fp, C.c_int, fp, fp, C.c_int, vp]
    lib.tetra_dos_select.argtypes = [vp, fp, fp, C.c_int, fp, C.c_int, ip, C.c_int, C.c_int, fp, fp, C.c_int, vp]
    lib.tetra_eigh.argtypes = [vp, fp, fp, fp, vp]
    lib.tetra_weights.argtypes = [vp, fp, C.c_int, fp, C.c_int, fp, fp, vp]
    lib.tetra_dos_partial.argtypes = [vp, fp, fp, C.c_int, fp, C.c_int, C.c_int, C.c_int, vp, vp]
    lib.tetra_dos_partial_slab.argtypes = [vp, fp, fp, C.c_int, fp, C.c_int, C.c_int, C.c_int, vp, vp]
    lib.tetra_dos_finalize.argtypes = [vp, vp, C.c_int, fp, fp, vp]
    lib.tetra_dos_simple.argtypes = [fp, fp, C.c_int, C.c_int, C.c_int, C.c_float, C.c_float, C.c_int, fp, fp]
    lib.tetra_dos_static.argtypes = [ip, C.c_int, C.c_int, fp, fp, C.c_int, fp, C.c_int, fp, fp, vp]
    lib.tdos_plan_info.argtypes = [vp, C.POINTER(C.c_longlong)]
    lib.tdos_last_counters.argtypes = [vp, C.POINTER(C.c_longlong)]
    lib.tdos_kernel_ms.argtypes = [vp, C.c_int, C.POINTER(C.c_float), C.POINTER(C.c_float)]
    lib.tdos_last_kernel_ms.argtypes = [vp, C.POINTER(C.c_float), C.POINTER(C.c_float)]
    lib.tdos_fp32_fma_probe.argtypes = [vp, C.c_int, C.POINTER(C.c_double)]
    for name in SYMBOLS:
        getattr(lib, name)
    _lib = lib
    return lib


def _ptr(t):
    """Raw address of a torch tensor / numpy array / None."""
    if t is None:
        return None
    if hasattr(t, "data_ptr"):
        return t.data_ptr()
    return t.ctypes.data


def _check(rc: int, where: str):
    if rc != TDOS_OK:
        raise TdosError(rc, where)


class Plan:
    """tdos_plan: owns device scratch for one (grid, nb, norb, nE_max) shape on one device."""

    def __init__(self, nk, nb: int, norb: int, nE_max: int, device: int = 0):
        lib = load()
        self._h = C.c_void_p()
        self.nk = tuple(int(x) for x in nk)
        self.nb, self.norb, self.nE_max, self.device = int(nb), int(norb), int(nE_max), int(device)
        arr = (C.c_int * 3)(*self.nk)
        _check(lib.tdos_plan_create(C.byref(self._h), self.device, arr, self.nb, self.norb, self.nE_max),
               "tdos_plan_create")

    def set_accumulation(self, fp64, weights_fp64: bool = False):
        """tdos_plan_set_accumulation(): fp64 sums after the single-precision corner weights;
        weights_fp64 (or fp64 == TDOS_ACC_FP64_ALL): the corner weights in double precision too."""
        mode = TDOS_ACC_FP64_ALL if (weights_fp64 or fp64 == TDOS_ACC_FP64_ALL) else (TDOS_ACC_FP64 if fp64 else TDOS_ACC_FP32)
        _check(load().tdos_plan_set_accumulation(self._h, mode), "tdos_plan_set_accumulation")

    def close(self):
        if getattr(self, "_h", None) is not None and self._h.value:
            load().tdos_plan_destroy(self._h)
            self._h = C.c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def __enter__(self):
        return self

    def __exit__(self, *a):
        self.close()

    # ---- the hot path
    def tetra_dos(self, E, W, omega, dos, nos=None, layout: int = TDOS_AOS, memspace: int = TDOS_DEVICE, stream=None):
        """tetra_dos(): E, W, omega, dos, nos are torch tensors (device or pinned host) or numpy
        arrays (host); shapes are the caller's business exactly as in C.  `stream` is a
        torch.cuda.Stream or None (current stream)."""
        nE = int(omega.shape[0])
        _check(load().tetra_dos(self._h, _ptr(E), _ptr(W), layout, _ptr(omega), nE, _ptr(dos), _ptr(nos), memspace,
                                _stream_ptr(stream, memspace)), "tetra_dos")

    def tetra_dos_complex(self, E, A, omega, dos, nos=None, layout: int = TDOS_AOS, memspace: int = TDOS_DEVICE,
                          stream=None):
        """tetra_dos_complex(): A holds the eigenvector elements as (re, im) float pairs (last axis of size 2, or a
        complex64 array viewed as float32)."""
        nE = int(omega.shape[0])
        _check(load().tetra_dos_complex(self._h, _ptr(E), _ptr(A), layout, _ptr(omega), nE, _ptr(dos), _ptr(nos),
                                        memspace, _stream_ptr(stream, memspace)), "tetra_dos_complex")

    def tetra_dos_select(self, E, W, omega, orbitals, want_total: bool, dos, nos=None, layout: int = TDOS_AOS,
                         memspace: int = TDOS_DEVICE, stream=None):
        """tetra_dos_select(): rows = the listed orbitals, then (want_total) the sum over all orbitals."""
        nE = int(omega.shape[0])
        orb = (C.c_int * max(len(orbitals), 1))(*[int(x) for x in orbitals])
        _check(load().tetra_dos_select(self._h, _ptr(E), _ptr(W), layout, _ptr(omega), nE, orb, len(orbitals),
                                       1 if want_total else 0, _ptr(dos), _ptr(nos), memspace,
                                       _stream_ptr(stream, memspace)), "tetra_dos_select")

    def tetra_eigh(self, H, E, A, stream=None):
        """tetra_eigh(): device tensors H[nk][nb][nb] complex64 (or float pairs) -> E[nk][nb], A[nk][nb][nb] complex64."""
        _check(load().tetra_eigh(self._h, _ptr(H), _ptr(E), _ptr(A), _stream_ptr(stream, TDOS_DEVICE)), "tetra_eigh")

    def tetra_weights(self, E, energies, wk, dwk=None, layout: int = TDOS_AOS, stream=None):
        """tetra_weights(): per-k-point integration weights wk[nW][nb][nk] (and dwk) for device tensors."""
        _check(load().tetra_weights(self._h, _ptr(E), layout, _ptr(energies), int(energies.shape[0]), _ptr(wk), _ptr(dwk),
                                    _stream_ptr(stream, TDOS_DEVICE)), "tetra_weights")

    def tetra_dos_partial(self, E, W, omega, z_lo: int, z_hi: int, part, layout: int = TDOS_AOS, stream=None):
        nE = int(omega.shape[0])
        _check(load().tetra_dos_partial(self._h, _ptr(E), _ptr(W), layout, _ptr(omega), nE, int(z_lo), int(z_hi),
                                        _ptr(part), _stream_ptr(stream, TDOS_DEVICE)), "tetra_dos_partial")

    def tetra_dos_partial_slab(self, E, W, omega, z_lo: int, z_hi: int, part, layout: int = TDOS_AOS, stream=None):
        """tetra_dos_partial_slab(): E, W hold only the k-planes z_lo .. z_hi (slab + halo plane) of the grid."""
        nE = int(omega.shape[0])
        _check(load().tetra_dos_partial_slab(self._h, _ptr(E), _ptr(W), layout, _ptr(omega), nE, int(z_lo), int(z_hi),
                                             _ptr(part), _stream_ptr(stream, TDOS_DEVICE)), "tetra_dos_partial_slab")

    def tetra_dos_finalize(self, part, nE: int, dos, nos=None, stream=None):
        _check(load().tetra_dos_finalize(self._h, _ptr(part), int(nE), _ptr(dos), _ptr(nos),
                                         _stream_ptr(stream, TDOS_DEVICE)), "tetra_dos_finalize")

    # ---- diagnostics
    def info(self) -> dict:
        w = (C.c_longlong * 8)()
        _check(load().tdos_plan_info(self._h, w), "tdos_plan_info")
        return {"grid": w[0], "threads": w[1], "smem": w[2], "items": w[3], "launches": w[4], "tile": (w[5], w[6], w[7])}

    def last_counters(self) -> dict:
        w = (C.c_longlong * 4)()
        _check(load().tdos_last_counters(self._h, w), "tdos_last_counters")
        return {"n_tb": w[0], "n_eval": w[1], "n_eval_mid": w[2], "kernel": w[3]}

    def kernel_ms(self, ncalls: int = 1):
        """(main kernel ms, merge+finalize ms), mean over the last `ncalls` device-mode calls."""
        a, b = C.c_float(), C.c_float()
        _check(load().tdos_kernel_ms(self._h, int(ncalls), C.byref(a), C.byref(b)), "tdos_kernel_ms")
        return a.value, b.value

    def last_kernel_ms(self):
        return self.kernel_ms(1)

    def fp32_fma_probe(self, packed: bool = False) -> float:
        t = C.c_double()
        _check(load().tdos_fp32_fma_probe(self._h, 1 if packed else 0, C.byref(t)), "tdos_fp32_fma_probe")
        return t.value


def _stream_ptr(stream, memspace):
    if memspace == TDOS_HOST:
        return None
    if stream is None:
        import torch
        return torch.cuda.current_stream().cuda_stream
    return stream.cuda_stream if hasattr(stream, "cuda_stream") else int(stream)


def tetra_dos_simple(E, W, Nk: int, nb: int, norb: int, omega_min: float, omega_max: float, nE: int, dos, nos=None):
    """tetra_dos_simple(): host arrays, AoS, cubic grid, uniform omega; one-shot."""
    _check(load().tetra_dos_simple(_ptr(E), _ptr(W), int(Nk), int(nb), int(norb), float(omega_min), float(omega_max),
                                   int(nE), _ptr(dos), _ptr(nos)), "tetra_dos_simple")


def tetra_dos_static(nk, nb: int, norb: int, E, W, omega, dos, nos=None, layout: int = TDOS_AOS, stream=None):
    """tetra_dos_static(): tetra_dos on device tensors without a plan and without a single device allocation, for
    callers that are barred from cudaMalloc (a plug-in in a host code that owns all GPU memory through its own pools, a
    loop that cannot take cudaMalloc's device-wide synchronisation).  The scratch is a fixed buffer inside the library,
    so norb * (nE rounded up to 4) must not exceed TDOS_STATIC_MAX_CELLS (TdosError with code TDOS_ESIZE otherwise),
    and calls that could overlap on one GPU must be ordered by the caller: they all share that buffer.  Runs on the
    current device; the first call per device also does the one-time set-up (include/tetrados.h)."""
    arr = (C.c_int * 3)(*[int(x) for x in nk])
    _check(load().tetra_dos_static(arr, int(nb), int(norb), _ptr(E), _ptr(W), layout, _ptr(omega), int(omega.shape[0]),
                                   _ptr(dos), _ptr(nos), _stream_ptr(stream, TDOS_DEVICE)), "tetra_dos_static")


def tdos_version() -> int:
    return int(load().tdos_version())


def tdos_strerror(code: int) -> str:
    return load().tdos_strerror(int(code)).decode()
