"""B200-native linear-tetrahedron density of states (arxiv 1710.10789 hot path).

`Plan`, `tetra_dos_simple` & co. are thin ctypes bindings over the C-ABI library
(include/tetrados.h); every step of the path runs in the CUDA kernels under csrc/.
The library is loaded on first use and a missing build raises: there is no CPU
fallback.  `workloads` (seeded input generators) imports without the library.
"""
import importlib

_BINDING_NAMES = ("Plan", "TdosError", "tetra_dos_simple", "tdos_version", "tdos_strerror", "load",
                  "TDOS_AOS", "TDOS_SOA", "TDOS_DEVICE", "TDOS_HOST", "TDOS_MAX_NE", "SYMBOLS")


def __getattr__(name):
    # lazy: importing the package (e.g. for workloads) must not need the .so
    if name in _BINDING_NAMES:
        return getattr(importlib.import_module(__name__ + ".binding"), name)
    raise AttributeError("module %r has no attribute %r" % (__name__, name))
