"""B200-native linear-tetrahedron density of states (arxiv 1710.10789 hot path).

`tetra_dos` & co. are thin ctypes bindings over the C-ABI library
(include/tetrados.h); every step of the path runs in the CUDA kernels under csrc/.
The library is loaded on first use and a missing build raises: there is no CPU
fallback.  `workloads` (seeded input generators) imports without the library.
"""
from . import workloads  # noqa: F401


def __getattr__(name):
    # lazy: importing the package (e.g. for workloads) must not need the .so
    from . import binding
    if hasattr(binding, name):
        return getattr(binding, name)
    raise AttributeError(name)
