"""fp64 CPU oracle for the tetrahedron-DOS path -- TEST INFRASTRUCTURE ONLY.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference
legs may import this package.  It shares nothing with paper_1710_10789_b200/.
"""
from .oracle import (  # noqa: F401
    build, corner_weights, sort4, table_I, corner_offset, tetra_dos, tetra_weights, eigh_bands, max_threads,
    AOS, SOA,
)
