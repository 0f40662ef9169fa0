"""fp64 CPU oracle for the long-range P3T force path -- TEST INFRASTRUCTURE, NOT THE PRODUCT.

Only ``tests/``, ``__graft_entry__.smoke()`` and ``bench.py``'s ``cpu_baseline`` /
``--impl reference`` legs may import this package.  It wraps ``petar_oracle.c`` (plain C,
fp64, built with gcc at first use) through ctypes and imports nothing from the CUDA package.
"""
from . import artificial  # noqa: F401  (part (E): kick, pseudoparticles, tidal tensors; numpy)
from .binding import (  # noqa: F401
    OracleParams, OracleTree, K, W, f, direct, neighbors_direct, build_library, num_threads, set_num_threads,
    search_radii, pericentre, neighbors_orbit_direct, clusters, dK, short_range,
)
