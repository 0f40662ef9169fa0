"""Seeded synthetic inputs shaped like the paper's workloads (Table 3 :659-672).

This package serves BOTH the fp64 oracle (``oracle/``) and the CUDA path
(``paper_2006_16560_b200/``).  It holds input generation only -- sampling of
positions, masses, binary orbits and the per-particle radii that are *inputs*
of the library (Eq. 12) -- and none of the method's force,
tree or neighbour arithmetic.  It imports neither ``oracle`` nor the package.
"""
from .generators import (  # noqa: F401
    CONFIGS,
    Workload,
    make_workload,
    plummer_positions,
    kroupa_masses,
    changeover_radii,
    PLUMMER_A,
)
