"""B200-native long-range P3T force path of PeTar (arxiv 2006.16560).

The product is the C-ABI library ``libpetar_b200.so`` (include/petar.h, hand-written CUDA for
sm_100a).  This package is the thin Python binding with the same names: it marshals arguments
only -- every step of the path runs in the library's kernels.  PyTorch supplies device memory and
streams.  There is no CPU fallback: if the library is missing or no CUDA device is present the
calls raise.
"""
from .binding import (  # noqa: F401
    PetarParams, PetarCounts, PetarError, Tree,
    lib, library_path, exported_symbols,
    petar_workspace_bytes, petar_tree_build, petar_tree_rebuild, petar_long_range_force, petar_neighbor_list,
    petar_tree_status, petar_tree_destroy, petar_strerror, petar_debug_export,
    petar_set_profiling, petar_stage_times, petar_launch_count, petar_probe_fp32,
    petar_search_radii, petar_neighbor_list_orbit, petar_clusters_workspace_bytes, petar_clusters,
    petar_short_range_workspace_bytes, petar_short_range_force, petar_short_range_force_noalloc, SHORT_RANGE_NOALLOC_MAX_N,
    petar_kick, petar_artificial_particles, petar_tidal_tensor_fit, petar_orbit_sampling, art_count,
    STAGE_NAMES,
)
