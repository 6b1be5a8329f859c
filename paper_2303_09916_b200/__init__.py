"""B200-native docking hot path of DSDP (arxiv 2303.09916): C-ABI library + thin Python binding.

The product is `libdock_b200.so` (hand-written sm_100a CUDA behind include/dock.h).  This package
only marshals arguments; it never computes any step of the path on the CPU.
"""
from .binding import (  # noqa: F401
    DOCK_EXIT_CAP,
    DOCK_EXIT_GTOL,
    DOCK_EXIT_LINESEARCH,
    DOCK_ITER_HEADER,
    DOCK_TRACE_HEADER,
    DockError,
    EXPORTS,
    GridMaps,
    LigandHandle,
    dock_box,
    dock_build_grids,
    dock_build_grids_batch,
    dock_default_params,
    dock_grid,
    dock_grid_bytes,
    dock_grid_dims,
    dock_init_poses,
    dock_init_poses_site,
    dock_ligand,
    dock_local_opt_batch,
    dock_params,
    dock_probe_peaks,
    dock_score_batch,
    dock_score_batch_host,
    dock_search,
    dock_system_host,
    dock_topk,
    dock_topk_fixed,
    launch_count,
    load_library,
    make_box,
    score_jit_cache,
)
