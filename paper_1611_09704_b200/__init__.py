"""spd-b200: single-pulse detection (arXiv 1611.09704) as hand-written sm_100a CUDA kernels behind a C ABI.

`binding` is a thin ctypes layer over libspd.so (include/spd.h); `build` compiles the library in-tree; `shard`
(DM-row sharding over torch.distributed) and `stream` (copy / compute overlap over consecutive chunks) are plumbing.
Nothing here computes on the CPU; the package is independent of the CPU checker used by the tests.
"""
from .binding import (  # noqa: F401
    SpdError, lib, LIB_PATH, STATS_DTYPE, CAND_DTYPE,
    SPD_SIGMA_SQRT, SPD_SIGMA_LINEAR, SPD_SIGMA_LINEAR_ANCHORED,
    workspace_bytes, new_workspace, new_stats, read_stats, write_stats, new_candidates, read_candidates,
    spd_stats, spd_stats_merge, spd_boxcar_snr, spd_candidates, spd_search_fused,
    search_host_arena_bytes, spd_search_host, search_host_decimated_arena_bytes, spd_search_host_decimated,
    new_workspace_rows, spd_stats_rows, spd_boxcar_snr_rows, spd_search_fused_rows, spd_stats_rows_noalloc, noalloc_max_rows,
    decimated_level_offset, spd_boxcar_snr_decimated, spd_candidates_decimated, spd_search_fused_decimated,
)
