"""B200-native single-pulse detection (arXiv:1910.08324 hot path).

``libspd_b200.so`` (hand-written sm_100a CUDA behind the C ABI of ``include/spd.h``)
does all the work; this package only builds it (``build()``) and marshals
arguments (``binding``).  There is no CPU fallback and nothing here imports the
test oracle.
"""
from ._build import LIB_PATH, build
from .binding import (  # noqa: F401
    CANDIDATE_DTYPE, EXPORTS, Plan, SpdError,
    SPD_FLAG_FORCE_GENERIC, SPD_FLAG_BLOCK_TREE, SPD_FLAG_GENERIC_WORKSPACE, SPD_FLAG_WIDTH_U8,
    SPD_OPT_SEGMENTS_PER_ROW, SPD_OPT_HOST_ROWS_PER_BLOCK, spd_plan_set_option, spd_row_stats_converge, spd_cluster_candidates,
    spd_run_host_candidates, SPD_PATH_DYADIC_TREE, SPD_PATH_GENERIC, SPD_PATH_IGRID_TREE, SPD_PATH_GRID,
    spd_separation_generate, spd_plan_create_grid, spd_width_sigma, spd_run_sigma_w,
    candidates_to_numpy, load, spd_destroy, spd_find_candidates, spd_last_error_string,
    spd_plan_create, spd_plan_destroy, spd_plan_get_info, spd_plan_get_widths, spd_run,
    spd_run_flagged, spd_find_candidates_flagged, spd_row_stats, spd_row_stats_static,
    SPD_STATIC_MAX_ROWS, SPD_STATIC_MAX_PARTIALS, spd_plan_get_iterations, spd_run_iterations,
    spd_run_host, spd_version, spd_width_set_generate,
)

__all__ = [
    "LIB_PATH", "build", "load", "Plan", "SpdError", "EXPORTS", "CANDIDATE_DTYPE",
    "SPD_FLAG_FORCE_GENERIC", "SPD_FLAG_BLOCK_TREE", "SPD_FLAG_GENERIC_WORKSPACE", "SPD_FLAG_WIDTH_U8",
    "SPD_OPT_SEGMENTS_PER_ROW", "SPD_OPT_HOST_ROWS_PER_BLOCK", "spd_plan_set_option", "spd_row_stats_converge", "spd_cluster_candidates",
    "spd_run_host_candidates", "SPD_PATH_DYADIC_TREE", "SPD_PATH_GENERIC", "SPD_PATH_IGRID_TREE", "SPD_PATH_GRID",
    "spd_separation_generate", "spd_plan_create_grid", "spd_width_sigma", "spd_run_sigma_w",
    "spd_width_set_generate", "spd_plan_create", "spd_plan_destroy", "spd_destroy",
    "spd_plan_get_widths", "spd_plan_get_info", "spd_run", "spd_find_candidates",
    "spd_run_flagged", "spd_find_candidates_flagged", "spd_row_stats", "spd_row_stats_static",
    "SPD_STATIC_MAX_ROWS", "SPD_STATIC_MAX_PARTIALS", "spd_plan_get_iterations", "spd_run_iterations",
    "spd_run_host", "spd_last_error_string", "spd_version", "candidates_to_numpy",
]
