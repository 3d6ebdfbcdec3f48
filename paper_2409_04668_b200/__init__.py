"""paper_2409_04668_b200 -- B200-native hot path of MC/DC (arXiv 2409.04668): the time-dependent
multigroup Monte Carlo particle-history transport loop as a C-ABI CUDA library (libmcdc.so, sm_100a)
plus this thin binding.  Every step of the path runs in the library's kernels; Python only marshals
arguments and lends PyTorch device memory and a stream.  There is no CPU fallback.
"""
from .api import (  # noqa: F401
    McdcError,
    Problem,
    lib,
    lib_path,
    mcdc_problem_create,
    mcdc_problem_create_csg,
    mcdc_problem_destroy,
    mcdc_problem_reset,
    mcdc_problem_info_get,
    mcdc_kernel_info_get,
    mcdc_workspace_size,
    mcdc_workspace_size_async,
    mcdc_workspace_bind,
    mcdc_run,
    mcdc_run_ex,
    mcdc_run_eigenvalue,
    mcdc_tallies_get,
    mcdc_tally_sums_get,
    mcdc_collision_tally_enable,
    mcdc_collision_tallies_get,
    mcdc_counters_get,
    mcdc_census_get,
    mcdc_history_events_get,
    mcdc_technique_set,
    mcdc_census_after_get,
    mcdc_state_size,
    mcdc_state_export,
    mcdc_state_import,
    mcdc_strerror,
    mcdc_version,
    EXPORTED_SYMBOLS,
)
