"""B200-native Dykstra projection onto multi-scale window balls (arXiv 1503.03492 hot path).

Thin Python binding over the C ABI of include/smre.h (argument marshalling only; PyTorch
supplies device memory and streams).  Shares nothing with the test oracle.
"""
from .smre import (  # noqa: F401
    SMRE_INCOMPLETE, SMRE_SCHED_AUTO, SMRE_SCHED_GRAPH, SMRE_SCHED_PERSISTENT, SMRE_SCHED_STRIPS, SMRE_STANDARD,
    SmreError, Solver, exported_symbols, lib_path, load_library, smre_create, smre_destroy,
    smre_export_increments, smre_family, smre_info, smre_last_error, smre_last_launch,
    smre_plan_check, smre_project, smre_project_host, calibrate, cumulant2, admm, psf_apply, smre_admm, smre_psf_apply, AdmmParams, smre_calibrate, smre_cumulant2, smre_project_noalloc, smre_project_tol, smre_export_tile_cycles, smre_set_schedule,
)
