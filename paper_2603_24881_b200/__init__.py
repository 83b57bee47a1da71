"""B200-native multigrid Gaussian-Plane-Wave collocation / integration (arxiv 2603.24881 hot path).

The product is the C-ABI library built from csrc/ (include/gpw.h); this package only marshals
arguments (binding.py), builds the library (build.py) and generates seeded inputs (inputs.py).
"""
from .binding import (GpwError, Plan, gpw_build_pairs, gpw_dfma_peak, gpw_eval_mat, gpw_eval_rho, gpw_free_plan,  # noqa: F401
                      gpw_interp_up, gpw_plan_export_tasks, gpw_plan_get_timing, gpw_plan_info,
                      gpw_plan_set_timing, gpw_restrict_down,
                      load_library, model_flops)
