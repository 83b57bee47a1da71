"""B200-native multigrid Gaussian-Plane-Wave collocation / integration (arxiv 2603.24881 hot path).

The product is the C-ABI library built from csrc/ (include/gpw.h); this package only marshals
arguments (binding.py), builds the library (build.py) and generates seeded inputs (inputs.py).
"""
from .binding import *  # noqa: F401,F403
from .binding import EXPORTS, GpwError, Plan, load_library, model_flops  # noqa: F401
