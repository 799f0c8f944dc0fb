"""B200-native open-boundary RPY mobility (M.F) and Lanczos sqrt(M).W -- Python binding of liblm.

The product is the C-ABI CUDA library ``liblm.so`` (``include/lm.h``).  This package only
marshals arguments (``binding.py``); every step of the path runs in the library's kernels.
``workloads.py`` holds the seeded synthetic inputs of the five benchmark configs.
"""
from . import workloads  # noqa: F401
from .binding import (  # noqa: F401
    LM_E_ANGULAR, LM_E_CUDA, LM_E_INVALID, LM_E_NOCONV, LM_E_NOPOS, LM_E_NULL, LM_F32, LM_F64, LM_OK,
    LM_OPT_ACCUMULATE_F64, LM_OPT_GATHER_IN_PLACE, LM_OPT_GRAPH_REPLAY, LM_OPT_J_SPLITS, LM_OPT_LANCZOS_RULE, LM_OPT_SHARE_FIRST_APPLY, LM_OPT_SMALL_KERNEL, LM_RULE_ESTIMATE, LM_RULE_STEP,
    LmError, Solver, lib, lm_dist_row_block, lm_dist_unique_id, lm_mdot_static_max_n, lm_version, mdot_static,
)
