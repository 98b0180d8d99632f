"""paper_1612_09491_b200 -- B200 (sm_100a) phase-space-element mass deposit (arXiv:1612.09491).

The product is the C-ABI CUDA library `libpsd.so` (include/psd.h); this package is its thin
ctypes binding (argument marshalling only).  There is no CPU fallback: importing the binding
without the built library, or creating a context without a CUDA device, fails loudly.
"""
from .binding import (  # noqa: F401
    F32, F64, OPT_WEIGHT_MODE, OPT_KERNEL, OPT_COUNTERS, OPT_CHUNK, OPT_CHORD_AXIS, OPT_REFINE_SUBBLOCK, OPT_CLASS_SMALL_CELLS,
    OPT_PATCH_RESTRICT, OPT_PAIR_RECORDS, OPT_ROWS_FP32, OPT_FACE_SHARING,
    SUBBLOCK_UNIT,
    RULE_LITERAL_TOP_DOWN, RULE_BOTTOM_UP_LEVEL_MEAN, PsdError, PsdStats, Context, lib, version,
    EXPORTS, psd_deposit_uniform_static, STATIC_MAX_N, STATIC_MAX_G, STATIC_MAX_PAIRS,
)
