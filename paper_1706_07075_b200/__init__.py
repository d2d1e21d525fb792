"""paper_1706_07075_b200 -- B200-native list-mode TOF-MLEM hot path (arxiv 1706.07075).

`csrc/` holds the hand-written sm_100a CUDA kernels and the C ABI (include/tofmlem.h);
`tofmlem.py` is the ctypes binding (argument marshalling only); `build.py` compiles libtofmlem.so in-tree.
"""
from .tofmlem import (Context, Events, Grid, Scanner, Stats, TofMlemError, lib, make_grid, version,  # noqa: F401
                      em_correction_static,
                      OPT_PROJECTOR, OPT_SAMPLES_K, OPT_SENS_FLOOR_REL, OPT_SHELL_MM, OPT_TILE_LOG2,
                      OPT_TRUNC_SIGMAS, OPT_CTA_INTERLEAVE, OPT_EM_VARIANT, OPT_SUBBINS, OPT_MEDIAN, OPT_CACHE_SHARE, OPT_CORR_BRICKS, OPT_DETERMINISTIC, OPT_TILE_MIN_EVENTS, OPT_TILE_CHECK, OPT_TILE_MAX_EVENTS, OPT_REGION_PLAN, OPT_REGION_OVERLAP, OPT_L2_PERSIST, OPT_TILE_MIN_ITEMS, OPT_SENS_SORT, OPT_CONCURRENT, OPT_WARP_WALK, Plan, PROJECTOR_SIDDON, PROJECTOR_SAMPLED, SYMBOLS, EVENT_FIELDS)
