"""B200-native VRC (volumetric-ray-casting) fluence-tally hot path of arXiv:1706.07476.

The product is the C-ABI CUDA library libmonteray.so (include/monteray.h, csrc/); this package
is its thin Python binding.  Importing the package does not load the library; the first use
does, and fails loudly if it has not been built.  There is no CPU fallback.
"""
from .binding import (  # noqa: F401
    EXPORTS,
    LIB_PATH,
    MR_INFO_COARSE_SHIFT,
    MR_INFO_DEFER_DIRECT_PAIRS,
    MR_INFO_DEFERRED,
    MR_INFO_DISTINCT_RECORDS,
    MR_INFO_RECORD_PATH,
    MR_OPT_AGGREGATE_FIRST,
    MR_OPT_BLOCK_THREADS,
    MR_OPT_COARSE_RECORDS,
    MR_OPT_COOP_FLUSH,
    MR_OPT_COPY_THREADS,
    MR_OPT_DEFERRED_TALLY,
    MR_OPT_DEFER_POOL_ENTRIES,
    MR_OPT_DEFER_REGION_SHIFT,
    MR_OPT_FUSED_TALLY,
    MR_OPT_ORDER_MODE,
    MR_OPT_PAIR_RECORDS,
    MR_OPT_PERSISTENT_LANES,
    MR_OPT_RZ_BLOCK_THREADS,
    MR_OPT_TILED_TALLY,
    MR_OPT_WHOLE_BATCH,
    MR_OPT_SORT_RAYS,
    MR_OPT_STAGE_RAYS,
    MR_OPT_TILED_INDEX,
    MR_PATH_NAMES,
    MR_PRECISION_DOUBLE,
    MR_PRECISION_MIXED,
    MR_WHERE_DEVICE,
    MR_WHERE_HOST,
    MonteRay,
    MonteRayError,
    Stats,
    load_library,
    microbench_red,
)
