"""B200-native box-least-squares periodogram (arxiv 1112.1701, section 2.2.2): Python binding of the
C-ABI library libbls_b200.so.  The CUDA kernels are the product; this package only marshals
arguments.  Importing it never builds or falls back to anything on the CPU."""
from .binding import (  # noqa: F401
    BLS_ERR_ARG,
    BLS_ERR_BATCH,
    BLS_ERR_CONFIG,
    BLS_ERR_CUDA,
    BLS_ERR_NULL,
    BLS_ERR_UNSUPPORTED,
    BLS_OK,
    BLS_FLAG_CANONICAL_PHASE,
    BLS_FLAG_FOLD_DEPTH,
    BLS_FLAG_FOLD_WARPS,
    BLS_FLAG_MERGE_WARPS,
    BLS_FLAG_WS_SHAPE,
    BLS_FLAG_NONE,
    BLS_FLAG_NO_SMALL_CTAS,
    BLS_FLAG_WARP_PER_TILE,
    BLS_FLAG_SINGLE_BUFFER,
    BLS_FLAG_WARPS,
    BlsError,
    EXPORTS,
    LIB_PATH,
    PEAK_DTYPE,
    REFINED_DTYPE,
    Plan,
    debug_fold_bins,
    detection_efficiency,
    lib,
    variability,
)
from . import binding  # noqa: F401
