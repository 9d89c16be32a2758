"""B200-native multi-view Richardson-Lucy deconvolution (arXiv 1308.0730): Python binding of libmvd.so.

The product is the C-ABI library (include/mvd.h; sources under csrc/).  This package only marshals
arguments; importing it does not load the library and does not need a GPU.  Using it does: there
is no CPU path (oracle/ is test infrastructure and is never imported from here).
"""
from .binding import (  # noqa: F401
    KERNEL_MODES,
    LIB_PATH,
    SYMBOLS,
    VARIANTS,
    Deconvolver,
    MvdError,
    ViewParallelDeconvolver,
    reduce_sum,
    reduce_sum_static,
    split_views,
    deconvolve_blocked,
    load_library,
    plan_dims,
    workspace_size,
)
