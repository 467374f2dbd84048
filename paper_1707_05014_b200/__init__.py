"""pct-b200: the hot path of proton-CT reconstruction (arxiv 1707.05014) as CUDA kernels for B200.

The product is ``libpct.so`` (C ABI, ``include/pct.h``); this package is its thin ctypes binding
with the same names.  Importing it requires the built CUDA library -- there is no CPU path.
"""
from ._build import build  # noqa: F401
from .binding import (  # noqa: F401
    EXPORTS,
    FIELDS,
    PCT_PATH_MLP,
    PCT_PATH_SPLINE,
    PCT_TVS_STATIC_MAX_SLOTS,
    PCT_WALK_EXACT,
    PCT_WALK_MIDPOINT,
    PctError,
    lib,
    pct_create,
    pct_debug_block,
    pct_debug_rows,
    pct_destroy,
    pct_get_image,
    pct_get_stats,
    pct_get_tvs_state,
    pct_image_storage,
    pct_iterate,
    pct_iterate_carp,
    pct_measure_peaks,
    pct_profile_sweep,
    pct_set_histories,
    pct_set_histories_host,
    pct_set_histories_xyz,
    pct_set_image,
    pct_set_path_model,
    pct_set_step,
    pct_set_tvs,
    pct_set_walk,
    pct_synchronize,
    pct_tvs_step,
    pct_tvs_step_static,
    pct_version,
)
