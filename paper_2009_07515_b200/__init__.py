"""B200-native TPC sector track finder (hot path of arXiv 2009.07515): C-ABI CUDA library + thin binding.

The product is ``libtpc_tracker.so`` (csrc/, sm_100a, ``include/tpc_tracker.h``); this package only
marshals arguments.  Nothing here imports ``oracle/``.
"""
from .binding import (  # noqa: F401
    EXPORTS,
    APEX_CUTS,
    MERGE_CUTS,
    PROTECT_STATIC_MAX_CLUSTERS,
    REMOVAL_CUTS,
    STATUS_BITS,
    Tracker,
    Tracks,
    library_path,
    load_library,
    max_bins_bound,
    pack_params,
    suggest_capacities,
)
