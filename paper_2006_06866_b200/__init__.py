"""gce-b200: Conditional Entropy (P, Pdot) period search for NVIDIA B200 (sm_100a).

The product is the C-ABI library declared in include/gce_ce.h (built in-tree as libgce_ce.so from
csrc/gce_ce.cu); this package is its ctypes binding.  Importing it without the built library raises --
there is no CPU fallback.  Build with `python -m paper_2006_06866_b200.build`.
"""
from .binding import (  # noqa: F401
    EXPORTS, GceError, Params, SearchResult, gce_ce_debug_bins, gce_ce_debug_histogram, gce_ce_launch_count,
    gce_ce_search, gce_ce_search_host, gce_ce_validate_host, gce_ce_version, gce_ce_workspace_bytes, make_params,
    search,
)
