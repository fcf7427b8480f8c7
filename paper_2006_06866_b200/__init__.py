"""gce-b200: Conditional Entropy (P, Pdot) period search for NVIDIA B200 (sm_100a).

The product is the C-ABI library declared in include/gce_ce.h (built in-tree as libgce_ce.so from
csrc/gce_ce.cu and csrc/gce_search_family.cu); this package is its ctypes binding.  The binding is loaded on first use of any of its
names and raises ImportError if the library has not been built -- there is no CPU fallback.  Build with
`python -m paper_2006_06866_b200.build` (the build module itself must be importable before the library
exists, hence the lazy load).
"""
import importlib

_BINDING_NAMES = (
    "EXPORTS", "GceError", "Params", "SearchResult", "gce_ce_debug_bins", "gce_ce_debug_histogram",
    "gce_ce_launch_count", "gce_ce_search", "gce_ce_search_host", "gce_ce_validate_host", "gce_ce_version",
    "gce_ce_workspace_bytes", "make_params", "search", "gce_ce_partial_words", "gce_ce_search_partial",
    "gce_ce_merge_partials", "search_period_chunks", "gce_ce_host_release", "gce_ce_probe_rate",
    "gce_ce_search_static", "STATIC_SCRATCH_BYTES", "ERR_STATIC_LIMIT",
)


def __getattr__(name):
    if name in _BINDING_NAMES or name == "binding":
        mod = importlib.import_module(".binding", __name__)
        return mod if name == "binding" else getattr(mod, name)
    raise AttributeError(f"module {__name__!r} has no attribute {name!r}")


def __dir__():
    return sorted(list(globals()) + list(_BINDING_NAMES))
