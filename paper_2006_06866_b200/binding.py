"""Thin ctypes binding of include/gce_ce.h (argument marshalling only).

Every step of the path runs in the CUDA kernels of libgce_ce.so.  PyTorch is used for device memory and
the stream handle; nothing here computes.  There is no CPU fallback: if the library has not been built
(`python -m paper_2006_06866_b200.build`) importing this module raises.
"""
from __future__ import annotations

import contextlib
import ctypes as C
import os

import numpy as np
import torch

from .build import LIB

if not os.path.exists(LIB):
    raise ImportError(f"{LIB} is missing: run `python -m paper_2006_06866_b200.build` (nvcc, sm_100a). "
                      "There is no CPU fallback.")

_lib = C.CDLL(LIB)

MAX_BINS, MAX_TOPK, MAX_POINTS, MAX_POINTS_OVERLAP, MAX_POINTS_WIDE = 64, 32, 65535, 32767, 1 << 26
OK, ERR_POINTER, ERR_RANGE, ERR_WORKSPACE, ERR_CUDA = 0, -1, -2, -3, -4
ERR_STATIC_LIMIT = -5                 # gce_ce_search_static: the call needs more than STATIC_SCRATCH_BYTES of scratch
STATIC_SCRATCH_BYTES = 8 << 20        # GCE_CE_STATIC_SCRATCH_BYTES
FOLD_AUTO, FOLD_PLAIN, FOLD_PAIR, FOLD_QUAD, FOLD_GENERIC, FOLD_PDOT_ZERO = range(6)   # gce_ce_debug_bins fold_mode


class Params(C.Structure):
    _fields_ = [("n_phase_bins", C.c_int32), ("n_mag_bins", C.c_int32), ("top_k", C.c_int32),
                ("ce_fp64", C.c_int32), ("want_stats", C.c_int32), ("overlap", C.c_int32),
                ("max_lc_points", C.c_int32), ("normalise", C.c_int32), ("ev_search_begin", C.c_void_p),
                ("ev_search_end", C.c_void_p), ("filter_ids", C.c_void_p)]


_vp, _i32, _i64, _sz = C.c_void_p, C.c_int32, C.c_int64, C.c_size_t
_lib.gce_ce_workspace_bytes.argtypes = [_i64, _i32, _i64, _i64, C.POINTER(Params), C.POINTER(_sz)]
_lib.gce_ce_search.argtypes = [_vp, _vp, _vp, _i32, _i64, _vp, _i64, _vp, _i64, C.POINTER(Params),
                               _vp, _vp, _vp, _vp, _vp, _sz, _vp]
_lib.gce_ce_search_static.argtypes = [_vp, _vp, _vp, _i32, _i64, _vp, _i64, _vp, _i64, C.POINTER(Params),
                                      _vp, _vp, _vp, _vp, _vp]
_lib.gce_ce_search_static.restype = C.c_int
_lib.gce_ce_search_host.argtypes = [_vp, _vp, _vp, _i32, _vp, _i64, _vp, _i64, C.POINTER(Params), _vp, _vp, _vp, _vp]
_lib.gce_ce_debug_histogram.argtypes = [_vp, _vp, _vp, _i32, _i64, _vp, _i64, _vp, _i64, C.POINTER(Params),
                                        _vp, _i64, _vp, _vp, _vp, _sz, _vp]
_lib.gce_ce_debug_bins.argtypes = [_vp, _vp, _vp, _i32, _vp, _i64, _vp, _i64, C.POINTER(Params), _i32, _i64, _i32,
                                   _vp, _vp, _vp, _vp]
_lib.gce_ce_partial_words.argtypes = [_i32]
_lib.gce_ce_partial_words.restype = _sz
_lib.gce_ce_search_partial.argtypes = [_vp, _vp, _vp, _i32, _i64, _vp, _i64, _vp, _i64, C.POINTER(Params), _i64, _i64,
                                       _vp, _vp, _vp, _sz, _vp]
_lib.gce_ce_merge_partials.argtypes = [_vp, _i32, _i32, C.POINTER(Params), _vp, _vp, _vp, _vp]
_lib.gce_ce_merge_partials_to_partial.argtypes = [_vp, _i32, _i32, C.POINTER(Params), _vp, _vp]
_lib.gce_ce_merge_partials_to_partial.restype = C.c_int
_lib.gce_ce_validate_host.argtypes = [_vp, _vp, _vp, _i32, _vp, _i64, _vp, _i64, C.POINTER(Params)]
_lib.gce_ce_launch_count.argtypes = [_i32, _i64, C.POINTER(Params), C.c_int]
_lib.gce_ce_probe_rate.argtypes = [_i32, C.POINTER(C.c_double)]
_lib.gce_ce_strerror.argtypes = [C.c_int]
_lib.gce_ce_strerror.restype = C.c_char_p
_lib.gce_ce_version.restype = C.c_char_p
for _f in ("gce_ce_workspace_bytes", "gce_ce_search", "gce_ce_search_host", "gce_ce_debug_histogram",
           "gce_ce_debug_bins", "gce_ce_validate_host", "gce_ce_launch_count", "gce_ce_last_cuda_error",
           "gce_ce_search_partial", "gce_ce_merge_partials", "gce_ce_merge_partials_to_partial", "gce_ce_host_release",
           "gce_ce_probe_rate"):
    getattr(_lib, _f).restype = C.c_int

EXPORTS = ("gce_ce_workspace_bytes", "gce_ce_search", "gce_ce_search_host", "gce_ce_debug_histogram",
           "gce_ce_debug_bins", "gce_ce_validate_host", "gce_ce_launch_count", "gce_ce_strerror",
           "gce_ce_last_cuda_error", "gce_ce_version", "gce_ce_partial_words", "gce_ce_search_partial",
           "gce_ce_merge_partials", "gce_ce_merge_partials_to_partial", "gce_ce_host_release", "gce_ce_probe_rate",
           "gce_ce_search_static")


class GceError(RuntimeError):
    def __init__(self, code):
        self.code = int(code)
        msg = _lib.gce_ce_strerror(self.code).decode()
        if self.code == ERR_CUDA:
            msg += f" [cudaError {_lib.gce_ce_last_cuda_error()}]"
        super().__init__(f"gce_ce error {self.code}: {msg}")


def _check(rc):
    if rc != OK:
        raise GceError(rc)


def gce_ce_version() -> str:
    return _lib.gce_ce_version().decode()


def make_params(n_phase_bins, n_mag_bins, top_k=0, ce_fp64=False, want_stats=False, overlap=False,
                ev_search_begin=None, ev_search_end=None, max_lc_points=0, normalise=False, filter_ids=None) -> Params:
    """ev_search_begin / ev_search_end: optional torch.cuda.Event(enable_timing=True) objects that have been
    recorded at least once (torch creates the cudaEvent_t lazily).  max_lc_points: upper bound on the longest light
    curve when that exceeds MAX_POINTS (32-bit counters).  normalise / filter_ids: the paper's per-filter median / std
    normalisation; filter_ids is an int32 tensor [total_points] on the device (on the host for gce_ce_search_host)
    or None.  The caller keeps the events and filter_ids alive."""
    def _ev(e):
        return None if e is None else C.c_void_p(e.cuda_event)
    if filter_ids is not None:
        if filter_ids.dtype != torch.int32 or not filter_ids.is_contiguous():
            raise TypeError("filter_ids: contiguous int32 tensor expected")
    return Params(int(n_phase_bins), int(n_mag_bins), int(top_k), int(bool(ce_fp64)), int(bool(want_stats)),
                  int(bool(overlap)), int(max_lc_points), int(bool(normalise)), _ev(ev_search_begin), _ev(ev_search_end),
                  None if filter_ids is None else C.c_void_p(filter_ids.data_ptr()))


def gce_ce_workspace_bytes(total_points, n_lc, n_p, n_pdot, prm: Params) -> int:
    out = _sz(0)
    _check(_lib.gce_ce_workspace_bytes(int(total_points), int(n_lc), int(n_p), int(n_pdot), C.byref(prm), C.byref(out)))
    return int(out.value)


def gce_ce_launch_count(n_lc, n_p, prm: Params, partial=False) -> int:
    return int(_lib.gce_ce_launch_count(int(n_lc), int(n_p), C.byref(prm), int(bool(partial))))


def _dev(t, dtype):
    if t is None:
        return None
    if not (isinstance(t, torch.Tensor) and t.is_cuda and t.dtype == dtype and t.is_contiguous()):
        raise TypeError(f"expected a contiguous CUDA tensor of {dtype}")
    return t


def _ptr(t):
    return None if t is None else C.c_void_p(t.data_ptr())


def _stream(stream):
    s = torch.cuda.current_stream() if stream is None else stream
    return C.c_void_p(s.cuda_stream)


def gce_ce_search(times, mags, lc_offsets, periods, pdots, prm: Params, out_ce=None, out_best_idx=None,
                  out_best_ce=None, out_stats=None, workspace=None, stream=None):
    """Enqueue the search on `stream` (default: torch's current stream).  All tensors are CUDA tensors the caller
    owns; see include/gce_ce.h for layouts.  Returns nothing; outputs are the tensors passed in."""
    times, mags = _dev(times, torch.float64), _dev(mags, torch.float64)
    lc_offsets = _dev(lc_offsets, torch.int64)
    periods, pdots = _dev(periods, torch.float64), _dev(pdots, torch.float64)
    n_lc = lc_offsets.numel() - 1
    ce_dtype = torch.float64 if prm.ce_fp64 else torch.float32
    if out_ce is not None:
        _dev(out_ce, ce_dtype)
        if out_ce.numel() != n_lc * periods.numel() * pdots.numel():
            raise ValueError("out_ce has the wrong number of elements")
    if out_best_idx is not None:
        _dev(out_best_idx, torch.int64)
        if out_best_idx.numel() != n_lc * prm.top_k:
            raise ValueError("out_best_idx has the wrong number of elements")
    if out_best_ce is not None:
        _dev(out_best_ce, torch.float32)
        if out_best_ce.numel() != n_lc * prm.top_k:
            raise ValueError("out_best_ce has the wrong number of elements")
    if out_stats is not None:
        _dev(out_stats, torch.float64)
    if workspace is None or not workspace.is_cuda:
        raise TypeError("workspace must be a CUDA tensor (see gce_ce_workspace_bytes)")
    _check(_lib.gce_ce_search(_ptr(times), _ptr(mags), _ptr(lc_offsets), n_lc, times.numel(), _ptr(periods),
                              periods.numel(), _ptr(pdots), pdots.numel(), C.byref(prm), _ptr(out_ce),
                              _ptr(out_best_idx), _ptr(out_best_ce), _ptr(out_stats), _ptr(workspace),
                              workspace.numel() * workspace.element_size(), _stream(stream)))


def gce_ce_search_static(times, mags, lc_offsets, periods, pdots, prm: Params, out_ce=None, out_best_idx=None,
                         out_best_ce=None, out_stats=None, stream=None):
    """gce_ce_search without a workspace argument, for callers that are not allowed to allocate device memory.

    Meant for code that is a guest in another program's GPU process (an alert broker, a pipeline plug-in): the host
    program passes in input and output tensors and a stream but owns all the memory, and cudaMalloc is ruled out there
    because it stalls the whole device and can fail once the host has taken the card's memory.  The scratch the search
    needs sits in an 8 MiB array (STATIC_SCRATCH_BYTES) built into libgce_ce.so, so this call -- the wrapper included --
    creates no tensor and the library calls no allocator.  Same kernels, same results as gce_ce_search.

    Raises GceError with code ERR_STATIC_LIMIT (nothing enqueued) when gce_ce_workspace_bytes(...) for these sizes is
    larger than STATIC_SCRATCH_BYTES.  The first call on a device looks up the array's address; make it before any
    stream capture starts.  All calls on a device share the one array: calls that can run on the GPU at the same time
    (unordered streams, several threads) corrupt each other, so keep them ordered on one stream or with events."""
    times, mags = _dev(times, torch.float64), _dev(mags, torch.float64)
    lc_offsets = _dev(lc_offsets, torch.int64)
    periods, pdots = _dev(periods, torch.float64), _dev(pdots, torch.float64)
    n_lc = lc_offsets.numel() - 1
    _dev(out_ce, torch.float64 if prm.ce_fp64 else torch.float32)
    _dev(out_best_idx, torch.int64)
    _dev(out_best_ce, torch.float32)
    _dev(out_stats, torch.float64)
    for t, n, what in ((out_ce, n_lc * periods.numel() * pdots.numel(), "out_ce"), (out_best_idx, n_lc * prm.top_k, "out_best_idx"),
                       (out_best_ce, n_lc * prm.top_k, "out_best_ce"), (out_stats, n_lc * 4, "out_stats")):
        if t is not None and t.numel() != n:
            raise ValueError(f"{what} has the wrong number of elements")
    _check(_lib.gce_ce_search_static(_ptr(times), _ptr(mags), _ptr(lc_offsets), n_lc, times.numel(), _ptr(periods),
                                     periods.numel(), _ptr(pdots), pdots.numel(), C.byref(prm), _ptr(out_ce),
                                     _ptr(out_best_idx), _ptr(out_best_ce), _ptr(out_stats), _stream(stream)))


def gce_ce_host_release() -> None:
    """Return the cached device memory of the host entry points to the driver."""
    _lib.gce_ce_host_release.restype = C.c_int
    _check(_lib.gce_ce_host_release())


PROBE_FP64, PROBE_SHARED = 0, 1


def gce_ce_probe_rate(kind) -> float:
    """Measured per-SM issue rate on the current device: FP64 lane-ops / SM / clk or shared wavefronts / SM / clk."""
    out = C.c_double(0.0)
    _check(_lib.gce_ce_probe_rate(int(kind), C.byref(out)))
    return float(out.value)


def gce_ce_partial_words(top_k) -> int:
    return int(_lib.gce_ce_partial_words(int(top_k)))


def gce_ce_search_partial(times, mags, lc_offsets, periods, pdots, prm: Params, ip_begin, ip_end, out_partial,
                          out_ce=None, workspace=None, stream=None):
    """Search the periods [ip_begin, ip_end) of the grid; out_partial int64 [n_lc][gce_ce_partial_words(top_k)]."""
    times, mags = _dev(times, torch.float64), _dev(mags, torch.float64)
    lc_offsets = _dev(lc_offsets, torch.int64)
    periods, pdots = _dev(periods, torch.float64), _dev(pdots, torch.float64)
    n_lc = lc_offsets.numel() - 1
    _dev(out_partial, torch.int64)
    if out_partial.numel() != n_lc * gce_ce_partial_words(prm.top_k):
        raise ValueError("out_partial has the wrong number of elements")
    if out_ce is not None:
        _dev(out_ce, torch.float64 if prm.ce_fp64 else torch.float32)
        if out_ce.numel() != n_lc * (int(ip_end) - int(ip_begin)) * pdots.numel():
            raise ValueError("out_ce has the wrong number of elements")
    if workspace is None or not workspace.is_cuda:
        raise TypeError("workspace must be a CUDA tensor (see gce_ce_workspace_bytes)")
    _check(_lib.gce_ce_search_partial(_ptr(times), _ptr(mags), _ptr(lc_offsets), n_lc, times.numel(), _ptr(periods),
                                      periods.numel(), _ptr(pdots), pdots.numel(), C.byref(prm), int(ip_begin),
                                      int(ip_end), _ptr(out_ce), _ptr(out_partial), _ptr(workspace),
                                      workspace.numel() * workspace.element_size(), _stream(stream)))


def gce_ce_merge_partials(partials, n_parts, n_lc, prm: Params, out_best_idx=None, out_best_ce=None, out_stats=None,
                          stream=None):
    """Merge int64 [n_parts][n_lc][words] partial blobs into the final selection / Eq. 5 statistics."""
    _dev(partials, torch.int64)
    if partials.numel() != int(n_parts) * int(n_lc) * gce_ce_partial_words(prm.top_k):
        raise ValueError("partials has the wrong number of elements")
    if out_best_idx is not None:
        _dev(out_best_idx, torch.int64)
    if out_best_ce is not None:
        _dev(out_best_ce, torch.float32)
    if out_stats is not None:
        _dev(out_stats, torch.float64)
    _check(_lib.gce_ce_merge_partials(_ptr(partials), int(n_parts), int(n_lc), C.byref(prm), _ptr(out_best_idx),
                                      _ptr(out_best_ce), _ptr(out_stats), _stream(stream)))


def gce_ce_debug_histogram(times, mags, lc_offsets, periods, pdots, prm: Params, trial_q, out_counts, out_ce_at=None,
                           workspace=None, stream=None):
    """The search kernel of this grid in dump mode: count tables (and CE) of the listed flat trials."""
    n_lc = lc_offsets.numel() - 1
    _dev(trial_q, torch.int64)
    _dev(out_counts, torch.int32)  # uint32 counts viewed as int32 storage
    if out_counts.numel() != n_lc * trial_q.numel() * prm.n_phase_bins * prm.n_mag_bins:
        raise ValueError("out_counts has the wrong number of elements")
    if out_ce_at is not None:
        _dev(out_ce_at, torch.float64)
    _check(_lib.gce_ce_debug_histogram(_ptr(times), _ptr(mags), _ptr(lc_offsets), n_lc, times.numel(), _ptr(periods),
                                       periods.numel(), _ptr(pdots), pdots.numel(), C.byref(prm), _ptr(trial_q),
                                       trial_q.numel(), _ptr(out_counts), _ptr(out_ce_at), _ptr(workspace),
                                       workspace.numel() * workspace.element_size(), _stream(stream)))


def gce_ce_debug_bins(times, mags, lc_offsets, periods, pdots, prm: Params, lc, q, out_phase_bin, out_mag_bin,
                      fold_mode=FOLD_AUTO, out_fold_mode=None, stream=None):
    n_lc = lc_offsets.numel() - 1
    _dev(out_phase_bin, torch.int32)
    _dev(out_mag_bin, torch.int32)
    if out_fold_mode is not None:
        _dev(out_fold_mode, torch.int32)
    _check(_lib.gce_ce_debug_bins(_ptr(times), _ptr(mags), _ptr(lc_offsets), n_lc, _ptr(periods), periods.numel(),
                                  _ptr(pdots), pdots.numel(), C.byref(prm), int(lc), int(q), int(fold_mode),
                                  _ptr(out_phase_bin), _ptr(out_mag_bin), _ptr(out_fold_mode), _stream(stream)))


def _host(a, dtype):
    """Host buffer -> (object keeping it alive, address).  Accepts numpy arrays and (pinned) CPU torch tensors."""
    if a is None:
        return None, None
    if isinstance(a, torch.Tensor):
        if a.is_cuda or not a.is_contiguous():
            raise TypeError("expected a contiguous CPU tensor")
        return a, C.c_void_p(a.data_ptr())
    a = np.ascontiguousarray(a, dtype=dtype)
    return a, C.c_void_p(a.ctypes.data)


def gce_ce_search_host(times, mags, lc_offsets, periods, pdots, prm: Params, out_ce=None, out_best_idx=None,
                       out_best_ce=None, out_stats=None):
    """Same call with HOST buffers (numpy or CPU torch tensors); copies in, runs, copies out, synchronises."""
    keep = []
    ptrs = []
    for a, dt in ((times, np.float64), (mags, np.float64), (lc_offsets, np.int64), (periods, np.float64),
                  (pdots, np.float64)):
        k, p = _host(a, dt)
        keep.append(k)
        ptrs.append(p)
    n_lc = (keep[2].numel() if isinstance(keep[2], torch.Tensor) else keep[2].shape[0]) - 1
    n_p = keep[3].numel() if isinstance(keep[3], torch.Tensor) else keep[3].shape[0]
    n_pdot = keep[4].numel() if isinstance(keep[4], torch.Tensor) else keep[4].shape[0]
    outs = []
    for a in (out_ce, out_best_idx, out_best_ce, out_stats):
        if a is None:
            outs.append(None)
        elif isinstance(a, torch.Tensor):
            outs.append(C.c_void_p(a.data_ptr()))
        else:
            if not a.flags["C_CONTIGUOUS"]:
                raise TypeError("output arrays must be C-contiguous")
            outs.append(C.c_void_p(a.ctypes.data))
    _check(_lib.gce_ce_search_host(ptrs[0], ptrs[1], ptrs[2], n_lc, ptrs[3], n_p, ptrs[4], n_pdot, C.byref(prm),
                                   outs[0], outs[1], outs[2], outs[3]))


def gce_ce_validate_host(times, mags, lc_offsets, periods, pdots, prm: Params) -> int:
    t, m = np.ascontiguousarray(times, np.float64), np.ascontiguousarray(mags, np.float64)
    o = np.ascontiguousarray(lc_offsets, np.int64)
    p, pd = np.ascontiguousarray(periods, np.float64), np.ascontiguousarray(pdots, np.float64)
    return int(_lib.gce_ce_validate_host(C.c_void_p(t.ctypes.data), C.c_void_p(m.ctypes.data), C.c_void_p(o.ctypes.data),
                                         o.shape[0] - 1, C.c_void_p(p.ctypes.data), p.shape[0],
                                         C.c_void_p(pd.ctypes.data), pd.shape[0], C.byref(prm)))


# ------------------------------------------------------------------------------------------ convenience
class SearchResult:
    __slots__ = ("ce", "best_idx", "best_ce", "stats")

    def __init__(self, ce, best_idx, best_ce, stats):
        self.ce, self.best_idx, self.best_ce, self.stats = ce, best_idx, best_ce, stats


def search(times, mags, lc_offsets, periods, pdots, n_phase_bins, n_mag_bins, top_k=0, want_cube=True,
           ce_fp64=False, want_stats=False, overlap=False, workspace=None, stream=None, normalise=False,
           filter_ids=None) -> SearchResult:
    """Allocate outputs + workspace with torch and call gce_ce_search (device tensors in, device tensors out).
    When the batch holds more points than one light curve may have with 16-bit counters, the longest light curve is read
    back (one synchronisation) to announce it to the library (max_lc_points)."""
    longest = 0
    if times.numel() > (MAX_POINTS_OVERLAP if overlap else MAX_POINTS) and lc_offsets.numel() > 1:
        longest = int((lc_offsets[1:] - lc_offsets[:-1]).max().item())
    prm = make_params(n_phase_bins, n_mag_bins, top_k, ce_fp64, want_stats, overlap, max_lc_points=longest,
                      normalise=normalise, filter_ids=filter_ids)
    dev = times.device
    n_lc = lc_offsets.numel() - 1
    n_p, n_pdot = periods.numel(), pdots.numel()
    ce = torch.empty((n_lc, n_p, n_pdot), dtype=torch.float64 if ce_fp64 else torch.float32, device=dev) if want_cube else None
    bidx = torch.empty((n_lc, top_k), dtype=torch.int64, device=dev) if top_k > 0 else None
    bce = torch.empty((n_lc, top_k), dtype=torch.float32, device=dev) if top_k > 0 else None
    stats = torch.empty((n_lc, 4), dtype=torch.float64, device=dev) if want_stats else None
    if workspace is None:
        nbytes = gce_ce_workspace_bytes(times.numel(), n_lc, n_p, n_pdot, prm)
        workspace = torch.empty(nbytes, dtype=torch.uint8, device=dev)
    gce_ce_search(times, mags, lc_offsets, periods, pdots, prm, ce, bidx, bce, stats, workspace, stream)
    return SearchResult(ce, bidx, bce, stats)


def search_period_chunks(times, mags, lc_offsets, periods, pdots, n_phase_bins, n_mag_bins, chunks, top_k=1,
                         want_stats=True, overlap=False, ce_fp64=False, cube_sink=None, dist=None, stream=None,
                         max_lc_points=0, normalise=False, filter_ids=None) -> SearchResult:
    """The search over a list of period ranges [(ip_begin, ip_end), ...] -- this process's share of the grid -- merged
    exactly (batches bound the memory, their minima are merged; period-axis split when
    there are fewer light curves than GPUs).  One workspace and one partial buffer are reused for every chunk.
    cube_sink(ip_begin, ip_end, ce_slice) receives each non-empty cube slice [n_lc][ip_end - ip_begin][n_pdot] (device
    tensor, overwritten by the next chunk) when given.  With `dist` (initialised torch.distributed) the partial blobs of
    all ranks are all-gathered -- n_lc x (2 top_k + 10) int64 per rank, the only exchange of the path -- and every rank
    merges them, so every rank returns the whole grid's selection.  NCCL gathers the device blobs in stream order; a
    backend without CUDA support (gloo) gets them staged through the host (kilobytes).  Argument marshalling and
    plumbing only: the merge runs in the library's kernels."""
    prm = make_params(n_phase_bins, n_mag_bins, top_k, ce_fp64, want_stats, overlap, max_lc_points=max_lc_points,
                      normalise=normalise, filter_ids=filter_ids)
    dev = times.device
    n_lc = lc_offsets.numel() - 1
    n_pdot = pdots.numel()
    words = gce_ce_partial_words(top_k)
    chunks = [(int(a), int(b)) for a, b in chunks]
    widest = max([b - a for a, b in chunks], default=0)
    # everything below is ordered on `stream`: torch allocations, the collective and the library's kernels alike
    with torch.cuda.stream(stream) if stream is not None else contextlib.nullcontext():
        ws = torch.empty(gce_ce_workspace_bytes(times.numel(), n_lc, widest, n_pdot, prm), dtype=torch.uint8, device=dev)
        parts = torch.empty((max(len(chunks), 1), n_lc, words), dtype=torch.int64, device=dev)
        ce = None
        if cube_sink is not None and widest > 0:
            ce = torch.empty(n_lc * widest * n_pdot, dtype=torch.float64 if ce_fp64 else torch.float32, device=dev)
        if not chunks:  # a rank with no periods still contributes a (neutral) blob
            gce_ce_search_partial(times, mags, lc_offsets, periods, pdots, prm, 0, 0, parts[0], None, ws, stream)
        for i, (a, b) in enumerate(chunks):
            sl = ce[: n_lc * (b - a) * n_pdot] if (ce is not None and b > a) else None
            gce_ce_search_partial(times, mags, lc_offsets, periods, pdots, prm, a, b, parts[i], sl, ws, stream)
            if cube_sink is not None and sl is not None:
                cube_sink(a, b, sl.view(n_lc, b - a, n_pdot))
        n_parts = parts.shape[0]
        if dist is not None and dist.is_initialized() and dist.get_world_size() > 1:
            # ranks may hold different numbers of chunks: merge locally first, then exchange one blob array per rank
            local = torch.empty((1, n_lc, words), dtype=torch.int64, device=dev)
            _merge_to_partial(parts, n_parts, n_lc, prm, local, stream)
            if str(dist.get_backend()) == "nccl":
                gathered = [torch.empty_like(local) for _ in range(dist.get_world_size())]
                dist.all_gather(gathered, local)
                parts = torch.cat(gathered, dim=0)
            else:
                host = local.cpu()  # synchronises this stream
                gathered = [torch.empty_like(host) for _ in range(dist.get_world_size())]
                dist.all_gather(gathered, host)
                parts = torch.cat(gathered, dim=0).to(dev)
            n_parts = parts.shape[0]
        bidx = torch.empty((n_lc, top_k), dtype=torch.int64, device=dev) if top_k > 0 else None
        bce = torch.empty((n_lc, top_k), dtype=torch.float32, device=dev) if top_k > 0 else None
        stats = torch.empty((n_lc, 4), dtype=torch.float64, device=dev) if want_stats else None
        gce_ce_merge_partials(parts, n_parts, n_lc, prm, bidx, bce, stats, stream)
    return SearchResult(None, bidx, bce, stats)


def _merge_to_partial(parts, n_parts, n_lc, prm, out_partial, stream=None):
    _check(_lib.gce_ce_merge_partials_to_partial(_ptr(parts), int(n_parts), int(n_lc), C.byref(prm), _ptr(out_partial),
                                                 _stream(stream)))
