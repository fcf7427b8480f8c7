"""ctypes front-end of the CPU oracle (oracle/gce_oracle.c).

TEST INFRASTRUCTURE, NOT THE PRODUCT: only tests/, __graft_entry__.smoke() and bench.py's
cpu_baseline / --impl reference legs may import this package.  It shares no code with
paper_2006_06866_b200 and does not import it.  Every function takes and returns host numpy
arrays; all arithmetic happens in the C file (this module only marshals arguments).
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "gce_oracle.c")
_LIB = os.path.join(_HERE, "libgce_oracle.so")
# -ffp-contract=off is required: a fused multiply-add would change phase-bin indices.
CFLAGS = ["-O2", "-std=c11", "-ffp-contract=off", "-fno-fast-math", "-fopenmp", "-shared", "-fPIC"]

_lib = None


def build(force: bool = False) -> str:
    """Compile the oracle with gcc (in-tree) if the .so is missing or older than the source."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        tmp = _LIB + f".tmp{os.getpid()}"
        subprocess.check_call(["gcc", *CFLAGS, "-o", tmp, _SRC, "-lm"])
        os.replace(tmp, _LIB)
    return _LIB


_f64p = C.POINTER(C.c_double)
_i64p = C.POINTER(C.c_int64)
_i32p = C.POINTER(C.c_int32)


def _p(a, typ):
    return a.ctypes.data_as(typ)


def _f64(a):
    return np.ascontiguousarray(a, dtype=np.float64)


def _i64(a):
    return np.ascontiguousarray(a, dtype=np.int64)


def lib():
    global _lib
    if _lib is None:
        build()
        L = C.CDLL(_LIB)
        L.gce_oracle_preprocess.argtypes = [_f64p, _f64p, C.c_int64, C.c_int32, _f64p, _f64p, _i32p]
        L.gce_oracle_fold_bins.argtypes = [_f64p, _f64p, C.c_int64, C.c_double, C.c_double, C.c_int32, _i32p, _f64p]
        L.gce_oracle_ce_from_counts.argtypes = [_i64p, C.c_int32, C.c_int32, C.c_int64]
        L.gce_oracle_ce_from_counts.restype = C.c_double
        L.gce_oracle_histogram.argtypes = [_f64p, _f64p, _i32p, C.c_int64, _f64p, C.c_int64, _f64p, C.c_int64,
                                           C.c_int32, C.c_int32, _i64p, C.c_int64, _i64p]
        L.gce_oracle_ce_search.argtypes = [_f64p, _f64p, _i64p, C.c_int32, _f64p, C.c_int64, _f64p, C.c_int64,
                                           C.c_int32, C.c_int32, _f64p, C.c_int32]
        L.gce_oracle_ce_at.argtypes = [_f64p, _f64p, _i64p, C.c_int32, _f64p, C.c_int64, _f64p, C.c_int64,
                                       C.c_int32, C.c_int32, _i64p, C.c_int64, _f64p, C.c_int32]
        L.gce_oracle_ce_search_overlap.argtypes = L.gce_oracle_ce_search.argtypes
        L.gce_oracle_ce_at_overlap.argtypes = L.gce_oracle_ce_at.argtypes
        L.gce_oracle_overlap_counts.argtypes = [_i64p, C.c_int32, C.c_int32, _i64p]
        L.gce_oracle_normalise_filters.argtypes = [_f64p, _i32p, C.c_int64, _f64p]
        L.gce_oracle_topk.argtypes = [_f64p, C.c_int64, C.c_int32, _i64p, _f64p]
        L.gce_oracle_significance.argtypes = [_f64p, C.c_int64, _f64p]
        L.gce_oracle_num_threads.restype = C.c_int
        _lib = L
    return _lib


def _check(rc):
    if rc != 0:
        raise ValueError(f"gce_oracle: invalid argument (rc={rc})")


def num_threads() -> int:
    return int(lib().gce_oracle_num_threads())


def preprocess(times, mags, n_mag_bins):
    """S1 for one light curve -> (dt, dt2, mbin)."""
    t, m = _f64(times), _f64(mags)
    n = t.shape[0]
    dt, dt2, mbin = np.empty(n), np.empty(n), np.empty(n, dtype=np.int32)
    _check(lib().gce_oracle_preprocess(_p(t, _f64p), _p(m, _f64p), n, int(n_mag_bins),
                                       _p(dt, _f64p), _p(dt2, _f64p), _p(mbin, _i32p)))
    return dt, dt2, mbin


def normalise(mags, filter_ids=None):
    """S0 (N4) for ONE light curve: per-filter (median, population std) normalisation -> u[N]."""
    m = _f64(mags)
    n = m.shape[0]
    u = np.empty(n)
    f = None if filter_ids is None else np.ascontiguousarray(filter_ids, dtype=np.int32)
    _check(lib().gce_oracle_normalise_filters(_p(m, _f64p), None if f is None else _p(f, _i32p), n, _p(u, _f64p)))
    return u


def normalise_batch(mags, lc_offsets, filter_ids=None):
    """S0 applied light curve by light curve to a CSR batch -> the magnitudes the search then bins."""
    m, offs = _f64(mags), _i64(lc_offsets)
    out = np.empty_like(m)
    for l in range(offs.shape[0] - 1):
        a, b = int(offs[l]), int(offs[l + 1])
        out[a:b] = normalise(m[a:b], None if filter_ids is None else np.asarray(filter_ids)[a:b])
    return out


def fold_bins(dt, dt2, P, Pdot, n_phase_bins):
    """S2 for one light curve and one trial -> (phase_bin[N], x[N] cycles)."""
    dt, dt2 = _f64(dt), _f64(dt2)
    n = dt.shape[0]
    pb, x = np.empty(n, dtype=np.int32), np.empty(n)
    _check(lib().gce_oracle_fold_bins(_p(dt, _f64p), _p(dt2, _f64p), n, float(P), float(Pdot),
                                      int(n_phase_bins), _p(pb, _i32p), _p(x, _f64p)))
    return pb, x


def ce_from_counts(counts):
    """S4 from a count table counts[j][i] (phase-major)."""
    cnt = _i64(counts)
    n_phase, n_mag = cnt.shape
    return float(lib().gce_oracle_ce_from_counts(_p(cnt, _i64p), n_phase, n_mag, int(cnt.sum())))


def histogram(times, mags, periods, pdots, n_phase_bins, n_mag_bins, trial_q):
    """S1..S3 for one light curve at flat trials q = ip*n_pdot + ipd -> counts[n_trials][n_phase][n_mag]."""
    dt, dt2, mbin = preprocess(times, mags, n_mag_bins)
    periods, pdots, trial_q = _f64(periods), _f64(pdots), _i64(trial_q)
    out = np.zeros((trial_q.shape[0], int(n_phase_bins), int(n_mag_bins)), dtype=np.int64)
    _check(lib().gce_oracle_histogram(_p(dt, _f64p), _p(dt2, _f64p), _p(mbin, _i32p), dt.shape[0],
                                      _p(periods, _f64p), periods.shape[0], _p(pdots, _f64p), pdots.shape[0],
                                      int(n_phase_bins), int(n_mag_bins), _p(trial_q, _i64p), trial_q.shape[0],
                                      _p(out, _i64p)))
    return out


def overlap_counts(counts):
    """N2: the 50 %-overlapping table c[k][i] = n[k][i] + n[k-1 mod n_phase][i] from plain counts n[j][i]."""
    cnt = _i64(counts)
    out = np.empty_like(cnt)
    _check(lib().gce_oracle_overlap_counts(_p(cnt, _i64p), cnt.shape[0], cnt.shape[1], _p(out, _i64p)))
    return out


def ce_search(times, mags, lc_offsets, periods, pdots, n_phase_bins, n_mag_bins, n_threads=0, overlap=False):
    """Full CE cube [n_lc][n_p][n_pdot] (fp64).  overlap=True: 50 %-overlapping phase bins (N2)."""
    t, m, offs, periods, pdots = _f64(times), _f64(mags), _i64(lc_offsets), _f64(periods), _f64(pdots)
    n_lc = offs.shape[0] - 1
    out = np.empty((n_lc, periods.shape[0], pdots.shape[0]), dtype=np.float64)
    fn = lib().gce_oracle_ce_search_overlap if overlap else lib().gce_oracle_ce_search
    _check(fn(_p(t, _f64p), _p(m, _f64p), _p(offs, _i64p), n_lc,
                                      _p(periods, _f64p), periods.shape[0], _p(pdots, _f64p), pdots.shape[0],
                                      int(n_phase_bins), int(n_mag_bins), _p(out, _f64p), int(n_threads)))
    return out


def ce_at(times, mags, lc_offsets, periods, pdots, n_phase_bins, n_mag_bins, trial_q, n_threads=0, overlap=False):
    """CE at sampled flat trials (same list for every light curve) -> [n_lc][n_trials] (fp64)."""
    t, m, offs, periods, pdots = _f64(times), _f64(mags), _i64(lc_offsets), _f64(periods), _f64(pdots)
    trial_q = _i64(trial_q)
    n_lc = offs.shape[0] - 1
    out = np.empty((n_lc, trial_q.shape[0]), dtype=np.float64)
    fn = lib().gce_oracle_ce_at_overlap if overlap else lib().gce_oracle_ce_at
    _check(fn(_p(t, _f64p), _p(m, _f64p), _p(offs, _i64p), n_lc,
                                  _p(periods, _f64p), periods.shape[0], _p(pdots, _f64p), pdots.shape[0],
                                  int(n_phase_bins), int(n_mag_bins), _p(trial_q, _i64p), trial_q.shape[0],
                                  _p(out, _f64p), int(n_threads)))
    return out


def topk(ce_row, k):
    """S5 for one light curve: the k smallest CE by (CE, q) -> (idx[k] i64, val[k] f64)."""
    ce = _f64(ce_row).ravel()
    idx, val = np.empty(k, dtype=np.int64), np.empty(k)
    _check(lib().gce_oracle_topk(_p(ce, _f64p), ce.shape[0], int(k), _p(idx, _i64p), _p(val, _f64p)))
    return idx, val


def significance(ce_row):
    """Eq. 5 for one light curve -> (mu, sigma, rho)."""
    ce = _f64(ce_row).ravel()
    out = np.empty(3)
    _check(lib().gce_oracle_significance(_p(ce, _f64p), ce.shape[0], _p(out, _f64p)))
    return tuple(float(v) for v in out)
