"""Pins for the CPU oracle (oracle/gce_oracle.c) -- everything here runs without a GPU.

The paper (arXiv 2006.06866) prints no worked numerical CE example, so the oracle is pinned to
what the paper's equations and the mathematics fix: hand-worked dyadic folds and count tables
(tests/golden/, each citing the passage), closed forms (Eq. 6), textbook identities evaluated by
library routines (scipy.stats.entropy, numpy.histogram), exact rational arithmetic, invariants
and brute force on tiny inputs.  SURVEY.md section 8(c) lists the pins; DESIGN.md repeats them.
"""
import math
import os
from fractions import Fraction

import numpy as np
import pytest
import scipy.stats

import gce_workloads as W
from conftest import GOLDEN


# ------------------------------------------------------------------ golden file readers
def _read_fold_cases():
    cases, cur = [], None
    for line in open(os.path.join(GOLDEN, "fold_hand_examples.txt")):
        line = line.strip()
        if not line or line.startswith("#"):
            continue
        tok = line.split()
        if tok[0] == "case":
            cur = {"name": tok[1], "P": float(tok[3]), "Pdot": float(tok[5]), "n_phase": int(tok[7]), "rows": []}
            cases.append(cur)
        else:
            cur["rows"].append((float(tok[0]), float(tok[1]), int(tok[2])))
    return cases


def _read_ce_tables():
    tables, cur = [], None
    for line in open(os.path.join(GOLDEN, "ce_hand_tables.txt")):
        line = line.strip()
        if not line or line.startswith("#"):
            continue
        tok = line.split()
        if tok[0] == "table":
            cur = {"name": tok[1], "rows": int(tok[3]), "cols": int(tok[5]), "expr": " ".join(tok[7:]), "cnt": []}
            tables.append(cur)
        else:
            cur["cnt"].append([int(v) for v in tok])
    return tables


# ------------------------------------------------------------------ S2: fold (Eq. 3)
@pytest.mark.parametrize("case", _read_fold_cases(), ids=lambda c: c["name"])
def test_fold_hand_examples(oracle, case):
    """Eq. 3 on dyadic inputs: exact cycles x and phase bins, worked by hand."""
    dt = np.array([r[0] for r in case["rows"]])
    pb, x = oracle.fold_bins(dt, dt * dt, case["P"], case["Pdot"], case["n_phase"])
    assert x.tolist() == [r[1] for r in case["rows"]]
    assert pb.tolist() == [r[2] for r in case["rows"]]


def test_fold_quadratic_term_matches_eq6(oracle):
    """Eq. 6: x(Pdot) - x(0) = +1/2 |Pdot| t^2 / P^2 for Pdot < 0; Fig. 2 system
    (P = 7 min, Pdot = -2.14e-11) after 10 yr -> 6.0408 cycles (sign and size)."""
    t = np.array([10 * 365.25 * 86400.0])
    _, x0 = oracle.fold_bins(t, t * t, 420.0, 0.0, 50)
    _, x1 = oracle.fold_bins(t, t * t, 420.0, -2.14e-11, 50)
    assert x1[0] - x0[0] == pytest.approx(6.0408, abs=2e-4)
    _, x2 = oracle.fold_bins(t, t * t, 420.0, +2.14e-11, 50)
    assert x2[0] - x0[0] == pytest.approx(-6.0408, abs=2e-4)


def test_fold_against_exact_rational_arithmetic(oracle):
    """The frozen fp64 order may differ from exact-real arithmetic only within 1e-6 of a bin edge.

    Exact value computed with python Fractions from the SAME fp64 inputs: x = dt/P - Pdot dt^2/(2 P^2)."""
    rng = np.random.default_rng(11)
    n_phase = 20
    dt = np.sort(rng.uniform(0, 3 * 365.25 * 86400.0, size=400))
    dt[0] = 0.0
    bad = 0
    for P, Pd in [(123.456, 0.0), (431.7, -3.3e-11), (95.0, -1.9e-9), (777.7, 4e-11), (3599.0, -1e-10)]:
        pb, _ = oracle.fold_bins(dt, dt * dt, P, Pd, n_phase)
        FP, FPd = Fraction(P), Fraction(Pd)
        for k in range(dt.shape[0]):
            Fd = Fraction(float(dt[k]))
            y = (Fd / FP - FPd * Fd * Fd / (2 * FP * FP)) * n_phase
            j_exact = math.floor(y) % n_phase
            if j_exact != int(pb[k]):
                dist = min(y - math.floor(y), math.ceil(y) - y)
                assert dist < Fraction(1, 10 ** 6), (P, Pd, k, float(y))
                assert (int(pb[k]) - j_exact) % n_phase in (1, n_phase - 1)
                bad += 1
    assert bad <= 2  # essentially never at these sizes


def test_fold_pdot_zero_is_textbook_frac(oracle):
    """Pdot = 0 reduces to the textbook fold frac(t/P): j = floor(n * ((t/P) mod 1)) away from edges."""
    rng = np.random.default_rng(5)
    dt = rng.uniform(0, 1e6, size=2000)
    P, n_phase = 311.0, 15
    pb, x = oracle.fold_bins(dt, dt * dt, P, 0.0, n_phase)
    phase = np.mod(dt / P, 1.0)
    safe = np.abs(phase * n_phase - np.round(phase * n_phase)) > 1e-6
    assert safe.sum() > 1900
    assert np.array_equal(pb[safe], np.floor(phase[safe] * n_phase).astype(np.int32))
    assert pb.min() >= 0 and pb.max() < n_phase


# ------------------------------------------------------------------ S1: preprocess
def test_preprocess_t0_invariance(oracle):
    """t0 = min t (reading Q1): integer times shifted by 1000 give identical dt and bins; order-free."""
    t = np.arange(50, dtype=np.float64)
    m = np.sin(t)
    a = oracle.preprocess(t, m, 7)
    b = oracle.preprocess(t + 1000.0, m, 7)
    for u, v in zip(a, b):
        assert np.array_equal(u, v)
    perm = np.random.default_rng(0).permutation(50)
    c = oracle.preprocess(t[perm] + 1000.0, m[perm], 7)
    assert np.array_equal(c[0], a[0][perm]) and np.array_equal(c[2], a[2][perm])
    assert np.array_equal(a[1], a[0] * a[0])


def test_preprocess_magnitude_bins_match_numpy_histogram(oracle):
    """Equal-width bins over [m_min, m_max], last bin closed = numpy.histogram's convention."""
    rng = np.random.default_rng(3)
    for n_mag in (2, 8, 10, 13):
        m = rng.normal(18.0, 0.3, size=777)
        _, _, mbin = oracle.preprocess(np.arange(777.0), m, n_mag)
        ref, _ = np.histogram(m, bins=n_mag, range=(m.min(), m.max()))
        assert np.array_equal(np.bincount(mbin, minlength=n_mag), ref)
        assert mbin[np.argmax(m)] == n_mag - 1 and mbin[np.argmin(m)] == 0


def test_preprocess_hand_example_and_degenerate(oracle):
    # m in {0, 0.25, 0.5, 0.75, 1.0}, 4 bins: edges at .25/.5/.75 belong to the upper bin; 1.0 to the last.
    _, _, mbin = oracle.preprocess(np.arange(5.0), np.array([0.0, 0.25, 0.5, 0.75, 1.0]), 4)
    assert mbin.tolist() == [0, 1, 2, 3, 3]
    # affine invariance (Q2): median/std normalisation gives the same equal-width bins
    m = np.array([3.0, 4.0, 5.0, 7.0, 11.0])
    _, _, b1 = oracle.preprocess(np.arange(5.0), m, 4)
    _, _, b2 = oracle.preprocess(np.arange(5.0), (m - 5.0) / 4.0, 4)
    assert b1.tolist() == b2.tolist() == [0, 0, 1, 2, 3]
    # all magnitudes equal -> bin 0 everywhere (Q12)
    _, _, b3 = oracle.preprocess(np.arange(4.0), np.full(4, 2.5), 6)
    assert b3.tolist() == [0, 0, 0, 0]


# ------------------------------------------------------------------ S4: conditional entropy (Eq. 4)
@pytest.mark.parametrize("tab", _read_ce_tables(), ids=lambda t: t["name"])
def test_ce_hand_tables(oracle, tab):
    cnt = np.array(tab["cnt"], dtype=np.int64)
    assert cnt.shape == (tab["rows"], tab["cols"])
    expect = eval(tab["expr"], {"log": math.log})
    got = oracle.ce_from_counts(cnt)
    assert got == pytest.approx(expect, rel=1e-14, abs=1e-16)
    if expect == 0.0:
        assert got == 0.0


def test_ce_asym3_printed_value(oracle):
    """[[3,1,0],[0,2,2],[1,0,3]] -> 0.6059391565991873 and H(m) = 1.0775563270668007."""
    cnt = np.array([[3, 1, 0], [0, 2, 2], [1, 0, 3]])
    assert oracle.ce_from_counts(cnt) == pytest.approx(0.6059391565991873, rel=1e-14)
    assert scipy.stats.entropy(cnt.sum(axis=0)) == pytest.approx(1.0775563270668007, rel=1e-14)


def test_ce_is_joint_minus_marginal_entropy(oracle):
    """Eq. 4 = H(m,phi) - H(phi) (textbook identity), evaluated by scipy.stats.entropy."""
    rng = np.random.default_rng(7)
    for shape in [(20, 10), (15, 8), (30, 10), (50, 10), (1, 5), (6, 1)]:
        for _ in range(5):
            cnt = rng.poisson(2.0, size=shape).astype(np.int64)
            cnt[rng.random(shape) < 0.3] = 0
            if cnt.sum() == 0:
                cnt[0, 0] = 1
            ref = scipy.stats.entropy(cnt.ravel()) - scipy.stats.entropy(cnt.sum(axis=1))
            got = oracle.ce_from_counts(cnt)
            assert got == pytest.approx(ref, rel=1e-12, abs=1e-13)
            h_m = scipy.stats.entropy(cnt.sum(axis=0))
            assert -1e-15 <= got <= h_m + 1e-12 <= math.log(shape[1]) + 1e-12


# ------------------------------------------------------------------ S1..S4 end to end, brute force
def _brute_counts(t, m, P, Pd, n_phase, n_mag):
    """Independent brute force with exact rational arithmetic (no floats after input conversion)."""
    Ft = [Fraction(float(v)) for v in t]
    Fm = [Fraction(float(v)) for v in m]
    t0, lo, hi = min(Ft), min(Fm), max(Fm)
    cnt = np.zeros((n_phase, n_mag), dtype=np.int64)
    FP, FPd = Fraction(P), Fraction(Pd)
    for tk, mk in zip(Ft, Fm):
        d = tk - t0
        x = d / FP - FPd * d * d / (2 * FP * FP)
        j = math.floor((x - math.floor(x)) * n_phase)
        i = 0 if hi == lo else min(math.floor((mk - lo) / (hi - lo) * n_mag), n_mag - 1)
        cnt[j, i] += 1
    return cnt


def test_end_to_end_half_ln2_example(oracle):
    """P=8, Pdot=0, n_phi=4, n_m=2, dt=0..7, m=0,0,0,1,1,1,0,1 -> [[2,0],[1,1],[0,2],[1,1]], 1/2 ln 2."""
    t = np.arange(8.0) + 100.0
    m = np.array([0, 0, 0, 1, 1, 1, 0, 1], dtype=np.float64)
    cnt = oracle.histogram(t, m, [8.0], [0.0], 4, 2, [0])[0]
    assert cnt.tolist() == [[2, 0], [1, 1], [0, 2], [1, 1]]
    cube = oracle.ce_search(t, m, [0, 8], [8.0], [0.0], 4, 2)
    assert cube.shape == (1, 1, 1)
    assert cube[0, 0, 0] == pytest.approx(0.5 * math.log(2), rel=1e-15)


def test_histogram_brute_force_dyadic(oracle):
    """Integer times, dyadic P and Pdot, dyadic magnitudes: fp64 is exact, so the oracle must equal the
    exact-rational brute force on every trial of a small (P, Pdot) grid."""
    rng = np.random.default_rng(21)
    t = rng.integers(0, 4096, size=60).astype(np.float64) + 7.0
    m = rng.integers(0, 64, size=60) / 64.0
    periods = np.array([8.0, 4.0, 16.0, 0.5, 32.0])   # powers of two: 1/P exact
    pdots = np.array([-0.5, 0.0, 0.25, -2.0 ** -6])
    n_phase, n_mag = 8, 4
    q = np.arange(periods.size * pdots.size)
    cnt = oracle.histogram(t, m, periods, pdots, n_phase, n_mag, q)
    cube = oracle.ce_search(t, m, [0, 60], periods, pdots, n_phase, n_mag)
    for ip, P in enumerate(periods):
        for ipd, Pd in enumerate(pdots):
            ref = _brute_counts(t, m, P, Pd, n_phase, n_mag)
            assert np.array_equal(cnt[ip * pdots.size + ipd], ref), (P, Pd)
            ce_ref = scipy.stats.entropy(ref.ravel()) - scipy.stats.entropy(ref.sum(axis=1))
            assert cube[0, ip, ipd] == pytest.approx(ce_ref, rel=1e-12, abs=1e-14)


def test_histogram_invariants_on_c1(oracle):
    """Sum of counts = N, permutation invariance, trial-independent magnitude marginal = numpy.histogram."""
    w = W.make("C1", n_p=64)
    q = np.arange(64)
    cnt = oracle.histogram(w.times, w.mags, w.periods, w.pdots, 20, 10, q)
    assert np.all(cnt.sum(axis=(1, 2)) == 200)
    ref, _ = np.histogram(w.mags, bins=10, range=(w.mags.min(), w.mags.max()))
    assert np.all(cnt.sum(axis=1) == ref[None, :])
    perm = np.random.default_rng(1).permutation(200)
    cnt2 = oracle.histogram(w.times[perm], w.mags[perm], w.periods, w.pdots, 20, 10, q)
    assert np.array_equal(cnt, cnt2)
    # numpy.histogram2d on (phase, u) agrees for trials whose points all sit away from bin edges
    dt, dt2, _ = oracle.preprocess(w.times, w.mags, 10)
    u = (w.mags - w.mags.min()) / (w.mags.max() - w.mags.min())
    checked = 0
    for s in range(64):
        _, x = oracle.fold_bins(dt, dt2, w.periods[s], 0.0, 20)
        ph = x - np.floor(x)
        edge = np.abs(ph * 20 - np.round(ph * 20))
        edge[ph == 0.0] = 1.0                                # dt = 0 sits exactly on edge 0: bin 0 either way
        if np.min(edge) < 1e-9:
            continue
        h2, _, _ = np.histogram2d(ph, u, bins=[20, 10], range=[[0, 1], [0, 1]])
        assert np.array_equal(h2.astype(np.int64), cnt[s])
        checked += 1
    assert checked > 50


def test_search_matches_histogram_path_and_ce_at(oracle):
    w = W.random_batch(4, n_lc=3, n_min=0, n_max=40, n_p=9, n_pdot=4, n_phase_bins=6, n_mag_bins=3)
    cube = oracle.ce_search(w.times, w.mags, w.lc_offsets, w.periods, w.pdots, 6, 3)
    q = np.array([0, 5, 35, 17])
    at = oracle.ce_at(w.times, w.mags, w.lc_offsets, w.periods, w.pdots, 6, 3, q)
    for l in range(3):
        a, b = w.lc_offsets[l], w.lc_offsets[l + 1]
        if b == a:
            assert np.all(np.isnan(cube[l])) and np.all(np.isnan(at[l]))
            continue
        assert np.array_equal(cube[l].ravel()[q], at[l])
        cnt = oracle.histogram(w.times[a:b], w.mags[a:b], w.periods, w.pdots, 6, 3, q)
        for s in range(q.size):
            assert oracle.ce_from_counts(cnt[s]) == cube[l].ravel()[q[s]]


# ------------------------------------------------------------------ special cases of the whole path
def test_special_cases(oracle):
    rng = np.random.default_rng(9)
    n = 300
    t = np.sort(rng.uniform(0, 1e6, size=n))
    m = rng.normal(0, 1, size=n)
    periods = 1.0 / np.linspace(1 / 900.0, 1 / 100.0, 40)
    pdots = np.array([-1e-9, 0.0])
    offs = [0, n]
    # n_phi = 1 -> CE = H(m) for every trial
    _, _, mbin = oracle.preprocess(t, m, 10)
    h_m = scipy.stats.entropy(np.bincount(mbin, minlength=10))
    cube = oracle.ce_search(t, m, offs, periods, pdots, 1, 10)
    assert np.allclose(cube, h_m, rtol=1e-13)
    # n_m = 1 -> CE = 0 exactly
    assert np.all(oracle.ce_search(t, m, offs, periods, pdots, 20, 1) == 0.0)
    # all magnitudes equal -> CE = 0 ; N = 1 -> CE = 0 ; N = 0 -> NaN (Q12)
    assert np.all(oracle.ce_search(t, np.full(n, 3.0), offs, periods, pdots, 20, 10) == 0.0)
    assert np.all(oracle.ce_search(t[:1], m[:1], [0, 1], periods, pdots, 20, 10) == 0.0)
    assert np.all(np.isnan(oracle.ce_search(t[:0], m[:0], [0, 0], periods, pdots, 20, 10)))
    # general bounds 0 <= CE <= H(m) <= ln n_m
    cube = oracle.ce_search(t, m, offs, periods, pdots, 20, 10)
    assert cube.min() >= 0.0 and cube.max() <= h_m + 1e-12 <= math.log(10) + 1e-12


def test_ce_zero_when_magnitude_is_function_of_phase_bin(oracle):
    """Perfectly phase-determined signal: m depends only on the phase bin at the true period -> CE = 0 there."""
    P, n_phase = 64.0, 8
    t = np.arange(0, 4096, 3, dtype=np.float64)           # dyadic -> exact folds
    j = np.floor((t / P - np.floor(t / P)) * n_phase).astype(int)
    levels = np.array([0.0, 0.3, 0.3, 0.9, 1.0, 0.1, 0.6, 0.6])
    m = levels[j]
    cube = oracle.ce_search(t, m, [0, t.size], [P, 48.0], [0.0], n_phase, 5)
    assert cube[0, 0, 0] == 0.0
    assert cube[0, 1, 0] > 0.1


def test_ce_equals_hm_when_all_points_share_one_phase(oracle):
    """All dt integer multiples of a dyadic P, Pdot = 0: every point in phase bin 0 -> CE = H(m)."""
    rng = np.random.default_rng(2)
    t = 16.0 * rng.integers(0, 1000, size=200)
    t[0] = 0.0
    m = rng.normal(size=200)
    _, _, mbin = oracle.preprocess(t, m, 10)
    cube = oracle.ce_search(t, m, [0, 200], [16.0, 8.0, 0.5], [0.0], 20, 10)
    assert np.allclose(cube, scipy.stats.entropy(np.bincount(mbin, minlength=10)), rtol=1e-14)


# ------------------------------------------------------------------ S5: selection
def test_topk_is_lexicographic_sort(oracle):
    rng = np.random.default_rng(13)
    ce = np.round(rng.uniform(0, 2, size=500), 2)          # many exact ties
    for k in (1, 5, 16, 32):
        idx, val = oracle.topk(ce, k)
        order = np.lexsort((np.arange(ce.size), ce))[:k]    # (CE asc, q asc)
        assert np.array_equal(idx, order) and np.array_equal(val, ce[order])
    idx, val = oracle.topk(np.array([0.5, 0.25, 0.25]), 5)  # k > n_trials: padding
    assert idx.tolist() == [1, 2, 0, -1, -1] and np.isnan(val[3:]).all()
    idx, val = oracle.topk(np.full(4, np.nan), 2)           # empty light curve
    assert idx.tolist() == [-1, -1]


def test_planted_minimum_and_noiseless_recovery(oracle):
    """Noiseless two-dip signal with injected (P, Pdot): on the dense local grid of SURVEY 8(c) the argmin
    trial folds every point to within one bin of the generating phase."""
    rng = np.random.default_rng(17)
    T = 3 * 365.25 * W.DAY
    t = np.sort(rng.uniform(0, T, size=600))
    t -= t[0]
    P_true, Pd_true, n_phase = 431.7, -4.0e-11, 20
    m = W.two_dip_mags(rng, t, P_true, Pd_true, 0.6, 0.3, 0.0)
    periods, pdots = W.dense_local_grid(P_true, Pd_true, t[-1], half_width=0.0005, n_pdot=33)
    # plant the generating trial exactly on the grid
    ip0, ipd0 = periods.size // 2, int(np.argmin(np.abs(pdots - Pd_true)))
    periods[ip0], pdots[ipd0] = P_true, Pd_true
    cube = oracle.ce_search(t, m, [0, t.size], periods, pdots, n_phase, 10)
    idx, _ = oracle.topk(cube[0], 1)
    ip, ipd = divmod(int(idx[0]), pdots.size)
    dt, dt2, _ = oracle.preprocess(t, m, 10)
    _, x_best = oracle.fold_bins(dt, dt2, periods[ip], pdots[ipd], n_phase)
    _, x_true = oracle.fold_bins(dt, dt2, P_true, Pd_true, n_phase)
    d = x_best - x_true
    d -= np.round(np.median(d))                            # a constant phase offset does not change CE
    assert np.max(np.abs(d - np.median(d))) < 1.0 / n_phase
    # and the Pdot = 0 column is clearly worse than the best (dephasing)
    assert cube[0, :, -1].min() > cube[0].min() + 0.05


def test_significance_matches_numpy(oracle):
    """Eq. 5: rho = (mu - min) / sigma, population sigma (Q13)."""
    ce = np.random.default_rng(0).uniform(1.0, 2.0, size=1000)
    ce[77] = 0.2
    mu, sigma, rho = oracle.significance(ce)
    assert mu == pytest.approx(ce.mean(), rel=1e-13)
    assert sigma == pytest.approx(ce.std(ddof=0), rel=1e-12)
    assert rho == pytest.approx((ce.mean() - 0.2) / ce.std(ddof=0), rel=1e-12)


# ------------------------------------------------------------------ N2: 50 %-overlapping phase bins
def _read_tables(fname):
    tables, cur = [], None
    for line in open(os.path.join(GOLDEN, fname)):
        line = line.strip()
        if not line or line.startswith("#"):
            continue
        tok = line.split()
        if tok[0] == "table":
            cur = {"name": tok[1], "rows": int(tok[3]), "cols": int(tok[5]), "expr": " ".join(tok[7:]), "cnt": []}
            tables.append(cur)
        else:
            cur["cnt"].append([int(v) for v in tok])
    return tables


@pytest.mark.parametrize("tab", _read_tables("ce_overlap_hand_tables.txt"), ids=lambda t: t["name"])
def test_overlap_hand_tables(oracle, tab):
    n = np.array(tab["cnt"], dtype=np.int64)
    assert n.shape == (tab["rows"], tab["cols"])
    expect = eval(tab["expr"], {"log": math.log})
    c = oracle.overlap_counts(n)
    assert c.sum() == 2 * n.sum()
    got = oracle.ce_from_counts(c)
    assert got == pytest.approx(expect, rel=1e-14, abs=1e-16)
    if expect == 0.0:
        assert got == 0.0


def _brute_overlap_counts(t, m, P, Pd, n_phase, n_mag):
    """Independent definition by interval membership, exact rationals: bin k holds the points whose phase lies in the
    cyclic interval [(k-1)/n_phase, (k+1)/n_phase) -- width 2/n_phase, 50 % shared with each neighbour."""
    Ft = [Fraction(float(v)) for v in t]
    Fm = [Fraction(float(v)) for v in m]
    t0, lo, hi = min(Ft), min(Fm), max(Fm)
    cnt = np.zeros((n_phase, n_mag), dtype=np.int64)
    FP, FPd = Fraction(P), Fraction(Pd)
    w = Fraction(1, n_phase)
    for tk, mk in zip(Ft, Fm):
        d = tk - t0
        x = d / FP - FPd * d * d / (2 * FP * FP)
        phi = x - math.floor(x)
        i = 0 if hi == lo else min(math.floor((mk - lo) / (hi - lo) * n_mag), n_mag - 1)
        for k in range(n_phase):
            rel = (phi - (k - 1) * w) % 1          # distance past the bin's left edge, cyclic
            if rel < 2 * w:
                cnt[k, i] += 1
    return cnt


def test_overlap_counts_equal_interval_membership_brute_force(oracle):
    """Dyadic inputs (fp64 exact): the oracle's overlapped table equals exact-rational interval membership, every
    point is counted exactly twice, and the search's CE equals scipy's H(m,phi) - H(phi) of that table."""
    rng = np.random.default_rng(31)
    t = rng.integers(0, 4096, size=70).astype(np.float64) + 3.0
    m = rng.integers(0, 64, size=70) / 64.0
    periods = np.array([8.0, 4.0, 16.0, 32.0])
    pdots = np.array([-0.5, 0.0, 0.25])
    for n_phase, n_mag in ((8, 4), (16, 3), (4, 2)):
        q = np.arange(periods.size * pdots.size)
        plain = oracle.histogram(t, m, periods, pdots, n_phase, n_mag, q)
        cube = oracle.ce_search(t, m, [0, 70], periods, pdots, n_phase, n_mag, overlap=True)
        at = oracle.ce_at(t, m, [0, 70], periods, pdots, n_phase, n_mag, q, overlap=True)
        for ip, P in enumerate(periods):
            for ipd, Pd in enumerate(pdots):
                ref = _brute_overlap_counts(t, m, P, Pd, n_phase, n_mag)
                got = oracle.overlap_counts(plain[ip * pdots.size + ipd])
                assert np.array_equal(got, ref), (n_phase, P, Pd)
                assert ref.sum() == 140 and np.array_equal(ref.sum(axis=0), 2 * plain[0].sum(axis=0))
                ce_ref = scipy.stats.entropy(ref.ravel()) - scipy.stats.entropy(ref.sum(axis=1))
                assert cube[0, ip, ipd] == pytest.approx(ce_ref, rel=1e-12, abs=1e-14)
                assert at[0, ip * pdots.size + ipd] == cube[0, ip, ipd]


def test_overlap_special_cases_and_bounds(oracle):
    """n_phase = 1 and 2: every bin holds every point -> CE = H(m); n_mag = 1 -> 0; 0 <= CE <= H(m); on a smooth
    light curve at its true period the overlapped CE stays low and within ln 2 of the plain one
    (each overlapped bin is the union of two plain cells)."""
    w = W.make("C1", n_p=200)
    _, _, mbin = oracle.preprocess(w.times, w.mags, 10)
    hm = scipy.stats.entropy(np.bincount(mbin, minlength=10))
    for n_phase in (1, 2):
        ce = oracle.ce_search(w.times, w.mags, w.lc_offsets, w.periods, w.pdots, n_phase, 10, overlap=True)
        assert np.allclose(ce, hm, rtol=1e-13)
    assert np.all(oracle.ce_search(w.times, w.mags, w.lc_offsets, w.periods, w.pdots, 20, 1, overlap=True) == 0.0)
    ov = oracle.ce_search(w.times, w.mags, w.lc_offsets, w.periods, w.pdots, 20, 10, overlap=True)
    pl = oracle.ce_search(w.times, w.mags, w.lc_offsets, w.periods, w.pdots, 20, 10)
    assert np.all(ov >= 0) and np.all(ov <= hm + 1e-12)
    # an overlapped bin's magnitude distribution is a two-component mixture of its cells' distributions, and every cell
    # enters two bins with weight 1/2: H(mixture) >= the weighted mean of the parts (concavity) and <= that mean + ln 2
    assert np.all(ov >= pl - 1e-12)
    assert np.all(ov <= pl + math.log(2) + 1e-12)


# ------------------------------------------------------------------------------------------ N4: per-filter median / std
def test_normalise_hand_examples(oracle):
    """PAPER.md:96 (reading Q19): u = (m - median) / population std, per filter.  Closed forms by hand:
    [1,2,3,4,10]: median 3, mean 4, var (9+4+1+0+36)/5 = 10;  [1,2,3,4]: median 2.5, var 1.25."""
    u = oracle.normalise(np.array([1.0, 2.0, 3.0, 4.0, 10.0]))
    np.testing.assert_allclose(u, (np.array([1.0, 2, 3, 4, 10]) - 3.0) / math.sqrt(10.0), rtol=1e-15)
    u = oracle.normalise(np.array([4.0, 1.0, 3.0, 2.0]))
    np.testing.assert_allclose(u, (np.array([4.0, 1, 3, 2]) - 2.5) / math.sqrt(1.25), rtol=1e-15)
    # dyadic case, exact: symmetric +-2 -> median 0, std 2
    assert np.array_equal(oracle.normalise(np.array([-2.0, 2.0, 2.0, -2.0])), np.array([-1.0, 1.0, 1.0, -1.0]))
    # degenerate filters: one point, all equal -> 0 (no NaN)
    assert np.array_equal(oracle.normalise(np.array([5.0])), np.zeros(1))
    assert np.array_equal(oracle.normalise(np.array([7.0, 7.0, 7.0])), np.zeros(3))
    assert oracle.normalise(np.zeros(0)).shape == (0,)


def test_normalise_matches_numpy_per_filter(oracle):
    """Library special case: numpy.median / numpy.std (ddof 0) on each filter's points; interleaved filters."""
    rng = np.random.default_rng(11)
    m = rng.normal(18.0, 0.4, 500)
    f = rng.integers(0, 3, 500).astype(np.int32)
    m[f == 1] += 1.3
    m[f == 2] *= 0.5
    u = oracle.normalise(m, f)
    for k in range(3):
        sel = f == k
        np.testing.assert_allclose(u[sel], (m[sel] - np.median(m[sel])) / np.std(m[sel]), rtol=1e-12, atol=1e-13)
        assert abs(np.median(u[sel])) < 1e-13 and abs(np.std(u[sel]) - 1.0) < 1e-12
    # filter ids outside 0..7 are refused
    with pytest.raises(Exception):
        oracle.normalise(m, np.full(500, 8, dtype=np.int32))


def test_single_filter_normalisation_does_not_change_the_bins(oracle):
    """Reading Q2: equal-width bins over the data range are invariant under positive affine maps, so with ONE filter the
    paper's median / std step leaves every magnitude bin where min/max normalisation puts it -- exactly on dyadic data,
    and on random data except for points within rounding of a bin edge."""
    m = np.array([-2.0, 2.0, 2.0, -2.0, -2.0, 2.0, 2.0, -2.0])   # median 0, std 2: u = m / 2 exactly
    t = np.arange(m.size, dtype=np.float64)
    raw = oracle.preprocess(t, m, 8)[2]
    norm = oracle.preprocess(t, oracle.normalise(m), 8)[2]
    assert np.array_equal(raw, norm) and set(raw) == {0, 7}
    rng = np.random.default_rng(3)
    mr = rng.normal(17.0, 0.3, 4000)
    tr = np.arange(4000.0)
    raw_r = oracle.preprocess(tr, mr, 10)[2]
    norm_r = oracle.preprocess(tr, oracle.normalise(mr), 10)[2]
    u = (mr - mr.min()) / (mr.max() - mr.min()) * 10
    near_edge = np.abs(u - np.round(u)) < 1e-9
    assert np.array_equal(raw_r[~near_edge], norm_r[~near_edge])
    assert np.mean(raw_r == norm_r) > 0.999


def test_two_filters_merged_into_one_light_curve(oracle):
    """What the option is for: two filters offset by 0.9 mag merged into one light curve.  After the
    per-filter median / std step both filters share one scale (median 0, std 1 each), the magnitude bins differ from the
    min/max bins of the raw merged magnitudes, and the CE minimum on a dense local grid sits at the injected period."""
    import gce_workloads as W
    w, filt = W.two_filter_batch(5, n_lc=3, n_obs=400, n_p=500, n_pdot=1)
    u = oracle.normalise_batch(w.mags, w.lc_offsets, filt)
    for lc in range(3):
        a, b = int(w.lc_offsets[lc]), int(w.lc_offsets[lc + 1])
        for k in (0, 1):
            sel = filt[a:b] == k
            assert abs(np.median(u[a:b][sel])) < 1e-13 and abs(np.std(u[a:b][sel]) - 1.0) < 1e-12
        raw_bins = oracle.preprocess(w.times[a:b], w.mags[a:b], 10)[2]
        norm_bins = oracle.preprocess(w.times[a:b], u[a:b], 10)[2]
        assert np.mean(raw_bins != norm_bins) > 0.3
        P = w.truth["P"][lc]
        periods = 1.0 / (1.0 / P + np.arange(-150, 151) / (3.0 * w.times[b - 1]))   # dense local grid around the truth
        offs = np.array([0, b - a], dtype=np.int64)
        ce_norm = oracle.ce_search(w.times[a:b], u[a:b], offs, periods, np.zeros(1), 20, 10)[0].ravel()
        assert abs(int(np.argmin(ce_norm)) - 150) <= 1
