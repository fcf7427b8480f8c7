"""Seeded synthetic workloads for the CE (P, Pdot) search.

This module holds ONLY input generators (numpy, host side).  It contains none of
the method's arithmetic (no fold-to-bin, no histogram, no entropy) and is the one
piece of code that both the oracle tests and the CUDA path's tests / bench share.

The five configurations are the ones fixed by BASELINE.json:configs[0..4]
("C1".."C5" = 1-based) with the draw order of SURVEY.md section 8(d).  They stand in for
the paper's COSMIC / "Burdge" ellc light curves observed with a VRO/ZTF-like
cadence, none of which are available here; DESIGN.md states the
recipe.

Light-curve model (C2..C5): a two-dip eclipsing-binary-like shape (two eclipses
half a period apart) whose phase drifts quadratically with an injected
Pdot -- the signal model uses the same closed form as Eq. 3 purely to
synthesise magnitudes; it is not used by either implementation of the search.
"""
from __future__ import annotations

from dataclasses import dataclass, field

import numpy as np

DAY = 86400.0
HOUR = 3600.0


@dataclass
class Workload:
    """One batch of light curves plus its trial grid (all host numpy arrays)."""

    name: str
    times: np.ndarray        # f64 [sum N], seconds, per-LC sorted, first time subtracted
    mags: np.ndarray         # f64 [sum N]
    lc_offsets: np.ndarray   # i64 [n_lc + 1]
    periods: np.ndarray      # f64 [n_p], seconds, grid order (descending P)
    pdots: np.ndarray        # f64 [n_pdot], s/s
    n_phase_bins: int
    n_mag_bins: int
    top_k: int               # 0 = no selection requested
    want_cube: bool          # True = full CE cube is part of the requested output
    truth: dict = field(default_factory=dict)  # injected P / Pdot per light curve

    @property
    def n_lc(self) -> int:
        return int(self.lc_offsets.shape[0] - 1)

    @property
    def n_p(self) -> int:
        return int(self.periods.shape[0])

    @property
    def n_pdot(self) -> int:
        return int(self.pdots.shape[0])

    @property
    def total_points(self) -> int:
        return int(self.lc_offsets[-1])

    @property
    def point_folds(self) -> int:
        """n_lc x n_p x n_pdot x N_obs summed over light curves (BASELINE.json:metric)."""
        return int(self.total_points) * self.n_p * self.n_pdot

    def subset(self, lcs=None, p_idx=None, pdot_idx=None, name=None) -> "Workload":
        """Same workload restricted to some light curves / a sub-grid (for sampled parity)."""
        lcs = np.arange(self.n_lc) if lcs is None else np.asarray(lcs, dtype=np.int64)
        t_parts, m_parts, offs = [], [], [0]
        for l in lcs:
            a, b = int(self.lc_offsets[l]), int(self.lc_offsets[l + 1])
            t_parts.append(self.times[a:b])
            m_parts.append(self.mags[a:b])
            offs.append(offs[-1] + (b - a))
        periods = self.periods if p_idx is None else self.periods[np.asarray(p_idx)]
        pdots = self.pdots if pdot_idx is None else self.pdots[np.asarray(pdot_idx)]
        truth = {k: np.asarray(v)[lcs] for k, v in self.truth.items()}
        return Workload(
            name=name or (self.name + "-subset"),
            times=np.ascontiguousarray(np.concatenate(t_parts)) if t_parts else np.zeros(0),
            mags=np.ascontiguousarray(np.concatenate(m_parts)) if m_parts else np.zeros(0),
            lc_offsets=np.asarray(offs, dtype=np.int64),
            periods=np.ascontiguousarray(periods, dtype=np.float64),
            pdots=np.ascontiguousarray(pdots, dtype=np.float64),
            n_phase_bins=self.n_phase_bins, n_mag_bins=self.n_mag_bins,
            top_k=self.top_k, want_cube=self.want_cube, truth=truth)


# ----------------------------------------------------------------------------- signal model
def _model_phase(t, P, Pdot):
    """Cycle count of the injected signal at time t (closed form of Eq. 3)."""
    x = t / P - 0.5 * Pdot * t * t / (P * P)
    return x - np.floor(x)


def two_dip_mags(rng, t, P, Pdot, d1, d2, sigma_n, sigma_phi=0.02, base=18.0):
    """Flat baseline with Gaussian dips at phase 0 and 0.5, plus white noise."""
    phi = _model_phase(t, P, Pdot)
    delta0 = np.minimum(phi, 1.0 - phi)
    delta_half = np.abs(phi - 0.5)
    shape = d1 * np.exp(-0.5 * (delta0 / sigma_phi) ** 2) + d2 * np.exp(-0.5 * (delta_half / sigma_phi) ** 2)
    return base + shape + rng.normal(0.0, sigma_n, size=t.shape[0])


# ----------------------------------------------------------------------------- cadences
def ztf_like_cadence(rng, years: int, n_obs: int) -> np.ndarray:
    """Nightly cadence: 1-3 visits per kept night, 30 % of nights dropped, 120-day seasonal gap."""
    nights = np.arange(365 * years)
    observable = nights[(nights % 365) < 245]
    kept = observable[rng.random(observable.shape[0]) < 0.7]
    visits = rng.integers(1, 4, size=kept.shape[0])
    night_of_visit = np.repeat(kept, visits)
    pool = night_of_visit * DAY + rng.uniform(0.0, 8.0 * HOUR, size=night_of_visit.shape[0])
    if pool.shape[0] >= n_obs:
        t = rng.choice(pool, size=n_obs, replace=False)
    else:
        extra_n = n_obs - pool.shape[0]
        extra_nights = rng.choice(kept, size=extra_n, replace=True)
        extra = extra_nights * DAY + rng.uniform(0.0, 8.0 * HOUR, size=extra_n)
        t = np.concatenate([pool, extra])
    t = np.sort(t)
    return t - t[0]


def lsst_like_cadence(rng, n_obs: int) -> np.ndarray:
    """Uniform over ten observable half-years [y*365.25, y*365.25 + 182.625) d, y = 0..9."""
    year = rng.integers(0, 10, size=n_obs)
    t = (year * 365.25 + rng.uniform(0.0, 182.625, size=n_obs)) * DAY
    t = np.sort(t)
    return t - t[0]


def high_cadence_blocks(rng, n_dense_nights=10, slots_kept=300, n_sparse=2000, years=3) -> np.ndarray:
    """Ten 4-hour blocks at 30 s cadence (300 of 480 slots kept) + sparse nightly visits."""
    n_nights = 365 * years
    dense_nights = rng.choice(n_nights, size=n_dense_nights, replace=False)
    parts = []
    for night in dense_nights:
        start = night * DAY + rng.uniform(0.0, 4.0 * HOUR)
        slots = rng.choice(480, size=slots_kept, replace=False)
        parts.append(start + 30.0 * slots)
    sparse_nights = rng.integers(0, n_nights, size=n_sparse)
    parts.append(sparse_nights * DAY + rng.uniform(0.0, 8.0 * HOUR, size=n_sparse))
    t = np.sort(np.concatenate(parts))
    return t - t[0]


def _pack(lcs):
    offs = np.zeros(len(lcs) + 1, dtype=np.int64)
    for i, (t, _m) in enumerate(lcs):
        offs[i + 1] = offs[i] + t.shape[0]
    times = np.ascontiguousarray(np.concatenate([t for t, _ in lcs]), dtype=np.float64)
    mags = np.ascontiguousarray(np.concatenate([m for _, m in lcs]), dtype=np.float64)
    return times, mags, offs


def _freq_grid(f_lo, f_hi, n):
    """Grid is built in frequency, handed over as periods."""
    return np.ascontiguousarray(1.0 / np.linspace(f_lo, f_hi, int(n)), dtype=np.float64)


# ----------------------------------------------------------------------------- the five configs
def config_c1(n_p=1000, seed=0) -> Workload:
    """BASELINE.json:configs[0] -- one sinusoid, 200 points over 30 days, 1000 frequencies."""
    rng = np.random.default_rng(seed)
    t = np.sort(rng.uniform(0.0, 30.0 * DAY, size=200))
    mag = 0.2 * np.sin(2.0 * np.pi * t / 420.0) + rng.normal(0.0, 0.05, size=200)
    t = t - t[0]
    times, mags, offs = _pack([(t, mag)])
    return Workload("C1", times, mags, offs, _freq_grid(1 / 3600.0, 1 / 180.0, n_p), np.zeros(1),
                    20, 10, top_k=1, want_cube=True, truth={"P": np.array([420.0]), "Pdot": np.array([0.0])})


def _two_dip_batch(seed, n_lc, cadence, p_lo, p_hi, pdot_log10, d1_rng, d2_rng, sigma_n):
    rng = np.random.default_rng(seed)
    lcs, Ps, Pds = [], [], []
    for _ in range(n_lc):
        t = cadence(rng)
        P = float(np.exp(rng.uniform(np.log(p_lo), np.log(p_hi))))
        Pd = 0.0 if pdot_log10 is None else -float(10.0 ** rng.uniform(*pdot_log10))
        d1 = rng.uniform(*d1_rng)
        d2 = rng.uniform(*d2_rng)
        lcs.append((t, two_dip_mags(rng, t, P, Pd, d1, d2, sigma_n)))
        Ps.append(P)
        Pds.append(Pd)
    return lcs, {"P": np.asarray(Ps), "Pdot": np.asarray(Pds)}


def config_c2(n_lc=100, n_p=10_000, seed=1) -> Workload:
    """BASELINE.json:configs[1] -- 100 ZTF-like LCs (N=500, 2 yr), 1e4 frequencies, Pdot={0}."""
    lcs, truth = _two_dip_batch(seed, n_lc, lambda r: ztf_like_cadence(r, 2, 500), 300.0, 3600.0, None,
                                (0.1, 0.8), (0.05, 0.4), 0.03)
    times, mags, offs = _pack(lcs)
    return Workload("C2", times, mags, offs, _freq_grid(1 / 7200.0, 1 / 180.0, n_p), np.zeros(1),
                    20, 10, top_k=1, want_cube=False, truth=truth)


def config_c3(n_lc=64, n_p=50_000, n_pdot=64, seed=2) -> Workload:
    """BASELINE.json:configs[2] -- the P-Pdot grid: 64 LCs (N=1000, 3 yr) x 5e4 freqs x 64 Pdots."""
    lcs, truth = _two_dip_batch(seed, n_lc, lambda r: ztf_like_cadence(r, 3, 1000), 180.0, 900.0, (-12.0, -10.0),
                                (0.1, 0.8), (0.05, 0.4), 0.05)
    times, mags, offs = _pack(lcs)
    return Workload("C3", times, mags, offs, _freq_grid(1 / 1200.0, 1 / 120.0, n_p),
                    np.ascontiguousarray(np.linspace(-1e-10, 0.0, int(n_pdot))),
                    20, 10, top_k=1, want_cube=True, truth=truth)


def config_c4(n_lc=1000, n_p=100_000, seed=3) -> Workload:
    """BASELINE.json:configs[3] -- LSST-like sparse batch: 1000 LCs (N=200, 10 yr), 1e5 freqs, top-5."""
    lcs, truth = _two_dip_batch(seed, n_lc, lambda r: lsst_like_cadence(r, 200), 600.0, 7200.0, None,
                                (0.05, 0.5), (0.05, 0.5), 0.08)
    times, mags, offs = _pack(lcs)
    return Workload("C4", times, mags, offs, _freq_grid(1 / 14400.0, 1 / 300.0, n_p), np.zeros(1),
                    15, 8, top_k=5, want_cube=False, truth=truth)


def config_c5(n_lc=16, n_p=1 << 17, n_pdot=256, seed=4) -> Workload:
    """BASELINE.json:configs[4] -- heavy high-cadence P-Pdot search: 16 LCs (N=5000), 2^17 x 256, top-16."""
    lcs, truth = _two_dip_batch(seed, n_lc, lambda r: high_cadence_blocks(r), 120.0, 600.0, (-11.0, -9.0),
                                (0.1, 0.8), (0.05, 0.4), 0.02)
    times, mags, offs = _pack(lcs)
    return Workload("C5", times, mags, offs, _freq_grid(1 / 900.0, 1 / 90.0, n_p),
                    np.ascontiguousarray(np.linspace(-2e-9, 0.0, int(n_pdot))),
                    30, 10, top_k=16, want_cube=False, truth=truth)


def fig3_batch(n_obs, n_search_points, n_phase_bins, n_lc=16, n_pdot=32, seed=7) -> Workload:
    """Workload of the paper's timing figure (Fig. 3): light curves of n_obs points (100 or 1000)
    over ten years (VRO-like, :90), a grid of n_search_points = n_p x n_pdot trials per light curve (the paper searches
    groups of 32 / 128 / 512 Pdot values, :158), 15 or 50 phase bins x 10 magnitude bins.  Two-dip model as C4."""
    n_p = max(1, int(round(n_search_points / n_pdot)))
    lcs, truth = _two_dip_batch(seed, n_lc, lambda r: lsst_like_cadence(r, n_obs), 600.0, 7200.0, (-12.0, -10.0),
                                (0.05, 0.5), (0.05, 0.5), 0.08)
    times, mags, offs = _pack(lcs)
    return Workload(f"fig3-N{n_obs}-phi{n_phase_bins}", times, mags, offs, _freq_grid(1 / 14400.0, 1 / 300.0, n_p),
                    np.ascontiguousarray(np.linspace(-1e-10, 0.0, int(n_pdot))), n_phase_bins, 10, top_k=1,
                    want_cube=False, truth=truth)


def vro_like_cadence(rng, n_obs: int, mean_dt_days=7.0, sigma_dt_days=1.0) -> np.ndarray:
    """"The time difference between each observation point is sampled from a Gaussian distribution with
    mean dt" -- VRO-like: ten-year baseline, about 7 days between observations, n ~ 500.  (The width of the Gaussian is
    not given; one day is this harness's choice.)"""
    dt = np.maximum(rng.normal(mean_dt_days, sigma_dt_days, size=n_obs), 0.01) * DAY
    t = np.cumsum(dt)
    return t - t[0]


def config_paper(n_lc=100, n_p=5_183_995, n_pdot=32, seed=9) -> Workload:
    """NEXT item N4 -- the paper's production search: 5,183,995 frequencies linearly spaced
    from 2/B (B = 10 yr) to 1/(3 min), 32 / 128 / 512 Pdot values log-spaced from -1e-12 to -1e-10, 100 light curves of
    about 500 points, 50 overlapping phase bins x 10 magnitude bins.  The cube (1.7e10 values at 32 Pdots) is never
    materialised: fused top-k + Eq. 5 statistics.  Synthetic two-dip light curves stand in for the COSMIC / ellc set."""
    lcs, truth = _two_dip_batch(seed, n_lc, lambda r: vro_like_cadence(r, 500), 300.0, 3600.0, (-12.0, -10.3),
                                (0.1, 0.8), (0.05, 0.4), 0.2)
    times, mags, offs = _pack(lcs)
    B = 10.0 * 365.25 * DAY
    pdots = -np.logspace(-12.0, -10.0, int(n_pdot))
    return Workload("P1", times, mags, offs, _freq_grid(2.0 / B, 1.0 / 180.0, n_p), np.ascontiguousarray(pdots),
                    50, 10, top_k=5, want_cube=False, truth=truth)


CONFIGS = {"C1": config_c1, "C2": config_c2, "C3": config_c3, "C4": config_c4, "C5": config_c5, "P1": config_paper}


def make(name: str, **kw) -> Workload:
    """make("C3") -> full-size workload; keyword overrides shrink n_lc / n_p / n_pdot (same ranges); `seed`
    overrides the configuration's own seed (used for the other ranks' batches in weak-scaling runs)."""
    return CONFIGS[name.upper()](**kw)


def two_filter_batch(seed, n_lc=4, n_obs=400, n_p=600, n_pdot=4, offset=0.9, scale=0.6):
    """N4: light curves observed in two filters merged into one time series.  Filter 1 sees the same
    two-dip signal `offset` mag fainter with its dips scaled by `scale` (a colour term) and its own noise; about 40 % of
    the points are in filter 1.  Returns (Workload, filter_ids int32[sum N])."""
    rng = np.random.default_rng(seed)
    lcs, filt, truth_p = [], [], []
    for _ in range(n_lc):
        t = np.sort(rng.uniform(0.0, 2.0 * 365.25 * DAY, size=n_obs))
        P = float(np.exp(rng.uniform(np.log(400.0), np.log(2000.0))))
        f = (rng.uniform(size=n_obs) < 0.4).astype(np.int32)
        clean = two_dip_mags(rng, t, P, 0.0, 0.5, 0.25, 0.0)
        m = np.where(f == 0, clean, 18.0 + offset + scale * (clean - 18.0))
        m = m + rng.normal(0.0, np.where(f == 0, 0.03, 0.05))
        lcs.append((t, m))
        filt.append(f)
        truth_p.append(P)
    times, mags, offs = _pack(lcs)
    w = Workload(f"twofilter{seed}", times, mags, offs, _freq_grid(1 / 2400.0, 1 / 350.0, n_p),
                 np.ascontiguousarray(np.linspace(-2e-11, 0.0, int(n_pdot))) if n_pdot > 1 else np.zeros(1), 20, 10, 3, True,
                 truth={"P": np.array(truth_p)})
    return w, np.ascontiguousarray(np.concatenate(filt), dtype=np.int32)


# ----------------------------------------------------------------------------- small helpers for tests
def random_batch(seed, n_lc, n_min, n_max, n_p, n_pdot, n_phase_bins=20, n_mag_bins=10, top_k=3,
                 pdot_range=(-1e-9, 1e-10), baseline_days=400.0) -> Workload:
    """Ragged batch (lengths n_min..n_max, possibly 0) of noise-plus-sinusoid light curves."""
    rng = np.random.default_rng(seed)
    lcs = []
    for _ in range(n_lc):
        n = int(rng.integers(n_min, n_max + 1))
        t = np.sort(rng.uniform(0.0, baseline_days * DAY, size=n)) + 5.0e8  # unsorted-origin: t0 != 0
        P = float(np.exp(rng.uniform(np.log(200.0), np.log(5000.0))))
        m = 15.0 + 0.3 * np.sin(2 * np.pi * t / P) + rng.normal(0.0, 0.1, size=n)
        lcs.append((t, m))
    if lcs:
        times, mags, offs = _pack(lcs)
    else:
        times, mags, offs = np.zeros(0), np.zeros(0), np.zeros(1, dtype=np.int64)
    periods = _freq_grid(1 / 6000.0, 1 / 150.0, n_p)
    pdots = np.ascontiguousarray(np.linspace(pdot_range[0], pdot_range[1], int(n_pdot))) if n_pdot > 1 else np.zeros(1)
    return Workload(f"rand{seed}", times, mags, offs, periods, pdots, n_phase_bins, n_mag_bins, top_k, True)


def dense_local_grid(P_true, Pdot_true, baseline_s, half_width=0.02, n_pdot=33):
    """Recovery grid of SURVEY 8(c): f_true(1 +- 2 %) at step 1/(3T) x Pdot in [2 Pdot_true, 0]."""
    f0 = 1.0 / P_true
    step = 1.0 / (3.0 * baseline_s)
    n_side = int(np.ceil(half_width * f0 / step))
    freqs = f0 + step * np.arange(-n_side, n_side + 1)
    pdots = np.linspace(2.0 * Pdot_true, 0.0, n_pdot) if Pdot_true != 0.0 else np.zeros(1)
    return np.ascontiguousarray(1.0 / freqs), np.ascontiguousarray(pdots)
