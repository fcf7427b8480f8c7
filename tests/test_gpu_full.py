"""GPU parity at BASELINE.json's FULL sizes (the launch configuration bench.py times) and on the kernel's
less-travelled paths (streamed light curves, cells with >= 1024 points, R = 2 trials per thread).

At full size the oracle cannot produce the whole cube in seconds, so the comparison is on sampled outputs the
oracle computes one by one (oracle.ce_at), plus properties that hold at any size: the fused selection equals a
CPU reduction of the GPU's own cube, every reported best CE equals the oracle's CE of that trial, and no sampled
trial beats the reported minimum.
"""
import numpy as np
import pytest
import torch

import gce_workloads as W
from test_gpu_parity import (RTOL32, RTOL64, assert_ce_close, assert_counts_match_oracle, assert_topk_matches, dev,
                             run_search)

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def gce():
    from paper_2006_06866_b200.build import build
    build()
    import paper_2006_06866_b200 as g
    return g


def sample_trials(n_trials, n, seed):
    """Seeded sample of flat trial indices that always holds the first / last trial and a tile boundary."""
    rng = np.random.default_rng(seed)
    q = rng.choice(n_trials, size=min(n, n_trials), replace=False)
    edge = np.array([0, 1, 2047, 2048, 2049, n_trials - 2, n_trials - 1])
    return np.unique(np.concatenate([q, edge[(edge >= 0) & (edge < n_trials)]])).astype(np.int64)


def check_selection_against_oracle(w, res, k, oracle, q_sample, ref_sample):
    """Properties of the fused top-k that need no full oracle cube."""
    idx = res.best_idx.cpu().numpy()
    val = res.best_ce.cpu().numpy()
    for lc in range(w.n_lc):
        gi = idx[lc]
        assert len(set(gi.tolist())) == k and gi.min() >= 0 and gi.max() < w.periods.size * w.pdots.size
        exact = oracle.ce_at(w.times, w.mags, w.lc_offsets, w.periods, w.pdots, w.n_phase_bins, w.n_mag_bins, gi)[lc]
        # reported values are the oracle's CE of the reported trials, ascending
        assert np.all(np.abs(val[lc] - exact) <= RTOL32 * np.abs(exact) + 1e-12), lc
        assert np.all(np.diff(exact) >= -RTOL64 * np.abs(exact[1:]) - 1e-13), lc
        # nothing in the oracle's sample beats the k-th reported trial unless it is itself reported (or ties it)
        better = ref_sample[lc] < exact[-1] * (1 - RTOL64) - 1e-13
        assert set(q_sample[better].tolist()) <= set(gi.tolist()), lc


def test_c2_full(gce, oracle):
    """configs[1] at full size (100 x 500 points x 1e4 periods, Pdot = {0}): whole cube + per-LC best."""
    w = W.make("C2")
    ref = oracle.ce_search(w.times, w.mags, w.lc_offsets, w.periods, w.pdots, w.n_phase_bins, w.n_mag_bins)
    res = run_search(gce, w, top_k=1)
    assert_ce_close(res.ce.cpu().numpy(), ref, RTOL32)
    for lc in range(w.n_lc):
        assert_topk_matches(ref[lc], res.best_idx[lc].cpu().numpy(), res.best_ce[lc].cpu().numpy(), 1, RTOL32, oracle)
    res2 = run_search(gce, w, top_k=1, want_cube=False)
    assert torch.equal(res2.best_idx, res.best_idx)


def test_c3_full_sampled(gce, oracle):
    """configs[2] at full size, exactly as bench.py launches it (fp32 cube 64 x 50000 x 64 + per-LC best)."""
    w = W.make("C3")
    res = run_search(gce, w, top_k=1)
    n_trials = w.periods.size * w.pdots.size
    q = sample_trials(n_trials, 3000, seed=33)
    ref = oracle.ce_at(w.times, w.mags, w.lc_offsets, w.periods, w.pdots, w.n_phase_bins, w.n_mag_bins, q)
    cube = res.ce.reshape(w.n_lc, n_trials)
    got = cube[:, torch.from_numpy(q).cuda()].cpu().numpy()
    assert_ce_close(got, ref, RTOL32)
    # the fused argmin equals a reduction of the GPU's own cube up to fp32 rounding of the stored values:
    # the cube's minimum value is the reported trial's value
    mn = cube.min(dim=1).values.cpu().numpy()
    assert np.array_equal(mn, res.best_ce[:, 0].cpu().numpy())
    assert np.array_equal(cube.gather(1, res.best_idx).cpu().numpy()[:, 0], mn)
    check_selection_against_oracle(w, res, 1, oracle, q, ref)
    assert bool(torch.all(cube >= 0)) and float(cube.max()) <= np.log(w.n_mag_bins) + 1e-6


def test_c4_full_top5(gce, oracle):
    """configs[3] at full size: 1000 light curves x 200 points x 1e5 periods, 15 x 8 bins, fused top-5, no cube."""
    w = W.make("C4")
    res = run_search(gce, w, top_k=5, want_cube=False)
    assert res.ce is None
    q = sample_trials(w.periods.size, 1500, seed=44)
    ref = oracle.ce_at(w.times, w.mags, w.lc_offsets, w.periods, w.pdots, w.n_phase_bins, w.n_mag_bins, q)
    check_selection_against_oracle(w, res, 5, oracle, q, ref)
    # full oracle cube for a few light curves: ordered top-5 with the near-tie rule
    for lc in (0, 499, 999):
        a, b = w.lc_offsets[lc], w.lc_offsets[lc + 1]
        row = oracle.ce_search(w.times[a:b], w.mags[a:b], np.array([0, b - a]), w.periods, w.pdots, 15, 8)[0]
        assert_topk_matches(row, res.best_idx[lc].cpu().numpy(), res.best_ce[lc].cpu().numpy(), 5, RTOL32, oracle)


def test_c5_full_top16(gce, oracle):
    """configs[4] at full size: 16 x 5000 points x 2^17 periods x 256 Pdots, 30 x 10 bins, fused top-16."""
    w = W.make("C5")
    res = run_search(gce, w, top_k=16, want_cube=False)
    n_trials = w.periods.size * w.pdots.size
    q = sample_trials(n_trials, 1200, seed=55)
    ref = oracle.ce_at(w.times, w.mags, w.lc_offsets, w.periods, w.pdots, w.n_phase_bins, w.n_mag_bins, q)
    check_selection_against_oracle(w, res, 16, oracle, q, ref)
    # every reported trial and its +-2 neighbours along both axes: the reported one is not beaten by a neighbour
    # that is missing from the list
    n_pd = w.pdots.size
    for lc in (0, 15):
        gi = res.best_idx[lc].cpu().numpy()
        nb = set()
        for g in gi:
            ip, ipd = divmod(int(g), n_pd)
            for dp in range(-2, 3):
                for dd in range(-2, 3):
                    if 0 <= ip + dp < w.periods.size and 0 <= ipd + dd < n_pd:
                        nb.add((ip + dp) * n_pd + ipd + dd)
        nb = np.array(sorted(nb), dtype=np.int64)
        a, b = w.lc_offsets[lc], w.lc_offsets[lc + 1]
        ce_nb = oracle.ce_at(w.times[a:b], w.mags[a:b], np.array([0, b - a]), w.periods, w.pdots, 30, 10, nb)[0]
        kth = ce_nb[np.searchsorted(nb, gi[-1])]
        better = nb[ce_nb < kth * (1 - RTOL64) - 1e-13]
        assert set(better.tolist()) <= set(gi.tolist())


# ------------------------------------------------------------------------------------------ counts of the timed kernels
def _fold_modes_of(gce, w, lc, qs):
    """Fold variant the owning thread of each trial qualifies for (gce_ce_debug_bins, FOLD_AUTO)."""
    prm = gce.make_params(w.n_phase_bins, w.n_mag_bins)
    t, m, o, p, pd = dev(w.times), dev(w.mags), dev(w.lc_offsets), dev(w.periods), dev(w.pdots)
    n = int(w.lc_offsets[lc + 1] - w.lc_offsets[lc])
    pb = torch.empty(n, dtype=torch.int32, device="cuda")
    mb = torch.empty(n, dtype=torch.int32, device="cuda")
    mode = torch.empty(1, dtype=torch.int32, device="cuda")
    out = []
    for q in qs:
        gce.gce_ce_debug_bins(t, m, o, p, pd, prm, lc, int(q), pb, mb, out_fold_mode=mode)
        out.append(int(mode.item()))
    return out


def _tile_edge_trials(n_trials, tile, rng, n_random):
    """First / last trial, both sides of the first tile boundaries and of a boundary deep in the grid, plus a random sample.
    A tile is threads x trials-per-thread; the kernels run 512 or 384 threads, so the edges of both tilings are taken."""
    edge = [0, 1, 3, 4, n_trials - 2, n_trials - 1]
    for t in (tile, tile * 3 // 4):
        deep = (n_trials // t // 2) * t
        edge += [t - 1, t, t + 1, 2 * t - 1, 2 * t, deep - 1, deep, deep + 5]
    q = np.concatenate([np.array(edge), rng.integers(0, n_trials, size=n_random)])
    return np.unique(q[(q >= 0) & (q < n_trials)]).astype(np.int64)


def test_c3_full_counts_of_the_timed_kernel(gce, oracle):
    """configs[2] at full size: the kernel bench.py times (n_phi = 20, 4 trials per thread sharing a period, shared floors,
    512 threads: k_search<20,1,4,1,.,1,512>) in dump mode -- histogram counts bit-exact against the oracle on all 64 light
    curves, at tile edges, and in both the quad (long periods) and the pair (short periods) shared-floor variants."""
    w = W.make("C3")
    n_pd = w.pdots.size
    n_trials = w.periods.size * n_pd
    rng = np.random.default_rng(303)
    short_p = (w.periods.size - 1 - rng.integers(0, 2000, size=6)) * n_pd + rng.integers(0, n_pd, size=6)  # P ~ 120 s
    q = np.unique(np.concatenate([_tile_edge_trials(n_trials, 2048, rng, 24), short_p]))
    modes = set(_fold_modes_of(gce, w, 0, q))
    assert {gce.binding.FOLD_QUAD, gce.binding.FOLD_PAIR} <= modes, modes
    assert_counts_match_oracle(gce, oracle, w, q)


def test_c5_full_counts_of_the_timed_kernel(gce, oracle):
    """configs[4] at full size: k_search<30,1,4,1,.,0,384> in dump mode, all 16 light curves of 5000 points (magnitude bins
    above 1024 points: the table's global tail), counts bit-exact at tile edges and on a random sample."""
    w = W.make("C5")
    n_trials = w.periods.size * w.pdots.size
    rng = np.random.default_rng(505)
    q = _tile_edge_trials(n_trials, 2048, rng, 20)
    assert_counts_match_oracle(gce, oracle, w, q)


def test_c4_full_counts_of_the_timed_kernel(gce, oracle):
    """configs[3] at full size: k_search<15,1,4,0,.,0,512> (Pdot = {0}: the 4 trials of a thread are 4 periods) in dump
    mode, bit-exact counts on a sample of the 1000 light curves (the dump runs all of them)."""
    w = W.make("C4")
    rng = np.random.default_rng(404)
    q = _tile_edge_trials(w.periods.size, 2048, rng, 20)
    assert_counts_match_oracle(gce, oracle, w, q, lcs=[0, 1, 2, 250, 499, 777, 998, 999])


def test_c2_full_counts_of_the_timed_kernel(gce, oracle):
    w = W.make("C2")
    rng = np.random.default_rng(202)
    q = _tile_edge_trials(w.periods.size, 2048, rng, 20)
    assert_counts_match_oracle(gce, oracle, w, q, lcs=[0, 1, 50, 98, 99])


def test_paper_binning_counts_of_the_timed_kernel(gce, oracle):
    """The paper's production binning (50 overlapping phase bins x 10) on the C3 grid: k_search<50,1,2,1,.,0,512>
    in dump mode writes the overlapped table; bit-exact against oracle.overlap_counts(oracle.histogram)."""
    w = W.make("C3", n_lc=8)
    w.n_phase_bins, w.n_mag_bins = 50, 10
    rng = np.random.default_rng(5050)
    q = _tile_edge_trials(w.periods.size * w.pdots.size, 1024, rng, 16)
    assert_counts_match_oracle(gce, oracle, w, q, overlap=True)
    assert_counts_match_oracle(gce, oracle, w, q[:8], overlap=False)


def test_c5_cube_mode_sampled(gce, oracle):
    """The C5 shape with the cube written (reduced period axis so the cube stays small): fp64 output, 30 x 10 bins,
    magnitude bins with more than 1024 points (the table's global-memory tail)."""
    w = W.make("C5", n_lc=2, n_p=2048, n_pdot=256)
    res = run_search(gce, w, top_k=16, ce_fp64=True)
    n_trials = w.periods.size * w.pdots.size
    q = sample_trials(n_trials, 1500, seed=56)
    ref = oracle.ce_at(w.times, w.mags, w.lc_offsets, w.periods, w.pdots, 30, 10, q)
    got = res.ce.reshape(2, n_trials)[:, torch.from_numpy(q).cuda()].cpu().numpy()
    assert_ce_close(got, ref, RTOL64)
    cube = res.ce.reshape(2, n_trials).cpu().numpy()
    for lc in range(2):
        order = np.lexsort((np.arange(n_trials), cube[lc]))[:16]
        assert np.array_equal(order, res.best_idx[lc].cpu().numpy())


@pytest.mark.parametrize("n_obs,n_phi,n_m,n_pdot", [(20000, 20, 10, 4), (9000, 30, 10, 2), (30000, 15, 2, 1),
                                                    (65535, 20, 10, 4)])
def test_long_light_curves_are_streamed(gce, oracle, n_obs, n_phi, n_m, n_pdot):
    """Light curves longer than the shared-memory point buffer (NEXT item N3: streamed through two half buffers),
    cells with far more than 1024 points, next to a short light curve in the same batch."""
    rng = np.random.default_rng(n_obs)
    t_long = np.sort(rng.uniform(0, 3e7, n_obs))
    m_long = W.two_dip_mags(rng, t_long, 611.0, -2e-11, 0.5, 0.2, 0.05)
    t_short = np.sort(rng.uniform(0, 3e7, 300))
    m_short = rng.normal(size=300)
    times = np.concatenate([t_long, t_short])
    mags = np.concatenate([m_long, m_short])
    offs = np.array([0, n_obs, n_obs + 300], dtype=np.int64)
    periods = 1.0 / np.linspace(1 / 900.0, 1 / 300.0, 700)
    pdots = np.linspace(-4e-11, 0.0, n_pdot)
    w = W.Workload("long", times, mags, offs, periods, pdots, n_phi, n_m, 4, True)
    ref = oracle.ce_search(times, mags, offs, periods, pdots, n_phi, n_m)
    res = run_search(gce, w, top_k=4, ce_fp64=True)
    assert_ce_close(res.ce.cpu().numpy(), ref, RTOL64)
    for lc in range(2):
        assert_topk_matches(ref[lc], res.best_idx[lc].cpu().numpy(), res.best_ce[lc].cpu().numpy(), 4, RTOL64, oracle)
    # bit-exact counts of a few trials of the long light curve
    q = torch.tensor([0, 1, 699 * n_pdot + n_pdot - 1], dtype=torch.int64, device="cuda")
    prm = gce.make_params(n_phi, n_m)
    counts = torch.empty((2, 3, n_phi, n_m), dtype=torch.int32, device="cuda")
    ws = torch.empty(gce.gce_ce_workspace_bytes(times.size, 2, 700, n_pdot, prm), dtype=torch.uint8, device="cuda")
    gce.gce_ce_debug_histogram(dev(times), dev(mags), dev(offs), dev(periods), dev(pdots), prm, q, counts, None, ws)
    torch.cuda.synchronize()
    refc = oracle.histogram(t_long, m_long, periods, pdots, n_phi, n_m, q.cpu().numpy())
    assert np.array_equal(counts[0].cpu().numpy().astype(np.int64), refc)


def _long_batch(n_obs, seed):
    rng = np.random.default_rng(seed)
    t_long = np.sort(rng.uniform(0, 3e7, n_obs))
    m_long = W.two_dip_mags(rng, t_long, 611.0, -2e-11, 0.5, 0.2, 0.05)
    t_short = np.sort(rng.uniform(0, 3e7, 300))
    m_short = rng.normal(size=300)
    return (np.concatenate([t_long, t_short]), np.concatenate([m_long, m_short]),
            np.array([0, n_obs, n_obs + 300], dtype=np.int64), t_long, m_long)


@pytest.mark.parametrize("n_obs,n_phi,n_m,n_pdot,overlap", [(100000, 20, 10, 4, False), (70001, 30, 7, 2, False),
                                                            (100000, 50, 10, 2, True), (40000, 15, 10, 1, True)])
def test_light_curves_beyond_the_16_bit_counters(gce, oracle, n_obs, n_phi, n_m, n_pdot, overlap):
    """NEXT item N3 (light curves of any length): a call that announces light curves longer than 65 535
    points (32 767 with overlapping bins) runs with 32-bit counters and a k ln k table as long as the light curve
    (whose fixed-point shift drops below 42 once it has more than 2^17 entries).  Cube, selection, Eq. 5 and bit-exact
    counts against the oracle, next to a short light curve in the same batch."""
    times, mags, offs, t_long, m_long = _long_batch(n_obs, n_obs + n_phi)
    periods = 1.0 / np.linspace(1 / 900.0, 1 / 300.0, 300)
    pdots = np.linspace(-4e-11, 0.0, n_pdot) if n_pdot > 1 else np.zeros(1)
    ref = oracle.ce_search(times, mags, offs, periods, pdots, n_phi, n_m, overlap=overlap)
    res = gce.search(dev(times), dev(mags), dev(offs), dev(periods), dev(pdots), n_phi, n_m, top_k=4, want_cube=True,
                     ce_fp64=True, want_stats=True, overlap=overlap)
    torch.cuda.synchronize()
    assert_ce_close(res.ce.cpu().numpy(), ref, RTOL64)
    for lc in range(2):
        assert_topk_matches(ref[lc], res.best_idx[lc].cpu().numpy(), res.best_ce[lc].cpu().numpy(), 4, RTOL64, oracle)
        mu, sigma, rho = oracle.significance(ref[lc])
        st = res.stats[lc].cpu().numpy()
        np.testing.assert_allclose(st[:3], [mu, sigma, ref[lc].min()], rtol=1e-9)
    # bit-exact counts of a few trials of the long light curve, from the kernel the search ran (with overlap = 1 the
    # dump holds the overlapped table the entropy is taken from)
    q = torch.tensor([0, 1, 299 * n_pdot + n_pdot - 1], dtype=torch.int64, device="cuda")
    prm = gce.make_params(n_phi, n_m, overlap=overlap, max_lc_points=n_obs)
    counts = torch.empty((2, 3, n_phi, n_m), dtype=torch.int32, device="cuda")
    ws = torch.empty(gce.gce_ce_workspace_bytes(times.size, 2, 300, n_pdot, prm), dtype=torch.uint8, device="cuda")
    gce.gce_ce_debug_histogram(dev(times), dev(mags), dev(offs), dev(periods), dev(pdots), prm, q, counts, None, ws)
    torch.cuda.synchronize()
    refc = oracle.histogram(t_long, m_long, periods, pdots, n_phi, n_m, q.cpu().numpy())
    if overlap:
        refc = np.stack([oracle.overlap_counts(r) for r in refc])
    assert np.array_equal(counts[0].cpu().numpy().astype(np.int64), refc)
    # the host entry sees the lengths and switches to the 32-bit counters itself: same bits
    ce_h = np.empty((2, 300, n_pdot), dtype=np.float64)
    idx_h = np.empty((2, 4), dtype=np.int64)
    gce.gce_ce_search_host(times, mags, offs, periods, pdots, gce.make_params(n_phi, n_m, top_k=4, ce_fp64=True, overlap=overlap),
                           ce_h, idx_h, None)
    assert np.array_equal(ce_h, res.ce.cpu().numpy()) and np.array_equal(idx_h, res.best_idx.cpu().numpy())


def test_unannounced_long_light_curve_is_treated_as_empty(gce):
    """Device-pointer call without max_lc_points: the lengths live on the device, so a light curve beyond the 16-bit
    range cannot be refused up front; it is never folded with wrapped counters but treated as empty (NaN, -1), and the
    other light curves of the batch are unaffected.  When total_points alone proves it the call is refused."""
    times, mags, offs, _, _ = _long_batch(70000, 5)
    periods = 1.0 / np.linspace(1 / 900.0, 1 / 300.0, 64)
    pdots = np.zeros(1)
    prm = gce.make_params(20, 10, top_k=2)
    ce = torch.empty((2, 64, 1), dtype=torch.float32, device="cuda")
    idx = torch.empty((2, 2), dtype=torch.int64, device="cuda")
    ws = torch.empty(gce.gce_ce_workspace_bytes(times.size, 2, 64, 1, prm), dtype=torch.uint8, device="cuda")
    gce.gce_ce_search(dev(times), dev(mags), dev(offs), dev(periods), dev(pdots), prm, ce, idx, None, None, ws)
    torch.cuda.synchronize()
    assert torch.isnan(ce[0]).all() and (idx[0] == -1).all()
    assert torch.isfinite(ce[1]).all() and (idx[1] >= 0).all()
    one = np.array([0, 70000], dtype=np.int64)
    with pytest.raises(gce.GceError) as e:
        gce.gce_ce_search(dev(times[:70000]), dev(mags[:70000]), dev(one), dev(periods), dev(pdots), prm, ce[:1], idx[:1], None, None, ws)
    assert e.value.code == -2


def test_wide_counters_period_split_is_exact(gce):
    """The partial blob carries the table's fixed-point shift, so a period-split search of a long light curve merges to
    the bits of the unsplit call."""
    times, mags, offs, _, _ = _long_batch(140000, 6)
    periods = 1.0 / np.linspace(1 / 900.0, 1 / 300.0, 96)
    pdots = np.linspace(-4e-11, 0.0, 2)
    args = (dev(times), dev(mags), dev(offs), dev(periods), dev(pdots), 20, 10)
    whole = gce.search(*args, top_k=3, want_cube=False, want_stats=True)
    # search_period_chunks builds its own params: announce the length through the keyword
    split = gce.search_period_chunks(*args, [(0, 40), (40, 41), (41, 96)], top_k=3, want_stats=True, max_lc_points=140000)
    torch.cuda.synchronize()
    assert torch.equal(whole.best_idx, split.best_idx) and torch.equal(whole.best_ce, split.best_ce)
    assert torch.equal(whole.stats, split.stats)


def test_eq5_sums_of_a_clean_long_light_curve_do_not_wrap(gce, oracle):
    """The warp-level Eq. 5 reduction adds up to 128 squares of d = S - K in 128 bits, so |d| must stay below 2^60.5.
    Worst case: a noiseless signal (CE ~ 0, d ~ -K) in a long light curve with 64 magnitude bins (K = N H(m) 2^shift),
    many Pdots sharing the true period so that all 128 trials of a warp sit at the minimum.  With the table shift at 42
    for N = 1e5 this K is 2^60.7 and the sum of squares wrapped; the shift of tables beyond the 16-bit range is now
    chosen from L(k_max) (gce_ce.cu table_shift), K = 2^58.7.  mean / std / min / rho against the oracle's Eq. 5."""
    n_obs, n_phi, n_m, P = 100000, 64, 64, 611.0
    rng = np.random.default_rng(77)
    t = np.sort(rng.uniform(0, 3e7, n_obs))
    m = np.mod(t / P, 1.0)                       # sawtooth: the magnitude is the phase, H(m) = ln 64, CE ~ 0 at P
    offs = np.array([0, n_obs], dtype=np.int64)
    periods = np.array([P, P * 1.37, P, P * 0.71, P, P * 1.11, P, P], dtype=np.float64)   # rows at P: 128 trials near CE = 0
    pdots = np.linspace(-1e-19, 0.0, 128)        # no measurable drift: every Pdot of a row gives the same low CE
    ref = oracle.ce_search(t, m, offs, periods, pdots, n_phi, n_m)
    assert ref[0, 0].max() < 0.3 * np.log(64) and ref[0, 1].min() > 0.8 * np.log(64)
    res = gce.search(dev(t), dev(m), dev(offs), dev(periods), dev(pdots), n_phi, n_m, top_k=2, want_cube=True,
                     ce_fp64=True, want_stats=True)
    torch.cuda.synchronize()
    assert_ce_close(res.ce.cpu().numpy(), ref, RTOL64)
    mu, sigma, rho = oracle.significance(ref[0])
    np.testing.assert_allclose(res.stats[0].cpu().numpy(), [mu, sigma, ref[0].min(), rho], rtol=RTOL_STATS)


# ------------------------------------------------------------------------------------------ N1: fused Eq. 5 statistics
RTOL_STATS = 1e-9   # exact integer sums of N*CE*2^42, one fp64 conversion; the per-trial CE values
                    # differ from the oracle's by <= 1e-12 relative, the variance subtraction amplifies that by mean^2/var


def _stats_ref(oracle, ref_cube):
    out = []
    for row in ref_cube:
        mu, sigma, rho = oracle.significance(row)
        out.append((mu, sigma, float(np.min(row)) if row.size else np.nan, rho))
    return np.array(out)


@pytest.mark.parametrize("name,kw", [
    ("C2", dict(n_lc=6, n_p=3000)),
    ("C3", dict(n_lc=4, n_p=1500, n_pdot=64)),
    ("C3", dict(n_lc=2, n_p=1111, n_pdot=7)),
    ("C4", dict(n_lc=9, n_p=5000)),
    ("C5", dict(n_lc=2, n_p=300, n_pdot=16)),
])
def test_fused_significance_matches_oracle(gce, oracle, name, kw):
    """out_stats = {mean CE, population std, min CE, rho} (Eq. 5) against the oracle's Eq. 5 over the
    oracle's cube; with and without the cube / top-k outputs (the no-cube mode is what N1 is for)."""
    w = W.make(name, **kw)
    ref = oracle.ce_search(w.times, w.mags, w.lc_offsets, w.periods, w.pdots, w.n_phase_bins, w.n_mag_bins)
    want = _stats_ref(oracle, ref.reshape(w.n_lc, -1))
    d = lambda a: torch.from_numpy(np.ascontiguousarray(a)).cuda()
    args = (d(w.times), d(w.mags), d(w.lc_offsets), d(w.periods), d(w.pdots), w.n_phase_bins, w.n_mag_bins)
    for top_k, cube in ((0, False), (3, False), (1, True)):
        res = gce.search(*args, top_k=top_k, want_cube=cube, want_stats=True)
        torch.cuda.synchronize()
        got = res.stats.cpu().numpy()
        np.testing.assert_allclose(got, want, rtol=RTOL_STATS, atol=1e-13)
        if top_k:
            assert np.allclose(got[:, 2], res.best_ce[:, 0].cpu().numpy().astype(np.float64), rtol=1e-6)


def test_fused_significance_degenerate_and_split_invariance(gce, oracle):
    """N = 0 -> NaN; constant CE (n_phi = 1, or all magnitudes equal) -> std exactly 0 and rho NaN like the oracle's 0/0;
    the statistics do not depend on how the trials are split over CTAs (exact integer partial sums)."""
    rng = np.random.default_rng(3)
    lcs = [(np.zeros(0), np.zeros(0)), (np.sort(rng.uniform(0, 1e6, 400)), np.full(400, 3.0)),
           (np.sort(rng.uniform(0, 1e6, 700)), rng.normal(size=700))]
    times = np.concatenate([t for t, _ in lcs]); mags = np.concatenate([m for _, m in lcs])
    offs = np.cumsum([0] + [t.size for t, _ in lcs]).astype(np.int64)
    periods = 1.0 / np.linspace(1 / 5000.0, 1 / 50.0, 4099)
    pdots = np.linspace(-1e-9, 0, 3)
    d = lambda a: torch.from_numpy(np.ascontiguousarray(a)).cuda()
    res = gce.search(d(times), d(mags), d(offs), d(periods), d(pdots), 20, 10, top_k=0, want_cube=True, ce_fp64=True,
                     want_stats=True)
    torch.cuda.synchronize()
    st = res.stats.cpu().numpy()
    assert np.all(np.isnan(st[0]))
    assert st[1, 0] == 0.0 and st[1, 1] == 0.0 and st[1, 2] == 0.0 and np.isnan(st[1, 3])
    cube = res.ce.cpu().numpy().reshape(3, -1)
    assert st[2, 0] == pytest.approx(cube[2].mean(), rel=1e-12)
    assert st[2, 1] == pytest.approx(cube[2].std(), rel=1e-9)
    assert st[2, 2] == cube[2].min()
    # n_phi = 1: CE = H(m) for every trial -> spread exactly 0
    res1 = gce.search(d(times), d(mags), d(offs), d(periods), d(pdots), 1, 10, top_k=0, want_cube=False, want_stats=True)
    torch.cuda.synchronize()
    s1 = res1.stats.cpu().numpy()
    assert s1[2, 1] == 0.0 and s1[2, 0] == s1[2, 2] > 0 and np.isnan(s1[2, 3])
    # a different CTA split (one light curve alone gets more jobs per light curve) gives the same bits
    a, b = offs[2], offs[3]
    res2 = gce.search(d(times[a:b]), d(mags[a:b]), d(np.array([0, b - a])), d(periods), d(pdots), 20, 10, top_k=0,
                      want_cube=False, want_stats=True)
    torch.cuda.synchronize()
    assert np.array_equal(res2.stats.cpu().numpy()[0], st[2])
    # a one-trial grid on a long light curve: N * CE * 2^42 needs more than 53 bits, mean and min must still be the same
    # number and rho NaN (not +-inf from two differently rounded conversions)
    t5 = np.sort(rng.uniform(0, 1e7, 5000)); m5 = rng.normal(size=5000)
    res3 = gce.search(d(t5), d(m5), d(np.array([0, 5000])), d(np.array([733.0])), d(np.zeros(1)), 20, 10, top_k=1,
                      want_cube=True, ce_fp64=True, want_stats=True)
    torch.cuda.synchronize()
    s3 = res3.stats.cpu().numpy()[0]
    assert s3[0] == s3[2] == float(res3.ce.ravel()[0]) > 1.0 and s3[1] == 0.0 and np.isnan(s3[3])


def test_c4_full_stats_sampled_light_curves(gce, oracle):
    """configs[3] at full size in the no-cube mode with Eq. 5 fused: statistics of three light curves against the
    oracle's full rows, the rest against bounds (min = best CE, 0 <= min <= mean <= ln n_m, std > 0)."""
    w = W.make("C4")
    d = lambda a: torch.from_numpy(np.ascontiguousarray(a)).cuda()
    res = gce.search(d(w.times), d(w.mags), d(w.lc_offsets), d(w.periods), d(w.pdots), 15, 8, top_k=5, want_cube=False,
                     want_stats=True)
    torch.cuda.synchronize()
    st = res.stats.cpu().numpy()
    assert np.all(st[:, 2] >= 0) and np.all(st[:, 2] <= st[:, 0]) and np.all(st[:, 0] <= np.log(8) + 1e-12)
    assert np.all(st[:, 1] > 0) and np.all(st[:, 3] > 0)
    assert np.allclose(st[:, 2], res.best_ce[:, 0].cpu().numpy().astype(np.float64), rtol=1e-6)
    for lc in (0, 500, 999):
        a, b = w.lc_offsets[lc], w.lc_offsets[lc + 1]
        row = oracle.ce_search(w.times[a:b], w.mags[a:b], np.array([0, b - a]), w.periods, w.pdots, 15, 8)[0]
        np.testing.assert_allclose(st[lc], _stats_ref(oracle, row.reshape(1, -1))[0], rtol=RTOL_STATS)


# ------------------------------------------------------------------------------------------ N2: 50 %-overlapping phase bins
@pytest.mark.parametrize("name,kw,n_phi,n_m,k", [
    ("C3", dict(n_lc=3, n_p=900, n_pdot=64), 50, 10, 4),     # the paper's production binning: generic n_phi
    ("C3", dict(n_lc=2, n_p=1111, n_pdot=7), 50, 10, 1),     # trials of a thread do not share a period
    ("C3", dict(n_lc=3, n_p=1500, n_pdot=64), 20, 10, 3),    # compile-time n_phi, register marginals
    ("C2", dict(n_lc=6, n_p=3000), 50, 10, 1),               # Pdot = {0}
    ("C4", dict(n_lc=9, n_p=5000), 15, 8, 5),
    ("C5", dict(n_lc=2, n_p=300, n_pdot=16), 30, 10, 16),    # 2 x points per magnitude bin above the shared table
    ("C1", dict(), 1, 10, 1), ("C1", dict(), 2, 10, 1), ("C1", dict(), 64, 64, 2),
    ("P1", dict(n_lc=2, n_p=2000, n_pdot=32), 50, 10, 5),    # the paper's production grid shape (N4), log-spaced Pdots
])
def test_overlapping_phase_bins_match_oracle(gce, oracle, name, kw, n_phi, n_m, k):
    """overlap = 1 against the oracle's N2 variant (bin k = plain cells k-1 and k, 2N entries): whole fp64 / fp32 cube,
    fused top-k and Eq. 5 statistics."""
    w = W.make(name, **kw)
    ref = oracle.ce_search(w.times, w.mags, w.lc_offsets, w.periods, w.pdots, n_phi, n_m, overlap=True)
    d = lambda a: torch.from_numpy(np.ascontiguousarray(a)).cuda()
    args = (d(w.times), d(w.mags), d(w.lc_offsets), d(w.periods), d(w.pdots), n_phi, n_m)
    for fp64, rtol in ((True, RTOL64), (False, RTOL32)):
        res = gce.search(*args, top_k=k, want_cube=True, ce_fp64=fp64, want_stats=True, overlap=True)
        torch.cuda.synchronize()
        assert_ce_close(res.ce.cpu().numpy(), ref, rtol)
        for lc in range(w.n_lc):
            assert_topk_matches(ref[lc], res.best_idx[lc].cpu().numpy(), res.best_ce[lc].cpu().numpy(), k, rtol, oracle)
    want = _stats_ref(oracle, ref.reshape(w.n_lc, -1))
    got = res.stats.cpu().numpy()
    # constant CE (n_phi = 1 or 2: every bin holds every point): the oracle's two-pass sigma is rounding noise of
    # order 1e-14, the GPU's integer sums give exactly 0 and rho = NaN; compare mean and min there
    ok = want[:, 1] > 1e-10 * np.abs(want[:, 0])
    np.testing.assert_allclose(got[ok], want[ok], rtol=RTOL_STATS, atol=1e-13)
    np.testing.assert_allclose(got[~ok][:, [0, 2]], want[~ok][:, [0, 2]], rtol=RTOL_STATS, atol=1e-13)
    assert np.all(got[~ok][:, 1] == 0.0)
    # the plain search on the same inputs is unchanged by the option and never above the overlapped CE
    plain = gce.search(*args, top_k=0, want_cube=True, ce_fp64=True)
    torch.cuda.synchronize()
    assert bool(torch.all(res.ce.double() >= plain.ce - 1e-5))


def test_overlap_paper_binning_sampled_at_c3_size(gce, oracle):
    """The paper's production setting (50 overlapping phase bins x 10 magnitude bins) on the full C3
    grid without a cube: sampled oracle values against the reported best, selection properties."""
    w = W.make("C3")
    w.n_phase_bins, w.n_mag_bins = 50, 10
    d = lambda a: torch.from_numpy(np.ascontiguousarray(a)).cuda()
    res = gce.search(d(w.times), d(w.mags), d(w.lc_offsets), d(w.periods), d(w.pdots), 50, 10, top_k=3, want_cube=False,
                     want_stats=True, overlap=True)
    torch.cuda.synchronize()
    idx = res.best_idx.cpu().numpy()
    val = res.best_ce.cpu().numpy()
    q = sample_trials(w.periods.size * w.pdots.size, 1500, seed=77)
    ref = oracle.ce_at(w.times, w.mags, w.lc_offsets, w.periods, w.pdots, 50, 10, q, overlap=True)
    for lc in range(w.n_lc):
        exact = oracle.ce_at(w.times, w.mags, w.lc_offsets, w.periods, w.pdots, 50, 10, idx[lc], overlap=True)[lc]
        assert np.all(np.abs(val[lc] - exact) <= RTOL32 * np.abs(exact) + 1e-12)
        better = ref[lc] < exact[-1] * (1 - RTOL64) - 1e-13
        assert set(q[better].tolist()) <= set(idx[lc].tolist())
    st = res.stats.cpu().numpy()
    assert np.allclose(st[:, 2], val[:, 0].astype(np.float64), rtol=1e-6) and np.all(st[:, 1] > 0)


# ------------------------------------------------------------------------------------------ extended-row variant (pair floors)
@pytest.mark.parametrize("n_phi,pdots", [
    (20, np.linspace(-1e-10, 0.0, 64)),                       # C3's own grid: every pair within one cycle
    (20, np.linspace(0.0, -1e-10, 64)),                       # descending Pdot: the other slot of each pair is the base
    (20, np.linspace(-5e-9, 5e-9, 8)),                        # both signs, pairs more than a cycle apart at short periods:
                                                              # the warp falls back to its own floor per trial there
    (15, np.random.default_rng(5).permutation(np.linspace(-3e-10, 1e-10, 16))),   # unordered Pdots: mixed swaps
    (20, np.array([-1e-10, -1e-10, -1e-10, 0.0])),            # equal Pdots inside a pair, Pdot = 0 inside a thread
])
def test_pair_floor_variant_matches_oracle(gce, oracle, n_phi, pdots):
    """k_search's extended-row variant (two trials of a counter word share one floor(x), rows up to 2 n_phi folded back
    when the bin closes) against the oracle: fp64 cube to 1e-12, top-k, Eq. 5; odd tile tails and a short light curve."""
    w = W.make("C3", n_lc=3, n_p=1531, n_pdot=4)
    pd = np.ascontiguousarray(pdots, dtype=np.float64)
    n_m = 10 if n_phi == 20 else 8
    ref = oracle.ce_search(w.times, w.mags, w.lc_offsets, w.periods, pd, n_phi, n_m)
    d = lambda a: torch.from_numpy(np.ascontiguousarray(a)).cuda()
    res = gce.search(d(w.times), d(w.mags), d(w.lc_offsets), d(w.periods), d(pd), n_phi, n_m, top_k=4, want_cube=True,
                     ce_fp64=True, want_stats=True)
    torch.cuda.synchronize()
    assert_ce_close(res.ce.cpu().numpy(), ref, RTOL64)
    for lc in range(w.n_lc):
        assert_topk_matches(ref[lc], res.best_idx[lc].cpu().numpy(), res.best_ce[lc].cpu().numpy(), 4, RTOL64, oracle)
    np.testing.assert_allclose(res.stats.cpu().numpy(), _stats_ref(oracle, ref.reshape(w.n_lc, -1)), rtol=RTOL_STATS)
    res32 = gce.search(d(w.times), d(w.mags), d(w.lc_offsets), d(w.periods), d(pd), n_phi, n_m, top_k=4, want_cube=True)
    torch.cuda.synchronize()
    assert_ce_close(res32.ce.cpu().numpy(), ref, RTOL32)
    assert torch.equal(res32.best_idx, res.best_idx)


def test_pair_floor_variant_streams_a_long_light_curve(gce, oracle):
    """The extended-row variant is planned from the AVERAGE light-curve length; one light curve that is longer than the
    remaining shared-memory buffer (3420 points beside 168 KB of counters) is streamed through two half buffers."""
    rng = np.random.default_rng(17)
    lcs = []
    for n in [300] * 11 + [6001]:
        t = np.sort(rng.uniform(0, 9e7, n))
        lcs.append((t, W.two_dip_mags(rng, t, 533.0, -4e-11, 0.5, 0.2, 0.05)))
    times = np.concatenate([t for t, _ in lcs]); mags = np.concatenate([m for _, m in lcs])
    offs = np.cumsum([0] + [t.size for t, _ in lcs]).astype(np.int64)
    periods = 1.0 / np.linspace(1 / 1200.0, 1 / 400.0, 520)
    pdots = np.linspace(-8e-11, 0.0, 8)
    ref = oracle.ce_search(times, mags, offs, periods, pdots, 20, 10)
    d = lambda a: torch.from_numpy(np.ascontiguousarray(a)).cuda()
    res = gce.search(d(times), d(mags), d(offs), d(periods), d(pdots), 20, 10, top_k=3, want_cube=True, ce_fp64=True,
                     want_stats=True)
    torch.cuda.synchronize()
    assert_ce_close(res.ce.cpu().numpy(), ref, RTOL64)
    for lc in range(12):
        assert_topk_matches(ref[lc], res.best_idx[lc].cpu().numpy(), res.best_ce[lc].cpu().numpy(), 3, RTOL64, oracle)
    np.testing.assert_allclose(res.stats.cpu().numpy(), _stats_ref(oracle, ref.reshape(12, -1)), rtol=RTOL_STATS)


@pytest.mark.parametrize("n_phi,overlap,step", [(20, False, 0.30), (20, False, 0.45), (20, False, 3.0), (15, False, 0.30),
                                                (50, True, 0.33), (50, False, 0.6), (50, True, 5.0)])
def test_pdot_zero_grids_fine_and_coarse(gce, oracle, n_phi, overlap, step):
    """Pdot = {0} on frequency grids from properly oversampled (step x 1/T between neighbouring trials; the paper uses
    1/(3T)) to coarse, with the paper's VRO-like time sampling: the trials of a thread have different
    periods (no shared a = dt/P, no shared floors).  (Sharing floors between neighbouring periods was measured: +5 % on
    this kind of grid, -2 to -10 % on every BASELINE config through the larger kernels, so it is not built.)"""
    rng = np.random.default_rng(23)
    lcs = []
    for n in (500, 731, 64):
        t = W.vro_like_cadence(rng, n)
        lcs.append((t, W.two_dip_mags(rng, t, 1234.5, 0.0, 0.4, 0.2, 0.1)))
    times = np.concatenate([t for t, _ in lcs]); mags = np.concatenate([m for _, m in lcs])
    offs = np.cumsum([0] + [t.size for t, _ in lcs]).astype(np.int64)
    T = max(float(t[-1]) for t, _ in lcs)
    freqs = 1 / 1500.0 + (step / T) * np.arange(3001)
    periods = np.ascontiguousarray(1.0 / freqs)
    n_m = 10 if n_phi != 15 else 8
    ref = oracle.ce_search(times, mags, offs, periods, np.zeros(1), n_phi, n_m, overlap=overlap)
    d = lambda a: torch.from_numpy(np.ascontiguousarray(a)).cuda()
    res = gce.search(d(times), d(mags), d(offs), d(periods), d(np.zeros(1)), n_phi, n_m, top_k=3, want_cube=True,
                     ce_fp64=True, want_stats=True, overlap=overlap)
    torch.cuda.synchronize()
    assert_ce_close(res.ce.cpu().numpy(), ref, RTOL64)
    for lc in range(3):
        assert_topk_matches(ref[lc], res.best_idx[lc].cpu().numpy(), res.best_ce[lc].cpu().numpy(), 3, RTOL64, oracle)
    np.testing.assert_allclose(res.stats.cpu().numpy(), _stats_ref(oracle, ref.reshape(3, -1)), rtol=RTOL_STATS)
    # ascending periods (descending 1/P) give the same cube, reversed
    res_r = gce.search(d(times), d(mags), d(offs), d(periods[::-1].copy()), d(np.zeros(1)), n_phi, n_m, top_k=0,
                       want_cube=True, ce_fp64=True, overlap=overlap)
    torch.cuda.synchronize()
    assert torch.equal(res_r.ce.flip(1), res.ce)


# ------------------------------------------------------------------------------------------ N4: per-filter median / std
def test_two_filter_normalisation_matches_the_oracle(gce, oracle):
    """NEXT item N4: normalise = 1 with per-point filter ids.  The GPU's S0 follows the same frozen
    arithmetic as oracle.normalise (order-statistic median, sequential sums), so magnitude bins and counts are bit-exact
    and the cube agrees at the fp64 tolerance; selection and Eq. 5 follow."""
    w, filt = W.two_filter_batch(21, n_lc=5, n_obs=401, n_p=500, n_pdot=4)
    u = oracle.normalise_batch(w.mags, w.lc_offsets, filt)
    ref = oracle.ce_search(w.times, u, w.lc_offsets, w.periods, w.pdots, 20, 10)
    raw = oracle.ce_search(w.times, w.mags, w.lc_offsets, w.periods, w.pdots, 20, 10)
    assert np.max(np.abs(ref - raw)) > 1e-2          # the option changes the result on a two-filter light curve
    args = (dev(w.times), dev(w.mags), dev(w.lc_offsets), dev(w.periods), dev(w.pdots), 20, 10)
    res = gce.search(*args, top_k=3, want_cube=True, ce_fp64=True, want_stats=True, normalise=True, filter_ids=dev(filt))
    torch.cuda.synchronize()
    assert_ce_close(res.ce.cpu().numpy(), ref, RTOL64)
    for lc in range(w.n_lc):
        assert_topk_matches(ref[lc], res.best_idx[lc].cpu().numpy(), res.best_ce[lc].cpu().numpy(), 3, RTOL64, oracle)
    # bit-exact counts through the normalised magnitudes
    q = torch.tensor([0, 17, 500 * 4 - 1], dtype=torch.int64, device="cuda")
    fdev = dev(filt)   # the params hold a raw pointer: keep the tensor alive
    prm = gce.make_params(20, 10, normalise=True, filter_ids=fdev)
    counts = torch.empty((w.n_lc, 3, 20, 10), dtype=torch.int32, device="cuda")
    ws = torch.empty(gce.gce_ce_workspace_bytes(w.total_points, w.n_lc, 500, 4, prm), dtype=torch.uint8, device="cuda")
    gce.gce_ce_debug_histogram(dev(w.times), dev(w.mags), dev(w.lc_offsets), dev(w.periods), dev(w.pdots), prm, q, counts, None, ws)
    torch.cuda.synchronize()
    for lc in range(w.n_lc):
        a, b = int(w.lc_offsets[lc]), int(w.lc_offsets[lc + 1])
        refc = oracle.histogram(w.times[a:b], u[a:b], w.periods, w.pdots, 20, 10, q.cpu().numpy())
        assert np.array_equal(counts[lc].cpu().numpy().astype(np.int64), refc)
    # host entry: filter ids as a host array
    ce_h = np.empty((w.n_lc, 500, 4), dtype=np.float64)
    idx_h = np.empty((w.n_lc, 3), dtype=np.int64)
    gce.gce_ce_search_host(w.times, w.mags, w.lc_offsets, w.periods, w.pdots,
                           gce.make_params(20, 10, top_k=3, ce_fp64=True, normalise=True, filter_ids=torch.from_numpy(filt)),
                           ce_h, idx_h, None)
    assert np.array_equal(ce_h, res.ce.cpu().numpy()) and np.array_equal(idx_h, res.best_idx.cpu().numpy())


@pytest.mark.parametrize("n_obs,n_filters", [(1, 1), (2, 1), (777, 1), (5000, 3), (20001, 8)])
def test_normalised_magnitude_bins_are_bit_exact(gce, oracle, n_obs, n_filters):
    """S0 + S1 alone: with n_phase_bins = 1 every count table is the magnitude histogram of the normalised light curve
    (independent of the trial), compared bit for bit with the oracle's bins; even / odd filter sizes, a filter with one
    point, ties, light curves longer than one radix-select pass's worth of threads."""
    rng = np.random.default_rng(n_obs * 10 + n_filters)
    m = np.round(rng.normal(17.0, 0.5, n_obs), 2)               # rounded: many exact ties around the median
    f = rng.integers(0, n_filters, n_obs).astype(np.int32)
    if n_obs > 10:
        f[0] = n_filters - 1
        m[f == 0] += 2.5
    t = np.sort(rng.uniform(0, 1e7, n_obs))
    offs = np.array([0, n_obs], dtype=np.int64)
    u = oracle.normalise(m, f)
    mb = oracle.preprocess(t, u, 13)[2]
    fdev = dev(f)
    prm = gce.make_params(1, 13, normalise=True, filter_ids=fdev)
    counts = torch.empty((1, 1, 1, 13), dtype=torch.int32, device="cuda")
    ws = torch.empty(gce.gce_ce_workspace_bytes(n_obs, 1, 1, 1, prm), dtype=torch.uint8, device="cuda")
    gce.gce_ce_debug_histogram(dev(t), dev(m), dev(offs), dev(np.array([500.0])), dev(np.zeros(1)), prm,
                               torch.zeros(1, dtype=torch.int64, device="cuda"), counts, None, ws)
    torch.cuda.synchronize()
    assert np.array_equal(counts.cpu().numpy().ravel(), np.bincount(mb, minlength=13))


def test_one_filter_normalisation_equals_min_max(gce):
    """Reading Q2 on the GPU: with one filter the paper's normalisation leaves the search result unchanged up to points
    within rounding of a magnitude-bin edge -- here: the same best trials on C2-like light curves."""
    w = W.make("C2", n_lc=6, n_p=1500)
    args = (dev(w.times), dev(w.mags), dev(w.lc_offsets), dev(w.periods), dev(w.pdots), 20, 10)
    a = gce.search(*args, top_k=1, want_cube=True, ce_fp64=True)
    b = gce.search(*args, top_k=1, want_cube=True, ce_fp64=True, normalise=True)
    torch.cuda.synchronize()
    assert torch.equal(a.best_idx, b.best_idx)
    assert float((a.ce - b.ce).abs().max()) < 0.02   # a handful of edge points may move by one bin
