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
from test_gpu_parity import RTOL32, RTOL64, assert_ce_close, assert_topk_matches, dev, run_search

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
