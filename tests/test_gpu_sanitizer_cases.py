"""Small cases for compute-sanitizer (memcheck / racecheck on C1-size inputs -- the shared-memory
histograms, the volatile top-k state, the two mbarriers and the refill of streamed light curves are the race risk).

They are ordinary GPU parity tests, sized so that a run under `compute-sanitizer --tool racecheck` (or memcheck /
initcheck / synccheck) ends within minutes:
    compute-sanitizer --tool racecheck python -m pytest tests/test_gpu_sanitizer_cases.py -m gpu -q -x
On the round-3 pool the tool is closed (profiles/r3_sanitizer.md has the answer it gave), so for now these run plain,
as part of `-m gpu`.
Every case goes through the C ABI: C1 (Pdot = {0}, 20 x 10, cube + argmin), a streamed light curve next to a short
one, the shared-floor (EXT) kernels with top-k and Eq. 5 statistics, the 50-bin overlapping kernels, a wide
(32-bit counter) call, the dump-mode kernels, the period split with its merge, and the no-allocation entry point.
"""
import numpy as np
import pytest
import torch

import gce_workloads as W

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def gce():
    from paper_2006_06866_b200.build import build
    build()
    import paper_2006_06866_b200 as g
    return g


def dev(a):
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


def _check(gce, oracle, w, top_k, want_stats=False, overlap=False, ce_fp64=True):
    ref = oracle.ce_search(w.times, w.mags, w.lc_offsets, w.periods, w.pdots, w.n_phase_bins, w.n_mag_bins, overlap=overlap)
    res = gce.search(dev(w.times), dev(w.mags), dev(w.lc_offsets), dev(w.periods), dev(w.pdots), w.n_phase_bins,
                     w.n_mag_bins, top_k=top_k, want_cube=True, ce_fp64=ce_fp64, want_stats=want_stats, overlap=overlap)
    torch.cuda.synchronize()
    got = res.ce.cpu().numpy().astype(np.float64)
    np.testing.assert_allclose(got, ref, rtol=1e-12 if ce_fp64 else 1e-5, atol=1e-13)
    for lc in range(w.n_lc):
        flat = ref[lc].ravel()
        gi = res.best_idx[lc].cpu().numpy()
        want = np.sort(flat)[:top_k]
        np.testing.assert_allclose(flat[gi], want, rtol=1e-12, atol=1e-13)
        if want_stats:
            mu, sigma, _rho = oracle.significance(flat)
            np.testing.assert_allclose(res.stats[lc, :3].cpu().numpy(), [mu, sigma, flat.min()], rtol=1e-9, atol=1e-13)
    return res


def test_c1(gce, oracle):
    _check(gce, oracle, W.make("C1"), top_k=1, ce_fp64=False)


def test_streamed_light_curve_next_to_a_short_one(gce, oracle):
    rng = np.random.default_rng(5)
    n_long = 9000                                  # beyond the 8192-point shared-memory buffer: two half buffers, refilled per tile
    t_long = np.sort(rng.uniform(0, 3e7, n_long))
    m_long = W.two_dip_mags(rng, t_long, 611.0, -2e-11, 0.5, 0.2, 0.05)
    t_short = np.sort(rng.uniform(0, 3e7, 300))
    w = W.Workload("streamed", np.concatenate([t_long, t_short]), np.concatenate([m_long, rng.normal(size=300)]),
                   np.array([0, n_long, n_long + 300], dtype=np.int64), 1.0 / np.linspace(1 / 900.0, 1 / 300.0, 600),
                   np.linspace(-4e-11, 0.0, 4), 20, 10, 3, True)
    _check(gce, oracle, w, top_k=3, want_stats=True)


def test_shared_floor_kernels_with_topk_and_stats(gce, oracle):
    _check(gce, oracle, W.make("C3", n_lc=2, n_p=1300, n_pdot=8), top_k=4, want_stats=True)


def test_fifty_overlapping_bins(gce, oracle):
    w = W.make("C4", n_lc=3, n_p=2500)
    w.n_phase_bins, w.n_mag_bins = 50, 10
    _check(gce, oracle, w, top_k=5, want_stats=True, overlap=True)


def test_wide_counters(gce, oracle):
    rng = np.random.default_rng(6)
    n = 66000
    t = np.sort(rng.uniform(0, 3e7, n))
    w = W.Workload("wide", t, W.two_dip_mags(rng, t, 611.0, 0.0, 0.5, 0.2, 0.05), np.array([0, n], dtype=np.int64),
                   1.0 / np.linspace(1 / 900.0, 1 / 300.0, 128), np.linspace(-4e-11, 0.0, 2), 20, 10, 2, True)
    _check(gce, oracle, w, top_k=2, want_stats=True)


def test_dump_mode_and_debug_bins(gce, oracle):
    w = W.make("C3", n_lc=2, n_p=1300, n_pdot=8)
    n_trials = w.n_p * w.n_pdot
    q = torch.tensor([0, 7, n_trials // 2 + 3, n_trials - 1], dtype=torch.int64, device="cuda")
    prm = gce.make_params(20, 10)
    counts = torch.empty((2, 4, 20, 10), dtype=torch.int32, device="cuda")
    ce_at = torch.empty((2, 4), dtype=torch.float64, device="cuda")
    ws = torch.empty(gce.gce_ce_workspace_bytes(w.total_points, 2, w.n_p, w.n_pdot, prm), dtype=torch.uint8, device="cuda")
    gce.gce_ce_debug_histogram(dev(w.times), dev(w.mags), dev(w.lc_offsets), dev(w.periods), dev(w.pdots), prm, q, counts, ce_at, ws)
    torch.cuda.synchronize()
    for lc in range(2):
        a, b = w.lc_offsets[lc], w.lc_offsets[lc + 1]
        ref = oracle.histogram(w.times[a:b], w.mags[a:b], w.periods, w.pdots, 20, 10, q.cpu().numpy())
        assert np.array_equal(counts[lc].cpu().numpy().astype(np.int64), ref)


def test_period_split_and_merge(gce):
    w = W.make("C3", n_lc=2, n_p=1300, n_pdot=8)
    args = (dev(w.times), dev(w.mags), dev(w.lc_offsets), dev(w.periods), dev(w.pdots), 20, 10)
    whole = gce.search(*args, top_k=3, want_cube=False, want_stats=True)
    split = gce.search_period_chunks(*args, [(0, 500), (500, 501), (501, 1300)], top_k=3, want_stats=True)
    torch.cuda.synchronize()
    assert torch.equal(whole.best_idx, split.best_idx) and torch.equal(whole.stats, split.stats)


def test_no_allocation_entry_point(gce):
    w = W.make("C3", n_lc=2, n_p=1300, n_pdot=8)
    args = (dev(w.times), dev(w.mags), dev(w.lc_offsets), dev(w.periods), dev(w.pdots))
    ref = gce.search(*args, 20, 10, top_k=3, want_cube=True, want_stats=True)
    prm = gce.make_params(20, 10, top_k=3, want_stats=True)
    ce, idx = torch.empty_like(ref.ce), torch.empty_like(ref.best_idx)
    bce, st = torch.empty_like(ref.best_ce), torch.empty_like(ref.stats)
    gce.gce_ce_search_static(*args, prm, ce, idx, bce, st)
    torch.cuda.synchronize()
    assert torch.equal(idx, ref.best_idx) and torch.equal(ce, ref.ce) and torch.equal(st, ref.stats)
