"""N4: period sub-ranges and exact merging (PAPER.md:232-234 batch merge; SURVEY.md 8e period-axis split).

gce_ce_search_partial over disjoint period ranges + gce_ce_merge_partials must reproduce gce_ce_search on the whole grid
bit for bit (indices, fp32 CE, Eq. 5 statistics), however the grid is split, because every key and sum is an integer.
One two-"rank" case runs the ranks one after the other in one process and concatenates their blobs; the other runs
search_period_chunks(dist=...) in two real processes (world_size 2, gloo all-gather of the host-staged blobs, both ranks
on cuda:0 -- their kernels never wait on one another).
"""
import os

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


def d(a):
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


@pytest.mark.parametrize("name,kw,k,overlap", [
    ("C3", dict(n_lc=3, n_p=1300, n_pdot=64), 4, False),
    ("C3", dict(n_lc=2, n_p=777, n_pdot=7), 1, False),
    ("C2", dict(n_lc=5, n_p=4000), 3, True),
    ("C5", dict(n_lc=2, n_p=260, n_pdot=16), 16, False),
])
def test_period_chunks_merge_bit_exactly(gce, name, kw, k, overlap):
    w = W.make(name, **kw)
    args = (d(w.times), d(w.mags), d(w.lc_offsets), d(w.periods), d(w.pdots), w.n_phase_bins, w.n_mag_bins)
    whole = gce.search(*args, top_k=k, want_cube=True, want_stats=True, overlap=overlap)
    torch.cuda.synchronize()
    n_p = w.n_p
    for cuts in ([0, n_p], [0, 1, n_p], [0, n_p // 3, n_p // 3, 2 * n_p // 3 + 5, n_p], [0, 7, 8, 9, n_p - 1, n_p]):
        chunks = list(zip(cuts[:-1], cuts[1:]))
        slices = {}
        res = gce.search_period_chunks(*args, chunks, top_k=k, want_stats=True, overlap=overlap,
                                       cube_sink=lambda a, b, ce: slices.__setitem__((a, b), ce.clone()))
        torch.cuda.synchronize()
        assert torch.equal(res.best_idx, whole.best_idx), cuts
        assert torch.equal(res.best_ce, whole.best_ce), cuts
        assert np.array_equal(res.stats.cpu().numpy(), whole.stats.cpu().numpy()), cuts
        for (a, b) in chunks:
            if b > a:   # the sink is called for non-empty slices only
                assert torch.equal(slices[(a, b)], whole.ce[:, a:b, :]), (cuts, a)
            else:
                assert (a, b) not in slices


def test_two_ranks_split_the_period_axis(gce):
    """One deep target (fewer light curves than GPUs): each 'rank' searches half of the periods in two chunks, merges its
    chunks into one blob array, the blob arrays are concatenated (= all_gather) and merged."""
    w = W.make("C3", n_lc=1, n_p=3000, n_pdot=32)
    args = (d(w.times), d(w.mags), d(w.lc_offsets), d(w.periods), d(w.pdots))
    prm = gce.make_params(20, 10, top_k=5, want_stats=True)
    words = gce.gce_ce_partial_words(5)
    ws = torch.empty(gce.gce_ce_workspace_bytes(w.total_points, 1, 3000, 32, prm), dtype=torch.uint8, device="cuda")
    per_rank = []
    for lo, hi in ((0, 1400), (1400, 3000)):
        parts = torch.empty((2, 1, words), dtype=torch.int64, device="cuda")
        mid = (lo + hi) // 2
        gce.gce_ce_search_partial(*args, prm, lo, mid, parts[0], None, ws)
        gce.gce_ce_search_partial(*args, prm, mid, hi, parts[1], None, ws)
        one = torch.empty((1, 1, words), dtype=torch.int64, device="cuda")
        gce.binding._merge_to_partial(parts, 2, 1, prm, one)
        per_rank.append(one)
    gathered = torch.cat(per_rank, dim=0)
    idx = torch.empty((1, 5), dtype=torch.int64, device="cuda")
    val = torch.empty((1, 5), dtype=torch.float32, device="cuda")
    st = torch.empty((1, 4), dtype=torch.float64, device="cuda")
    gce.gce_ce_merge_partials(gathered, 2, 1, prm, idx, val, st)
    whole = gce.search(*args, 20, 10, top_k=5, want_cube=False, want_stats=True)
    torch.cuda.synchronize()
    assert torch.equal(idx, whole.best_idx) and torch.equal(val, whole.best_ce)
    assert np.array_equal(st.cpu().numpy(), whole.stats.cpu().numpy())


def test_empty_range_and_errors(gce):
    w = W.make("C2", n_lc=2, n_p=50)
    args = (d(w.times), d(w.mags), d(w.lc_offsets), d(w.periods), d(w.pdots))
    prm = gce.make_params(20, 10, top_k=2, want_stats=True)
    words = gce.gce_ce_partial_words(2)
    assert words == 2 * 2 + 10
    ws = torch.empty(gce.gce_ce_workspace_bytes(w.total_points, 2, 50, 1, prm), dtype=torch.uint8, device="cuda")
    parts = torch.empty((2, 2, words), dtype=torch.int64, device="cuda")
    gce.gce_ce_search_partial(*args, prm, 10, 10, parts[0], None, ws)      # empty range: a neutral blob
    gce.gce_ce_search_partial(*args, prm, 0, 50, parts[1], None, ws)
    res = gce.search(*args, 20, 10, top_k=2, want_cube=False, want_stats=True)
    idx = torch.empty((2, 2), dtype=torch.int64, device="cuda")
    st = torch.empty((2, 4), dtype=torch.float64, device="cuda")
    gce.gce_ce_merge_partials(parts, 2, 2, prm, idx, None, st)
    torch.cuda.synchronize()
    assert torch.equal(idx, res.best_idx) and np.array_equal(st.cpu().numpy(), res.stats.cpu().numpy())
    with pytest.raises(gce.GceError) as e:
        gce.gce_ce_search_partial(*args, prm, 40, 51, parts[0], None, ws)
    assert e.value.code == -2


def test_host_entry_pipelines_large_cubes_bit_exactly(gce):
    """gce_ce_search_host with a cube >= 64 MB splits the period axis into chunks and overlaps the device-to-host copy
    of each slice with the next chunk's search; outputs equal the single device call bit for bit."""
    w = W.make("C3", n_lc=6, n_p=45001, n_pdot=64)      # 69 MB fp32 cube, ragged last chunk
    prm = gce.make_params(20, 10, top_k=3, want_stats=True)
    ce = np.empty((6, 45001, 64), dtype=np.float32)
    idx = np.empty((6, 3), dtype=np.int64)
    val = np.empty((6, 3), dtype=np.float32)
    st = np.empty((6, 4), dtype=np.float64)
    gce.gce_ce_search_host(w.times, w.mags, w.lc_offsets, w.periods, w.pdots, prm, ce, idx, val, st)
    res = gce.search(d(w.times), d(w.mags), d(w.lc_offsets), d(w.periods), d(w.pdots), 20, 10, top_k=3, want_cube=True,
                     want_stats=True)
    torch.cuda.synchronize()
    assert np.array_equal(ce, res.ce.cpu().numpy())
    assert np.array_equal(idx, res.best_idx.cpu().numpy()) and np.array_equal(val, res.best_ce.cpu().numpy())
    assert np.array_equal(st, res.stats.cpu().numpy())
    # cube only (no selection, no statistics)
    prm0 = gce.make_params(20, 10)
    ce2 = np.zeros_like(ce)
    gce.gce_ce_search_host(w.times, w.mags, w.lc_offsets, w.periods, w.pdots, prm0, ce2, None, None, None)
    assert np.array_equal(ce2, ce)


def _period_split_rank(rank, world, port, result_dir):
    """One real process per rank (both on cuda:0; the exchange is gloo's all_gather of the host-staged blobs: NCCL
    refuses two ranks on one GPU).  The ranks' kernels never wait on one another: each rank searches its own period
    ranges, the only exchange is the all-gather of n_lc x (2k + 10) int64 blobs, after which every rank merges."""
    import torch.distributed as dist
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        import paper_2006_06866_b200 as gce
        torch.cuda.set_device(0)
        w = W.make("C3", n_lc=1, n_p=3000, n_pdot=32)     # one deep target: fewer light curves than ranks
        args = (d(w.times), d(w.mags), d(w.lc_offsets), d(w.periods), d(w.pdots), 20, 10)
        chunks = [[(0, 700), (700, 1400)], [(1400, 3000)]][rank]   # complementary halves, unequal chunk counts
        side = torch.cuda.Stream()
        got = gce.search_period_chunks(*args, chunks, top_k=5, want_stats=True, dist=dist, stream=side)
        whole = gce.search(*args, top_k=5, want_cube=False, want_stats=True)
        torch.cuda.synchronize()
        ok = (torch.equal(got.best_idx, whole.best_idx) and torch.equal(got.best_ce, whole.best_ce)
              and np.array_equal(got.stats.cpu().numpy(), whole.stats.cpu().numpy()))
        # a rank with no periods at all still takes part in the exchange
        chunks2 = [[(0, 3000)], []][rank]
        got2 = gce.search_period_chunks(*args, chunks2, top_k=5, want_stats=True, dist=dist)
        torch.cuda.synchronize()
        ok = ok and torch.equal(got2.best_idx, whole.best_idx) and np.array_equal(got2.stats.cpu().numpy(), whole.stats.cpu().numpy())
        with open(os.path.join(result_dir, f"rank{rank}.txt"), "w") as f:
            f.write("ok" if ok else "mismatch")
    finally:
        dist.destroy_process_group()


def test_period_axis_split_in_two_processes(gce, tmp_path):
    """SURVEY.md 8(e) / PAPER.md:234: the period-axis split with its one collective, run in two real processes
    (world_size 2): every rank's selection and Eq. 5 statistics are bit-equal to the unsplit call."""
    import socket
    import torch.multiprocessing as mp
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        port = s.getsockname()[1]
    mp.spawn(_period_split_rank, args=(2, port, str(tmp_path)), nprocs=2, join=True)
    for r in range(2):
        assert (tmp_path / f"rank{r}.txt").read_text() == "ok"
