"""N > 1 host logic on CPU: partition by light curve, world_size-2 gloo run.

No GPU here, so each gloo rank stands in for its GPU with the oracle on its own shard; what is under test is
the sharding / gather / timing-reduction plumbing of paper_2006_06866_b200.sharding, which the GPU path uses
unchanged (bench.py, N > 1).
"""
import os
import socket

import numpy as np
import pytest

import gce_workloads as W
from paper_2006_06866_b200 import sharding


def test_partition_covers_every_light_curve_once():
    rng = np.random.default_rng(0)
    for n_lc in (0, 1, 2, 7, 64, 1000):
        sizes = rng.integers(0, 3000, size=n_lc)
        offs = np.concatenate([[0], np.cumsum(sizes)]).astype(np.int64)
        for world in (1, 2, 3, 8):
            ranges = sharding.partition_light_curves(offs, world)
            assert len(ranges) == world
            assert ranges[0][0] == 0 and ranges[-1][1] == n_lc
            assert all(a[1] == b[0] for a, b in zip(ranges, ranges[1:]))
            assert all(lo <= hi for lo, hi in ranges)
            if n_lc >= 8 * world and offs[-1] > 0:
                # balanced by points to within the largest light curve
                pts = [int(offs[hi] - offs[lo]) for lo, hi in ranges]
                assert max(pts) - min(pts) <= 2 * int(sizes.max())


def test_shard_arrays_rebases_offsets():
    w = W.random_batch(3, n_lc=6, n_min=10, n_max=50, n_p=4, n_pdot=1)
    t, m, o = sharding.shard_arrays(w.times, w.mags, w.lc_offsets, 2, 5)
    assert o[0] == 0 and o.shape[0] == 4 and t.shape[0] == o[-1] == m.shape[0]
    assert np.array_equal(t, w.times[w.lc_offsets[2]:w.lc_offsets[5]])


def test_single_process_helpers_are_identity():
    assert sharding.reduce_timing(3.0, 10.0) == (3.0, 10.0)
    x = np.arange(6).reshape(3, 2)
    assert np.array_equal(sharding.gather_per_light_curve(x, 3, [(0, 3)], 0), x)


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, out_dir):
    import torch.distributed as dist
    import oracle
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        w = W.make("C3", n_lc=5, n_p=60, n_pdot=4)
        ranges = sharding.partition_light_curves(w.lc_offsets, world)
        lo, hi = ranges[rank]
        t, m, o = sharding.shard_arrays(w.times, w.mags, w.lc_offsets, lo, hi)
        ce = oracle.ce_search(t, m, o, w.periods, w.pdots, w.n_phase_bins, w.n_mag_bins).reshape(hi - lo, -1)
        best = np.stack([oracle.topk(row, 3)[0] for row in ce]) if hi > lo else np.zeros((0, 3), dtype=np.int64)
        best_all = sharding.gather_per_light_curve(best, w.n_lc, ranges, rank, dist)
        ms, pf = sharding.reduce_timing(10.0 + rank, float(int(o[-1]) * w.n_p * w.n_pdot), dist)
        if rank == 0:
            np.save(os.path.join(out_dir, "best.npy"), best_all)
            np.save(os.path.join(out_dir, "acct.npy"), np.array([ms, pf]))
    finally:
        dist.destroy_process_group()


@pytest.mark.timeout(300)
def test_world_size_2_gloo_matches_single_process(tmp_path, oracle):
    import torch.multiprocessing as mp
    world = 2
    mp.spawn(_worker, args=(world, _free_port(), str(tmp_path)), nprocs=world, join=True)
    w = W.make("C3", n_lc=5, n_p=60, n_pdot=4)
    ce = oracle.ce_search(w.times, w.mags, w.lc_offsets, w.periods, w.pdots, w.n_phase_bins, w.n_mag_bins)
    ref = np.stack([oracle.topk(row, 3)[0] for row in ce.reshape(w.n_lc, -1)])
    assert np.array_equal(np.load(tmp_path / "best.npy"), ref)
    ms, pf = np.load(tmp_path / "acct.npy")
    assert ms == 11.0                       # max over ranks
    assert pf == float(w.point_folds)       # sum over ranks = the whole job
