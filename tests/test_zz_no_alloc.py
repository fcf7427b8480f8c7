"""gce_ce_search_static: the search for callers that may not allocate device memory.

Some users of this library run as guests in a GPU process they do not own (an alert broker, a plug-in of a pipeline
that took the whole card for its own pool): they get input and output buffers and a stream, never an allocator, and
cudaMalloc is forbidden to them because it stalls the device and can fail late.  For them the library carries its
scratch memory inside its own device image (8 MiB, include/gce_ce.h).  These tests check that this entry point gives
exactly what the workspace-taking gce_ce_search gives -- it launches the same kernels -- on two calls made straight
after each other, the second with a different shape, so that it runs on whatever the first left behind in the shared
array; that an over-sized call is refused with its own error code; and that nothing was allocated through torch on the
way.  The file sorts last on purpose: `pytest -x` stops at the first failure, and a failure here must not hide any
other test.  It passes alone in a fresh process (first call on the device = the address look-up) and after the suite.
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


def _dev(a):
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


class _Case:
    """Device inputs of one workload, the existing path's outputs, and empty outputs for the static entry point."""

    def __init__(self, gce, w, top_k, want_stats, overlap=False, ce_fp64=False):
        self.t, self.m, self.off = _dev(w.times), _dev(w.mags), _dev(w.lc_offsets)
        self.p, self.pd = _dev(w.periods), _dev(w.pdots)
        self.prm = gce.make_params(w.n_phase_bins, w.n_mag_bins, top_k, ce_fp64, want_stats, overlap)
        self.ref = gce.search(self.t, self.m, self.off, self.p, self.pd, w.n_phase_bins, w.n_mag_bins, top_k=top_k,
                              want_cube=True, ce_fp64=ce_fp64, want_stats=want_stats, overlap=overlap)
        self.need = gce.gce_ce_workspace_bytes(w.total_points, w.n_lc, w.n_p, w.n_pdot, self.prm)
        # outputs are the caller's; filled with a pattern no result can equal, so an unwritten element is noticed
        self.ce = torch.full_like(self.ref.ce, -7.0)
        self.idx = torch.full_like(self.ref.best_idx, -99)
        self.bce = torch.full_like(self.ref.best_ce, -7.0)
        self.stats = torch.full_like(self.ref.stats, -7.0) if want_stats else None

    def run_static(self, gce):
        gce.gce_ce_search_static(self.t, self.m, self.off, self.p, self.pd, self.prm, self.ce, self.idx, self.bce, self.stats)

    def check(self):
        # same kernels, same plan, integer accumulation: equal bits, which is inside every tolerance the parity tests
        # use (1e-5 relative on the fp32 cube, 1e-12 on the fp64 cube, exact indices)
        assert torch.equal(self.idx, self.ref.best_idx)
        assert torch.equal(self.ce.view(torch.int32 if self.ce.dtype == torch.float32 else torch.int64),
                           self.ref.ce.view(torch.int32 if self.ce.dtype == torch.float32 else torch.int64))
        np.testing.assert_array_equal(self.bce.cpu().numpy(), self.ref.best_ce.cpu().numpy())
        if self.stats is not None:
            np.testing.assert_array_equal(self.stats.cpu().numpy(), self.ref.stats.cpu().numpy())


def test_static_scratch_matches_workspace_path_on_two_calls_in_a_row(gce):
    # A: the P-Pdot shape of C3 (20 x 10 bins, 8 Pdots per period, shared-floor kernels), top-4 and Eq. 5 statistics
    a = _Case(gce, W.make("C3", n_lc=5, n_p=900, n_pdot=8), top_k=4, want_stats=True)
    # B: the Pdot = {0} shape of C4 with the paper's 50 overlapping bins, more and shorter light curves, fp64 cube
    wb = W.make("C4", n_lc=37, n_p=3001)
    wb.n_phase_bins, wb.n_mag_bins = 50, 10
    b = _Case(gce, wb, top_k=5, want_stats=False, overlap=True, ce_fp64=True)
    assert 0 < a.need <= gce.STATIC_SCRATCH_BYTES and 0 < b.need <= gce.STATIC_SCRATCH_BYTES and a.need != b.need
    torch.cuda.synchronize()
    before = torch.cuda.memory_stats()["allocation.all.allocated"]
    a.run_static(gce)   # two calls back to back on one stream, no synchronisation between them:
    b.run_static(gce)   # B works on the scratch exactly as A left it
    after = torch.cuda.memory_stats()["allocation.all.allocated"]
    torch.cuda.synchronize()
    assert after == before, "the static entry point's wrapper must not create device tensors"
    a.check()
    b.check()
    # and once more in the other order, over B's leftovers
    a.ce.fill_(-7.0); a.idx.fill_(-99); a.bce.fill_(-7.0); a.stats.fill_(-7.0)
    a.run_static(gce)
    torch.cuda.synchronize()
    a.check()


def test_static_scratch_refuses_what_does_not_fit(gce):
    """More scratch than the built-in array holds: a dedicated error code, nothing launched, outputs untouched."""
    n_lc, n_obs = 3000, 200
    prm = gce.make_params(15, 8, top_k=5)
    total = n_lc * n_obs
    assert gce.gce_ce_workspace_bytes(total, n_lc, 1000, 1, prm) > gce.STATIC_SCRATCH_BYTES
    t = torch.zeros(total, dtype=torch.float64, device="cuda")
    off = torch.arange(0, total + 1, n_obs, dtype=torch.int64, device="cuda")
    p = torch.full((1000,), 100.0, dtype=torch.float64, device="cuda")
    pd = torch.zeros(1, dtype=torch.float64, device="cuda")
    idx = torch.full((n_lc, 5), -99, dtype=torch.int64, device="cuda")
    with pytest.raises(gce.GceError) as e:
        gce.gce_ce_search_static(t, t, off, p, pd, prm, None, idx, None, None)
    assert e.value.code == gce.ERR_STATIC_LIMIT == -5
    assert "GCE_CE_STATIC_SCRATCH_BYTES" in str(e.value)
    torch.cuda.synchronize()
    assert bool((idx == -99).all())
    # the ordinary argument checks still come first
    with pytest.raises(gce.GceError) as e2:
        gce.gce_ce_search_static(t, t, off, p, pd, gce.make_params(0, 8, top_k=5), None, idx, None, None)
    assert e2.value.code == -2
