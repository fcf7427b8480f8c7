"""bench.py on the GPU box (shrunk grids: the contract of the JSON line, not a reported number) and the library's own
peak probe behind the roofline denominators."""
import json
import os
import subprocess
import sys

import pytest

pytestmark = pytest.mark.gpu
ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _bench(*args):
    out = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--quick", "--steps", "2", "--warmup", "3",
                          "--no-cpu-baseline", *args], capture_output=True, text=True, timeout=900, cwd=ROOT)
    assert out.returncode == 0, out.stderr[-3000:]
    lines = [l for l in out.stdout.splitlines() if l.strip()]
    assert len(lines) == 1
    return json.loads(lines[0])


def test_default_line_carries_both_p_pdot_grids():
    d = _bench()
    assert d["config"]["workload"].startswith("C5") and d["secondary"]["config"]["workload"].startswith("C3")
    for rec in (d, d["secondary"]):
        r = rec["roofline"]
        assert r["bound"] == "alu" and r["pipe"] in ("fp64", "shared-memory wavefronts")
        assert 0.0 < r["frac"] < 1.0 and 0.0 < r["other_bound"]["frac"] < 1.0
        assert r["frac"] >= r["other_bound"]["frac"]            # "bound" names the ceiling the kernel is closer to
        assert abs(r["frac"] - r["achieved"] / r["peak"]) < 1e-12
        assert r["traffic"] is None                              # shrunk grid: no ncu capture applies
        assert rec["e2e"]["value"] > 0 and rec["e2e"]["h2d_bytes_per_step"] > 0 and rec["e2e"]["d2h_bytes_per_step"] > 0
        assert rec["gpu_launches"] > 0 and set(rec["config"]["sha256_16"]) == {"times", "mags", "lc_offsets", "periods", "pdots"}
        assert rec["clocks"]["sm_mhz"] is None or rec["clocks"]["sm_mhz"] > 0
    assert d["metric"] == "CE point-folds/sec" and d["unit"] == "point-folds/s" and d["dtype"] == "f64" and d["n_gpus"] == 1
    assert 55.0 < d["roofline"]["probe_measured_per_sm_clk"] < 66.0      # FP64 lane-ops / SM / clk, nominal 64


def test_pdot_zero_grid_reports_both_ceilings():
    d = _bench("--config", "C4")
    r = d["roofline"]
    assert {r["pipe"], r["other_bound"]["pipe"]} == {"fp64", "shared-memory wavefronts"}
    assert r["algorithmic_per_point_fold"] > 0 and "secondary" not in d
    fp64 = r if r["pipe"] == "fp64" else r["other_bound"]
    assert fp64["algorithmic_per_point_fold"] == 3.0            # Pdot = {0}: a, y, floor


def test_probe_rates_are_near_the_nominal_figures():
    import paper_2006_06866_b200 as gce
    f = gce.gce_ce_probe_rate(gce.binding.PROBE_FP64)
    s = gce.gce_ce_probe_rate(gce.binding.PROBE_SHARED)
    assert 55.0 < f < 66.0 and 0.85 < s < 1.05
    with pytest.raises(gce.GceError):
        gce.gce_ce_probe_rate(7)


def test_design_ablation_kernel_matches_the_oracle(oracle):
    """csrc/gce_ablation.cu (the north_star's warp-per-trial + match_any sketch, its own shared object, timed by
    bench.py --ablation) computes the same CE as the oracle on a small C3-shaped case with a ragged last warp of points."""
    import ctypes as C

    import numpy as np
    import torch

    import bench
    import gce_workloads as W
    lib = bench.load_ablation()
    w = W.make("C3", n_lc=3, n_p=257, n_pdot=8)
    d = lambda a: torch.from_numpy(np.ascontiguousarray(a)).cuda()
    t, m, offs, per, pd = d(w.times), d(w.mags), d(w.lc_offsets), d(w.periods), d(w.pdots)
    out = torch.full((3, 257, 8), -1.0, dtype=torch.float32, device="cuda")
    err = C.c_int32(0)
    rc = lib.gce_ablation_warp_per_trial(t.data_ptr(), m.data_ptr(), offs.data_ptr(), 3, int(np.max(np.diff(w.lc_offsets))),
                                         per.data_ptr(), 257, pd.data_ptr(), 8, 20, 10, out.data_ptr(), C.byref(err), None)
    torch.cuda.synchronize()
    assert rc == 0, err.value
    ref = oracle.ce_search(w.times, w.mags, w.lc_offsets, w.periods, w.pdots, 20, 10)
    np.testing.assert_allclose(out.cpu().numpy().astype(np.float64), ref, rtol=1e-5, atol=1e-7)
