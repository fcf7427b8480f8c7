"""bench.py contract on CPU: the reference arm (the oracle on the host cores) prints ONE JSON line with the keys the
driver reads; the product arm refuses to run without a CUDA device instead of falling back."""
import json
import os
import subprocess
import sys

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def test_reference_arm_prints_one_json_line():
    out = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--quick", "--steps", "1",
                          "--warmup", "0", "--config", "C2"], capture_output=True, text=True, timeout=600, cwd=ROOT)
    assert out.returncode == 0, out.stderr[-2000:]
    lines = [l for l in out.stdout.splitlines() if l.strip()]
    assert len(lines) == 1
    d = json.loads(lines[0])
    assert d["impl"] == "reference" and d["metric"] == "CE point-folds/sec" and d["unit"] == "point-folds/s"
    assert d["higher_is_better"] is True and d["value"] > 0 and d["n_gpus"] == 1 and d["steps"] == 1
    assert d["cpu_baseline"]["kind"] == "oracle" and d["cpu_baseline"]["cores"] >= 1 and d["cpu_baseline"]["sample"]
    assert d["e2e"] == {"value": d["value"], "unit": d["unit"], "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}
    assert d["config"]["workload"].startswith("C2") and "model" not in d["config"]


def test_reference_arm_other_ranks_exit_silently():
    env = dict(os.environ, RANK="1", WORLD_SIZE="2")
    out = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--quick", "--gpus", "2"],
                         capture_output=True, text=True, timeout=120, cwd=ROOT, env=env)
    assert out.returncode == 0 and out.stdout.strip() == ""


def test_product_arm_has_no_cpu_fallback():
    import torch
    if torch.cuda.is_available():
        return
    out = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--quick", "--steps", "1", "--warmup", "0"],
                         capture_output=True, text=True, timeout=300, cwd=ROOT)
    assert out.returncode != 0 and "no CPU fallback" in (out.stderr + out.stdout)


def _bench(*argv, env=None, timeout=600):
    return subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), *argv], capture_output=True, text=True,
                          timeout=timeout, cwd=ROOT, env=env)


def _clean_env():
    return {k: v for k, v in os.environ.items() if k not in ("RANK", "LOCAL_RANK", "WORLD_SIZE", "MASTER_ADDR", "MASTER_PORT")}


def test_gpus_n_launches_n_ranks_itself_strong_scaling_by_light_curve():
    """`python bench.py --gpus 2` with no RANK in the environment -- the form of the driver's N = 1 command -- starts two
    ranks itself (world_size 2, gloo in --dry-run) instead of silently running one; --scaling strong partitions the GIVEN
    config by light curve: C5's 16 light curves -> 8 + 8, the same grid on both ranks, all point-folds accounted for."""
    out = _bench("--gpus", "2", "--dry-run", "--config", "C5", "--scaling", "strong", env=_clean_env())
    assert out.returncode == 0, out.stderr[-2000:]
    lines = [l for l in out.stdout.splitlines() if l.startswith("{")]
    assert len(lines) == 1
    d = json.loads(lines[0])
    assert d["dry_run"] is True and d["n_gpus"] == 2 and d["scaling"] == "strong"
    assert [r["rank"] for r in d["ranks"]] == [0, 1]
    assert [r["lc_range"] for r in d["ranks"]] == [[0, 8], [8, 16]]
    assert all(r["period_range"] == [0, 1 << 17] for r in d["ranks"])
    assert d["point_folds_total"] == 16 * 5000 * (1 << 17) * 256 == d["config"]["point_folds_per_step_per_gpu"]
    assert d["ranks"][0]["sha256_16"]["periods"] == d["ranks"][1]["sha256_16"]["periods"]
    assert d["ranks"][0]["sha256_16"]["times"] != d["ranks"][1]["sha256_16"]["times"]


def test_strong_scaling_with_fewer_light_curves_than_gpus_splits_the_period_axis():
    out = _bench("--gpus", "2", "--dry-run", "--config", "C1", "--scaling", "strong", env=_clean_env())
    assert out.returncode == 0, out.stderr[-2000:]
    d = json.loads([l for l in out.stdout.splitlines() if l.startswith("{")][0])
    assert [r["period_range"] for r in d["ranks"]] == [[0, 500], [500, 1000]]
    assert all(r["lc_range"] == [0, 1] for r in d["ranks"]) and d["point_folds_total"] == 200 * 1000


def test_weak_scaling_dry_run_re_seeds_the_batch_per_rank():
    out = _bench("--gpus", "2", "--dry-run", "--config", "C3", "--quick", env=_clean_env())
    assert out.returncode == 0, out.stderr[-2000:]
    d = json.loads([l for l in out.stdout.splitlines() if l.startswith("{")][0])
    assert d["scaling"] == "weak" and d["n_gpus"] == 2
    assert d["ranks"][0]["point_folds"] == d["ranks"][1]["point_folds"] and d["point_folds_total"] == 2 * d["ranks"][0]["point_folds"]
    assert d["ranks"][0]["sha256_16"]["mags"] != d["ranks"][1]["sha256_16"]["mags"]


def test_gpus_n_without_n_devices_exits_non_zero():
    import torch
    have = torch.cuda.device_count() if torch.cuda.is_available() else 0
    out = _bench("--gpus", str(have + 2), "--quick", "--steps", "1", "--warmup", "0", env=_clean_env(), timeout=300)
    assert out.returncode != 0 and "not starting" in out.stderr and out.stdout.strip() == ""


def test_world_size_that_contradicts_gpus_is_refused():
    env = dict(_clean_env(), RANK="0", WORLD_SIZE="2", LOCAL_RANK="0")
    out = _bench("--gpus", "4", "--dry-run", env=env, timeout=120)
    assert out.returncode != 0 and "WORLD_SIZE=2" in out.stderr
