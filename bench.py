#!/usr/bin/env python
"""bench.py -- CE (P, Pdot) search throughput on B200, one JSON line on stdout.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config C5] [--impl ours|reference]

A "step" is one pass of the whole hot path (S1..S5 of SURVEY.md section 8a: preprocess, fold + bin + entropy,
cube store and/or fused top-k) over one batch of seeded synthetic light curves (gce_workloads, DESIGN.md
section 5).  Default workload: C5 = BASELINE.json:configs[4], the largest single-GPU configuration (16 light
curves x 5000 points x 2^17 periods x 256 Pdots, 30 x 10 bins, fused top-16: 2.68e12 point-folds per step).
The north_star's roofline target is stated on the two P-Pdot grids, so the default run ALSO times C3 =
configs[2] (64 x 1000 points x 50 000 periods x 64 Pdots, full fp32 CE cube + per-LC best) with the same K / W and
carries it in the same JSON line under "secondary", with its own roofline, clocks, kernel_ms and e2e.
--config X times X alone.

metric  : CE point-folds per second = n_lc * n_p * n_pdot * N_obs / t   (BASELINE.json:metric)
value   : inputs already resident in HBM, CUDA-event time of the gce_ce_search enqueue, L2 flushed between steps
e2e     : the same through gce_ce_search_host with pinned HOST buffers (H2D of the inputs, D2H of the outputs
          and device allocation inside the timed region)
roofline: the fold+bin+entropy kernel (k_search), timed live with CUDA events recorded by the library around that
          kernel, against the two on-SM ceilings of SURVEY 8(d) -- FP64-pipe issue rate and shared-memory
          wavefronts -- "bound" names the one that binds (the larger fraction), the other is kept in "other_bound"
cpu_baseline: the oracle (oracle/, as it stands) on this box's host cores over a bounded sample of the workload

N > 1 (one process per GPU): started under torchrun the ranks come from the environment; started plainly as
`python bench.py --gpus N` (no RANK in the environment) bench.py launches the N ranks itself (torch.distributed.run on
127.0.0.1) and passes their one JSON line through.  Light curves are independent, so there is no data-path collective.
  --scaling weak   (default) each rank searches its own batch of the config's shape (seed offset by rank);
                   value = all ranks' point-folds / max-over-ranks time
  --scaling strong the GIVEN config is partitioned by light curve (sharding.partition_light_curves, balanced by points;
                   C5: 16 light curves -> 2 per GPU at N = 8), every rank searches its slice, the per-light-curve
                   selections are gathered and rank 0 checks them against its own search of the whole config; value =
                   the config's point-folds / max-over-ranks time.  Fewer light curves than GPUs (one deep target): the
                   period axis is split instead and the per-rank partial blobs are all-gathered and merged exactly
                   (search_period_chunks; the path's one real exchange step).
--dry-run stops before CUDA: the ranks rendezvous over gloo, build the workload and the partition, and rank 0 prints the
plan as one JSON line (tests/test_bench_contract.py runs it with 2 ranks on CPU).
--impl reference times the oracle instead (rank 0 only).
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import gce_workloads as W  # noqa: E402

METRIC = "CE point-folds/sec"
UNIT = "point-folds/s"
FP64_LANES_PER_SM_CLK = 64       # B200 FP64 pipe: 64 lane-ops / SM / clk (probe-measured)
N_SM = 148
OVERLAP = [False]   # set from --overlap; the oracle legs time the same binning
PROBED = {}         # gce_ce_probe_rate results of this run (rank 0)
SHARED_WAVEFRONTS_PER_SM_CLK = 1   # shared-memory data pipe: 1 wavefront / SM / clk (ncu's own denominator)
DEFAULT_CONFIG = "C5"              # BASELINE.json:configs[4]: the largest single-GPU configuration
SECONDARY_CONFIG = "C3"            # configs[2]: the other P-Pdot grid of the north_star's roofline target
# DRAM traffic of one k_search launch from the committed ncu --set full captures, keyed to the library sources
# (paper_2006_06866_b200.build.source_hash) they were captured from.  C3 writes the 819.2 MB fp32 cube (part of it is
# still in L2 at kernel end); C5 writes no cube.  Only workloads that were captured have an entry.
NCU_TRAFFIC = {
    "C3": {"bytes": 15.283456e6 + 769.811456e6, "source_hash": "25ab21d75632df2d", "profile": "profiles/r3_k_search_C3_full.md"},
    "C5": {"bytes": 2.521600e6, "source_hash": "25ab21d75632df2d", "profile": "profiles/r3_k_search_C5_full.md"},
    "C4": {"bytes": 4.464640e6, "source_hash": "25ab21d75632df2d", "profile": "profiles/r3_k_search_C4_full.md"},
}


def load_peaks():
    try:
        with open(os.path.join(ROOT, "MEASURED_PEAKS.json")) as f:
            return json.load(f), "measured"
    except Exception:
        return {"hbm_gbs": 6650.0, "sm_max_mhz": 1965.0}, "fallback"


class ClockSampler:
    """nvidia-smi clocks + throttle reasons during the timed region (B200_PROFILING.md recipe)."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        self.rows, self.proc, self.thr, self.index = [], None, None, index

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(self.index), f"--query-gpu={self.Q}",
                                          "--format=csv,noheader,nounits", "-lms", "100"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
        except Exception:
            self.proc = None
            return
        def pump():
            for line in self.proc.stdout:
                self.rows.append((time.time(), line.strip()))
        self.thr = threading.Thread(target=pump, daemon=True)
        self.thr.start()

    def stop(self, t0=None, t1=None):
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.15)
        self.proc.terminate()
        try:
            self.proc.wait(timeout=5)
        except Exception:
            self.proc.kill()
        sm, mx, pw, reasons = [], [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        rows = [r for (t, r) in self.rows if (t0 is None or t >= t0) and (t1 is None or t <= t1 + 0.1)] or \
               [r for (_, r) in self.rows]
        for r in rows:
            f = [x.strip() for x in r.split(",")]
            if len(f) < 7:
                continue
            try:
                sm.append(float(f[0])); mx.append(float(f[1])); pw.append(float(f[2]))
            except ValueError:
                continue
            for nm, v in zip(names, f[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(nm)
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "power_w_max": max(pw) if pw else None, "samples": len(sm), "reasons": sorted(reasons)}


def make_workload(name, rank, shrink, n_pdot=0):
    kw = {}
    if shrink:  # --quick: same ranges, smaller grid (for smoke-testing the bench itself; never a reported number)
        kw = {"C1": {}, "C2": dict(n_lc=8, n_p=2000), "C3": dict(n_lc=4, n_p=2000, n_pdot=64),
              "C4": dict(n_lc=16, n_p=4000), "C5": dict(n_lc=2, n_p=512, n_pdot=32),
              "P1": dict(n_lc=4, n_p=20000, n_pdot=32)}[name]
    if name == "P1" and n_pdot:
        kw = dict(kw, n_pdot=n_pdot)
    if rank > 0:
        # weak scaling: every rank owns a batch of the same shape; rank r re-draws it from seed + 1000 r
        kw = dict(kw, seed={"C1": 0, "C2": 1, "C3": 2, "C4": 3, "C5": 4, "P1": 9}[name] + 1000 * rank)
    return W.make(name, **kw)


def rank_workload(name, rank, world, args, n_pdot=0):
    """(this rank's workload, the whole config or None, the light-curve ranges or None).  weak: a batch of the config's
    shape per rank.  strong: the given config partitioned by light curve."""
    if args.scaling != "strong" or world == 1:
        return apply_binning(make_workload(name, rank, args.quick, n_pdot), args), None, None
    from paper_2006_06866_b200 import sharding
    full = apply_binning(make_workload(name, 0, args.quick, n_pdot), args)
    if full.n_lc < world:
        return full, full, None   # fewer light curves than ranks: the period axis is split instead (measure_period_split)
    ranges = sharding.partition_light_curves(full.lc_offsets, world)
    lo, hi = ranges[rank]
    t, m, offs = sharding.shard_arrays(full.times, full.mags, full.lc_offsets, lo, hi)
    mine = W.Workload(f"{full.name}[{lo}:{hi}]", t, m, np.ascontiguousarray(offs), full.periods, full.pdots,
                      full.n_phase_bins, full.n_mag_bins, full.top_k, full.want_cube)
    return mine, full, ranges


def apply_binning(w, args):
    """--n-phase-bins / --n-mag-bins / --overlap: the same light curves and grid with another binning, e.g. the paper's
    production setting 50 overlapping phase bins x 10.  Named in config; never the default."""
    if args.n_phase_bins:
        w.n_phase_bins = args.n_phase_bins
    if args.n_mag_bins:
        w.n_mag_bins = args.n_mag_bins
    return w


def algorithmic_fp64_ops_per_pointfold(w):
    """DMUL a=dt*invP (shared by the Pdot values of one period), DMUL b=dt2*c, DADD x=a+b,
    DMUL y=x*n_phi, DADD.RD floor  ->  4 + 1/n_pdot per point-fold; 3 when the grid is Pdot = {0} only."""
    if w.n_pdot == 1 and float(w.pdots[0]) == 0.0:
        return 3.0
    return 4.0 + 1.0 / w.n_pdot


# ----------------------------------------------------------------------------------------- reference arm
def oracle_sample(w, seconds_target):
    """Bounded sample of the workload for the oracle: all light curves, all Pdots, a strided subset of the
    periods sized from a short calibration run so one pass takes about `seconds_target` seconds."""
    import oracle
    oracle.build()
    n_cal = max(1, min(w.n_p, int(2e8 // max(1, w.total_points * w.n_pdot))))
    cal = w.subset(p_idx=np.linspace(0, w.n_p - 1, n_cal).astype(np.int64))
    t = time.perf_counter()
    oracle.ce_search(cal.times, cal.mags, cal.lc_offsets, cal.periods, cal.pdots, w.n_phase_bins, w.n_mag_bins,
                     overlap=OVERLAP[0])
    dt = max(time.perf_counter() - t, 1e-4)
    rate = cal.point_folds / dt
    n_s = int(min(w.n_p, max(n_cal, rate * seconds_target // max(1, w.total_points * w.n_pdot))))
    idx = np.unique(np.linspace(0, w.n_p - 1, n_s).astype(np.int64))
    return w.subset(p_idx=idx), f"all {w.n_lc} light curves x {idx.size} of {w.n_p} periods (uniform stride) x all {w.n_pdot} Pdots"


def time_oracle(sample, w):
    import oracle
    t = time.perf_counter()
    oracle.ce_search(sample.times, sample.mags, sample.lc_offsets, sample.periods, sample.pdots,
                     w.n_phase_bins, w.n_mag_bins, overlap=OVERLAP[0])
    return time.perf_counter() - t


def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return 0
    import oracle
    name = args.config or DEFAULT_CONFIG
    if name == "P1":
        args.overlap = True
        OVERLAP[0] = True
    w = apply_binning(make_workload(name, 0, args.quick, args.n_pdot), args)
    per_step = max(1.0, min(20.0, 150.0 / max(1, args.steps + args.warmup)))
    sample, desc = oracle_sample(w, per_step)
    for _ in range(args.warmup):
        time_oracle(sample, w)
    ts = [time_oracle(sample, w) for _ in range(args.steps)]
    tot = float(sum(ts))
    val = sample.point_folds * args.steps / tot
    line = {"impl": "reference", "metric": METRIC, "value": val, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": 1e3 * tot / args.steps, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": workload_config(w, args),
            "cpu_baseline": {"value": val, "unit": UNIT, "cores": oracle.num_threads(), "kind": "oracle", "sample": desc},
            "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line))
    return 0


def array_sha256(w):
    """SHA-256 of every generated input array (runs are comparable only on identical inputs)."""
    import hashlib
    h = lambda a: hashlib.sha256(np.ascontiguousarray(a).tobytes()).hexdigest()[:16]
    return {"times": h(w.times), "mags": h(w.mags), "lc_offsets": h(w.lc_offsets), "periods": h(w.periods), "pdots": h(w.pdots)}


def workload_config(w, args):
    src = (f"BASELINE.json:configs[{int(w.name[1]) - 1}]" if w.name[0] == "C" else
           "the paper's production grid, PAPER.md:166-170, 50 overlapping phase bins; not a BASELINE.json config")
    return {"workload": f"{w.name} ({src})" + (" QUICK-SHRUNK" if args.quick else ""),
            "n_lc": w.n_lc, "n_obs_total": w.total_points, "n_p": w.n_p, "n_pdot": w.n_pdot,
            "n_phase_bins": w.n_phase_bins, "n_mag_bins": w.n_mag_bins, "overlap": bool(args.overlap), "top_k": w.top_k, "ce_cube": bool(w.want_cube),
            "point_folds_per_step_per_gpu": w.point_folds, "parallelism": f"independent light-curve batches x{args.gpus}",
            "l2": "flushed between timed steps (256 MiB write), each step timed by its own CUDA-event pair",
            "sha256_16": array_sha256(w)}


def algorithmic_shared_wavefronts_per_pointfold(w):
    """SURVEY 8(d), shared-memory row: one conflict-free counter update per point-fold = 1 wavefront per 32 point-folds
    (an atomic RED is one wavefront: ncu counts 1.00 per ATOMS.ADD, profiles/r2_*), plus S4's visit of every cell of
    every trial: one counter read and one k ln k lookup = 2 wavefronts per 32 (trial, cell) pairs.  Per point-fold:
    (1 + 2 n_phi n_m / N) / 32 with N the mean light-curve length.  (Counting a counter update as a non-atomic
    read-modify-write, 2 per 32, is SURVEY's other figure; the kernel does not pay it.)"""
    n_avg = w.total_points / max(1, w.n_lc)
    return (1.0 + 2.0 * w.n_phase_bins * w.n_mag_bins / max(1.0, n_avg)) / 32.0


def traffic_record(w, args):
    """DRAM bytes of one k_search launch (dram__bytes_read.sum + dram__bytes_write.sum, ncu --set full), valid only for
    the library sources they were captured from: null when the kernel sources have changed since (never a stale number)."""
    from paper_2006_06866_b200.build import source_hash
    rec = NCU_TRAFFIC.get(w.name)
    if args.quick or rec is None or args.n_phase_bins or args.n_mag_bins or args.overlap:
        return None, "no ncu capture of this workload"
    if rec["source_hash"] != source_hash():
        return None, f"kernel sources changed since the capture {rec['profile']} (hash {rec['source_hash']})"
    return rec["bytes"], f"{rec['profile']}: dram__bytes_read.sum + dram__bytes_write.sum of one k_search launch, ncu --set full; bytes per launch"


# ----------------------------------------------------------------------------------------- our arm
def measure(gce, w, args, dev, dist, rank, world, local_rank, with_cpu_baseline, keep=None):
    """W warm-ups, K timed steps (device-resident), the end-to-end host-buffer leg, the roofline record; one dict."""
    import torch
    d = lambda a: torch.from_numpy(np.ascontiguousarray(a)).to(dev)
    times, mags, offs, periods, pdots = d(w.times), d(w.mags), d(w.lc_offsets), d(w.periods), d(w.pdots)
    k = w.top_k
    ev_a, ev_b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    ev_a.record(); ev_b.record()  # forces creation of the cudaEvent_t handles
    prm = gce.make_params(w.n_phase_bins, w.n_mag_bins, top_k=k, overlap=args.overlap, ev_search_begin=ev_a, ev_search_end=ev_b)
    ce = torch.empty((w.n_lc, w.n_p, w.n_pdot), dtype=torch.float32, device=dev) if w.want_cube else None
    bidx = torch.empty((w.n_lc, k), dtype=torch.int64, device=dev) if k else None
    bce = torch.empty((w.n_lc, k), dtype=torch.float32, device=dev) if k else None
    ws = torch.empty(gce.gce_ce_workspace_bytes(w.total_points, w.n_lc, w.n_p, w.n_pdot, prm), dtype=torch.uint8, device=dev)
    flush = torch.empty(256 << 20, dtype=torch.uint8, device=dev)
    launches_per_step = gce.gce_ce_launch_count(w.n_lc, w.n_p, prm)

    def step():
        gce.gce_ce_search(times, mags, offs, periods, pdots, prm, ce, bidx, bce, None, ws)

    def sync_all():
        torch.cuda.synchronize()
        if world > 1:
            dist.barrier()
            torch.cuda.synchronize()

    for _ in range(args.warmup):
        step()
    sync_all()

    sampler = ClockSampler(local_rank)
    if rank == 0:
        sampler.start()
        time.sleep(0.25)
    s_ev = [torch.cuda.Event(enable_timing=True) for _ in range(args.steps)]
    e_ev = [torch.cuda.Event(enable_timing=True) for _ in range(args.steps)]
    k_ms = []
    sync_all()
    t_wall0 = time.time()
    for i in range(args.steps):
        flush.zero_()                       # evict L2 (126 MB) between timed steps; not inside the event pair
        s_ev[i].record()
        step()
        e_ev[i].record()
        e_ev[i].synchronize()               # the library's kernel-only events are reused every step
        k_ms.append(ev_a.elapsed_time(ev_b))
    sync_all()
    t_wall1 = time.time()
    clocks = sampler.stop(t_wall0, t_wall1) if rank == 0 else None
    step_ms = [s.elapsed_time(e) for s, e in zip(s_ev, e_ev)]
    tot_ms = float(sum(step_ms))
    from paper_2006_06866_b200 import sharding
    tot_ms_max, pf_all = sharding.reduce_timing(tot_ms, float(w.point_folds), dist if world > 1 else None, dev)
    value = pf_all * args.steps / (tot_ms_max * 1e-3)

    # ---- end to end through the host entry point: pinned host buffers, H2D + D2H + allocation inside the timing
    pin = lambda a: torch.from_numpy(np.ascontiguousarray(a)).pin_memory()
    h_in = [pin(w.times), pin(w.mags), pin(w.lc_offsets), pin(w.periods), pin(w.pdots)]
    h_ce = torch.empty((w.n_lc, w.n_p, w.n_pdot), dtype=torch.float32).pin_memory() if w.want_cube else None
    h_idx = torch.empty((w.n_lc, k), dtype=torch.int64).pin_memory() if k else None
    h_bce = torch.empty((w.n_lc, k), dtype=torch.float32).pin_memory() if k else None
    prm_h = gce.make_params(w.n_phase_bins, w.n_mag_bins, top_k=k, overlap=args.overlap)
    h2d = sum(x.numel() * x.element_size() for x in h_in)
    d2h = sum(x.numel() * x.element_size() for x in (h_ce, h_idx, h_bce) if x is not None)
    n_e2e = max(1, min(args.steps, 5))
    gce.gce_ce_search_host(*h_in, prm_h, h_ce, h_idx, h_bce)   # warm-up (allocator pools)
    sync_all()
    t0 = time.perf_counter()
    for _ in range(n_e2e):
        gce.gce_ce_search_host(*h_in, prm_h, h_ce, h_idx, h_bce)  # synchronises before returning
    e2e_s = time.perf_counter() - t0
    te = torch.tensor([e2e_s], dtype=torch.float64, device=dev)
    if world > 1:
        dist.all_reduce(te, op=dist.ReduceOp.MAX)
    e2e_val = pf_all * n_e2e / float(te.item())
    if k and rank == 0:
        assert torch.equal(h_idx.to(dev), bidx), "host and device entry points disagree"
    if keep is not None and k:
        keep["best_idx"], keep["best_ce"] = bidx.cpu().numpy(), bce.cpu().numpy()
    del ce, ws, flush, h_ce
    gce.gce_ce_host_release()
    torch.cuda.empty_cache()
    if rank != 0:
        return None

    # ---- roofline of the dominant kernel (k_search): the two on-SM ceilings of SURVEY 8(d); the binding one is the
    # ceiling the kernel is closer to (the larger fraction = the smaller point-folds/s ceiling)
    peaks, peaks_src = load_peaks()
    k_ms_avg = float(np.mean(k_ms))
    sm_max = float(peaks.get("sm_max_mhz", 1965.0))
    pf_s = w.point_folds / (k_ms_avg * 1e-3)
    fp64_ops = algorithmic_fp64_ops_per_pointfold(w)
    fp64 = {"bound": "alu", "pipe": "fp64", "achieved": fp64_ops * pf_s / 1e9,
            "peak": FP64_LANES_PER_SM_CLK * N_SM * sm_max * 1e6 / 1e9, "unit": "G FP64 lane-ops/s",
            "algorithmic_per_point_fold": fp64_ops,
            "peak_source": f"nominal 64 FP64 lanes/SM/clk x 148 SMs x {sm_max:.0f} MHz (max SM clock, {peaks_src} MEASURED_PEAKS.json, "
                           "which has no FP64 entry); the library's probe of independent DMUL/DADD chains (gce_ce_probe_rate, "
                           "probe_measured_per_sm_clk) stays just below it, so the nominal figure is the stricter denominator"}
    wf = algorithmic_shared_wavefronts_per_pointfold(w)
    shm = {"bound": "alu", "pipe": "shared-memory wavefronts", "achieved": wf * pf_s / 1e9,
           "peak": SHARED_WAVEFRONTS_PER_SM_CLK * N_SM * sm_max * 1e6 / 1e9, "unit": "G wavefronts/s",
           "algorithmic_per_point_fold": wf,
           "peak_source": f"1 shared-memory wavefront/SM/clk x 148 SMs x {sm_max:.0f} MHz (the denominator of ncu's "
                          "l1tex__data_pipe_lsu_wavefronts_mem_shared pct_of_peak; DESIGN.md section 7); probe_measured_per_sm_clk is "
                          "the library's conflict-free RED.shared probe"}
    if not PROBED:   # once per run: the per-SM rates behind the two denominators, measured on this GPU by the library's probe
        PROBED["fp64"] = gce.gce_ce_probe_rate(gce.binding.PROBE_FP64)
        PROBED["shared"] = gce.gce_ce_probe_rate(gce.binding.PROBE_SHARED)
    fp64["probe_measured_per_sm_clk"], fp64["nominal_per_sm_clk"] = PROBED["fp64"], FP64_LANES_PER_SM_CLK
    shm["probe_measured_per_sm_clk"], shm["nominal_per_sm_clk"] = PROBED["shared"], SHARED_WAVEFRONTS_PER_SM_CLK
    for r in (fp64, shm):
        r["frac"] = r["achieved"] / r["peak"]
        r["ceiling_point_folds_per_s"] = r["peak"] * 1e9 / r["algorithmic_per_point_fold"]
    main, other = (fp64, shm) if fp64["frac"] >= shm["frac"] else (shm, fp64)
    traffic, traffic_src = traffic_record(w, args)
    roof = dict(main, kernel="k_search", traffic=traffic, traffic_source=traffic_src,
                kernel_ms=k_ms_avg, kernel_share_of_step=k_ms_avg * args.steps / tot_ms,
                frac_at_observed_clock=(main["frac"] * sm_max / clocks["sm_mhz"]) if clocks and clocks.get("sm_mhz") else None,
                ce_output_gbs=(w.n_lc * w.n_p * w.n_pdot * 4 / (k_ms_avg * 1e-3) / 1e9) if w.want_cube else 0.0,
                hbm_peak_gbs=peaks.get("hbm_gbs"), other_bound=other)

    # ---- the oracle on this box's host cores, bounded sample
    cpu = None
    if with_cpu_baseline:
        import oracle
        sample, desc = oracle_sample(w, 15.0)
        t_cpu = time_oracle(sample, w)
        cpu = {"value": sample.point_folds / t_cpu, "unit": UNIT, "cores": oracle.num_threads(), "kind": "oracle",
               "sample": desc, "seconds": t_cpu}

    return {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
            "ms_per_step": tot_ms_max / args.steps, "higher_is_better": True, "scaling": args.scaling, "vs_baseline": None,
            "dtype": "f64", "data": "synthetic", "config": workload_config(w, args),
            "e2e": {"value": e2e_val, "unit": UNIT, "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": d2h, "steps": n_e2e,
                    "api": "gce_ce_search_host (pinned host buffers; allocation + H2D + search + D2H + sync; with a cube the period "
                           "axis is searched in 8 chunks and each slice's D2H overlaps the next chunk on a second stream)"},
            "gpu_launches": launches_per_step * args.steps, "clocks": clocks, "roofline": roof, "cpu_baseline": cpu}


def period_ranges(n_p, world):
    """Contiguous period ranges [a, b) per rank (the work of a period does not depend on its value for the plain fold)."""
    return [(n_p * r // world, n_p * (r + 1) // world) for r in range(world)]


def measure_period_split(gce, w, args, dev, dist, rank, world, local_rank):
    """Strong scaling of a config with fewer light curves than GPUs (one deep target): every rank
    searches all light curves over its slice of the period axis (gce_ce_search_partial), the per-rank partial blobs --
    n_lc x (2 top_k + 10) int64, the path's one exchange -- are all-gathered (NCCL, in stream order) and merged exactly
    by every rank (gce_ce_merge_partials).  A step is that whole sequence; the cube, when the config asks for one, is
    left sharded by period on the ranks.  No roofline record: k_search is the same kernel the N = 1 line describes."""
    import torch
    from paper_2006_06866_b200 import sharding
    d = lambda a: torch.from_numpy(np.ascontiguousarray(a)).to(dev)
    args_dev = (d(w.times), d(w.mags), d(w.lc_offsets), d(w.periods), d(w.pdots), w.n_phase_bins, w.n_mag_bins)
    k = max(1, w.top_k)
    a, b = period_ranges(w.n_p, world)[rank]
    sink = (lambda lo, hi, sl: None) if w.want_cube else None
    flush = torch.empty(256 << 20, dtype=torch.uint8, device=dev)

    def step():
        return gce.search_period_chunks(*args_dev, [(a, b)] if b > a else [], top_k=k, want_stats=False, overlap=args.overlap,
                                        cube_sink=sink, dist=dist)

    def sync_all():
        torch.cuda.synchronize()
        dist.barrier()
        torch.cuda.synchronize()

    for _ in range(args.warmup):
        step()
    sync_all()
    sampler = ClockSampler(local_rank)
    if rank == 0:
        sampler.start()
        time.sleep(0.25)
    s_ev = [torch.cuda.Event(enable_timing=True) for _ in range(args.steps)]
    e_ev = [torch.cuda.Event(enable_timing=True) for _ in range(args.steps)]
    sync_all()
    t0 = time.time()
    for i in range(args.steps):
        flush.zero_()
        s_ev[i].record()
        res = step()
        e_ev[i].record()
    sync_all()
    t1 = time.time()
    clocks = sampler.stop(t0, t1) if rank == 0 else None
    tot_ms = float(sum(s.elapsed_time(e) for s, e in zip(s_ev, e_ev)))
    my_pf = float(w.total_points) * (b - a) * w.n_pdot
    tot_ms_max, pf_all = sharding.reduce_timing(tot_ms, my_pf, dist, dev)
    if rank != 0:
        return None
    whole = gce.search(*args_dev, top_k=k, want_cube=False, overlap=args.overlap)   # the N = 1 selection, outside the timing
    torch.cuda.synchronize()
    equal = bool(torch.equal(whole.best_idx, res.best_idx) and torch.equal(whole.best_ce, res.best_ce))
    assert equal, "period-split selection differs from the single-GPU search"
    prm = gce.make_params(w.n_phase_bins, w.n_mag_bins, top_k=k, overlap=args.overlap)
    cfg = workload_config(w, args)
    cfg["parallelism"] = f"period axis split x{world}, partial blobs all-gathered ({dist.get_backend()}) and merged exactly"
    return {"metric": METRIC, "value": pf_all * args.steps / (tot_ms_max * 1e-3), "unit": UNIT, "n_gpus": world, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": tot_ms_max / args.steps, "higher_is_better": True, "scaling": "strong",
            "vs_baseline": None, "dtype": "f64", "data": "synthetic", "config": cfg, "e2e": None,
            "gpu_launches": (gce.gce_ce_launch_count(w.n_lc, b - a, prm, partial=True) + 2) * args.steps, "clocks": clocks,
            "roofline": None, "cpu_baseline": None,
            "strong_check": {"mode": "period split", "period_ranges": period_ranges(w.n_p, world), "equal_to_single_gpu": equal}}


def measure_any(gce, name, args, dev, dist, rank, world, local_rank, with_cpu_baseline, n_pdot=0):
    """One config in the requested scaling mode; rank 0 gets the record."""
    import torch
    from paper_2006_06866_b200 import sharding
    w, full, ranges = rank_workload(name, rank, world, args, n_pdot)
    if full is not None and ranges is None:
        return measure_period_split(gce, full, args, dev, dist, rank, world, local_rank)
    keep = {} if full is not None else None
    line = measure(gce, w, args, dev, dist, rank, world, local_rank, with_cpu_baseline, keep=keep)
    if full is None:
        return line
    # strong scaling by light curve: gather the selections in light-curve order; rank 0 compares with the whole config
    k = full.top_k
    if k:
        gathered = sharding.gather_per_light_curve(keep.get("best_idx", np.zeros((0, k), dtype=np.int64)), full.n_lc, ranges, rank, dist)
        gathered_ce = sharding.gather_per_light_curve(keep.get("best_ce", np.zeros((0, k), dtype=np.float32)), full.n_lc, ranges, rank, dist)
    if rank != 0:
        return None
    equal = None
    if k:
        d = lambda a: torch.from_numpy(np.ascontiguousarray(a)).to(dev)
        whole = gce.search(d(full.times), d(full.mags), d(full.lc_offsets), d(full.periods), d(full.pdots), full.n_phase_bins,
                           full.n_mag_bins, top_k=k, want_cube=False, overlap=args.overlap)
        torch.cuda.synchronize()
        # A rank's call has fewer points than the whole config's, so its k ln k table may take a finer fixed-point shift
        # (gce_ce.cu table_shift): the selections agree except, possibly, inside a near tie (north_star's own exception),
        # where the two CE values are equal to fp32 precision.
        w_idx, w_ce = whole.best_idx.cpu().numpy(), whole.best_ce.cpu().numpy()
        differ = w_idx != gathered
        equal = bool(not differ.any())
        assert np.allclose(w_ce[differ], gathered_ce[differ], rtol=1e-6, atol=0.0), \
            "gathered per-light-curve selections differ from the single-GPU search of the whole config"
    line["config"] = dict(workload_config(full, args), point_folds_per_step_per_gpu=None, point_folds_per_step=full.point_folds,
                          parallelism=f"the config's light curves partitioned over {world} GPUs, balanced by points; no data-path collective")
    line["strong_check"] = {"mode": "light-curve partition", "lc_ranges": ranges, "equal_to_single_gpu": equal,
                            "near_tie_differences": int(differ.sum()) if k else 0}
    return line


def run_dry(args):
    """--dry-run: everything up to CUDA.  The ranks rendezvous over gloo, build the workload and the partition of the
    requested scaling mode, and rank 0 prints the plan."""
    import torch.distributed as dist
    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    if world > 1:
        os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
        dist.init_process_group("gloo")
    name = args.config or DEFAULT_CONFIG
    if name == "P1":
        args.overlap = True
        OVERLAP[0] = True
    w, full, ranges = rank_workload(name, rank, world, args, args.n_pdot)
    if full is not None and ranges is None:
        a, b = period_ranges(full.n_p, world)[rank]
        mine = {"rank": rank, "lc_range": [0, full.n_lc], "period_range": [a, b], "point_folds": full.total_points * (b - a) * full.n_pdot}
    else:
        mine = {"rank": rank, "lc_range": list(ranges[rank]) if ranges else [0, w.n_lc], "period_range": [0, w.n_p],
                "point_folds": w.point_folds, "sha256_16": array_sha256(w)}
    plans = [mine]
    if world > 1:
        plans = [None] * world
        dist.all_gather_object(plans, mine)
    if rank == 0:
        print(json.dumps({"dry_run": True, "n_gpus": world, "scaling": args.scaling, "config": workload_config(full or w, args),
                          "point_folds_total": sum(p["point_folds"] for p in plans), "ranks": plans}))
    if world > 1:
        dist.destroy_process_group()
    return 0


def self_launch(args, argv):
    """`python bench.py --gpus N` outside torchrun: start the N ranks (one process per GPU) and pass their output through."""
    import socket
    if not args.dry_run:
        import torch
        have = torch.cuda.device_count() if torch.cuda.is_available() else 0
        if have < args.gpus:
            sys.stderr.write(f"bench.py: --gpus {args.gpus} asked for, {have} CUDA device(s) visible; not starting\n")
            return 2
    with socket.socket() as sk:
        sk.bind(("127.0.0.1", 0))
        port = sk.getsockname()[1]
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", f"--nproc-per-node={args.gpus}",
           "--master-addr", "127.0.0.1", "--master-port", str(port), os.path.abspath(__file__), *argv]
    return subprocess.call(cmd)


def run_ours(args):
    import torch
    import torch.distributed as dist

    rank = int(os.environ.get("RANK", "0"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: there is no CPU fallback for the product path")
    torch.cuda.set_device(local_rank)
    dev = torch.device("cuda", local_rank)
    if world > 1:
        os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
        dist.init_process_group("nccl", device_id=dev)

    from paper_2006_06866_b200.build import build
    if rank == 0:
        build()
    if world > 1:
        dist.barrier()
    import paper_2006_06866_b200 as gce

    name = args.config or DEFAULT_CONFIG
    if name == "P1":
        args.overlap = True   # the paper's production binning
        OVERLAP[0] = True
    line = measure_any(gce, name, args, dev, dist, rank, world, local_rank, not args.no_cpu_baseline, args.n_pdot)
    if args.config is None:
        # the other P-Pdot grid the north_star's roofline target is stated on, same K / W, its own record
        sec = measure_any(gce, SECONDARY_CONFIG, args, dev, dist, rank, world, local_rank, False)
        if rank == 0:
            line["secondary"] = {key: sec.get(key) for key in ("value", "unit", "ms_per_step", "steps", "warmup", "config", "e2e",
                                                               "gpu_launches", "clocks", "roofline", "strong_check")}
    if rank == 0:
        print(json.dumps(line))
    if world > 1:
        dist.destroy_process_group()
    return 0


# ----------------------------------------------------------------------------------------- design ablation
def load_ablation():
    import ctypes as C
    from paper_2006_06866_b200.build import build_ablation
    lib = C.CDLL(build_ablation())
    vp, i32, i64 = C.c_void_p, C.c_int32, C.c_int64
    lib.gce_ablation_warp_per_trial.argtypes = [vp, vp, vp, i32, i32, vp, i64, vp, i64, i32, i32, vp, C.POINTER(i32), vp]
    lib.gce_ablation_warp_per_trial.restype = C.c_int
    return lib


def run_ablation(args):
    """The north_star's histogram sketch (one warp per trial, private 2-D table, match_any-aggregated shared atomics;
    csrc/gce_ablation.cu, its own shared object) timed beside the product's k_search on the same config, cube output only,
    same inputs, CUDA events, L2 flushed between steps; the two cubes are compared.  One JSON line."""
    import ctypes as C
    import torch
    from paper_2006_06866_b200.build import build
    build()
    import paper_2006_06866_b200 as gce
    lib = load_ablation()
    dev = torch.device("cuda", 0)
    torch.cuda.set_device(dev)
    w = apply_binning(make_workload(args.config or SECONDARY_CONFIG, 0, args.quick), args)
    d = lambda a: torch.from_numpy(np.ascontiguousarray(a)).to(dev)
    t, m, offs, per, pd = d(w.times), d(w.mags), d(w.lc_offsets), d(w.periods), d(w.pdots)
    longest = int(np.max(np.diff(w.lc_offsets)))
    cube_a = torch.empty((w.n_lc, w.n_p, w.n_pdot), dtype=torch.float32, device=dev)
    cube_p = torch.empty_like(cube_a)
    prm = gce.make_params(w.n_phase_bins, w.n_mag_bins, top_k=0)
    ws = torch.empty(gce.gce_ce_workspace_bytes(w.total_points, w.n_lc, w.n_p, w.n_pdot, prm), dtype=torch.uint8, device=dev)
    flush = torch.empty(256 << 20, dtype=torch.uint8, device=dev)
    err = C.c_int32(0)
    st = C.c_void_p(torch.cuda.current_stream().cuda_stream)

    def ablation():
        rc = lib.gce_ablation_warp_per_trial(t.data_ptr(), m.data_ptr(), offs.data_ptr(), w.n_lc, longest, per.data_ptr(), w.n_p,
                                             pd.data_ptr(), w.n_pdot, w.n_phase_bins, w.n_mag_bins, cube_a.data_ptr(), C.byref(err), st)
        if rc:
            raise SystemExit(f"gce_ablation_warp_per_trial failed: {rc} (cudaError {err.value})")

    def product():
        gce.gce_ce_search(t, m, offs, per, pd, prm, cube_p, None, None, None, ws)

    def timed(fn):
        for _ in range(args.warmup):
            fn()
        torch.cuda.synchronize()
        ms = []
        for _ in range(args.steps):
            flush.zero_()
            a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            a.record(); fn(); b.record(); b.synchronize()
            ms.append(a.elapsed_time(b))
        return float(np.mean(ms))

    sampler = ClockSampler(0)
    sampler.start()
    t0 = time.time()
    ms_a, ms_p = timed(ablation), timed(product)
    clocks = sampler.stop(t0, time.time())
    rel = float(((cube_a - cube_p).abs() / cube_p.abs().clamp_min(1e-30)).max().item())
    assert rel < 1e-5, f"the ablation kernel and k_search disagree: max relative difference {rel:.3e}"
    print(json.dumps({"ablation": "warp per trial, private n_phi x n_m table, match_any-aggregated shared atomics (north_star sketch)",
                      "config": workload_config(w, args), "steps": args.steps, "warmup": args.warmup, "unit": UNIT,
                      "ablation_ms": ms_a, "ablation_value": w.point_folds / (ms_a * 1e-3),
                      "product_ms": ms_p, "product_value": w.point_folds / (ms_p * 1e-3), "product_over_ablation": ms_a / ms_p,
                      "max_rel_diff_of_the_cubes": rel, "clocks": clocks}))
    return 0


# ----------------------------------------------------------------------------------------- Fig. 3 sweep
def run_sweep(args):
    """The paper's only timing result (Fig. 3): time per light curve per search point against the
    number of search points, for light curves of 100 / 1000 points and 15 plain / 50 overlapping phase bins.  Prints
    one JSON line per grid size and a markdown table on stderr; fused argmin + Eq. 5 statistics, no cube."""
    import torch
    from paper_2006_06866_b200.build import build
    build()
    import paper_2006_06866_b200 as gce
    dev = torch.device("cuda", 0)
    rows = []
    for n_obs in (100, 1000):
        for n_phi, ovl in ((15, False), (50, True)):
            for sp in (10 ** 3, 10 ** 4, 10 ** 5, 10 ** 6, 10 ** 7, 10 ** 8):
                w = W.fig3_batch(n_obs, sp, n_phi)
                d = lambda a: torch.from_numpy(np.ascontiguousarray(a)).to(dev)
                t_, m_, o_, p_, pd_ = d(w.times), d(w.mags), d(w.lc_offsets), d(w.periods), d(w.pdots)
                prm = gce.make_params(n_phi, 10, top_k=1, want_stats=True, overlap=ovl)
                bidx = torch.empty((w.n_lc, 1), dtype=torch.int64, device=dev)
                bce = torch.empty((w.n_lc, 1), dtype=torch.float32, device=dev)
                st = torch.empty((w.n_lc, 4), dtype=torch.float64, device=dev)
                ws = torch.empty(gce.gce_ce_workspace_bytes(w.total_points, w.n_lc, w.n_p, w.n_pdot, prm),
                                 dtype=torch.uint8, device=dev)
                reps = 3 if sp >= 10 ** 7 else 10
                for _ in range(3):
                    gce.gce_ce_search(t_, m_, o_, p_, pd_, prm, None, bidx, bce, st, ws)
                torch.cuda.synchronize()
                a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                a.record()
                for _ in range(reps):
                    gce.gce_ce_search(t_, m_, o_, p_, pd_, prm, None, bidx, bce, st, ws)
                b.record()
                b.synchronize()
                ms = a.elapsed_time(b) / reps
                trials = w.n_p * w.n_pdot
                row = {"sweep": "fig3", "n_obs": n_obs, "n_phase_bins": n_phi, "overlap": ovl, "n_lc": w.n_lc,
                       "search_points": trials, "ms": ms, "ns_per_lc_per_search_point": ms * 1e6 / (w.n_lc * trials),
                       "point_folds_per_s": w.point_folds / (ms * 1e-3)}
                rows.append(row)
                print(json.dumps(row), flush=True)
    print("| N_obs | phase bins | search points / LC | ms (16 LCs) | ns per LC per search point | point-folds/s |", file=sys.stderr)
    print("|---|---|---|---|---|---|", file=sys.stderr)
    for r in rows:
        print(f"| {r['n_obs']} | {r['n_phase_bins']}{' overlapping' if r['overlap'] else ''} | {r['search_points']:.0e} | "
              f"{r['ms']:.3f} | {r['ns_per_lc_per_search_point']:.3f} | {r['point_folds_per_s']:.3e} |", file=sys.stderr)
    return 0


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--config", default=None, choices=["C1", "C2", "C3", "C4", "C5", "P1"],
                    help="time this workload alone (default: C5 as the headline plus C3 under 'secondary')")
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--quick", action="store_true", help="shrunk grid, to test the bench itself; not a reportable number")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--n-phase-bins", type=int, default=0, help="override the config's phase bin count (named in config)")
    ap.add_argument("--n-mag-bins", type=int, default=0, help="override the config's magnitude bin count")
    ap.add_argument("--overlap", action="store_true", help="50 %% overlapping phase bins (N2, PAPER.md:106)")
    ap.add_argument("--n-pdot", type=int, default=0, help="P1 only: 32 / 128 / 512 log-spaced Pdot values (PAPER.md:170)")
    ap.add_argument("--sweep", action="store_true", help="the paper's Fig. 3 sweep instead of the benchmark line")
    ap.add_argument("--scaling", default="weak", choices=["weak", "strong"],
                    help="N > 1: weak = a batch of the config's shape per GPU; strong = the given config partitioned over the GPUs")
    ap.add_argument("--ablation", action="store_true",
                    help="time the north_star's warp-per-trial / match_any histogram sketch beside k_search (default config C3)")
    ap.add_argument("--dry-run", action="store_true", help="stop before CUDA: rendezvous (gloo), workload and partition only")
    args = ap.parse_args()
    args.warmup = max(args.warmup, 0)
    OVERLAP[0] = bool(args.overlap)
    if args.gpus < 1:
        ap.error("--gpus must be >= 1")
    in_launcher = "RANK" in os.environ and "WORLD_SIZE" in os.environ
    if in_launcher and int(os.environ["WORLD_SIZE"]) != args.gpus and args.impl == "ours":
        sys.stderr.write(f"bench.py: --gpus {args.gpus} but WORLD_SIZE={os.environ['WORLD_SIZE']}; launch one rank per GPU\n")
        return 2
    if args.gpus > 1 and not in_launcher and args.impl == "ours" and not args.sweep:
        return self_launch(args, sys.argv[1:])   # one process per GPU; never a silent single-rank run
    if args.ablation:
        return run_ablation(args)
    if args.dry_run:
        return run_dry(args)
    if args.sweep:
        return run_sweep(args)
    if args.impl == "reference":
        return run_reference(args)
    return run_ours(args)


if __name__ == "__main__":
    sys.exit(main())
