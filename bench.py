#!/usr/bin/env python
"""bench.py -- throughput of the KF hot path on B200 (contract: see DESIGN.md sec. 7).

  python bench.py [--gpus N] [--steps K] [--warmup W] [--workload fit_c1|fit_c2|fit_c0|build_c3|build_c4]
                  [--impl ours|reference] [--scaling weak|strong]

A "step" is one pass of the hot path over one batch of synthetic input: for the fit workloads one kf_fit call over
all tracks (steps F1-F9), for the build workloads kf_bin_hits + kf_build over all events (steps B0-B6).  The default
line is fit_c1 = BASELINE.json configs[1] (the configuration the roofline target is quoted on) and carries, under
"fit_c2", "build" (= build_c3) and "build_c4", the other BASELINE.json configs measured the same way in the same run,
each with its own clock sample, roofline and cpu_baseline.  With --gpus N > 1 and no torchrun environment bench.py starts
the N ranks itself (torch.distributed.run on 127.0.0.1).  `value` is whole-job throughput with
inputs resident in HBM; `e2e` is the same through the C-ABI call with pinned HOST buffers, H2D and D2H copies inside
the timed region.  `--impl reference` times the fp64 CPU oracle (oracle/) on a bounded sample of the same workload
on the host cores.  Under torchrun every rank works on its own shard of the same size (weak scaling, no collective
on the data path).
"""
from __future__ import annotations

import argparse
import json
import os
import statistics
import subprocess
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

from paper_1711_06571_b200 import synth  # noqa: E402

# Algorithmic work per unit (frozen before tuning).
FIT_FLOP_PER_TRACK_LAYER = 700.0          # re-count from the sec. 3 formulas
FIT_FLOP_PER_TRACK_LAYER_SURVEY = 800.0   # SURVEY.md sec. 8d hand count (reported as frac_survey_count)
FIT_BYTES_SEED_IN = 6 * 4 + 21 * 4 + 1            # par + cov + q
FIT_BYTES_OUT = 6 * 4 + 21 * 4 + 4 + 4 + 4        # par + cov + chi2 + nhits + status
FIT_BYTES_PER_HIT = 12
FIT_BYTES_PER_IDX = 4
BUILD_FLOP = dict(n_prop=458.0, n_scan=15.0, n_window=40.0, n_upd=250.0)
BIN_BYTES_PER_HIT = 28.0   # algorithmic: read x, y, z (12), write the sorted 16-byte record (16); + 4 per bin for bin_off
SM_COUNT, FP32_LANES = 148, 128
FIT_CFG = {"fit_c0": 0, "fit_c1": 1, "fit_c2": 2}
BUILD_CFG = {"build_c3": 3, "build_c4": 4, "build_lids": "lids", "build_lids_two_step": "lids"}
# building on the "cylinder with lids" (R22, R23): hits on the nominal surfaces / sensors
# staggered by +-0.3 cm with the second propagation step to every candidate hit (kf_geom.hit_mode = 1); not in the default line
BUILD_KW = {"build_lids_two_step": dict(jitter=0.3)}
BUILD_HIT_MODE = {"build_lids_two_step": 1}


def peaks():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(path):
        d = json.load(open(path))
        return dict(hbm_gbs=float(d["hbm_gbs"]), sm_max_mhz=float(d.get("sm_max_mhz", 1965.0)), source="measured")
    return dict(hbm_gbs=6650.0, sm_max_mhz=1965.0, source="fallback")


def fp32_peak_tflops(pk) -> float:
    return SM_COUNT * FP32_LANES * 2 * pk["sm_max_mhz"] * 1e6 / 1e12


class ClockSampler:
    """nvidia-smi clocks / throttle reasons during the timed region (B200_PROFILING.md clocks line)."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.rows = []
        self.proc = None
        try:
            self.proc = subprocess.Popen(["nvidia-smi", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits", "-lms", "100", "-i", str(index)],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.th = threading.Thread(target=self._read, daemon=True)
            self.th.start()
        except Exception:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append((time.time(), line.strip()))

    def stop(self, t0: float, t1: float) -> dict:
        if self.proc is None:
            return dict(sm_mhz=None, sm_max_mhz=None, reasons=["nvidia-smi unavailable"])
        time.sleep(0.15)
        self.proc.terminate()
        sm, mx, reasons = [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for ts, line in self.rows:
            if ts < t0 - 0.05 or ts > t1 + 0.05:
                continue
            f = [x.strip() for x in line.split(",")]
            try:
                sm.append(float(f[0])); mx.append(float(f[1]))
            except Exception:
                continue
            for nm, v in zip(names, f[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(nm)
        if not sm:   # region shorter than the sampling period: take the nearest samples
            for ts, line in self.rows[-3:]:
                f = [x.strip() for x in line.split(",")]
                try:
                    sm.append(float(f[0])); mx.append(float(f[1]))
                except Exception:
                    pass
        return dict(sm_mhz=statistics.median(sm) if sm else None, sm_max_mhz=max(mx) if mx else None,
                    reasons=sorted(reasons), samples=len(sm))


# ----------------------------------------------------------------------------------------------------------------
# algorithmic work
# ----------------------------------------------------------------------------------------------------------------
def fit_units(fi) -> dict:
    """Algorithmic flops / bytes of one kf_fit call over `fi`."""
    n_upd = int(fi.valid.sum())
    by = fi.n * (FIT_BYTES_SEED_IN + FIT_BYTES_OUT) + n_upd * FIT_BYTES_PER_HIT
    if fi.hit_idx is not None:
        by += fi.n * fi.geom.n_layers * FIT_BYTES_PER_IDX
    return dict(track_layers=n_upd, flops=n_upd * FIT_FLOP_PER_TRACK_LAYER, flops_survey=n_upd * FIT_FLOP_PER_TRACK_LAYER_SURVEY, bytes=by)


def fit_config(workload: str, fi) -> dict:
    """`config` of a fit line: the same keys and values from the GPU arm and the reference arm (the driver compares them)."""
    u = fit_units(fi)
    return dict(workload=workload, tracks_per_gpu=fi.n, layers=fi.geom.n_layers, track_layers=u["track_layers"],
                l2="inputs+outputs per step (%.0f MB) exceed the 126 MB L2; no explicit flush" % (u["bytes"] / 1e6))


def build_needs_flush(n_hits: int) -> bool:
    return n_hits * 28 < (160 << 20)      # working set of a step below the 126 MB L2


def build_config(workload: str, bi) -> dict:
    """`config` of a build line: the same keys and values from both arms."""
    n_hits = int(bi.seg_off[-1])
    return dict(workload=workload, events_per_gpu=bi.n_events, seeds_per_gpu=bi.n_seeds, hits_per_gpu=n_hits, layers=bi.geom.n_layers, K=bi.K,
                n_phi=bi.n_phi, n_z=bi.n_z, chi2_cut=bi.chi2_cut, n_sigma=bi.n_sigma,
                l2="192 MB fill between timed iterations (outside the timed segments)" if build_needs_flush(n_hits) else
                   "hits + sorted copy + candidates per step exceed the 126 MB L2; no explicit flush")


def build_units(counters: dict, n_seeds: int, K: int, L: int, scale: float = 1.0) -> dict:
    """Algorithmic flops / bytes of one kf_build call from the oracle's own counters."""
    c = {k: v * scale for k, v in counters.items()}
    fl = sum(BUILD_FLOP[k] * c[k] for k in BUILD_FLOP)
    by = 16.0 * c["n_scan"] + 8.0 * c["n_rows"] + 113.0 * n_seeds + (117.0 + 4.0 * L) * K * n_seeds
    return dict(flops=fl, bytes=by, counters={k: int(v) for k, v in c.items()})


# ----------------------------------------------------------------------------------------------------------------
# the oracle on the host cores (cpu_baseline leg and --impl reference)
# ----------------------------------------------------------------------------------------------------------------
class oracle_threads:
    """`with oracle_threads(1):` -- the oracle's OpenMP loops on n host threads, set through the libgomp the oracle is linked
    against (omp_set_num_threads), so that the oracle itself stays as it stands.  SURVEY.md sec. 8d asks for the single-thread
    rate beside the all-cores one."""

    def __init__(self, n: int):
        import ctypes
        from oracle import kf_oracle as o
        o.lib()                                   # libgomp is in the process once the oracle is loaded
        self.gomp = ctypes.CDLL("libgomp.so.1")
        self.n = n

    def __enter__(self):
        self.prev = int(self.gomp.omp_get_max_threads())
        self.gomp.omp_set_num_threads(self.n)
        return self

    def __exit__(self, *exc):
        self.gomp.omp_set_num_threads(self.prev)


def one_core(cb: dict, cb1: dict) -> dict:
    """adds the single-thread leg to a cpu_baseline object"""
    cb.update(value_1_core=cb1["value"], sample_1_core=cb1["sample"])
    return cb


def parity_summary(out, r, sample: str) -> dict:
    """The timed kernel's output against the oracle run of the cpu_baseline leg (same tracks), with the rules of tests/parity.py:
    a report, not a gate -- the gate is `pytest -m gpu`.  Worst errors are in units of their tolerance (1.0 = at tolerance)."""
    try:
        from tests.parity import compare_tracks, PHI_DIR_ABS
        n = len(r["chi2"])
        g = dict(par=out.par[:, :n].cpu().numpy(), cov=out.cov[:, :n].cpu().numpy(), chi2=out.chi2[:n].cpu().numpy(),
                 nhits=out.nhits[:n].cpu().numpy(), status=out.status[:n].cpu().numpy().view(np.uint32))
        same = (g["nhits"] == r["nhits"]) & (g["status"] == r["status"])
        rep = compare_tracks(g, r, sel=same & (r["nhits"] > 0))
        keys = ("n", "mom_viol", "pos_viol", "cov_viol", "chi2_viol", "phi_viol", "strict_phi_viol", "worst_mom", "worst_pos_norm", "worst_cov",
                "worst_chi2", "worst_phi_strict")
        return dict(sample=sample, decisions_differ=int((~same).sum()), worst_dphi_rad=rep["worst_phi_dir"] * PHI_DIR_ABS, **{k: rep[k] for k in keys})
    except Exception as e:                      # never let the report break the bench line
        return dict(error=f"{type(e).__name__}: {e}")


def oracle_fit(fi, n_s, steps, warmup, keep=None):
    """keep: a dict that receives the oracle's result of the last call under "r" (for the parity summary of the line)"""
    from oracle import kf_oracle as o
    n_s = min(fi.n, n_s)
    L, ld = fi.geom.n_layers, fi.ld
    hx = np.ascontiguousarray(fi.hit_x.reshape(L, ld)[:, :n_s]).reshape(-1).astype(np.float64)
    hy = np.ascontiguousarray(fi.hit_y.reshape(L, ld)[:, :n_s]).reshape(-1).astype(np.float64)
    hz = np.ascontiguousarray(fi.hit_z.reshape(L, ld)[:, :n_s]).reshape(-1).astype(np.float64)
    hi = None if fi.hit_idx is None else np.ascontiguousarray(fi.hit_idx[:, :n_s])
    par = np.ascontiguousarray(fi.par[:, :n_s]); cov = np.ascontiguousarray(fi.cov[:, :n_s]); q = fi.q[:n_s]
    seg = np.arange(L + 1) * n_s
    last = {}

    def call():
        last["r"] = o.fit(fi.geom.layer_table(), fi.geom.bz, par, cov, q, hx, hy, hz, seg, hi)
    for _ in range(warmup):
        call()
    t0 = time.perf_counter()
    for _ in range(steps):
        call()
    dt = (time.perf_counter() - t0) / steps
    if keep is not None:
        keep.update(last)
    return dict(value=n_s / dt, unit="tracks/s", cores=o.num_threads(), kind="oracle",
                sample=f"first {n_s} tracks of the {fi.n}-track workload per step", ms_per_step=dt * 1e3)


def oracle_build(bi, n_ev, steps, warmup, hit_mode=0):
    """kfo_bin_hits + kfo_build on the first n_ev events (whole events: seeds only see hits of their own event)."""
    from oracle import kf_oracle as o
    L = bi.geom.n_layers
    n_ev = min(n_ev, bi.n_events)
    n_h = int(bi.seg_off[n_ev * L])
    sel = np.nonzero(bi.seed_event < n_ev)[0]
    n_s = len(sel)
    assert n_s == 0 or sel[-1] == n_s - 1, "seeds are stored event by event"
    seg = bi.seg_off[: n_ev * L + 1]
    lt = bi.geom.layer_table()
    res = {}

    def call():
        rb = o.bin_hits(lt, n_ev, seg, bi.hit_x[:n_h], bi.hit_y[:n_h], bi.hit_z[:n_h], bi.n_phi, bi.n_z)
        res["r"] = o.kf_build(lt, bi.geom.bz, rb, seg, bi.par, bi.cov, bi.q[:n_s], bi.seed_event[:n_s], bi.seed_hit_idx, bi.first_layer,
                              bi.K, bi.chi2_cut, bi.n_sigma, n=n_s, hit_mode=hit_mode)
    for _ in range(warmup):
        call()
    t0 = time.perf_counter()
    for _ in range(steps):
        call()
    dt = (time.perf_counter() - t0) / steps
    return dict(value=n_s / dt, unit="seeds/s", cores=o.num_threads(), kind="oracle",
                sample=f"first {n_ev} of {bi.n_events} events ({n_s} of {bi.n_seeds} seeds, {n_h} hits), binning + building, per step",
                ms_per_step=dt * 1e3), res["r"]["counters"], n_s


def run_reference(args, workload):
    if workload in FIT_CFG:
        fi = synth.fit_inputs(FIT_CFG[workload], n=args.tracks)
        cb = oracle_fit(fi, args.ref_sample, args.steps, args.warmup)
        metric, cfg = "tracks_fitted_per_s", fit_config(workload, fi)
    elif workload == "mplex":
        from oracle import kf_oracle as o
        m = 2_000_000
        rng = np.random.default_rng(66)
        a_ = rng.normal(size=(m, 6, 6)).astype(np.float32); b_ = rng.normal(size=(m, 6, 6)).astype(np.float32)
        for _ in range(args.warmup):
            o.mat66_multiply(a_, b_)
        t0 = time.perf_counter()
        for _ in range(args.steps):
            o.mat66_multiply(a_, b_)
        dt = (time.perf_counter() - t0) / args.steps
        cb = dict(value=m / dt, unit="multiplies/s", cores=1, kind="oracle", sample=f"{m} matrices per step, numpy fp64 matmul", ms_per_step=dt * 1e3)
        metric, cfg = "mat66_multiplies_per_s", dict(workload=workload, matrices=args.tracks or 4_000_000)
    else:
        bi = synth.build_inputs(BUILD_CFG[workload], n_events=args.events, **BUILD_KW.get(workload, {}))
        cb, _, _ = oracle_build(bi, args.ref_events, args.steps, args.warmup, hit_mode=BUILD_HIT_MODE.get(workload, 0))
        metric, cfg = "seeds_built_per_s", build_config(workload, bi)
    ms = cb.pop("ms_per_step")
    return dict(impl="reference", metric=metric, value=cb["value"], unit=cb["unit"], n_gpus=args.gpus, steps=args.steps,
                warmup=args.warmup, ms_per_step=ms, higher_is_better=True, scaling="weak", vs_baseline=None,
                dtype="f64", data="synthetic", config=cfg, cpu_baseline=cb,
                e2e=dict(value=cb["value"], unit=cb["unit"], h2d_bytes_per_step=0, d2h_bytes_per_step=0), gpu_launches=0)


# ----------------------------------------------------------------------------------------------------------------
# GPU legs
# ----------------------------------------------------------------------------------------------------------------
class Dist:
    def __init__(self):
        self.rank = int(os.environ.get("RANK", "0"))
        self.world = int(os.environ.get("WORLD_SIZE", "1"))
        self.local = int(os.environ.get("LOCAL_RANK", "0"))

    def barrier(self):
        import torch
        if self.world > 1:
            import torch.distributed as dist
            dist.barrier()
        torch.cuda.synchronize()

    def max_ms(self, ms: float) -> float:
        from paper_1711_06571_b200 import shard
        return shard.max_over_ranks(ms, device="cuda")


def time_steps(step, steps, warmup, stream, d: Dist, marks=0):
    """W warm-up steps, then K steps between barrier + synchronize, CUDA events on the launching stream.
    `step(rec)` may call rec(i) to drop intermediate events (i < marks) for per-kernel shares.
    -> (ms per step as max over ranks, per-step ms list, per-mark ms lists, wall t0, t1)"""
    import torch
    for _ in range(warmup):
        step(lambda i: None)
    d.barrier()
    ev = [torch.cuda.Event(enable_timing=True) for _ in range(steps + 1)]
    mk = [[torch.cuda.Event(enable_timing=True) for _ in range(marks)] for _ in range(steps)]
    t0 = time.time()
    ev[0].record(stream)
    for i in range(steps):
        step(lambda j, i=i: mk[i][j].record(stream))
        ev[i + 1].record(stream)
    d.barrier()
    t1 = time.time()
    per = [ev[i].elapsed_time(ev[i + 1]) for i in range(steps)]
    seg = []
    for j in range(marks + 1 if marks else 0):
        a = [(ev[i] if j == 0 else mk[i][j - 1]) for i in range(steps)]
        b_ = [(mk[i][j] if j < marks else ev[i + 1]) for i in range(steps)]
        seg.append([x.elapsed_time(y) for x, y in zip(a, b_)])
    return d.max_ms(ev[0].elapsed_time(ev[-1]) / steps), per, seg, t0, t1


def pin(a):
    import torch
    return torch.from_numpy(np.ascontiguousarray(a)).pin_memory()


def nbytes(ts):
    return int(sum(t.numel() * t.element_size() for t in ts if t is not None))


def bench_fit(args, d: Dist, workload: str, sampler_cb=None):
    import torch
    from paper_1711_06571_b200 import binding as b
    # weak scaling (default): every rank its own shard of the configured size, events differ by rank;
    # strong scaling: the configured tracks split over the ranks (shard.track_range)
    from paper_1711_06571_b200 import shard
    n_cfg = args.tracks if args.tracks is not None else synth.FIT_CONFIGS[FIT_CFG[workload]]["n"]
    if args.scaling == "strong":
        lo_, hi_ = shard.track_range(n_cfg, d.rank, d.world)
        fi = synth.fit_inputs(FIT_CFG[workload], n=hi_ - lo_, event=d.rank)
    else:
        fi = synth.fit_inputs(FIT_CFG[workload], n=args.tracks, event=d.rank)
    n_job = n_cfg if args.scaling == "strong" else fi.n * d.world
    units = fit_units(fi)
    geom = b.Geom(fi.geom.layer_table(), fi.geom.bz)
    hits = b.Hits(fi.hit_x, fi.hit_y, fi.hit_z, fi.seg_off, 1)
    seeds = b.Tracks.from_host(fi.par, fi.cov, fi.q)
    hit_idx = None if fi.hit_idx is None else torch.from_numpy(fi.hit_idx).cuda()
    out = b.Tracks.empty(seeds.n, seeds.ld)
    out.q = seeds.q
    stream = torch.cuda.current_stream()

    def step(rec):
        b.kf_fit(geom, hits, hit_idx, None, seeds, out=out, stream=stream)

    W = max(args.warmup, 3)
    sampler = ClockSampler(d.local) if d.rank == 0 else None
    ms_per_step, per, _, t0, t1 = time_steps(step, args.steps, W, stream, d)
    clocks = sampler.stop(t0, t1) if sampler else None
    value = n_job / (ms_per_step * 1e-3)

    # ---- end to end: pinned host buffers -> H2D -> kf_fit -> D2H, all inside the timed region ----
    # pipeline.FitPipeline: the tracks in `args.e2e_streams` independent sub-batches, each with its own stream, pinned host
    # buffers and device buffers, so that the copies of one sub-batch overlap the fit of another ("multiple events in
    # flight ... to overlap expensive copy operations").
    from paper_1711_06571_b200 import pipeline
    pipe = pipeline.FitPipeline(geom, fi.n, fi.par, fi.cov, fi.q, fi.hit_x, fi.hit_y, fi.hit_z, fi.ld, hit_idx=fi.hit_idx, n_streams=args.e2e_streams or 4)
    n_sub, h2d, d2h = len(pipe.subs), pipe.h2d_bytes, pipe.d2h_bytes

    def e2e_step(rec):
        pipe.run(stream)

    e2e_ms, _, _, _, _ = time_steps(e2e_step, max(3, min(args.steps, 10)), 2, stream, d)
    e2e_value = n_job / (e2e_ms * 1e-3)
    if d.rank != 0:
        return None

    pk = peaks()
    kern_ms = statistics.mean(per)                    # one kernel per step: CUDA events on the launching stream
    peak = fp32_peak_tflops(pk)
    t_alu = units["flops"] / (peak * 1e12)
    t_hbm = units["bytes"] / (pk["hbm_gbs"] * 1e9)
    ach = units["flops"] / (kern_ms * 1e-3) / 1e12
    roofline = dict(bound="alu", achieved=ach, peak=peak, unit="TFLOP/s", frac=ach / peak, traffic=None,
                    kernel="kf_fit_pair_kernel" if fi.hit_idx is None else "kf_fit_kernel", kernel_ms=kern_ms, kernel_ms_min=min(per), kernel_share_of_step=1.0,
                    peak_source=f"148 SMs x 128 FP32 lanes x 2 x {pk['sm_max_mhz']:.0f} MHz (clocks.max.sm, {pk['source']})",
                    alg_flops_per_launch=units["flops"], alg_bytes_per_launch=units["bytes"],
                    alg_flop_per_track_layer=FIT_FLOP_PER_TRACK_LAYER,
                    frac_survey_count=units["flops_survey"] / (kern_ms * 1e-3) / 1e12 / peak,
                    hbm_achieved_gbs=units["bytes"] / (kern_ms * 1e-3) / 1e9, hbm_peak_gbs=pk["hbm_gbs"],
                    frac_of_slower_roof=max(t_alu, t_hbm) / (kern_ms * 1e-3))
    roofline["traffic"] = stored_traffic(workload)
    roofline["traffic_note"] = traffic_note(workload)
    line = dict(metric="tracks_fitted_per_s", value=value, unit="tracks/s", n_gpus=d.world, steps=args.steps, warmup=W,
                ms_per_step=ms_per_step, higher_is_better=True, scaling=args.scaling, vs_baseline=None, dtype="f32", data="synthetic",
                config=fit_config(workload, fi),
                clocks=clocks, e2e=dict(value=e2e_value, unit="tracks/s", h2d_bytes_per_step=h2d, d2h_bytes_per_step=d2h, ms_per_step=e2e_ms, streams=n_sub),
                gpu_launches=args.steps, roofline=roofline)
    if not args.no_cpu_baseline:
        keep = {}
        cb = oracle_fit(fi, args.cpu_sample, 1, 0, keep=keep)
        cb.pop("ms_per_step")
        line["parity_sample"] = parity_summary(out, keep.get("r"), cb["sample"])
        with oracle_threads(1):
            cb1 = oracle_fit(fi, max(args.cpu_sample // 10, 1), 1, 0)
            assert cb1["cores"] == 1
        line["cpu_baseline"] = one_core(cb, cb1)
    return line


def stored_traffic(workload):
    """dram bytes per launch of the dominant kernel from the committed ncu --set full capture (profiles/traffic.csv).
    A row counts only if it was captured with this version of the library (column kf_version): a stale number reads null."""
    import csv
    tr = os.path.join(ROOT, "profiles", "traffic.csv")
    if not os.path.exists(tr):
        return None
    try:
        from paper_1711_06571_b200 import binding as b
        ver = str(b.kf_version())
    except Exception:
        return None
    for row in csv.DictReader(open(tr)):
        if row["workload"] == workload and row["dram_bytes_per_launch"] and row.get("kf_version", "") == ver:
            return float(row["dram_bytes_per_launch"])
    return None


def traffic_note(workload):
    """why `traffic` is what it is: the capture it comes from, or why there is none for this library version"""
    import csv
    tr = os.path.join(ROOT, "profiles", "traffic.csv")
    try:
        from paper_1711_06571_b200 import binding as b
        ver = str(b.kf_version())
        rows = [r for r in csv.DictReader(open(tr)) if r["workload"] == workload and r["dram_bytes_per_launch"]]
    except Exception as e:
        return f"profiles/traffic.csv unreadable: {e}"
    if any(r.get("kf_version", "") == ver for r in rows):
        return f"ncu --set full capture at library version {ver} (profiles/traffic.csv)"
    have = sorted({r.get("kf_version", "?") for r in rows})
    return f"no capture at library version {ver} in profiles/traffic.csv (captures at: {', '.join(have) or 'none'}); a stale number is not reported"


BUILD_LAUNCHES_PER_STEP = 5   # bin: count, scan, scatter, place; build (the memset of bin_off is not a kernel)


def bench_build(args, d: Dist, workload: str, sample_clocks=True):
    import torch
    from paper_1711_06571_b200 import binding as b
    cfg = BUILD_CFG[workload]
    idle = False
    if args.scaling == "strong":      # the configured events dealt out whole, balanced by seed count (shard.assign_events)
        from paper_1711_06571_b200 import shard
        n_ev_cfg = args.events if args.events is not None else synth.BUILD_CONFIGS[cfg]["n_events"]
        per_event = synth.BUILD_CONFIGS[cfg]["tracks"] * (1.0 + synth.BUILD_CONFIGS[cfg]["fake_frac"])
        mine = shard.assign_events([per_event] * n_ev_cfg, d.world)[d.rank]
        idle = not mine           # more ranks than events: this rank holds placeholder inputs, launches nothing and counts no seeds
        bi = synth.build_inputs(cfg, events=mine if mine else [0], **BUILD_KW.get(workload, {}))      # exactly the events dealt to this rank
    else:
        bi = synth.build_inputs(cfg, n_events=args.events, event0=d.rank * 1000, **BUILD_KW.get(workload, {}))
    L, K = bi.geom.n_layers, bi.K
    geom = b.Geom(bi.geom.layer_table(), bi.geom.bz, hit_mode=BUILD_HIT_MODE.get(workload, 0))
    hits = b.Hits(bi.hit_x, bi.hit_y, bi.hit_z, bi.seg_off, bi.n_events)
    n_bins = bi.n_events * L * bi.n_phi * bi.n_z
    binned = b.Binned(hits.n_hits, n_bins, bi.n_phi, bi.n_z, soa=False)     # the records and bin_off: all the build reads
    ws = torch.empty(max(b.kf_bin_workspace_bytes(geom, hits, bi.n_phi, bi.n_z), 1), dtype=torch.uint8, device="cuda")
    seeds = b.Tracks.from_host(bi.par, bi.cov, bi.q)
    sev = torch.from_numpy(bi.seed_event).cuda(); shi = torch.from_numpy(bi.seed_hit_idx).cuda()
    out = b.Cands(bi.n_seeds, K, L)
    bws = torch.empty(max(b.kf_build_workspace_bytes(geom, bi.n_seeds, K), 1), dtype=torch.uint8, device="cuda")
    stream = torch.cuda.current_stream()
    flush = torch.empty(192 << 20, dtype=torch.uint8, device="cuda") if build_needs_flush(hits.n_hits) else None

    def step(rec):
        if flush is not None:
            flush.fill_(1)        # working set below the 126 MB L2: flush between timed iterations
        rec(0)
        if idle:
            rec(1)
            return
        b.kf_bin_hits(geom, hits, bi.n_phi, bi.n_z, out=binned, ws=ws, stream=stream)
        rec(1)
        b.kf_build(geom, hits, binned, seeds, sev, shi, bi.first_layer, K, bi.chi2_cut, bi.n_sigma, out=out, ws=bws, stream=stream)

    W = max(args.warmup, 3)
    sampler = ClockSampler(d.local) if (d.rank == 0 and sample_clocks) else None
    _, _, seg, t0, t1 = time_steps(step, args.steps, W, stream, d, marks=2)
    clocks = sampler.stop(t0, t1) if sampler else None
    bin_ms, build_ms = statistics.mean(seg[1]), statistics.mean(seg[2])
    ms_per_step = d.max_ms(bin_ms + build_ms)          # the L2 flush is not part of the step
    from paper_1711_06571_b200 import shard as _shard
    n_job = _shard.sum_over_ranks(0.0 if idle else float(bi.n_seeds), device="cuda")
    value = n_job / (ms_per_step * 1e-3)

    # ---- end to end: hits + seeds H2D, bin + build, candidates D2H ----
    # pipeline.BuildPipeline: the events in `args.e2e_streams` groups, each with its own stream and buffers: several events in
    # flight, copies of one group overlapping the building of another.
    from paper_1711_06571_b200 import pipeline
    pipe = pipeline.BuildPipeline(geom, bi.n_events, bi.hit_x, bi.hit_y, bi.hit_z, bi.seg_off, bi.n_phi, bi.n_z, bi.par, bi.cov, bi.q, bi.seed_event,
                                  bi.seed_hit_idx, bi.first_layer, K, bi.chi2_cut, bi.n_sigma, n_streams=args.e2e_streams or (8 if workload == "build_c4" else 4))
    n_sub = len(pipe.subs)

    def e2e_step(rec):
        if not idle:
            pipe.run(stream)

    e2e_ms, _, _, _, _ = time_steps(e2e_step, max(3, min(args.steps, 10)), 2, stream, d)
    if d.rank != 0:
        return None
    pk = peaks()
    res = dict(metric="seeds_built_per_s", value=value, unit="seeds/s", ms_per_step=ms_per_step, bin_ms=bin_ms, build_ms=build_ms,
               hits_binned_per_s=hits.n_hits / (bin_ms * 1e-3),
               config=build_config(workload, bi),
               e2e=dict(value=n_job / (e2e_ms * 1e-3), unit="seeds/s", h2d_bytes_per_step=pipe.h2d_bytes, d2h_bytes_per_step=pipe.d2h_bytes,
                        ms_per_step=e2e_ms, streams=n_sub),
               gpu_launches=args.steps * BUILD_LAUNCHES_PER_STEP, clocks=clocks)
    bin_bytes = BIN_BYTES_PER_HIT * hits.n_hits + 4.0 * n_bins
    res["bin_roofline"] = dict(bound="hbm", achieved=bin_bytes / (bin_ms * 1e-3) / 1e9, peak=pk["hbm_gbs"], unit="GB/s",
                               frac=bin_bytes / (bin_ms * 1e-3) / 1e9 / pk["hbm_gbs"], alg_bytes_per_step=bin_bytes, kernels="kf_bin_* (memset + 4 launches)")
    if not args.no_cpu_baseline:
        cb, counters, n_s = oracle_build(bi, args.cpu_events, 1, 0, hit_mode=BUILD_HIT_MODE.get(workload, 0))
        cb.pop("ms_per_step")
        with oracle_threads(1):
            cb1, _, _ = oracle_build(bi, 1, 1, 0, hit_mode=BUILD_HIT_MODE.get(workload, 0))
        one_core(cb, cb1)
        u = build_units(counters, bi.n_seeds, K, L, scale=bi.n_seeds / max(n_s, 1))
        peak = fp32_peak_tflops(pk)
        t_alu, t_hbm = u["flops"] / (peak * 1e12), u["bytes"] / (pk["hbm_gbs"] * 1e9)
        if t_alu >= t_hbm:
            ach = u["flops"] / (build_ms * 1e-3) / 1e12
            rf = dict(bound="alu", achieved=ach, peak=peak, unit="TFLOP/s", frac=ach / peak)
        else:
            ach = u["bytes"] / (build_ms * 1e-3) / 1e9
            rf = dict(bound="hbm", achieved=ach, peak=pk["hbm_gbs"], unit="GB/s", frac=ach / pk["hbm_gbs"])
        rf.update(traffic=stored_traffic(workload), traffic_note=traffic_note(workload), kernel="kf_build_kernel", kernel_ms=build_ms, kernel_share_of_step=build_ms / (bin_ms + build_ms),
                  alg_flops_per_launch=u["flops"], alg_bytes_per_launch=u["bytes"], counters=u["counters"],
                  counters_source="oracle run of the cpu_baseline sample, scaled by seeds")
        res["roofline"] = rf
        res["cpu_baseline"] = cb
    return res


def bench_mplex(args, d: Dist):
    """Layout micro-benchmark (sec. 4.3, Fig. 5): n 6x6 products per step in
    matrix-major layout (`value`), as an array of matrices, and through the library (cuBLAS batched GEMM via torch.bmm)."""
    import torch
    from paper_1711_06571_b200 import binding as b
    n = args.tracks or 4_000_000
    g = torch.Generator(device="cuda"); g.manual_seed(66 + d.rank)
    A1 = torch.randn((n, 36), generator=g, device="cuda"); B1 = torch.randn((n, 36), generator=g, device="cuda")
    A0 = A1.t().contiguous(); B0 = B1.t().contiguous()
    C0 = torch.empty_like(A0); C1 = torch.empty_like(A1); C2 = torch.empty((n, 6, 6), device="cuda")
    stream = torch.cuda.current_stream()
    W = max(args.warmup, 3)
    res = {}
    for name, fn in (("matrix_major", lambda rec: b.kf_mat66_multiply(0, A0, B0, out=C0, stream=stream)),
                     ("array_of_matrices", lambda rec: b.kf_mat66_multiply(1, A1, B1, out=C1, stream=stream)),
                     ("cublas_bmm", lambda rec: torch.bmm(A1.view(n, 6, 6), B1.view(n, 6, 6), out=C2))):
        sampler = ClockSampler(d.local) if (d.rank == 0 and name == "matrix_major") else None
        ms, per, _, t0, t1 = time_steps(fn, args.steps, W, stream, d)
        if sampler:
            clocks = sampler.stop(t0, t1)
        res[name] = dict(ms=ms, per_s=n * d.world / (ms * 1e-3))
    # end to end (matrix-major): pinned host A, B -> device, multiply, C -> pinned host
    hA, hB = A0.cpu().pin_memory(), B0.cpu().pin_memory(); hC = torch.empty_like(hA).pin_memory()

    def e2e_step(rec):
        A0.copy_(hA, non_blocking=True); B0.copy_(hB, non_blocking=True)
        b.kf_mat66_multiply(0, A0, B0, out=C0, stream=stream)
        hC.copy_(C0, non_blocking=True)

    e2e_ms, _, _, _, _ = time_steps(e2e_step, 3, 1, stream, d)
    if d.rank != 0:
        return None
    pk = peaks()
    by = 3 * 144.0 * n
    ach = by / (res["matrix_major"]["ms"] * 1e-3) / 1e9
    line = dict(metric="mat66_multiplies_per_s", value=res["matrix_major"]["per_s"], unit="multiplies/s", n_gpus=d.world, steps=args.steps, warmup=W,
                ms_per_step=res["matrix_major"]["ms"], higher_is_better=True, scaling="weak", vs_baseline=None, dtype="f32", data="synthetic",
                config=dict(workload="mplex", matrices_per_gpu=n, l2="3 x %.0f MB per step exceed the 126 MB L2; no explicit flush" % (144.0 * n / 1e6)),
                clocks=clocks, layouts=res,
                e2e=dict(value=n * d.world / (e2e_ms * 1e-3), unit="multiplies/s", h2d_bytes_per_step=2 * 144 * n, d2h_bytes_per_step=144 * n, ms_per_step=e2e_ms),
                gpu_launches=args.steps,
                roofline=dict(bound="hbm", achieved=ach, peak=pk["hbm_gbs"], unit="GB/s", frac=ach / pk["hbm_gbs"], traffic=stored_traffic("mplex") if n == 4_000_000 else None, kernel="kf_mat66_soa_kernel",
                              alg_bytes_per_launch=by, alg_flops_per_launch=432.0 * n))
    if not args.no_cpu_baseline:
        from oracle import kf_oracle as o
        m = min(n, 2_000_000)
        a_ = A1[:m].cpu().numpy().reshape(m, 6, 6); b_ = B1[:m].cpu().numpy().reshape(m, 6, 6)
        t0 = time.perf_counter(); o.mat66_multiply(a_, b_); dt = time.perf_counter() - t0
        line["cpu_baseline"] = dict(value=m / dt, unit="multiplies/s", cores=1, kind="oracle", sample=f"first {m} matrices, numpy fp64 matmul")
    return line


def spawn_ranks(n: int) -> int:
    """--gpus N without a torchrun environment: start the N ranks here (one process per GPU, rendezvous on 127.0.0.1)."""
    import socket
    with socket.socket() as sk:
        sk.bind(("127.0.0.1", 0))
        port = sk.getsockname()[1]
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", f"--nproc-per-node={n}", "--master-addr", "127.0.0.1",
           "--master-port", str(port), os.path.abspath(__file__)] + sys.argv[1:]
    return subprocess.call(cmd)


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=5)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", default="fit_c1", choices=list(FIT_CFG) + list(BUILD_CFG) + ["mplex"])
    ap.add_argument("--scaling", default="weak", choices=["weak", "strong"], help="weak: every rank a full-size shard; strong: the configured work split over the ranks")
    ap.add_argument("--tracks", type=int, default=None, help="override the track count (debug only; invalidates the metric)")
    ap.add_argument("--events", type=int, default=None, help="override the event count of a build workload (debug only)")
    ap.add_argument("--ref-sample", type=int, default=100_000, help="--impl reference: tracks per step")
    ap.add_argument("--ref-events", type=int, default=16, help="--impl reference: events per step (build workloads)")
    ap.add_argument("--cpu-sample", type=int, default=200_000)
    ap.add_argument("--cpu-events", type=int, default=None, help="events the oracle builds for cpu_baseline and the build counters (default: 16 for build_c3, 4 for build_c4)")
    ap.add_argument("--e2e-streams", type=int, default=None, help="sub-batches in flight in the end-to-end leg (copies overlap compute); default 4, build_c4: 8 (measured: 40.9 / 37.4 / 36.6 ms with 4 / 8 / 16 groups of events; build_c3 1.44 / 1.64 ms with 4 / 8)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-build", action="store_true", help="default line without the extra legs (fit_c2, build_c3, build_c4)")
    args = ap.parse_args()
    if args.gpus > 1 and "WORLD_SIZE" not in os.environ and args.impl == "ours":
        return spawn_ranks(args.gpus)
    d = Dist()

    if args.impl == "reference":
        if d.rank == 0:
            print(json.dumps(run_reference(args, args.workload)), flush=True)
        return 0

    import torch
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device (there is no CPU fallback for the product path)")
    torch.cuda.set_device(d.local)
    if d.world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=torch.device("cuda", d.local))

    def build_leg(wl):
        a2 = argparse.Namespace(**vars(args))
        if a2.cpu_events is None:
            a2.cpu_events = 4 if wl == "build_c4" else 16
        return bench_build(a2, d, wl)

    if args.workload == "mplex":
        line = bench_mplex(args, d)
    elif args.workload in FIT_CFG:
        line = bench_fit(args, d, args.workload)
        if not args.no_build and args.tracks is None and args.workload == "fit_c1":
            # the other BASELINE.json configs in the same run, each a compact line of its own
            f2 = bench_fit(args, d, "fit_c2")
            b3 = build_leg("build_c3")
            torch.cuda.empty_cache()
            b4 = build_leg("build_c4")
            if line is not None:
                keep = ("metric", "value", "unit", "ms_per_step", "config", "clocks", "roofline", "cpu_baseline", "parity_sample", "e2e", "gpu_launches")
                line["fit_c2"] = {k: f2[k] for k in keep if k in f2}
                line["build"] = b3
                line["build_c4"] = b4
                line["gpu_launches"] += f2["gpu_launches"] + b3["gpu_launches"] + b4["gpu_launches"]
    else:
        r = build_leg(args.workload)
        line = None
        if r is not None:
            line = dict(metric=r.pop("metric"), value=r.pop("value"), unit=r.pop("unit"), n_gpus=d.world, steps=args.steps,
                        warmup=max(args.warmup, 3), ms_per_step=r.pop("ms_per_step"), higher_is_better=True, scaling=args.scaling,
                        vs_baseline=None, dtype="f32", data="synthetic", **r)
    if d.rank == 0:
        print(json.dumps(line), flush=True)
    if d.world > 1:
        import torch.distributed as dist
        dist.destroy_process_group()
    return 0


if __name__ == "__main__":
    sys.exit(main())
