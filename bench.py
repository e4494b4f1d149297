#!/usr/bin/env python
"""bench.py -- throughput of the KF hot path on B200 (contract: see DESIGN.md sec. 7).

  python bench.py [--gpus N] [--steps K] [--warmup W] [--workload fit_c1|fit_c2|build_c3] [--impl ours|reference]

A "step" is one pass of the whole hot path over one batch of synthetic input (for the fit workloads: one kf_fit
call over all tracks).  `value` is whole-job throughput with inputs resident in HBM; `e2e` is the same through the
C-ABI call with pinned HOST buffers, H2D and D2H copies inside the timed region.  `--impl reference` times the fp64
CPU oracle (oracle/) on a bounded sample of the same workload on the host cores.
Under torchrun every rank fits its own shard of the same size (weak scaling, no collective on the data path).
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
FIT_FLOP_PER_TRACK_LAYER = 800.0
FIT_BYTES_SEED_IN = 6 * 4 + 21 * 4 + 1            # par + cov + q
FIT_BYTES_OUT = 6 * 4 + 21 * 4 + 4 + 4 + 4        # par + cov + chi2 + nhits + status
FIT_BYTES_PER_HIT = 12
FIT_BYTES_PER_IDX = 4
SM_COUNT, FP32_LANES = 148, 128


def peaks():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(path):
        d = json.load(open(path))
        return dict(hbm_gbs=float(d["hbm_gbs"]), sm_max_mhz=float(d.get("sm_max_mhz", 1965.0)), source="measured")
    return dict(hbm_gbs=6650.0, sm_max_mhz=1965.0, source="fallback")


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


def fit_units(fi) -> dict:
    """Algorithmic flops / bytes of one kf_fit call over `fi`."""
    n_upd = int(fi.valid.sum())
    by = fi.n * (FIT_BYTES_SEED_IN + FIT_BYTES_OUT) + n_upd * FIT_BYTES_PER_HIT
    if fi.hit_idx is not None:
        by += fi.n * fi.geom.n_layers * FIT_BYTES_PER_IDX
    return dict(track_layers=n_upd, flops=n_upd * FIT_FLOP_PER_TRACK_LAYER, bytes=by)


def run_reference(args, fi, workload):
    from oracle import kf_oracle as o
    n_s = min(fi.n, args.ref_sample)
    idx = np.arange(n_s)
    L, ld = fi.geom.n_layers, fi.ld
    hx = np.ascontiguousarray(fi.hit_x.reshape(L, ld)[:, :n_s]).reshape(-1).astype(np.float64)
    hy = np.ascontiguousarray(fi.hit_y.reshape(L, ld)[:, :n_s]).reshape(-1).astype(np.float64)
    hz = np.ascontiguousarray(fi.hit_z.reshape(L, ld)[:, :n_s]).reshape(-1).astype(np.float64)
    hi = None if fi.hit_idx is None else np.ascontiguousarray(fi.hit_idx[:, :n_s])
    par = np.ascontiguousarray(fi.par[:, :n_s]); cov = np.ascontiguousarray(fi.cov[:, :n_s]); q = fi.q[:n_s]
    seg = np.arange(L + 1) * n_s
    call = lambda: o.fit(fi.geom.layer_table(), fi.geom.bz, par, cov, q, hx, hy, hz, seg, hi)
    for _ in range(args.warmup):
        call()
    t0 = time.perf_counter()
    for _ in range(args.steps):
        call()
    dt = (time.perf_counter() - t0) / args.steps
    v = n_s / dt
    sample = f"first {n_s} tracks of the {fi.n}-track workload per step"
    return dict(impl="reference", metric="tracks_fitted_per_s", value=v, unit="tracks/s", n_gpus=args.gpus, steps=args.steps,
                warmup=args.warmup, ms_per_step=dt * 1e3, higher_is_better=True, scaling="weak", vs_baseline=None,
                dtype="f64", data="synthetic", config=dict(workload=workload, tracks=fi.n, layers=L),
                cpu_baseline=dict(value=v, unit="tracks/s", cores=o.num_threads(), kind="oracle", sample=sample),
                e2e=dict(value=v, unit="tracks/s", h2d_bytes_per_step=0, d2h_bytes_per_step=0), gpu_launches=0)


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=5)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", default="fit_c1", choices=["fit_c1", "fit_c2", "fit_c0"])
    ap.add_argument("--tracks", type=int, default=None, help="override the track count (debug only; invalidates the metric)")
    ap.add_argument("--ref-sample", type=int, default=100_000)
    ap.add_argument("--cpu-sample", type=int, default=200_000)
    ap.add_argument("--no-cpu-baseline", action="store_true")
    args = ap.parse_args()

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    cfg_id = {"fit_c0": 0, "fit_c1": 1, "fit_c2": 2}[args.workload]

    if args.impl == "reference":
        if rank != 0:
            return 0
        fi = synth.fit_inputs(cfg_id, n=args.tracks)
        print(json.dumps(run_reference(args, fi, args.workload)), flush=True)
        return 0

    import torch
    import torch.distributed as dist
    from paper_1711_06571_b200 import binding as b

    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device (there is no CPU fallback for the product path)")
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    # every rank: its own shard of the configured size (weak scaling); events differ by rank
    fi = synth.fit_inputs(cfg_id, n=args.tracks, event=rank)
    units = fit_units(fi)
    geom = b.Geom(fi.geom.layer_table(), fi.geom.bz)
    hits = b.Hits(fi.hit_x, fi.hit_y, fi.hit_z, fi.seg_off, 1)
    seeds = b.Tracks.from_host(fi.par, fi.cov, fi.q)
    hit_idx = None if fi.hit_idx is None else torch.from_numpy(fi.hit_idx).cuda()
    out = b.Tracks.empty(seeds.n, seeds.ld)
    out.q = seeds.q
    stream = torch.cuda.current_stream()

    def step():
        b.kf_fit(geom, hits, hit_idx, None, seeds, out=out, stream=stream)

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    for _ in range(max(args.warmup, 3)):
        step()
    barrier()
    sampler = ClockSampler(local) if rank == 0 else None
    ev = [torch.cuda.Event(enable_timing=True) for _ in range(args.steps + 1)]
    t0 = time.time()
    ev[0].record(stream)
    for i in range(args.steps):
        step()
        ev[i + 1].record(stream)
    barrier()
    t1 = time.time()
    total_ms = ev[0].elapsed_time(ev[-1])
    per = [ev[i].elapsed_time(ev[i + 1]) for i in range(args.steps)]
    clocks = sampler.stop(t0, t1) if sampler else None
    ms = torch.tensor([total_ms / args.steps], device="cuda")
    if world > 1:
        dist.all_reduce(ms, op=dist.ReduceOp.MAX)
    ms_per_step = float(ms.item())
    value = fi.n * world / (ms_per_step * 1e-3)

    # ---- end to end: pinned host buffers -> H2D -> kf_fit -> D2H, all inside the timed region ----
    pin = lambda a: torch.from_numpy(np.ascontiguousarray(a)).pin_memory()
    h_par, h_cov, h_q = pin(fi.par), pin(fi.cov), pin(fi.q)
    h_x, h_y, h_z = pin(fi.hit_x), pin(fi.hit_y), pin(fi.hit_z)
    h_idx = None if fi.hit_idx is None else pin(fi.hit_idx)
    o_par = torch.empty((6, seeds.ld), dtype=torch.float32).pin_memory(); o_cov = torch.empty((21, seeds.ld), dtype=torch.float32).pin_memory()
    o_chi2 = torch.empty(fi.n, dtype=torch.float32).pin_memory(); o_nh = torch.empty(fi.n, dtype=torch.int32).pin_memory()
    o_st = torch.empty(fi.n, dtype=torch.int32).pin_memory()
    h2d = sum(t.numel() * t.element_size() for t in (h_par, h_cov, h_q, h_x, h_y, h_z) + ((h_idx,) if h_idx is not None else ()))
    d2h = sum(t.numel() * t.element_size() for t in (o_par, o_cov, o_chi2, o_nh, o_st))

    def e2e_step():
        seeds.par.copy_(h_par, non_blocking=True); seeds.cov.copy_(h_cov, non_blocking=True); seeds.q.copy_(h_q, non_blocking=True)
        hits.x.copy_(h_x, non_blocking=True); hits.y.copy_(h_y, non_blocking=True); hits.z.copy_(h_z, non_blocking=True)
        if h_idx is not None:
            hit_idx.copy_(h_idx, non_blocking=True)
        b.kf_fit(geom, hits, hit_idx, None, seeds, out=out, stream=stream)
        o_par.copy_(out.par, non_blocking=True); o_cov.copy_(out.cov, non_blocking=True); o_chi2.copy_(out.chi2, non_blocking=True)
        o_nh.copy_(out.nhits, non_blocking=True); o_st.copy_(out.status, non_blocking=True)

    e2e_steps = max(3, min(args.steps, 10))
    for _ in range(2):
        e2e_step()
    barrier()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record(stream)
    for _ in range(e2e_steps):
        e2e_step()
    e1.record(stream)
    barrier()
    ems = torch.tensor([e0.elapsed_time(e1) / e2e_steps], device="cuda")
    if world > 1:
        dist.all_reduce(ems, op=dist.ReduceOp.MAX)
    e2e_value = fi.n * world / (float(ems.item()) * 1e-3)

    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return 0

    pk = peaks()
    kern_ms = statistics.mean(per)                    # one kernel per step: CUDA events on the launching stream
    fp32_peak = SM_COUNT * FP32_LANES * 2 * pk["sm_max_mhz"] * 1e6 / 1e12     # TFLOP/s
    t_alu = units["flops"] / (fp32_peak * 1e12)
    t_hbm = units["bytes"] / (pk["hbm_gbs"] * 1e9)
    achieved_tflops = units["flops"] / (kern_ms * 1e-3) / 1e12
    roofline = dict(bound="alu", achieved=achieved_tflops, peak=fp32_peak, unit="TFLOP/s", frac=achieved_tflops / fp32_peak,
                    traffic=None, kernel="kf_fit_kernel", kernel_ms=kern_ms, kernel_ms_min=min(per),
                    peak_source=f"148 SMs x 128 FP32 lanes x 2 x {pk['sm_max_mhz']:.0f} MHz (clocks.max.sm, {pk['source']})",
                    alg_flops_per_launch=units["flops"], alg_bytes_per_launch=units["bytes"],
                    hbm_achieved_gbs=units["bytes"] / (kern_ms * 1e-3) / 1e9, hbm_peak_gbs=pk["hbm_gbs"],
                    frac_of_slower_roof=max(t_alu, t_hbm) / (kern_ms * 1e-3))
    tr = os.path.join(ROOT, "profiles", "traffic.json")
    if os.path.exists(tr):
        try:
            roofline["traffic"] = json.load(open(tr)).get(args.workload)
        except Exception:
            pass
    line = dict(metric="tracks_fitted_per_s", value=value, unit="tracks/s", n_gpus=world, steps=args.steps, warmup=max(args.warmup, 3),
                ms_per_step=ms_per_step, higher_is_better=True, scaling="weak", vs_baseline=None, dtype="f32", data="synthetic",
                config=dict(workload=args.workload, tracks_per_gpu=fi.n, layers=fi.geom.n_layers, track_layers=units["track_layers"],
                            l2="inputs+outputs per step (%.0f MB) exceed the 126 MB L2; no explicit flush" % (units["bytes"] / 1e6)),
                clocks=clocks, e2e=dict(value=e2e_value, unit="tracks/s", h2d_bytes_per_step=h2d, d2h_bytes_per_step=d2h,
                                        ms_per_step=float(ems.item())),
                gpu_launches=args.steps, roofline=roofline)
    if not args.no_cpu_baseline:
        from oracle import kf_oracle as o
        sub = argparse.Namespace(**vars(args)); sub.steps = 1; sub.warmup = 0; sub.ref_sample = args.cpu_sample
        ref = run_reference(sub, fi, args.workload)
        line["cpu_baseline"] = ref["cpu_baseline"]
    print(json.dumps(line), flush=True)
    if world > 1:
        dist.destroy_process_group()
    return 0


if __name__ == "__main__":
    sys.exit(main())
