#!/usr/bin/env python
"""bench.py — headline benchmark of the reprojection hot path (BASELINE.json `metric`).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference]

A "step" is one pass of the whole hot path over one batch
of synthetic input: configs[2] of BASELINE.json — 32 float32 2048x2048 TAN-SIP3
exposures reprojected onto one shared 2048x2048 TAN-SIP3 grid, bilinear — through
the C ABI (dfr_reproject). Prints ONE JSON line (rank 0).

  value     output Mpix/s with inputs resident in HBM (CUDA events, max over ranks)
  e2e       the same through dfr_reproject_host: HOST (pinned) buffers in and out,
            host<->device copies inside the timed region
  roofline  dominant kernel vs the measured HBM copy bandwidth (MEASURED_PEAKS.json)
  cpu_baseline  the oracle, as it stands, on this box's host cores (bounded sample)

With N > 1 (torchrun) every rank reprojects its own batch of 32 (exposures are
independent: no collective on the data path; weak scaling).
`--impl reference` times the oracle (oracle/) on the host cores instead.
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

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

import numpy as np  # noqa: E402

import dfr_synth as S  # noqa: E402

METRIC = "output Mpix/s reprojected (2048^2 TAN-SIP3 bilinear, batch 32)"
UNIT = "Mpix/s"
BATCH, NPIX = 32, 2048
FALLBACK_HBM_GBS = 6650.0          # B200_PROFILING.md fallback if MEASURED_PEAKS.json is absent
# dram__bytes_read.sum + dram__bytes_write.sum of one tiled_reproject_kernel launch on this
# workload, from the `ncu --set full` capture summarised in profiles/ (cannot be measured live)
NCU_TRAFFIC_BYTES = 536.94e6 + 493.84e6
NCU_TRAFFIC_SOURCE = "profiles/r01_main_kernel_ncu.md"


def peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        d = json.load(open(p))
        return float(d["hbm_gbs"]), "measured", float(d.get("sm_max_mhz", 1965.0))
    return FALLBACK_HBM_GBS, "fallback", 1965.0


class ClockSampler(threading.Thread):
    """nvidia-smi clocks/throttle reasons DURING the timed region (B200_PROFILING.md)."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index=0):
        super().__init__(daemon=True)
        self.index, self.rows, self._stop = index, [], threading.Event()
        self.proc = None

    def run(self):
        try:
            self.proc = subprocess.Popen(
                ["nvidia-smi", "-i", str(self.index), f"--query-gpu={self.Q}",
                 "--format=csv,noheader,nounits", "-lms", "100"],
                stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            for line in self.proc.stdout:
                self.rows.append([t.strip() for t in line.split(",")])
                if self._stop.is_set():
                    break
        except Exception:
            pass

    def stop(self):
        self._stop.set()
        if self.proc:
            try:
                self.proc.terminate()
            except Exception:
                pass

    def summary(self):
        sm, mx, reasons = [], 0.0, set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for r in self.rows:
            try:
                sm.append(float(r[0]))
                mx = max(mx, float(r[1]))
            except (ValueError, IndexError):
                continue
            for k, nm in enumerate(names):
                if len(r) > 3 + k and r[3 + k].lower().startswith("active"):
                    reasons.add(nm)
        return {"sm_mhz": statistics.median(sm) if sm else None, "sm_max_mhz": mx or None,
                "reasons": sorted(reasons), "samples": len(sm)}


def time_oracle(w, n_exp, passes=1):
    """The oracle as it stands on all host cores: `passes` passes over the first n_exp
    exposures, full frames. Returns (Mpix/s over all passes, wall seconds, threads used)."""
    import oracle
    oracle.build()
    t0 = time.perf_counter()
    for _ in range(passes):
        oracle.reproject(w.images[:n_exp], w.src_wcs[:n_exp], w.tgt_wcs, w.shape_out, 1)
    dt = time.perf_counter() - t0
    mpix = passes * n_exp * w.shape_out[0] * w.shape_out[1] / 1e6
    return mpix / dt, dt, oracle.max_threads()


def run_reference(args):
    """--impl reference: the oracle (test infrastructure) timed on the host cores."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return 0
    n_exp = 2
    w = S.config2(batch=n_exp)
    for _ in range(args.warmup):
        time_oracle(S.Workload("w", w.images[:1], w.src_wcs[:1], w.tgt_wcs, (256, 2048), (1,)), 1)
    t0 = time.perf_counter()
    for _ in range(args.steps):
        v, dt, cores = time_oracle(w, n_exp)
    el = time.perf_counter() - t0
    mpix = n_exp * NPIX * NPIX / 1e6
    value = mpix * args.steps / el
    sample = f"{n_exp} of the 32 exposures of configs[2], full 2048x2048 frames, per step"
    line = {"impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * el / args.steps,
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64",
            "data": "synthetic",
            "config": {"workload": "configs[2] sample: " + sample},
            "cpu_baseline": {"value": value, "unit": UNIT, "cores": cores, "kind": "oracle",
                             "sample": sample},
            "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line))
    return 0


def run_stack(args):
    """--mode stack: dfr_reproject_stack on configs[2] (32 exposures -> one sum + one weight
    frame). Same timing discipline as the headline; one JSON line with its own metric."""
    import torch
    import paper_2505_03932_b200 as P
    P.lib()
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device (there is no CPU fallback)")
    torch.cuda.set_device(int(os.environ.get("LOCAL_RANK", "0")))
    w = S.config2(batch=BATCH)
    src = torch.from_numpy(w.images).cuda()
    ws_arr, tw = P.pack_wcs_array(w.src_wcs), P.pack_wcs(w.tgt_wcs)
    ssum = torch.empty((NPIX, NPIX), dtype=torch.float32, device="cuda")
    wsum = torch.empty_like(ssum)

    def step():
        P.dfr_reproject_stack(src, ws_arr, tw, (NPIX, NPIX), P.BILINEAR, sum=ssum, wsum=wsum)

    for _ in range(max(args.warmup, 3)):
        step()
    torch.cuda.synchronize()
    sampler = ClockSampler(0)
    sampler.start()
    time.sleep(0.3)
    ev = [torch.cuda.Event(enable_timing=True) for _ in range(args.steps + 1)]
    torch.cuda.synchronize()
    ev[0].record()
    for k in range(args.steps):
        step()
        ev[k + 1].record()
    torch.cuda.synchronize()
    total_ms = ev[0].elapsed_time(ev[-1])
    per_step = [ev[k].elapsed_time(ev[k + 1]) for k in range(args.steps)]
    time.sleep(0.2)
    sampler.stop()
    P.dfr_profile_enable(True)
    ms = []
    for _ in range(min(args.steps, 10)):
        step()
        ms.append(P.dfr_profile_last())
    P.dfr_profile_enable(False)
    main_ms = statistics.mean(m[1] for m in ms)
    stats = P.dfr_last_stats()
    in_mpix = BATCH * NPIX * NPIX / 1e6
    hbm, which, _ = peaks()
    alg = 4.0 * BATCH * NPIX * NPIX + 8.0 * NPIX * NPIX       # sources read once + sum and wsum written
    achieved = alg / (main_ms * 1e-3) / 1e9
    line = {"metric": "input exposure Mpix/s reprojected and stacked (32 x 2048^2 TAN-SIP3 bilinear -> one 2048^2 sum + weight)",
            "value": in_mpix * args.steps / (total_ms * 1e-3), "unit": UNIT, "n_gpus": 1, "steps": args.steps,
            "warmup": max(args.warmup, 3), "ms_per_step": total_ms / args.steps, "higher_is_better": True,
            "scaling": "weak", "vs_baseline": None, "dtype": "f32", "data": "synthetic",
            "config": {"workload": "configs[2] through dfr_reproject_stack", "depth_mean": float(wsum.mean().item()),
                       "l2": "inputs per step are 537 MB > 126 MB L2 (no flush needed)", "tiles": stats},
            "ms_per_step_median": statistics.median(per_step),
            "roofline": {"bound": "hbm", "achieved": achieved, "peak": hbm, "unit": "GB/s", "frac": achieved / hbm,
                         "traffic": None, "peak_source": which, "kernel": "tiled_stack_kernel", "kernel_ms": main_ms,
                         "setup_kernels_ms": statistics.mean(m[0] for m in ms), "algorithmic_bytes_per_launch": alg,
                         "note": "issue-bound, not HBM-bound: see DESIGN.md §6.5"},
            "cpu_baseline": None, "e2e": None, "gpu_launches": int(stats["kernels"]) * args.steps,
            "clocks": sampler.summary()}
    print(json.dumps(line))
    return 0


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--e2e-steps", type=int, default=3)
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--path", default="auto", choices=["auto", "exact"])
    ap.add_argument("--mode", default="reproject", choices=["reproject", "stack"],
                    help="stack: the fused reproject-and-stack entry point (SURVEY.md §8(f) f1) on the same "
                         "workload; not the headline metric")
    args = ap.parse_args()
    if args.mode == "stack" and args.impl == "ours":
        return run_stack(args)
    args.warmup = max(args.warmup, 3) if args.impl == "ours" else args.warmup
    if args.impl == "reference":
        return run_reference(args)

    import torch
    import torch.distributed as dist
    import paper_2505_03932_b200 as P
    from paper_2505_03932_b200.shard import max_over_ranks
    P.lib()                                    # fail loudly if the CUDA library is missing
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device (there is no CPU fallback)")

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    # ---- inputs: configs[2]; rank r draws exposures with seeds [2, 32 r + k] via its own batch
    w = S.config2(batch=BATCH)
    if rank > 0:                               # distinct exposures per rank, same recipe
        for k in range(BATCH):
            img, ws = S.jittered_exposure([2, BATCH * rank + k])
            w.images[k] = img
            w.src_wcs[k] = ws
    path = P.PATH_EXACT if args.path == "exact" else P.PATH_AUTO
    src = torch.from_numpy(w.images).cuda()
    out = torch.empty((BATCH, NPIX, NPIX), dtype=torch.float32, device="cuda")
    ws_arr = P.pack_wcs_array(w.src_wcs)
    tw = P.pack_wcs(w.tgt_wcs)
    out_mpix = BATCH * NPIX * NPIX / 1e6

    def step():
        P.dfr_reproject(src, ws_arr, tw, (NPIX, NPIX), P.BILINEAR, out=out, path=path)

    for _ in range(args.warmup):
        step()
    barrier()
    stats = P.dfr_last_stats()

    sampler = ClockSampler(local)
    if rank == 0:
        sampler.start()
        time.sleep(0.3)
    # ---- timed region: K steps, CUDA events on the launching (current) stream
    ev = [torch.cuda.Event(enable_timing=True) for _ in range(args.steps + 1)]
    barrier()
    ev[0].record()
    for k in range(args.steps):
        step()
        ev[k + 1].record()
    barrier()
    total_ms = ev[0].elapsed_time(ev[-1])
    per_step = [ev[k].elapsed_time(ev[k + 1]) for k in range(args.steps)]
    if rank == 0:
        time.sleep(0.2)
        sampler.stop()
    total_ms = max_over_ranks(total_ms, device="cuda")
    value = out_mpix * world * args.steps / (total_ms * 1e-3)

    # ---- dominant kernel, timed live by the library's own events on the launching stream
    kern_ms = None
    if path == P.PATH_AUTO:
        P.dfr_profile_enable(True)
        ms = []
        for _ in range(min(args.steps, 10)):
            step()
            ms.append(P.dfr_profile_last())          # waits for the call's last event
        P.dfr_profile_enable(False)
        kern_ms = {"setup_ms": statistics.mean(m[0] for m in ms), "main_ms": statistics.mean(m[1] for m in ms)}
    nan_frac = float(torch.isnan(out).float().mean().item())

    # ---- e2e: HOST pinned buffers through dfr_reproject_host (copies inside the timed region)
    e2e = None
    if args.e2e_steps > 0:
        hsrc = torch.from_numpy(w.images).pin_memory()
        hout = torch.empty((BATCH, NPIX, NPIX), dtype=torch.float32).pin_memory()
        P.dfr_reproject_host(hsrc, ws_arr, tw, (NPIX, NPIX), P.BILINEAR, out_host=hout, batch=4)
        barrier()
        t0 = time.perf_counter()
        for _ in range(args.e2e_steps):
            P.dfr_reproject_host(hsrc, ws_arr, tw, (NPIX, NPIX), P.BILINEAR, out_host=hout, batch=4)
        torch.cuda.synchronize()
        el = max_over_ranks(time.perf_counter() - t0, device="cuda")
        e2e = {"value": out_mpix * world * args.e2e_steps / el, "unit": UNIT,
               "h2d_bytes_per_step": int(w.images.nbytes), "d2h_bytes_per_step": int(hout.numel() * 4),
               "steps": args.e2e_steps, "api": "dfr_reproject_host(batch=4), pinned host buffers"}
        same = bool(torch.equal(torch.nan_to_num(hout[:2], nan=-1.0), torch.nan_to_num(out[:2].cpu(), nan=-1.0)))
        e2e["matches_device_path"] = same

    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return 0

    # ---- roofline: algorithmic bytes = 4 B stored per output pixel + 4 B per source pixel read once
    hbm, which, sm_max = peaks()
    # (8 B per output pixel is the upper bound SURVEY.md §8(d) states; the
    # source pixels outside every output footprint and the NaN pixels are NOT subtracted)
    alg_bytes = 8.0 * BATCH * NPIX * NPIX
    dom_ms = kern_ms["main_ms"] if kern_ms else statistics.median(per_step)
    achieved = alg_bytes / (dom_ms * 1e-3) / 1e9
    roofline = {"bound": "hbm", "achieved": achieved, "peak": hbm, "unit": "GB/s",
                "frac": achieved / hbm, "traffic": NCU_TRAFFIC_BYTES if kern_ms else None,
                "traffic_source": NCU_TRAFFIC_SOURCE, "peak_source": which,
                "kernel": "tiled_reproject_kernel" if kern_ms else "whole dfr_reproject call",
                "kernel_ms": dom_ms, "setup_kernels_ms": kern_ms["setup_ms"] if kern_ms else None,
                "algorithmic_bytes_per_launch": alg_bytes}

    cpu = None
    if not args.no_cpu_baseline:
        # bounded sample: one pass sizes the run, then enough passes for ~10 s of wall time
        n_exp = BATCH
        v1, dt1, cores = time_oracle(w, n_exp)
        passes = int(min(8, max(1, round(10.0 / max(dt1, 1e-3)))))
        v, dt, cores = time_oracle(w, n_exp, passes)
        cpu = {"value": v, "unit": UNIT, "cores": cores, "kind": "oracle",
               "sample": f"all {n_exp} exposures of the step, full 2048x2048 frames, {passes} pass(es) after "
                         f"one sizing pass ({dt:.1f} s wall, {dt * cores:.0f} core-seconds)"}

    line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": total_ms / args.steps, "higher_is_better": True,
            "scaling": "weak", "vs_baseline": None, "dtype": "f32", "data": "synthetic",
            "config": {"workload": "configs[2]: 32 x 2048^2 TAN-SIP3 -> shared 2048^2 TAN-SIP3, bilinear",
                       "batch_per_gpu": BATCH, "path": args.path,
                       "l2": "inputs+outputs per step are 1074 MB > 126 MB L2 (no flush needed)",
                       "nan_fraction": nan_frac, "tiles": stats},
            "ms_per_step_median": statistics.median(per_step),
            "roofline": roofline, "cpu_baseline": cpu, "e2e": e2e,
            "gpu_launches": int(stats["kernels"]) * args.steps,
            "clocks": sampler.summary()}
    print(json.dumps(line))
    if world > 1:
        dist.destroy_process_group()
    return 0


if __name__ == "__main__":
    sys.exit(main())
