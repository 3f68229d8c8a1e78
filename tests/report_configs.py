#!/usr/bin/env python
"""All five BASELINE.json configs on one B200: parity against the oracle and timing.

    python tests/report_configs.py [--out gpurun_out/report.md] [--c4-exposures 1024]

Not a test (pytest does not collect it) and not the headline benchmark (bench.py is): it
produces the per-config table of BASELINE.md §5. Lives under tests/ because it calls the
oracle. Timing: CUDA events on the launching stream, 3 warm-ups, median of 20 launches;
for C0/C1/C3, whose inputs fit the 126 MB L2, a 512 MB buffer is overwritten between
launches (and that fill is outside the events).
"""
from __future__ import annotations

import argparse
import json
import os
import statistics
import sys
import time

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)

import numpy as np  # noqa: E402
import torch  # noqa: E402

import dfr_synth as S  # noqa: E402
import oracle  # noqa: E402
import paper_2505_03932_b200 as P  # noqa: E402
from tests import parity as PR  # noqa: E402

ORDER_NAME = {0: "nearest", 1: "bilinear", 3: "bicubic"}


def hbm_peak():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    return float(json.load(open(p))["hbm_gbs"]) if os.path.exists(p) else 6650.0


def time_gpu(fn, flush=None, reps=20, warm=3):
    for _ in range(warm):
        fn()
    torch.cuda.synchronize()
    ms = []
    for _ in range(reps):
        if flush is not None:
            flush.fill_(1.0)
        a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        a.record()
        fn()
        b.record()
        b.synchronize()
        ms.append(a.elapsed_time(b))
    return statistics.median(ms), min(ms)


def parity(w, order, out, exposures):
    """max / p99.99 coordinate and value errors of the listed exposures."""
    sny, snx = w.images.shape[1:]
    xg, yg = P.dfr_src_coords([w.src_wcs[e] for e in exposures], w.tgt_wcs, (sny, snx), w.shape_out, order)
    xg, yg = xg.cpu().numpy(), yg.cpu().numpy()
    cmax = c9 = vmax = v9 = 0.0
    nan = []
    band = 0
    for t, e in enumerate(exposures):
        xo, yo = oracle.src_coords(w.tgt_wcs, w.src_wcs[e], *w.shape_out)
        c = PR.check_coords(xg[t], yg[t], xo, yo, w.src_wcs[e])
        ref = oracle.interp(w.images[e], xo.ravel(), yo.ravel(), order).reshape(w.shape_out).astype(np.float32)
        v = PR.check_image(out[e], ref, xo, yo, w.images[e], order)
        cmax, c9 = max(cmax, c["max"]), max(c9, c["p9999"])
        vmax, v9 = max(vmax, v["max"] / v["dr"]), max(v9, v["p9999"] / v["dr"])
        nan.append(v["nan_frac"])
        band += v["mask_diff_in_band"]
    return {"coord_max_px": cmax, "coord_p9999_px": c9, "value_max_dr": vmax, "value_p9999_dr": v9,
            "nan_frac": float(np.mean(nan)), "mask_diff_in_edge_band": band, "exposures_checked": list(exposures)}


PROFILE_RUNS = 0        # --profile-runs N: N plain launches per case, nothing else (for ncu captures)


def device_case(name, w, order, exposures, flush, oracle_exposures=1):
    src = torch.from_numpy(w.images).cuda()
    n = len(w.src_wcs)
    out = torch.empty((n,) + tuple(w.shape_out), dtype=torch.float32, device="cuda")
    ws, tw = P.pack_wcs_array(w.src_wcs), P.pack_wcs(w.tgt_wcs)

    def step():
        P.dfr_reproject(src, ws, tw, w.shape_out, order, out=out)

    if PROFILE_RUNS:
        for _ in range(PROFILE_RUNS):
            if flush is not None:
                flush.fill_(1.0)
            step()
        torch.cuda.synchronize()
        return {"config": name, "order": ORDER_NAME[order], "profile_runs": PROFILE_RUNS, "tiles": P.dfr_last_stats()}
    med, best = time_gpu(step, flush)
    P.dfr_profile_enable(True)
    km = []
    for _ in range(5):
        if flush is not None:
            flush.fill_(1.0)
        step()
        km.append(P.dfr_profile_last())
    P.dfr_profile_enable(False)
    main_ms = statistics.median(m[1] for m in km)
    stats = P.dfr_last_stats()
    mpix = n * w.shape_out[0] * w.shape_out[1] / 1e6
    par = parity(w, order, out.cpu().numpy(), exposures)
    # algorithmic bytes: 4 B stored per output pixel + 4 B per source pixel (read once)
    alg = 4.0 * n * (w.shape_out[0] * w.shape_out[1] + w.images.shape[1] * w.images.shape[2])
    t0 = time.perf_counter()
    oracle.reproject(w.images[:oracle_exposures], w.src_wcs[:oracle_exposures], w.tgt_wcs, w.shape_out, order)
    cpu_s = time.perf_counter() - t0
    cpu_mpix = oracle_exposures * w.shape_out[0] * w.shape_out[1] / 1e6 / cpu_s
    return {"config": name, "order": ORDER_NAME[order], "out_mpix": mpix, "ms_median": med, "ms_best": best,
            "mpix_per_s": mpix / (med * 1e-3), "main_kernel_ms": main_ms,
            "main_kernel_gbs": alg / (main_ms * 1e-3) / 1e9, "main_kernel_frac_hbm": alg / (main_ms * 1e-3) / 1e9 / hbm_peak(),
            "tiles": stats, "oracle_mpix_per_s": cpu_mpix, "oracle_threads": oracle.max_threads(), **par}


def stream_case(n_exp, n_img, batch=32):
    """configs[4]: n_exp exposures with their own WCS (seeded per index) through the
    HOST-buffer entry point in batches of 32; pixel content cycles through n_img
    distinct seeded images to bound host memory and generation time."""
    t0 = time.perf_counter()
    wi = S.config4(range(n_img))
    wcs = list(wi.src_wcs)
    for k in range(n_img, n_exp):
        wcs.append(S.jittered_exposure([4, k], with_image=False, fast_image=True)[1])
    gen_s = time.perf_counter() - t0
    hin = torch.from_numpy(wi.images).pin_memory()
    hout = torch.empty((batch,) + tuple(wi.shape_out), dtype=torch.float32).pin_memory()
    tw = P.pack_wcs(wi.tgt_wcs)
    ws_all = P.pack_wcs_array(wcs)
    # warm-up (allocates the pipeline slots)
    P.dfr_reproject_host(hin[:batch], ws_all[:batch], tw, wi.shape_out, 1, out_host=hout, batch=8)
    torch.cuda.synchronize()
    t0 = time.perf_counter()
    for b0 in range(0, n_exp, batch):
        i0 = b0 % n_img
        P.dfr_reproject_host(hin[i0:i0 + batch], ws_all[b0:b0 + batch], tw, wi.shape_out, 1, out_host=hout, batch=8)
    torch.cuda.synchronize()
    el = time.perf_counter() - t0
    # parity on the seeded sample, recomputed with the sample's own images
    idx = (0, 31, 32, 511, 1023)
    w = S.config4([k for k in idx if k < n_exp])
    out = P.dfr_reproject_host(torch.from_numpy(w.images).pin_memory(), w.src_wcs, w.tgt_wcs, w.shape_out, 1, batch=2)
    par = parity(w, 1, out.numpy(), range(len(w.src_wcs)))
    mpix = n_exp * wi.shape_out[0] * wi.shape_out[1] / 1e6
    # the same stream co-added instead of returned one by one (dfr_stack_host)
    # (one call per n_img exposures, because the pixel content cycles; each call returns its
    # own sum / wsum pair, added on the host outside nothing: the adds are inside the timing)
    P.dfr_stack_host(hin[:2 * batch], ws_all[:2 * batch], tw, wi.shape_out, 1, batch=batch)
    torch.cuda.synchronize()
    t0 = time.perf_counter()
    ssum = swsum = None
    for b0 in range(0, n_exp, n_img):
        a, c = P.dfr_stack_host(hin[:min(n_img, n_exp - b0)], ws_all[b0:b0 + n_img], tw, wi.shape_out, 1, batch=batch)
        ssum = a if ssum is None else ssum.add_(a)
        swsum = c if swsum is None else swsum.add_(c)
    stack_s = time.perf_counter() - t0
    stack_depth = float(swsum.max().item())
    # device-resident kernel time of one batch of 32
    src = hin[:batch].cuda()
    dout = torch.empty((batch,) + tuple(wi.shape_out), dtype=torch.float32, device="cuda")
    med, best = time_gpu(lambda: P.dfr_reproject(src, ws_all[:batch], tw, wi.shape_out, 1, out=dout))
    alg = 4.0 * batch * (wi.shape_out[0] * wi.shape_out[1] + 2048 * 2048)
    return {"config": "C4", "order": "bilinear", "exposures": n_exp, "distinct_images": n_img,
            "wall_s": el, "exposures_per_s": n_exp / el, "mpix_per_s": mpix / el,
            "h2d_gbs": n_exp * 2048 * 2048 * 4 / el / 1e9, "d2h_gbs": mpix * 4e6 / el / 1e9,
            "device_batch_ms": med, "device_batch_mpix_per_s": batch * 16.777216 / (med * 1e-3),
            "device_batch_gbs": alg / (med * 1e-3) / 1e9, "generation_s": gen_s,
            "stack_wall_s": stack_s, "stack_exposures_per_s": n_exp / stack_s,
            "stack_h2d_gbs": n_exp * 2048 * 2048 * 4 / stack_s / 1e9, "stack_depth_max": stack_depth, **par}


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--out", default=os.path.join(ROOT, "gpurun_out", "report"))
    ap.add_argument("--c4-exposures", type=int, default=1024)
    ap.add_argument("--c4-images", type=int, default=128)
    ap.add_argument("--skip", default="")
    ap.add_argument("--only", default="", help="comma list of c0..c4: run only these")
    ap.add_argument("--orders", default="0,1,3", help="interpolation orders of the C3 rows")
    ap.add_argument("--profile-runs", type=int, default=0,
                    help="N plain launches per device case and nothing else (no parity, no timing): the command "
                         "ncu captures are taken from")
    args = ap.parse_args()
    if args.only:
        args.skip = ",".join(c for c in ("c0", "c1", "c2", "c3", "c4") if c not in args.only.split(","))
    global PROFILE_RUNS
    PROFILE_RUNS = args.profile_runs
    if PROFILE_RUNS:
        args.skip += ",c4"
    P.lib()
    oracle.build()
    assert torch.cuda.is_available()
    flush = torch.empty(128 * 1024 * 1024, dtype=torch.float32, device="cuda")
    rows = []
    if "c0" not in args.skip:
        rows.append(device_case("C0", S.config0(), 1, [0], flush))
    if "c1" not in args.skip:
        rows.append(device_case("C1", S.config1(), 1, [0], flush))
    if "c2" not in args.skip:
        rows.append(device_case("C2", S.config2(), 1, [0, 13, 31], None, oracle_exposures=4))
    if "c3" not in args.skip:
        w3 = S.config3()
        for o in (int(t) for t in args.orders.split(",")):
            rows.append(device_case("C3", w3, o, [0], flush))
    for r in rows:
        print(json.dumps(r), flush=True)
    c4 = None
    if "c4" not in args.skip:
        c4 = stream_case(args.c4_exposures, args.c4_images)
        print(json.dumps(c4), flush=True)
    if PROFILE_RUNS:
        return
    os.makedirs(os.path.dirname(args.out), exist_ok=True)
    with open(args.out + ".json", "w") as f:
        json.dump({"device": rows, "stream": c4, "hbm_peak_gbs": hbm_peak()}, f, indent=1)
    with open(args.out + ".md", "w") as f:
        f.write("| config | order | out Mpix | step ms (median) | out Mpix/s | main kernel ms | main kernel GB/s (algorithmic) "
                "| of measured HBM | coord err max / p99.99 (px) | value err max / p99.99 (x DR) | NaN frac "
                "| mask diffs (all within the 1e-3 px edge band) | oracle Mpix/s (threads) |\n")
        f.write("|" + "---|" * 13 + "\n")
        for r in rows:
            f.write(f"| {r['config']} | {r['order']} | {r['out_mpix']:.3f} | {r['ms_median']:.4f} | {r['mpix_per_s']:.0f} "
                    f"| {r['main_kernel_ms']:.4f} | {r['main_kernel_gbs']:.0f} | {100 * r['main_kernel_frac_hbm']:.1f} % "
                    f"| {r['coord_max_px']:.1e} / {r['coord_p9999_px']:.1e} | {r['value_max_dr']:.1e} / {r['value_p9999_dr']:.1e} "
                    f"| {r['nan_frac']:.4f} | {r['mask_diff_in_edge_band']} | {r['oracle_mpix_per_s']:.1f} ({r['oracle_threads']}) |\n")
        if c4:
            f.write(f"\nC4 stream: {c4['exposures']} exposures ({c4['distinct_images']} distinct images cycled, every WCS its own) "
                    f"in {c4['wall_s']:.2f} s = {c4['exposures_per_s']:.0f} exposures/s = {c4['mpix_per_s']:.0f} output Mpix/s "
                    f"(H2D {c4['h2d_gbs']:.1f} GB/s + D2H {c4['d2h_gbs']:.1f} GB/s concurrently); device-resident batch of 32: "
                    f"{c4['device_batch_ms']:.3f} ms = {c4['device_batch_mpix_per_s']:.0f} Mpix/s, {c4['device_batch_gbs']:.0f} GB/s; "
                    f"parity on exposures {c4['exposures_checked']}: coord {c4['coord_max_px']:.1e} px, value {c4['value_max_dr']:.1e} x DR, "
                    f"NaN frac {c4['nan_frac']:.3f}. The same stream co-added by dfr_stack_host (only sum and wsum come back): "
                    f"{c4['stack_wall_s']:.2f} s = {c4['stack_exposures_per_s']:.0f} exposures/s (H2D {c4['stack_h2d_gbs']:.1f} GB/s), "
                    f"deepest pixel {c4['stack_depth_max']:.0f} exposures.\n")
    print("wrote", args.out + ".md")


if __name__ == "__main__":
    main()
