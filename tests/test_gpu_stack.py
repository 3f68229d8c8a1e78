"""-m gpu: dfr_reproject_stack (fused reproject-and-stack) against the
oracle's orc_stack on the same seeded inputs, through the C ABI.

Tolerances: every exposure's value is within VALUE_TOL x DR of the oracle's,
so |sum_gpu - sum_orc| <= VALUE_TOL x DR x sum_e |w_e| (+ float32 accumulation, which is far
below it); wsum must be identical; pixels where ANY exposure's oracle coordinate lies
within EDGE_BAND of its footprint edge are compared only for consistency (wsum may differ
by that exposure's weight there)."""
import numpy as np
import pytest

import dfr_synth as S
import oracle
from tests import parity as PR

torch = pytest.importorskip("torch")
pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def P():
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    import paper_2505_03932_b200 as pkg
    pkg.lib()
    return pkg


def check_stack(P, w, order, weights=None, tol_scale=1.0):
    n = len(w.src_wcs)
    sny, snx = w.images.shape[1:]
    src = torch.from_numpy(w.images).cuda()
    s, ws = P.dfr_reproject_stack(src, w.src_wcs, w.tgt_wcs, w.shape_out, order, weights=weights)
    torch.cuda.synchronize()
    s, ws = s.cpu().numpy(), ws.cpu().numpy()
    so, wo = oracle.stack(w.images, w.src_wcs, w.tgt_wcs, w.shape_out, order, weights)
    band = np.zeros(w.shape_out, dtype=bool)
    tie = np.zeros(w.shape_out, dtype=bool)
    for e in range(n):
        xo, yo = oracle.src_coords(w.tgt_wcs, w.src_wcs[e], *w.shape_out)
        band |= PR.edge_band(xo, yo, sny, snx)
        if order == 0:
            tie |= ((np.abs(xo - np.floor(xo) - 0.5) < PR.TIE_BAND) | (np.abs(yo - np.floor(yo) - 0.5) < PR.TIE_BAND))
    assert not np.isnan(s).any() and not np.isnan(ws).any()
    assert np.array_equal(ws[~band], wo[~band]), "weight sums differ away from footprint edges"
    wabs = np.abs(np.ones(n) if weights is None else np.asarray(weights, dtype=np.float64)).sum()
    dr = max(PR.dyn_range(im) for im in w.images)
    ok = ~band & ~tie
    err = np.abs(s[ok].astype(np.float64) - so[ok])
    lim = tol_scale * PR.VALUE_TOL * dr * wabs
    assert err.max() <= lim, f"stack parity: max {err.max():.3e} > {lim:.3e}"
    return {"max": float(err.max()), "lim": lim, "depth_max": float(wo.max()), "depth0_frac": float((wo == 0).mean()),
            "band_px": int(band.sum())}


@pytest.mark.parametrize("order", [0, 1, 3])
def test_stack_small_batch_all_orders(P, order):
    """Ragged shapes, rotated + SIP exposures overlapping partially, random weights."""
    rng = np.random.default_rng(61)
    sny, snx, ony, onx = 140, 212, 150, 177
    n = 5
    imgs = np.stack([S.make_image(sny, snx, 30, rng) for _ in range(n)])
    srcs = [S.add_sip(S.make_wcs(snx, sny, 150.0 + 0.004 * rng.uniform(-1, 1), 2.0 + 0.004 * rng.uniform(-1, 1),
                                 rng.uniform(-20, 20), S.PIXSCALE), 3, snx / 2.0, rng, amp=1e-4) for _ in range(n)]
    tgt = S.add_sip(S.make_wcs(onx, ony, 150.001, 2.0005, 4.0, S.PIXSCALE * 1.03), 3, onx / 2.0, rng, amp=1e-4)
    w = S.Workload("stack-ragged", imgs, srcs, tgt, (ony, onx), (order,))
    wts = rng.integers(4, 17, n) / 8.0          # multiples of 1/8: every partial sum is exact in float32
    st = check_stack(P, w, order, wts)
    assert st["depth_max"] > 3.0 and st["depth0_frac"] < 0.5
    print("stack ragged", order, st)


def test_stack_single_exposure_equals_reproject(P):
    w = S.config0()
    src = torch.from_numpy(w.images).cuda()
    out = P.dfr_reproject(src, w.src_wcs, w.tgt_wcs, w.shape_out, 1)[0]
    s, ws = P.dfr_reproject_stack(src, w.src_wcs, w.tgt_wcs, w.shape_out, 1)
    m = torch.isnan(out)
    assert torch.equal(ws, (~m).float())
    assert torch.equal(s[~m], out[~m]) and bool((s[m] == 0).all())        # bit exact: w = 1
    mean = P.dfr_stack_finalize(s, ws)
    assert torch.equal(torch.isnan(mean), m) and torch.equal(mean[~m], out[~m])


def test_stack_accumulate_over_batches_and_nan_pixels(P):
    """Two calls with accumulate=True equal one call over all exposures up to float32
    re-association (the second batch is summed before it is added); a NaN source pixel is
    skipped by its exposure only."""
    w = S.config2(batch=6, n=512, nstars=300)
    w.images[2, 100:110, 200:230] = np.nan
    src = torch.from_numpy(w.images).cuda()
    s_all, w_all = P.dfr_reproject_stack(src, w.src_wcs, w.tgt_wcs, w.shape_out, 1)
    s, ws = P.dfr_reproject_stack(src[:4], w.src_wcs[:4], w.tgt_wcs, w.shape_out, 1)
    P.dfr_reproject_stack(src[4:], w.src_wcs[4:], w.tgt_wcs, w.shape_out, 1, sum=s, wsum=ws, accumulate=True)
    assert torch.equal(ws, w_all) and torch.allclose(s, s_all, rtol=5e-7, atol=0)
    st = check_stack(P, w, 1)
    so, wo = oracle.stack(w.images, w.src_wcs, w.tgt_wcs, w.shape_out, 1)
    assert (wo == 5.0).sum() > 100 and not np.isnan(so).any()
    print("stack nan/accumulate", st)


def test_stack_config2_full_size(P):
    """configs[2] (32 x 2048^2 -> 2048^2) in the launch configuration bench.py --mode stack
    times: the WHOLE sum and wsum frames against orc_stack, element by element."""
    w = S.config2()
    st = check_stack(P, w, 1)
    stats = P.dfr_last_stats()
    assert st["depth_max"] == 32.0
    print("C2 stack", stats, st)


def test_stack_unaligned_pitch_and_exact_tiles(P):
    """nx % 4 != 0 (no TMA staging) and a map that defeats the polynomial fit (EXACT tiles)."""
    rng = np.random.default_rng(71)
    imgs = np.stack([S.make_image(301, 403, 60, rng) for _ in range(3)])
    srcs = [S.make_wcs(403, 301, 150.0 + 1e-3 * k, 2.0, 3.0 * k, S.PIXSCALE) for k in range(3)]
    tgt = S.make_wcs(390, 310, 150.001, 2.0005, -2.0, S.PIXSCALE)
    w = S.Workload("odd", imgs, srcs, tgt, (310, 390), (1,))
    check_stack(P, w, 1)
    assert P.dfr_last_stats()["tiles_fast"] > 0
    imgs = np.stack([S.make_image(512, 512, 100, rng) for _ in range(2)])
    srcs = [S.make_wcs(512, 512, 150.0, 2.0, 0.0, S.PIXSCALE), S.make_wcs(512, 512, 150.001, 2.0, 5.0, S.PIXSCALE)]
    tgt = S.make_wcs(512, 512, 150.0005, 2.0003, 0.7, S.PIXSCALE)
    tgt.a_order = tgt.b_order = 4
    tgt.a[4][0] = 1e-8
    w = S.Workload("quartic", imgs, srcs, tgt, (512, 512), (1,))
    check_stack(P, w, 1)
    assert P.dfr_last_stats()["tiles_exact"] > 0


def test_stack_host_stream(P):
    """dfr_stack_host on a configs[4]-like stream (mosaic target, one batch per 2 exposures so
    batches overlap on the pipeline's streams): equals the device entry point up to float32
    re-association, and the oracle within the stack tolerance."""
    idx = (0, 31, 32, 511, 1023)
    w = S.config4(idx, n=512, nstars=200, mosaic=1024)
    wts = np.array([1.0, 2.0, 0.5, 1.0, 4.0])
    src = torch.from_numpy(w.images).pin_memory()
    s, c = P.dfr_stack_host(src, w.src_wcs, w.tgt_wcs, w.shape_out, 1, weights=wts, batch=2)
    st = P.dfr_last_stats()
    ds, dc = P.dfr_reproject_stack(torch.from_numpy(w.images).cuda(), w.src_wcs, w.tgt_wcs, w.shape_out, 1, weights=wts)
    assert torch.equal(c, dc.cpu()) and torch.allclose(s, ds.cpu(), rtol=1e-6, atol=1e-3)
    assert st["tiles_fast"] + st["tiles_empty"] + st["tiles_exact"] == 5 * 32 * 32
    so, wo = oracle.stack(w.images, w.src_wcs, w.tgt_wcs, w.shape_out, 1, wts)
    band = np.zeros(w.shape_out, dtype=bool)
    for e in range(len(idx)):
        xo, yo = oracle.src_coords(w.tgt_wcs, w.src_wcs[e], *w.shape_out)
        band |= PR.edge_band(xo, yo, 512, 512)
    assert np.array_equal(c.numpy()[~band], wo[~band])
    dr = max(PR.dyn_range(im) for im in w.images)
    assert np.abs(s.numpy()[~band] - so[~band]).max() <= PR.VALUE_TOL * dr * wts.sum()
    assert 0.5 < (wo == 0).mean() < 0.95                  # a mosaic: most of it is empty


def test_stack_many_exposures_few_tiles(P):
    """40 exposures onto a 3 x 3-tile target: the grid is cut into the maximum number of
    exposure chunks, including chunks of unequal length; signed weights."""
    rng = np.random.default_rng(81)
    n, sn, on = 40, 128, 160
    imgs = np.stack([S.make_image(sn, sn, 8, rng) for _ in range(n)])
    srcs = [S.make_wcs(sn, sn, 150.0 + 0.01 * rng.uniform(-1, 1), 2.0 + 0.01 * rng.uniform(-1, 1),
                       rng.uniform(0, 360), S.PIXSCALE) for _ in range(n)]
    tgt = S.make_wcs(on, on, 150.0, 2.0, 10.0, S.PIXSCALE * 1.2)
    w = S.Workload("many", imgs, srcs, tgt, (on, on), (1,))
    wts = rng.integers(-8, 17, n) / 4.0
    st = check_stack(P, w, 1, wts)
    # accumulate=True on top of existing contents with several chunks
    src = torch.from_numpy(imgs).cuda()
    s0 = torch.full((on, on), 3.0, device="cuda")
    w0 = torch.full((on, on), 1.0, device="cuda")
    s, c = P.dfr_reproject_stack(src, srcs, tgt, (on, on), 1, weights=wts)
    P.dfr_reproject_stack(src, srcs, tgt, (on, on), 1, weights=wts, sum=s0, wsum=w0, accumulate=True)
    assert torch.equal(w0, c + 1.0) and torch.allclose(s0, s + 3.0, rtol=1e-6, atol=1e-3)
    print("stack many", st)


def test_stack_is_deterministic_run_to_run(P):
    """Every output pixel has one owner (or, with exposure chunks, a fixed order of partial sums):
    the same call must give the same BITS every time, for a chunked launch (few tiles, many
    exposures) and for an unchunked one (many tiles)."""
    for n, npx, out_px in ((12, 256, 200), (3, 512, 2048)):
        w = S.config2(batch=n, n=npx, nstars=100)
        tgt = S.make_wcs(out_px, out_px, 150.0, 2.0, 0.3, S.PIXSCALE * npx / out_px)
        src = torch.from_numpy(w.images).cuda()
        wts = np.linspace(0.3, 1.7, n).astype(np.float32)         # not exactly representable sums
        ref_s, ref_w = P.dfr_reproject_stack(src, w.src_wcs, tgt, (out_px, out_px), 1, weights=wts)
        ref_s, ref_w = ref_s.clone(), ref_w.clone()
        for _ in range(4):
            s, c = P.dfr_reproject_stack(src, w.src_wcs, tgt, (out_px, out_px), 1, weights=wts)
            assert torch.equal(s, ref_s) and torch.equal(c, ref_w)
        assert float(ref_w.max()) > 0
