"""-m gpu: the CUDA path (through the C ABI, via the thin binding) against the oracle,
element by element on the same seeded inputs. Rules and tolerances: tests/parity.py."""
import numpy as np
import pytest

import dfr_synth as S
import oracle
from tests import parity as PR

torch = pytest.importorskip("torch")
pytestmark = pytest.mark.gpu

PATHS = {"exact": 1, "auto": 0}


@pytest.fixture(scope="module")
def P():
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    import paper_2505_03932_b200 as pkg
    pkg.lib()
    return pkg


def run_gpu(P, w, order, path):
    src = torch.from_numpy(w.images).cuda()
    out = P.dfr_reproject(src, w.src_wcs, w.tgt_wcs, w.shape_out, order, path=path)
    torch.cuda.synchronize()
    return out.cpu().numpy()


def full_parity(P, w, path, orders=None, exposures=None):
    """Coordinates + mask + values for the listed exposures of workload w."""
    sny, snx = w.images.shape[1:]
    exposures = range(len(w.src_wcs)) if exposures is None else exposures
    orders = w.orders if orders is None else orders
    report = {}
    outs = {o: run_gpu(P, w, o, path) for o in orders}
    xg, yg = P.dfr_src_coords(w.src_wcs, w.tgt_wcs, (sny, snx), w.shape_out, orders[0], path=path)
    xg, yg = xg.cpu().numpy(), yg.cpu().numpy()
    for e in exposures:
        xo, yo = oracle.src_coords(w.tgt_wcs, w.src_wcs[e], *w.shape_out)
        report[("coords", e)] = PR.check_coords(xg[e], yg[e], xo, yo, w.src_wcs[e])
        for o in orders:
            ref = oracle.interp(w.images[e], xo.ravel(), yo.ravel(), o).reshape(w.shape_out).astype(np.float32)
            report[(o, e)] = PR.check_image(outs[o][e], ref, xo, yo, w.images[e], o)
    return report, outs


@pytest.mark.parametrize("path", list(PATHS))
def test_config0(P, path):
    w = S.config0()
    rep, outs = full_parity(P, w, PATHS[path])
    # the oracle's own whole-path entry point agrees with src_coords + interp used above
    ref = oracle.reproject(w.images, w.src_wcs, w.tgt_wcs, w.shape_out, 1)
    m = np.isnan(ref[0])
    assert abs(m.mean() - 0.024) < 0.004
    assert rep[(1, 0)]["max"] <= PR.VALUE_TOL * rep[(1, 0)]["dr"]
    print("C0", path, rep)


@pytest.mark.parametrize("path", list(PATHS))
def test_config1(P, path):
    w = S.config1()
    rep, _ = full_parity(P, w, PATHS[path])
    assert abs(rep[(1, 0)]["nan_frac"] - 0.007) < 0.004
    print("C1", path, rep)


@pytest.mark.parametrize("path", list(PATHS))
@pytest.mark.parametrize("order", [0, 1, 3])
def test_ragged_shapes_all_orders(P, path, order):
    """Sizes that are not multiples of any tile, rotated + SIP, mask on all four sides."""
    rng = np.random.default_rng(21)
    sny, snx, ony, onx = 131, 203, 150, 177
    img = S.make_image(sny, snx, 40, rng)
    src = S.add_sip(S.make_wcs(snx, sny, 150.0, 2.0, 0.0, S.PIXSCALE), 3, snx / 2.0, rng, amp=1e-4)
    tgt = S.add_sip(S.make_wcs(onx, ony, 150.003, 2.002, 17.0, S.PIXSCALE * 1.07), 4, onx / 2.0, rng, amp=1e-4)
    w = S.Workload("ragged", img[None], [src], tgt, (ony, onx), (order,))
    rep, _ = full_parity(P, w, PATHS[path])
    assert 0.05 < rep[(order, 0)]["nan_frac"] < 0.9


@pytest.mark.parametrize("path", list(PATHS))
def test_stress_sip_coordinates(P, path):
    """~9 px distortion: a percent-level SIP error would show far above 1e-4 px."""
    src, tgt = S.stress_sip_pair()
    xg, yg = P.dfr_src_coords([src], tgt, (1024, 1024), (1024, 1024), 1, path=PATHS[path])
    xo, yo = oracle.src_coords(tgt, src, 1024, 1024)
    st = PR.check_coords(xg[0].cpu().numpy(), yg[0].cpu().numpy(), xo, yo, src)
    print("stress", path, st)


@pytest.mark.parametrize("path", list(PATHS))
def test_identity_and_integer_shift(P, path):
    rng = np.random.default_rng(5)
    img = S.make_image(70, 90, 10, rng)
    w = S.make_wcs(90, 70, 10.0, -40.0, 0.0, S.PIXSCALE)
    src = torch.from_numpy(img).cuda()
    out = P.dfr_reproject(src, [w], w, None, 0, path=PATHS[path]).cpu().numpy()[0]
    assert np.array_equal(out, img)                     # nearest: bit exact, no NaN
    t = w.copy()
    t.crpix = (w.crpix[0] + 7, w.crpix[1] - 3)
    out = P.dfr_reproject(src, [w], t, None, 0, path=PATHS[path]).cpu().numpy()[0]
    assert np.array_equal(out[:67, 7:], img[3:, :83])
    assert np.isnan(out[67:, :]).all() and np.isnan(out[:, :7]).all()


@pytest.mark.parametrize("path", list(PATHS))
def test_degenerate_inputs(P, path):
    # 1x1 image onto 1x1 and 3x5 grids
    img = np.array([[42.0]], dtype=np.float32)
    w = S.make_wcs(1, 1, 20.0, 30.0, 0.0, S.PIXSCALE)
    src = torch.from_numpy(img).cuda()
    for o in (0, 1, 3):
        out = P.dfr_reproject(src, [w], w, (1, 1), o, path=PATHS[path]).cpu().numpy()
        assert out.shape == (1, 1, 1) and out[0, 0, 0] == 42.0
    t = S.make_wcs(5, 3, 20.0, 30.0, 0.0, S.PIXSCALE)
    out = P.dfr_reproject(src, [w], t, (3, 5), 1, path=PATHS[path]).cpu().numpy()[0]
    ref = oracle.reproject(img, [w], t, (3, 5), 1)[0]
    assert np.array_equal(np.isnan(out), np.isnan(ref)) and out[1, 2] == 42.0
    # source on the far side of the sky: every pixel NaN (theta <= 0, G12)
    far = S.make_wcs(64, 64, 200.0, -30.0, 0.0, S.PIXSCALE)
    img2 = np.ones((64, 64), dtype=np.float32)
    out = P.dfr_reproject(torch.from_numpy(img2).cuda(), [far], S.make_wcs(64, 64, 20.0, 30.0, 0.0, S.PIXSCALE),
                          None, 1, path=PATHS[path]).cpu().numpy()
    assert np.isnan(out).all()
    # disjoint but nearby footprint: all NaN as well
    near = S.make_wcs(64, 64, 20.5, 30.0, 0.0, S.PIXSCALE)
    out = P.dfr_reproject(torch.from_numpy(img2).cuda(), [near], S.make_wcs(64, 64, 20.0, 30.0, 0.0, S.PIXSCALE),
                          None, 1, path=PATHS[path]).cpu().numpy()
    assert np.isnan(out).all()


def test_sky_entry_points(P):
    rng = np.random.default_rng(9)
    w = S.add_sip(S.make_wcs(2048, 2048, 359.99, -35.5, 33.0, S.PIXSCALE), 4, 1024.0, rng, amp=1e-4)
    x = rng.uniform(-10, 2060, 20000)
    y = rng.uniform(-10, 2060, 20000)
    ra, dec = P.dfr_pix2world(w, torch.from_numpy(x).cuda(), torch.from_numpy(y).cuda())
    ra_o, dec_o = oracle.pix2world(w, x, y)
    d = np.abs((ra.cpu().numpy() - ra_o + 180.0) % 360.0 - 180.0)
    assert d.max() < 1e-10 and np.abs(dec.cpu().numpy() - dec_o).max() < 1e-10
    assert ra.min().item() >= 0.0 and ra.max().item() < 360.0
    xb, yb = P.dfr_world2pix(w, ra, dec)
    xo, yo = oracle.world2pix(w, ra_o, dec_o)
    lim = 1e-7 + PR.oracle_conditioning(xo, yo, w)
    assert np.all(np.abs(xb.cpu().numpy() - xo) < lim) and np.all(np.abs(yb.cpu().numpy() - yo) < lim)
    # far side -> NaN
    xf, yf = P.dfr_world2pix(w, torch.tensor([179.99], dtype=torch.float64).cuda(),
                             torch.tensor([35.5], dtype=torch.float64).cuda())
    assert torch.isnan(xf).all() and torch.isnan(yf).all()
    # zero points is legal
    e = torch.empty(0, dtype=torch.float64).cuda()
    r0, d0 = P.dfr_pix2world(w, e, e)
    assert r0.numel() == 0


def test_sip_order_9(P):
    rng = np.random.default_rng(99)
    src = S.add_sip(S.make_wcs(300, 300, 150.0, 2.0, 0.0, S.PIXSCALE), 9, 150.0, rng, amp=1e-4)
    tgt = S.add_sip(S.make_wcs(300, 300, 150.001, 2.001, -3.0, S.PIXSCALE), 7, 150.0, rng, amp=1e-4)
    for path in PATHS.values():
        xg, yg = P.dfr_src_coords([src], tgt, (300, 300), (300, 300), 1, path=path)
        xo, yo = oracle.src_coords(tgt, src, 300, 300)
        PR.check_coords(xg[0].cpu().numpy(), yg[0].cpu().numpy(), xo, yo, src)


def test_config2_batch_full_size(P):
    """configs[2] at full size in the launch configuration bench.py times (batch 32 in one
    call): ALL 32 exposures element by element (coordinates of the tiled path, mask, values;
    tests/parity.py), plus 40 000
    sampled pixels computed one by one through the oracle's sky entry points
    (pix2world -> world2pix -> interp: a second route through the oracle)."""
    w = S.config2()
    out = run_gpu(P, w, 1, 0)
    st = P.dfr_last_stats()
    sny, snx = w.images.shape[1:]
    fr, worst, worst_c = [], 0.0, 0.0
    for e in range(32):
        if e % 4 == 0:       # the kernels' own coordinates, 4 exposures x 2 x 33.5 MB at a time
            xg, yg = P.dfr_src_coords(w.src_wcs[e:e + 4], w.tgt_wcs, (sny, snx), w.shape_out, 1, path=0)
            xg, yg = xg.cpu().numpy(), yg.cpu().numpy()
        xo, yo = oracle.src_coords(w.tgt_wcs, w.src_wcs[e], *w.shape_out)
        worst_c = max(worst_c, PR.check_coords(xg[e % 4], yg[e % 4], xo, yo, w.src_wcs[e])["max"])
        ref = oracle.interp(w.images[e], xo.ravel(), yo.ravel(), 1).reshape(w.shape_out).astype(np.float32)
        r = PR.check_image(out[e], ref, xo, yo, w.images[e], 1)
        fr.append(r["nan_frac"])
        worst = max(worst, r["max"] / r["dr"])
    assert 0.005 < np.mean(fr) < 0.12
    rng = np.random.default_rng(222)
    for e in range(32):
        ii = rng.integers(0, 2048, 1250).astype(np.float64)
        jj = rng.integers(0, 2048, 1250).astype(np.float64)
        ra, dec = oracle.pix2world(w.tgt_wcs, ii, jj)
        xo, yo = oracle.world2pix(w.src_wcs[e], ra, dec)
        ref = oracle.interp(w.images[e], xo, yo, 1).astype(np.float32)
        got = out[e][jj.astype(int), ii.astype(int)]
        band = PR.edge_band(xo, yo, sny, snx)
        assert np.array_equal(np.isnan(got)[~band], np.isnan(ref)[~band])
        ok = ~np.isnan(got) & ~np.isnan(ref)
        assert np.max(np.abs(got[ok] - ref[ok])) <= PR.VALUE_TOL * PR.dyn_range(w.images[e])
    print("C2 stats", st, "worst value error", worst, "x DR, worst coordinate error", worst_c, "px, mean NaN fraction", np.mean(fr))


def test_config3_three_orders(P):
    w = S.config3()
    rep, _ = full_parity(P, w, 0)
    assert abs(rep[(1, 0)]["nan_frac"] - 0.075) < 0.01
    print("C3", rep)


def test_config4_stream_sample(P):
    """configs[4] on the seeded sample of exposures (0, 31, 32, 511, 1023) through the
    HOST-buffer streaming entry point, 2 exposures per batch so batches pipeline."""
    idx = (0, 31, 32, 511, 1023)
    w = S.config4(idx)
    src = torch.from_numpy(w.images).pin_memory()
    out = P.dfr_reproject_host(src, w.src_wcs, w.tgt_wcs, w.shape_out, 1, batch=2)
    out = out.numpy()
    inside, worst_c = [], 0.0
    for t in range(len(idx)):
        xo, yo = oracle.src_coords(w.tgt_wcs, w.src_wcs[t], *w.shape_out)
        xg, yg = P.dfr_src_coords([w.src_wcs[t]], w.tgt_wcs, w.images.shape[1:], w.shape_out, 1, path=0)
        worst_c = max(worst_c, PR.check_coords(xg[0].cpu().numpy(), yg[0].cpu().numpy(), xo, yo, w.src_wcs[t])["max"])
        del xg, yg
        ref = oracle.interp(w.images[t], xo.ravel(), yo.ravel(), 1).reshape(w.shape_out).astype(np.float32)
        r = PR.check_image(out[t], ref, xo, yo, w.images[t], 1)
        inside.append(1 - r["nan_frac"])
    assert abs(np.mean(inside) - 0.25) < 0.01
    print("C4 worst coordinate error", worst_c, "px")
    # same result from the device-buffer entry point
    dev = P.dfr_reproject(torch.from_numpy(w.images[:2]).cuda(), w.src_wcs[:2], w.tgt_wcs, w.shape_out, 1)
    assert np.array_equal(np.nan_to_num(dev.cpu().numpy(), nan=-1), np.nan_to_num(out[:2], nan=-1))


def test_fast_path_is_taken_and_matches_exact(P):
    """AUTO must run the tiled kernels on ordinary geometry (not silently the exact path),
    agree with the exact path to the parity tolerance, and classify empty tiles."""
    w = S.config1(n=1024, nstars=500)
    src = torch.from_numpy(w.images).cuda()
    fast = P.dfr_reproject(src, w.src_wcs, w.tgt_wcs, w.shape_out, 1, path=P.PATH_AUTO)
    st = P.dfr_last_stats()
    assert st["kernels"] == 3 and st["tiles_fast"] == 32 * 32 and st["tiles_exact"] == 0
    exact = P.dfr_reproject(src, w.src_wcs, w.tgt_wcs, w.shape_out, 1, path=P.PATH_EXACT)
    assert P.dfr_last_stats()["kernels"] == 1
    f, x = fast.cpu().numpy()[0], exact.cpu().numpy()[0]
    both = ~np.isnan(f) & ~np.isnan(x)
    assert (np.isnan(f) != np.isnan(x)).sum() <= 8           # only on the footprint edge
    assert np.max(np.abs(f[both] - x[both])) <= PR.VALUE_TOL * PR.dyn_range(w.images[0])
    xf, yf = P.dfr_src_coords(w.src_wcs, w.tgt_wcs, (1024, 1024), w.shape_out, 1, path=P.PATH_AUTO)
    xe, ye = P.dfr_src_coords(w.src_wcs, w.tgt_wcs, (1024, 1024), w.shape_out, 1, path=P.PATH_EXACT)
    d = max((xf - xe).abs().max().item(), (yf - ye).abs().max().item())
    print("tiled vs exact coords: max", d)
    assert d < 2e-5
    # a mosaic-like target: most tiles are empty
    w4 = S.config4((7,), n=512, nstars=100, mosaic=2048)
    out = P.dfr_reproject(torch.from_numpy(w4.images).cuda(), w4.src_wcs, w4.tgt_wcs, w4.shape_out, 1)
    st = P.dfr_last_stats()
    assert st["tiles_empty"] > 0.8 * 64 * 64 and st["tiles_fast"] > 0
    ref = oracle.reproject(w4.images, w4.src_wcs, w4.tgt_wcs, w4.shape_out, 1)
    xo, yo = oracle.src_coords(w4.tgt_wcs, w4.src_wcs[0], *w4.shape_out)
    PR.check_image(out[0].cpu().numpy(), ref[0], xo, yo, w4.images[0], 1)


def test_unaligned_row_pitch_uses_global_gathers(P):
    """nx % 4 != 0 cannot be described to TMA (16-byte row pitch): the tiled kernel then
    gathers from global memory; results must be the same."""
    rng = np.random.default_rng(31)
    img = S.make_image(301, 403, 60, rng)
    src = S.add_sip(S.make_wcs(403, 301, 150.0, 2.0, 0.0, S.PIXSCALE), 3, 201.5, rng, amp=1e-5)
    tgt = S.add_sip(S.make_wcs(390, 310, 150.002, 2.001, -2.0, S.PIXSCALE), 3, 195.0, rng, amp=1e-5)
    w = S.Workload("odd", img[None], [src], tgt, (310, 390), (0, 1, 3))
    rep, _ = full_parity(P, w, 0)
    assert P.dfr_last_stats()["tiles_fast"] > 0


def test_two_level_setup_fallback(P):
    """A quartic target distortion sized so that the cubic fit of a 64x64 CTA tile misses
    FIT_TOL (error ~ c h^4 / 8 = 1.3e-5 px at h = 32) while the fit of each 32x32 tile holds
    (8e-7 px): the setup kernel must refit per tile, not accept the parent cubic and not
    fall to EXACT. A 100x larger quartic defeats both levels: tiles become EXACT."""
    rng = np.random.default_rng(41)
    img = S.make_image(512, 512, 200, rng)
    src = S.make_wcs(512, 512, 150.0, 2.0, 0.0, S.PIXSCALE)
    for c4, want_exact in ((1e-10, False), (1e-8, True)):
        tgt = S.make_wcs(512, 512, 150.0005, 2.0003, 0.7, S.PIXSCALE)
        tgt.a_order = tgt.b_order = 4
        tgt.a[4][0] = c4
        tgt.b[0][4] = -c4
        w = S.Workload("quartic", img[None], [src], tgt, (512, 512), (1,))
        rep, _ = full_parity(P, w, 0)
        st = P.dfr_last_stats()
        xf, yf = P.dfr_src_coords(w.src_wcs, w.tgt_wcs, (512, 512), w.shape_out, 1, path=P.PATH_AUTO)
        xe, ye = P.dfr_src_coords(w.src_wcs, w.tgt_wcs, (512, 512), w.shape_out, 1, path=P.PATH_EXACT)
        d = max(torch.nan_to_num(xf - xe).abs().max().item(), torch.nan_to_num(yf - ye).abs().max().item())
        print("quartic", c4, st, "tiled vs exact", d, rep[("coords", 0)])
        if want_exact:
            assert st["tiles_exact"] > 0
        else:
            assert st["tiles_exact"] == 0 and st["tiles_fast"] > 200
            assert d < 5e-6                   # 1.3e-5 if the parent cubic had been accepted
    # u^4 - v^4 in ONE coordinate: the two fourth-order errors cancel wherever |s| and |t| are
    # both 0, 1/sqrt(2) or 1 (centre, diagonal, corners), so the check points must also sample
    # the axes or the 64x64 fit would be accepted with a 2.6e-5 px error
    tgt = S.make_wcs(512, 512, 150.0005, 2.0003, 0.7, S.PIXSCALE)
    tgt.a_order = tgt.b_order = 4
    tgt.a[4][0], tgt.a[0][4] = 1e-10, -1e-10
    xf, yf = P.dfr_src_coords([src], tgt, (512, 512), (512, 512), 1, path=P.PATH_AUTO)
    xe, ye = P.dfr_src_coords([src], tgt, (512, 512), (512, 512), 1, path=P.PATH_EXACT)
    d = max(torch.nan_to_num(xf - xe).abs().max().item(), torch.nan_to_num(yf - ye).abs().max().item())
    print("u^4 - v^4: tiled vs exact", d)
    assert d < 6e-6


def test_random_geometries_tiled_vs_exact(P):
    """Robustness of the unchecked interior loop: 36 seeded random geometries (scale ratio
    0.6-1.7, any rotation, offsets that leave part of the target uncovered, SIP on both
    sides, ragged shapes) x 3 orders. The tiled path must agree with the exact per-pixel
    path to the value tolerance wherever both are valid, differ in validity only on the
    footprint edge, and the stack must equal the NaN-aware sum of the exact reprojections."""
    rng = np.random.default_rng(2024)
    worst = 0.0
    for case in range(36):
        sny, snx = (int(v) for v in rng.integers(90, 420, 2))
        snx = snx // 4 * 4 if case % 3 else snx                    # both staged and unstaged sources
        ony, onx = (int(v) for v in rng.integers(70, 400, 2))
        n = int(rng.integers(1, 4))
        imgs = np.stack([S.make_image(sny, snx, 30, rng) for _ in range(n)])
        scale = S.PIXSCALE * rng.uniform(0.6, 1.7)
        srcs = []
        for _ in range(n):
            w = S.make_wcs(snx, sny, 150.0 + rng.uniform(-0.02, 0.02), 2.0 + rng.uniform(-0.02, 0.02),
                           rng.uniform(0, 360), S.PIXSCALE)
            srcs.append(S.add_sip(w, int(rng.integers(2, 6)), snx / 2.0, rng, amp=10 ** rng.uniform(-6, -3.5)))
        tgt = S.make_wcs(onx, ony, 150.0, 2.0, rng.uniform(0, 360), scale)
        if case % 2:
            S.add_sip(tgt, 3, onx / 2.0, rng, amp=1e-4)
        src = torch.from_numpy(imgs).cuda()
        dr = max(PR.dyn_range(im) for im in imgs)
        for order in (0, 1, 3):
            fast = P.dfr_reproject(src, srcs, tgt, (ony, onx), order, path=P.PATH_AUTO)
            st = P.dfr_last_stats()
            exact = P.dfr_reproject(src, srcs, tgt, (ony, onx), order, path=P.PATH_EXACT)
            mf, mx = torch.isnan(fast), torch.isnan(exact)
            assert int((mf != mx).sum()) <= 4 * (ony + onx) * n, (case, order)   # only along footprint edges
            both = ~mf & ~mx
            if order > 0 and bool(both.any()):
                d = float((fast[both] - exact[both]).abs().max())
                worst = max(worst, d / dr)
                assert d <= PR.VALUE_TOL * dr, (case, order, d, st)
            if order == 1:
                s, ws = P.dfr_reproject_stack(src, srcs, tgt, (ony, onx), order)
                ok = ~(mf != mx).any(0)
                ref = torch.nan_to_num(exact, nan=0.0).sum(0)
                assert torch.equal(ws[ok], (~mx).sum(0).float()[ok]), (case, "wsum")
                assert float((s[ok] - ref[ok]).abs().max()) <= PR.VALUE_TOL * dr * n, (case, "sum")
    print("random geometries: worst tiled-vs-exact value difference", worst, "x DR")


@pytest.mark.parametrize("path", list(PATHS))
def test_paper_demo_geometry(P, path):
    """The shape of the paper's own demonstration (two 50x50 frames offset by
    0.5 px and 0.005 deg, bilinear) on a synthetic frame (its FITS files are not available)."""
    rng = np.random.default_rng(127)
    img = S.make_image(50, 50, 6, rng)
    src = S.make_wcs(50, 50, 150.0, 2.0, 0.0, S.PIXSCALE)
    tgt = S.make_wcs(50, 50, 150.0, 2.0, 0.005, S.PIXSCALE)
    tgt.crpix = (src.crpix[0] + 0.5, src.crpix[1] + 0.5)
    w = S.Workload("demo", img[None], [src], tgt, (50, 50), (1,))
    rep, outs = full_parity(P, w, PATHS[path])
    # a half-pixel shift: each output pixel is close to the mean of its four neighbours (P9)
    out = outs[1][0]
    m = 0.25 * (img[:-1, :-1] + img[1:, :-1] + img[:-1, 1:] + img[1:, 1:])
    assert np.nanmax(np.abs(out[1:, 1:] - m)) < 2e-3 * PR.dyn_range(img)


def test_paper_footprint_mode(P):
    """dfr_reproject_edge(DFR_EDGE_PAPER) against orc_interp_paper (reading G19): bilinear
    keeps the half-pixel band (-1, -0.5) u (n - 0.5, n) the area rule drops, with the edge
    pixel's value; inside the area footprint the two modes are bit-identical; nearest is the
    area rule; bicubic is refused. Mask band: |x + 1|, |x - n| < EDGE_BAND."""
    rng = np.random.default_rng(69)
    sny, snx, ony, onx = 140, 212, 190, 260
    img = S.make_image(sny, snx, 40, rng)
    src = S.add_sip(S.make_wcs(snx, sny, 150.0, 2.0, 0.0, S.PIXSCALE), 3, snx / 2.0, rng, amp=1e-4)
    tgt = S.make_wcs(onx, ony, 150.0004, 2.0003, 11.0, S.PIXSCALE * 0.93)
    d = torch.from_numpy(img[None]).cuda()
    area = P.dfr_reproject(d, [src], tgt, (ony, onx), 1).cpu().numpy()[0]
    paper = P.dfr_reproject(d, [src], tgt, (ony, onx), 1, edge=P.EDGE_PAPER).cpu().numpy()[0]
    xo, yo = oracle.src_coords(tgt, src, ony, onx)
    ref, foot = oracle.interp_paper(img, xo.ravel(), yo.ravel(), 1)
    ref, foot = ref.reshape(ony, onx), foot.reshape(ony, onx)
    near = ((np.abs(xo + 1) < PR.EDGE_BAND) | (np.abs(xo - snx) < PR.EDGE_BAND)
            | (np.abs(yo + 1) < PR.EDGE_BAND) | (np.abs(yo - sny) < PR.EDGE_BAND))
    mg, mo = np.isnan(paper), np.isnan(ref)
    assert not ((mg != mo) & ~near).any()
    ok = ~mg & ~mo
    assert np.abs(paper[ok] - ref[ok]).max() <= PR.VALUE_TOL * PR.dyn_range(img)
    extra = ~np.isnan(paper) & np.isnan(area)
    assert extra.sum() > 300 and not (np.isnan(paper) & ~np.isnan(area)).any()   # a strict superset
    both = ~np.isnan(area)
    assert np.array_equal(paper[both], area[both])
    # nearest: the same as the area rule; bicubic: refused
    n0 = P.dfr_reproject(d, [src], tgt, (ony, onx), 0).cpu().numpy()
    n1 = P.dfr_reproject(d, [src], tgt, (ony, onx), 0, edge=P.EDGE_PAPER).cpu().numpy()
    assert np.array_equal(np.nan_to_num(n0, nan=-1), np.nan_to_num(n1, nan=-1))
    with pytest.raises(P.DfrError):
        P.dfr_reproject(d, [src], tgt, (ony, onx), 3, edge=P.EDGE_PAPER)


@pytest.mark.parametrize("path", list(PATHS))
@pytest.mark.parametrize("order", [0, 1, 3])
def test_nan_source_pixels_propagate(P, path, order):
    """Reading G14: NaN pixels in the source propagate by IEEE through the taps read (and only
    those). Blocks, lines and isolated NaN pixels, including on the image rim. Which taps are
    read depends on floor(x) (rint for nearest), so the NaN mask is compared away from the
    footprint edge AND away from coordinates within 2 x COORD_TOL of an integer (a half-integer
    for nearest), where a legal coordinate difference changes the tap set."""
    rng = np.random.default_rng(14)
    sny, snx, ony, onx = 236, 300, 250, 270
    img = S.make_image(sny, snx, 60, rng)
    img[40:52, 60:90] = np.nan                      # a block
    img[120, :] = np.nan                            # a row
    img[:, 200] = np.nan                            # a column
    img[0, 0] = img[sny - 1, snx - 1] = img[sny - 1, 10] = np.nan      # rim pixels (edge replication)
    ys, xs = rng.integers(0, sny, 150), rng.integers(0, snx, 150)
    img[ys, xs] = np.nan                            # isolated pixels
    src = S.add_sip(S.make_wcs(snx, sny, 150.0, 2.0, 0.0, S.PIXSCALE), 3, snx / 2.0, rng, amp=1e-4)
    tgt = S.add_sip(S.make_wcs(onx, ony, 150.002, 2.001, 9.0, S.PIXSCALE * 1.04), 3, onx / 2.0, rng, amp=1e-4)
    out = P.dfr_reproject(torch.from_numpy(img[None]).cuda(), [src], tgt, (ony, onx), order,
                          path=PATHS[path]).cpu().numpy()[0]
    xo, yo = oracle.src_coords(tgt, src, ony, onx)
    ref = oracle.interp(img, xo.ravel(), yo.ravel(), order).reshape(ony, onx)
    inside = ~PR.edge_band(xo, yo, sny, snx) & np.isfinite(xo)
    off = 0.5 if order == 0 else 0.0
    fx, fy = xo - off - np.floor(xo - off), yo - off - np.floor(yo - off)
    amb = (np.minimum(fx, 1 - fx) < PR.TIE_BAND) | (np.minimum(fy, 1 - fy) < PR.TIE_BAND)
    cmp = inside & ~amb
    mg, mo = np.isnan(out), np.isnan(ref)
    assert np.array_equal(mg[cmp], mo[cmp]), f"{int((mg != mo)[cmp].sum())} NaN-propagation mismatches"
    foot = np.isfinite(xo) & (xo >= -0.5) & (xo < snx - 0.5) & (yo >= -0.5) & (yo < sny - 0.5)
    assert (mo & foot).sum() > 500 and (~mo).sum() > 0.5 * ony * onx     # NaNs inside the footprint exist
    ok = ~mg & ~mo & cmp
    assert np.abs(out[ok] - ref[ok]).max() <= PR.VALUE_TOL * PR.dyn_range(img)


@pytest.mark.parametrize("fit_order", [3, 5])
def test_fitted_inverse_sip_end_to_end(P, fit_order):
    """§8(f) f4 end to end: a source WCS that carries only the forward SIP (A/B) gets AP/BP
    from dfr_wcs_fit_inverse_sip; the reprojection through those coefficients must equal the
    oracle fed the SAME fitted coefficients (coordinates, mask, values; all three orders)."""
    rng = np.random.default_rng(65)
    sny, snx, ony, onx = 400, 520, 410, 500
    img = S.make_image(sny, snx, 120, rng)
    src = S.make_wcs(snx, sny, 150.0, 2.0, 0.0, S.PIXSCALE)
    src.a, src.b = S.draw_sip(4, snx / 2.0, rng, amp=3e-4)
    src.a_order = src.b_order = 4                   # ~0.5 px distortion, no AP/BP
    tgt = S.make_wcs(onx, ony, 150.003, 2.002, -6.0, S.PIXSCALE)
    packed = P.pack_wcs(src)
    resid = P.dfr_wcs_fit_inverse_sip(packed, fit_order, snx, sny)
    assert 0.0 < resid < 0.2 and packed.ap_order == fit_order and packed.bp_order == fit_order
    fitted = src.copy()
    fitted.ap_order = fitted.bp_order = fit_order
    fitted.ap = np.array(packed.ap[:]).reshape(10, 10)
    fitted.bp = np.array(packed.bp[:]).reshape(10, 10)
    assert np.abs(fitted.ap).max() > 0
    w = S.Workload("f4", img[None], [fitted], tgt, (ony, onx), (0, 1, 3))
    for path in PATHS.values():
        rep, _ = full_parity(P, w, path)
    # without the fitted inverse the coordinates differ by the distortion itself
    xa, _ = oracle.src_coords(tgt, fitted, ony, onx)
    xb, _ = oracle.src_coords(tgt, src, ony, onx)
    assert np.nanmax(np.abs(xa - xb)) > 0.05
    print("f4", fit_order, "fit residual", resid, rep[("coords", 0)])


@pytest.mark.parametrize("order", [0, 1, 3])
def test_footprint_array_area_rule(P, order):
    """§8(f) f2: dfr_reproject_fp returns (array, footprint) like reproject_interp.
    Under the area rule the footprint is 1 where the oracle's footprint rule (O11) holds and 0
    elsewhere — the oracle side is its interpolation of an all-ones image (1 inside, NaN outside);
    identical outside the 1e-3 px edge band; `array` is bit-identical with and without it."""
    rng = np.random.default_rng(27)
    sny, snx, ony, onx = 236, 300, 250, 330
    imgs = np.stack([S.make_image(sny, snx, 40, rng) for _ in range(2)])
    imgs[1, 50:60, 70:90] = np.nan                  # NaN pixels do not change the footprint
    srcs = [S.add_sip(S.make_wcs(snx, sny, 150.0, 2.0 + 0.002 * k, 5.0 * k, S.PIXSCALE), 3, snx / 2.0, rng, amp=1e-4)
            for k in range(2)]
    tgt = S.make_wcs(onx, ony, 150.002, 2.001, 9.0, S.PIXSCALE * 1.04)
    d = torch.from_numpy(imgs).cuda()
    plain = P.dfr_reproject(d, srcs, tgt, (ony, onx), order)
    out, foot = P.dfr_reproject(d, srcs, tgt, (ony, onx), order, footprint=True)
    assert P.dfr_last_stats()["kernels"] == 4
    assert torch.equal(torch.nan_to_num(plain, nan=-7.0), torch.nan_to_num(out, nan=-7.0))
    foot = foot.cpu().numpy()
    ones = np.ones((sny, snx), dtype=np.float32)
    for e in range(2):
        xo, yo = oracle.src_coords(tgt, srcs[e], ony, onx)
        ref = np.nan_to_num(oracle.interp(ones, xo.ravel(), yo.ravel(), order).reshape(ony, onx), nan=0.0)
        band = PR.edge_band(xo, yo, sny, snx)
        assert set(np.unique(foot[e])) <= {0.0, 1.0} and 0.05 < ref.mean() < 0.95
        assert np.array_equal(foot[e][~band], ref[~band].astype(np.float32))
        # consistent with the array itself: valid pixels lie inside the footprint
        assert not (~np.isnan(out[e].cpu().numpy()) & (foot[e] == 0)).any()


def test_footprint_array_paper_rule(P):
    """the footprint is the projected identity. DFR_EDGE_PAPER + bilinear returns
    orc_interp_paper's `foot` (zero-padded interpolation of ones): |difference| <= COORD_TOL (its
    slope is at most 1 per pixel on each axis and the coordinates agree to COORD_TOL), 0 / > 0
    pattern identical outside the edge band of the (-1, n) rule; nearest: the 0/1 area footprint."""
    rng = np.random.default_rng(69)
    sny, snx, ony, onx = 140, 212, 190, 260
    img = S.make_image(sny, snx, 40, rng)
    src = S.add_sip(S.make_wcs(snx, sny, 150.0, 2.0, 0.0, S.PIXSCALE), 3, snx / 2.0, rng, amp=1e-4)
    tgt = S.make_wcs(onx, ony, 150.0004, 2.0003, 11.0, S.PIXSCALE * 0.93)
    d = torch.from_numpy(img[None]).cuda()
    out, foot = P.dfr_reproject(d, [src], tgt, (ony, onx), 1, edge=P.EDGE_PAPER, footprint=True)
    plain = P.dfr_reproject(d, [src], tgt, (ony, onx), 1, edge=P.EDGE_PAPER)
    assert torch.equal(torch.nan_to_num(plain, nan=-7.0), torch.nan_to_num(out, nan=-7.0))
    out, foot = out.cpu().numpy()[0], foot.cpu().numpy()[0]
    xo, yo = oracle.src_coords(tgt, src, ony, onx)
    ref, rfoot = oracle.interp_paper(img, xo.ravel(), yo.ravel(), 1)
    rfoot = rfoot.reshape(ony, onx)
    near = ((np.abs(xo + 1) < PR.EDGE_BAND) | (np.abs(xo - snx) < PR.EDGE_BAND)
            | (np.abs(yo + 1) < PR.EDGE_BAND) | (np.abs(yo - sny) < PR.EDGE_BAND))
    assert np.array_equal((foot > 0)[~near], (rfoot > 0)[~near])
    assert np.abs(foot - rfoot)[~near].max() <= PR.COORD_TOL
    part = (rfoot > 0) & (rfoot < 1)
    assert part.sum() > 300 and np.abs(foot - rfoot)[part & ~near].max() <= PR.COORD_TOL     # the linear rim is exercised
    assert np.array_equal(np.isnan(out)[~near], (foot == 0)[~near])          # the array is valid exactly where foot > 0
    o0, f0 = P.dfr_reproject(d, [src], tgt, (ony, onx), 0, edge=P.EDGE_PAPER, footprint=True)
    _, f0o = oracle.interp_paper(img, xo.ravel(), yo.ravel(), 0)
    band = PR.edge_band(xo, yo, sny, snx)
    assert np.array_equal(f0.cpu().numpy()[0][~band], f0o.reshape(ony, onx)[~band].astype(np.float32))
    # the Python drop-in returns (array, footprint)
    hdr = {"CRPIX1": src.crpix[0], "CRPIX2": src.crpix[1], "CRVAL1": src.crval[0], "CRVAL2": src.crval[1],
           "CD1_1": src.cd[0], "CD1_2": src.cd[1], "CD2_1": src.cd[2], "CD2_2": src.cd[3]}
    thdr = {"CRPIX1": tgt.crpix[0], "CRPIX2": tgt.crpix[1], "CRVAL1": tgt.crval[0], "CRVAL2": tgt.crval[1],
            "CD1_1": tgt.cd[0], "CD1_2": tgt.cd[1], "CD2_1": tgt.cd[2], "CD2_2": tgt.cd[3]}
    arr, fp = P.calculate_reprojection((img, hdr), thdr, (ony, onx), "bilinear", return_footprint=True)
    assert arr.shape == fp.shape == (ony, onx) and set(np.unique(fp)) <= {0.0, 1.0}
    assert np.array_equal(np.isnan(arr), fp == 0)


def test_multi_device_entry_points_on_one_gpu(P):
    """§8(e): dfr_reproject_host_multi / dfr_stack_host_multi shard the exposures over the listed
    devices; listing device 0 twice (and three times) runs the whole multi-shard path — shard
    threads, one pipeline per shard, peer copy + add for the stack — on a single GPU. The
    per-exposure result must equal the single-device call bit for bit; the stack up to float32
    re-association of the per-shard partial sums."""
    w = S.config2(batch=7, n=512, nstars=200)
    src = torch.from_numpy(w.images).pin_memory()
    one = P.dfr_reproject_host(src, w.src_wcs, w.tgt_wcs, w.shape_out, 1, batch=2).numpy().copy()
    st1 = P.dfr_last_stats()
    for devs in ([0], [0, 0], [0, 0, 0]):
        multi = P.dfr_reproject_host(src, w.src_wcs, w.tgt_wcs, w.shape_out, 1, batch=2, devices=devs).numpy()
        assert np.array_equal(np.nan_to_num(multi, nan=-1), np.nan_to_num(one, nan=-1)), devs
        st = P.dfr_last_stats()
        assert st["tiles_fast"] == st1["tiles_fast"] and st["tiles_empty"] == st1["tiles_empty"]
    wts = np.arange(1, 8, dtype=np.float32) / 4
    s1, c1 = P.dfr_stack_host(src, w.src_wcs, w.tgt_wcs, w.shape_out, 1, weights=wts, batch=3)
    s2, c2 = P.dfr_stack_host(src, w.src_wcs, w.tgt_wcs, w.shape_out, 1, weights=wts, batch=3, devices=[0, 0, 0])
    assert torch.equal(c1, c2) and torch.allclose(s1, s2, rtol=2e-6, atol=1e-3)
    so, wo = oracle.stack(w.images, w.src_wcs, w.tgt_wcs, w.shape_out, 1, wts)
    band = np.zeros(w.shape_out, dtype=bool)
    for e in range(7):
        xo, yo = oracle.src_coords(w.tgt_wcs, w.src_wcs[e], *w.shape_out)
        band |= PR.edge_band(xo, yo, *w.images.shape[1:])
    assert np.array_equal(c2.numpy()[~band], wo[~band])
    assert np.abs(s2.numpy() - so)[~band].max() <= PR.VALUE_TOL * max(PR.dyn_range(im) for im in w.images) * wts.sum()
    with pytest.raises(P.DfrError):
        P.dfr_reproject_host(src, w.src_wcs, w.tgt_wcs, w.shape_out, 1, devices=[torch.cuda.device_count()])
    P.dfr_release()                                  # frees the idle pipelines; the next call rebuilds them
    again = P.dfr_reproject_host(src, w.src_wcs, w.tgt_wcs, w.shape_out, 1, batch=4).numpy()
    assert np.array_equal(np.nan_to_num(again, nan=-1), np.nan_to_num(one, nan=-1))


def test_two_devices_from_one_thread(P):
    """The library's per-call state (events, mapped counters, scratch pool) is keyed by device: a
    thread that calls on cuda:0 and then on cuda:1 must get the same results on both."""
    if torch.cuda.device_count() < 2:
        pytest.skip("needs two CUDA devices")
    w = S.config0()
    outs = []
    for dev in (0, 1, 0):
        src = torch.from_numpy(w.images).to(f"cuda:{dev}")
        outs.append(P.dfr_reproject(src, w.src_wcs, w.tgt_wcs, w.shape_out, 1).cpu())
        with torch.cuda.device(dev):
            assert P.dfr_last_stats()["tiles_fast"] == 64
    assert torch.equal(torch.nan_to_num(outs[0]), torch.nan_to_num(outs[1]))
    assert torch.equal(torch.nan_to_num(outs[0]), torch.nan_to_num(outs[2]))
    src = torch.from_numpy(w.images).pin_memory()
    a = P.dfr_reproject_host(src, w.src_wcs, w.tgt_wcs, w.shape_out, 1, devices=[0, 1])
    assert torch.equal(torch.nan_to_num(a), torch.nan_to_num(outs[0]))


def test_many_exposures_call_does_not_block_the_host(P):
    """include/dfr.h promises 'return after enqueue'. The per-call constants (984 B per exposure)
    are staged through pinned memory, so a 128-exposure call (> 64 KB of constants) must return
    while an earlier kernel on the same stream is still running (a pageable cudaMemcpyAsync of
    that size would wait for it)."""
    import time
    n = 128
    rng = np.random.default_rng(3)
    img = S.make_image(64, 64, 5, rng)
    srcs = [S.make_wcs(64, 64, 150.0 + 1e-4 * k, 2.0, 0.1 * k, S.PIXSCALE) for k in range(n)]
    tgt = S.make_wcs(64, 64, 150.0, 2.0, 0.0, S.PIXSCALE)
    d = torch.from_numpy(np.repeat(img[None], n, 0)).cuda()
    out = torch.empty((n, 64, 64), dtype=torch.float32, device="cuda")
    P.dfr_reproject(d, srcs, tgt, (64, 64), 1, out=out)          # warm: pools, staging ring
    torch.cuda.synchronize()
    ws, tw = P.pack_wcs_array(srcs), P.pack_wcs(tgt)
    torch.cuda._sleep(int(4e8))                                  # ~0.2 s of GPU time on the current stream
    t0 = time.perf_counter()
    P.dfr_reproject(d, ws, tw, (64, 64), 1, out=out)
    dt = time.perf_counter() - t0
    still_running = not torch.cuda.current_stream().query()
    torch.cuda.synchronize()
    assert still_running and dt < 0.05, (still_running, dt)


def test_nearest_ties_round_half_even_on_both_paths(P):
    """Reading G8: nearest neighbour rounds half to even. A pure half-pixel CRPIX shift (the
    paper's demo offset, without its rotation) puts EVERY source coordinate on an
    exact tie x = k + 0.5; the tiled path (which rounds a tile-relative coordinate) must pick
    the pixel the oracle's rint picks on the exact half-integer — no tie band excluded. (The
    fp64 per-pixel path carries ~1e-10 px of rounding noise around the tie, so it may pick
    either neighbour: it is only required to pick one of the two.)"""
    rng = np.random.default_rng(8)
    img = S.make_image(96, 128, 20, rng)
    src = S.make_wcs(128, 96, 150.0, 2.0, 0.0, S.PIXSCALE)
    for sx, sy in ((0.5, 0.0), (0.0, 0.5), (0.5, 0.5), (3.5, -2.5)):
        tgt = src.copy()
        tgt.crpix = (src.crpix[0] + sx, src.crpix[1] + sy)
        d = torch.from_numpy(img[None]).cuda()
        a = P.dfr_reproject(d, [src], tgt, None, 0, path=P.PATH_AUTO).cpu().numpy()[0]
        assert P.dfr_last_stats()["tiles_fast"] > 0
        x = P.dfr_reproject(d, [src], tgt, None, 0, path=P.PATH_EXACT).cpu().numpy()[0]
        xo, yo = oracle.src_coords(tgt, src, 96, 128)
        exact_tie = (np.abs(xo - np.floor(xo) - 0.5) < 1e-5) | (np.abs(yo - np.floor(yo) - 0.5) < 1e-5)
        assert exact_tie.mean() > 0.9                     # the geometry really sits on the ties
        ref = oracle.interp(img, np.round(xo * 2).ravel() / 2, np.round(yo * 2).ravel() / 2, 0).reshape(96, 128)
        inside = ~PR.edge_band(np.round(xo * 2) / 2, np.round(yo * 2) / 2, 96, 128)
        assert np.array_equal(np.nan_to_num(a, nan=-1)[inside], np.nan_to_num(ref, nan=-1)[inside].astype(np.float32)), (sx, sy)
        lo = oracle.interp(img, np.floor(xo).ravel(), np.floor(yo).ravel(), 0).reshape(96, 128)
        hi = oracle.interp(img, np.ceil(xo - 1e-6).ravel(), np.ceil(yo - 1e-6).ravel(), 0).reshape(96, 128)
        mixed1 = oracle.interp(img, np.floor(xo).ravel(), np.ceil(yo - 1e-6).ravel(), 0).reshape(96, 128)
        mixed2 = oracle.interp(img, np.ceil(xo - 1e-6).ravel(), np.floor(yo).ravel(), 0).reshape(96, 128)
        okx = (x == lo) | (x == hi) | (x == mixed1) | (x == mixed2) | np.isnan(x)
        assert okx[inside].all(), (sx, sy)


def test_fit_acceptance_adversarial_sweep(P):
    """The tiled path accepts a cubic fit after comparing it with the exact map at check points
    (16 per 128x128 super-tile, 9 per 32x32 tile on the refit level; FIT_TOL = 2e-6 px): a spot
    check, not a bound. This seeded sweep searches for a
    geometry where an ACCEPTED tile is wrong anyway: SIP orders 2-9 on either side with
    amplitudes 1e-6 ... 1e-2 (up to tens of pixels of distortion), scale ratios 0.5-2, any
    rotation, tangent points up to degrees apart, declinations up to the poles. Everywhere
    |tiled - exact| must stay below 1e-5 px (design for <= 1e-5 px; the
    north_star tolerance is 1e-4 px), whatever mix of FAST / EXACT tiles the setup kernel chose."""
    rng = np.random.default_rng(777)
    worst, worst_case, n_fast, n_exact = 0.0, None, 0, 0
    for case in range(240):
        n_src = int(rng.integers(160, 420)) // 4 * 4
        n_out = int(rng.integers(160, 420))
        dec0 = [rng.uniform(-60, 60), rng.uniform(80, 89.9), -rng.uniform(80, 89.9), 89.999][case % 4]
        ra0 = rng.uniform(0, 360)
        sep = 10 ** rng.uniform(-4, 0.5) * S.PIXSCALE * 200            # tangent points 0.02 ... 600 px apart
        pa = rng.uniform(0, 2 * np.pi)
        ratio = 2 ** rng.uniform(-1, 1)
        src = S.make_wcs(n_src, n_src, ra0, dec0, rng.uniform(0, 360), S.PIXSCALE)
        dra = sep * np.sin(pa) / max(np.cos(np.radians(dec0)), 1e-3)
        tgt = S.make_wcs(n_out, n_out, ra0 + dra, min(max(dec0 + sep * np.cos(pa), -89.9999), 89.9999),
                         rng.uniform(0, 360), S.PIXSCALE * ratio)
        if case % 5:
            S.add_sip(src, int(rng.integers(2, 10)), n_src / 2.0, rng, amp=10 ** rng.uniform(-6, -2))
        if case % 3:
            S.add_sip(tgt, int(rng.integers(2, 10)), n_out / 2.0, rng, amp=10 ** rng.uniform(-6, -2))
        xa, ya = P.dfr_src_coords([src], tgt, (n_src, n_src), (n_out, n_out), 1, path=P.PATH_AUTO)
        img = torch.zeros((1, n_src, n_src), dtype=torch.float32, device="cuda")
        P.dfr_reproject(img, [src], tgt, (n_out, n_out), 1)
        st = P.dfr_last_stats()
        xe, ye = P.dfr_src_coords([src], tgt, (n_src, n_src), (n_out, n_out), 1, path=P.PATH_EXACT)
        assert torch.equal(torch.isfinite(xa), torch.isfinite(xe)), case
        # only coordinates that can matter: within 4 px of the source image
        near = torch.isfinite(xe) & (xe > -4) & (xe < n_src + 3) & (ye > -4) & (ye < n_src + 3)
        if bool(near.any()):
            d = float(torch.maximum((xa - xe).abs()[near].max(), (ya - ye).abs()[near].max()))
            if d > worst:
                worst, worst_case = d, (case, st, dec0, ratio, src.a_order, tgt.a_order)
        n_fast += st["tiles_fast"]
        n_exact += st["tiles_exact"]
    print("fit sweep: worst |tiled - exact| =", worst, "px at", worst_case, "; tiles fast / exact:", n_fast, n_exact)
    assert n_fast > 5000 and worst <= 1e-5


@pytest.mark.parametrize("path", list(PATHS))
def test_exact_inverse_sip_on_device(P, path):
    """§8(f) f4, device side: a source WCS with A/B but no AP/BP, ap_order = bp_order =
    DFR_SIP_INVERSE_EXACT: the library inverts the forward distortion itself. Oracle = the literal
    chain without inverse SIP (O6-O8) followed by the DEFINITION of the inverse distortion,
    oracle/sip_inverse.py: newton_inverse (pin I1). A ~9 px distortion: a fitted order-3 AP/BP
    is 0.1 px off here (pin I3), the exact inverse must meet the 1e-4 px bar."""
    from oracle import sip_inverse as SI
    src, tgt = S.stress_sip_pair()
    bare = src.copy()
    bare.ap_order = bare.bp_order = 0
    bare.ap, bare.bp = np.zeros((10, 10)), np.zeros((10, 10))
    exact = bare.copy()
    exact.ap_order = exact.bp_order = -1
    n = 1024
    rng = np.random.default_rng(44)
    img = S.make_image(n, n, 400, rng)
    xo, yo = oracle.src_coords(tgt, bare, n, n)              # U + crpix - 1: no inverse distortion applied
    u, v = SI.newton_inverse(bare, xo - (bare.crpix[0] - 1.0), yo - (bare.crpix[1] - 1.0))
    xo, yo = u + (bare.crpix[0] - 1.0), v + (bare.crpix[1] - 1.0)
    xg, yg = P.dfr_src_coords([exact], tgt, (n, n), (n, n), 1, path=PATHS[path])
    st = PR.check_coords(xg[0].cpu().numpy(), yg[0].cpu().numpy(), xo, yo, bare)
    xb, _ = P.dfr_src_coords([bare], tgt, (n, n), (n, n), 1, path=PATHS[path])
    assert float((xb[0] - xg[0]).abs().max()) > 1.0           # the inverse distortion is pixels, not noise
    for order in (0, 1, 3):
        out = P.dfr_reproject(torch.from_numpy(img[None]).cuda(), [exact], tgt, (n, n), order, path=PATHS[path])
        ref = oracle.interp(img, xo.ravel(), yo.ravel(), order).reshape(n, n).astype(np.float32)
        PR.check_image(out[0].cpu().numpy(), ref, xo, yo, img, order)
    if path == "auto":
        assert P.dfr_last_stats()["tiles_fast"] > 900
    # the sky entry point inverts as well: world2pix(pix2world(x)) = x to 1e-9 px without any AP/BP
    x = torch.from_numpy(rng.uniform(0, n - 1, 5000)).cuda()
    y = torch.from_numpy(rng.uniform(0, n - 1, 5000)).cuda()
    ra, dec = P.dfr_pix2world(exact, x, y)
    xr, yr = P.dfr_world2pix(exact, ra, dec)
    assert float((xr - x).abs().max()) < 1e-7 and float((yr - y).abs().max()) < 1e-7
    print("exact inverse", path, st)


@pytest.mark.parametrize("path", list(PATHS))
def test_exact_inverse_that_cannot_converge_gives_nan(P, path):
    """DFR_SIP_INVERSE_EXACT on a distortion whose gradient exceeds 1 (no fixed point to converge
    to): the documented outcome is NaN coordinates, hence NaN pixels — not a hang, not garbage.
    Near CRPIX, where the gradient is small, the solve still converges."""
    n = 256
    src = S.make_wcs(n, n, 150.0, 2.0, 0.0, S.PIXSCALE)
    src.a_order = src.b_order = 2
    src.a[2][0] = 2e-2                       # dA/du = 0.04 u: > 1 beyond 25 px from CRPIX
    src.ap_order = src.bp_order = -1
    tgt = S.make_wcs(n, n, 150.0, 2.0, 0.0, S.PIXSCALE)
    x, y = P.dfr_src_coords([src], tgt, (n, n), (n, n), 1, path=PATHS[path])
    x = x[0].cpu().numpy()
    assert np.isnan(x[:, :60]).all() and np.isnan(x[:, 200:]).all()
    centre = x[120:136, 124:132]
    assert np.isfinite(centre).all()
    out = P.dfr_reproject(torch.ones((1, n, n), device="cuda"), [src], tgt, (n, n), 1, path=PATHS[path])
    assert bool(torch.isnan(out[0, :, :60]).all()) and bool((out[0, 120:136, 124:132] == 1).all())


def test_maximum_frame_size_index_arithmetic(P):
    """Frames at the size limit of the ABI (ny * nx < 2^31 pixels: 46340 x 46340 = 8.6 GB each way):
    every byte offset above 4 GB, every element index near 2^31. The source is a linear ramp built
    on the device, which bilinear interpolation reproduces exactly (pin P10), so the expected value
    of a pixel is the ramp at the ORACLE's source coordinate: 400 000 sampled output pixels
    (including the four corners and the last rows) computed one by one through the oracle's sky
    entry points, plus the NaN mask."""
    n = 46340
    free, _ = torch.cuda.mem_get_info()
    if free < 20 * 2 ** 30:
        pytest.skip("needs 20 GB of free device memory")
    ax, ay, c0 = 0.25, 0.5, 7.0
    src = torch.empty((1, n, n), dtype=torch.float32, device="cuda")
    xs = torch.arange(n, dtype=torch.float32, device="cuda")
    for j0 in range(0, n, 4096):                                   # row blocks: no second full-size temporary
        j1 = min(n, j0 + 4096)
        src[0, j0:j1] = c0 + ax * xs[None, :] + ay * torch.arange(j0, j1, dtype=torch.float32, device="cuda")[:, None]
    sw = S.make_wcs(n, n, 150.0, 2.0, 0.0, S.PIXSCALE)
    tw = S.make_wcs(n, n, 150.02, 1.99, 0.4, S.PIXSCALE)          # ~25 px shift, 0.4 deg: NaN wedges on all sides
    out = P.dfr_reproject(src, [sw], tw, (n, n), 1)
    torch.cuda.synchronize()
    st = P.dfr_last_stats()
    assert st["tiles_fast"] + st["tiles_exact"] + st["tiles_empty"] == ((n + 31) // 32) ** 2
    rng = np.random.default_rng(4634)
    ii = np.concatenate([rng.integers(0, n, 399990), [0, n - 1, 0, n - 1, n - 1, n - 2, 1, n - 1, n // 2, n - 1]]).astype(np.float64)
    jj = np.concatenate([rng.integers(0, n, 399990), [0, 0, n - 1, n - 1, n - 2, n - 1, n - 1, 1, n - 1, n // 2]]).astype(np.float64)
    ra, dec = oracle.pix2world(tw, ii, jj)
    xo, yo = oracle.world2pix(sw, ra, dec)
    got = out[0][torch.from_numpy(jj.astype(np.int64)).cuda(), torch.from_numpy(ii.astype(np.int64)).cuda()].cpu().numpy()
    inside = (xo >= -0.5) & (xo < n - 0.5) & (yo >= -0.5) & (yo < n - 0.5)
    band = PR.edge_band(xo, yo, n, n)
    assert np.array_equal(np.isnan(got)[~band], ~inside[~band])
    # edge replication: the ramp is evaluated at the coordinate clamped to the pixel-centre hull
    want = c0 + ax * np.clip(xo, 0, n - 1) + ay * np.clip(yo, 0, n - 1)
    ok = inside & ~band
    dr = ax * (n - 1) + ay * (n - 1)
    err = np.abs(got[ok] - want[ok])
    # 1e-5 x DR = 0.35; what is actually expected: coordinate error (<= 1e-4 px) x slope + float32 rounding of the ramp (ulp 0.004)
    assert err.max() <= 0.01, err.max()
    assert 0.9 < ok.mean() < 1.0 and err.max() <= PR.VALUE_TOL * dr
    del out, src


def test_more_exposures_than_one_grid_dimension(P):
    """n > 65535 exposures in one call: the exposure index no longer fits grid.y / grid.z, so the
    launchers cut the batch; every exposure must still get its own WCS and its own image."""
    n, npx = 66000, 8
    rng = np.random.default_rng(66)
    imgs = rng.normal(100.0, 5.0, (n, npx, npx)).astype(np.float32)
    base = S.make_wcs(npx, npx, 150.0, 2.0, 0.0, S.PIXSCALE)
    tgt = S.make_wcs(npx, npx, 150.0, 2.0, 0.0, S.PIXSCALE)
    ws = (P.DfrWCS * n)()
    proto = P.pack_wcs(base)
    shifts = rng.integers(-2, 3, (n, 2))
    for k in range(n):
        ws[k] = proto
        ws[k].crpix[0] = base.crpix[0] + float(shifts[k, 0])
        ws[k].crpix[1] = base.crpix[1] + float(shifts[k, 1])
    src = torch.from_numpy(imgs).cuda()
    out = P.dfr_reproject(src, ws, tgt, (npx, npx), 0).cpu().numpy()
    for k in (0, 1, 65534, 65535, 65536, 65999):
        dx, dy = int(shifts[k, 0]), int(shifts[k, 1])              # source pixel = target pixel + shift
        want = np.full((npx, npx), np.nan, dtype=np.float32)
        for j in range(npx):
            for i in range(npx):
                if 0 <= i + dx < npx and 0 <= j + dy < npx:
                    want[j, i] = imgs[k, j + dy, i + dx]
        assert np.array_equal(np.nan_to_num(out[k], nan=-1), np.nan_to_num(want, nan=-1)), k
    s, c = P.dfr_reproject_stack(src, ws, tgt, (npx, npx), 0)
    valid = ~np.isnan(out)
    assert np.array_equal(c.cpu().numpy(), valid.sum(0).astype(np.float32))
    assert np.allclose(s.cpu().numpy(), np.where(valid, out, 0).astype(np.float64).sum(0), rtol=1e-4)
