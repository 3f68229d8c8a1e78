"""Pins P1-P5, P14-P16: the oracle's coordinate chain
(oracle/orc.c, §3.2) against what the paper and the mathematics fix.
CPU only. Nothing here touches the CUDA path."""
import math

import numpy as np
import pytest

import dfr_synth as S
import oracle
from oracle import mp_chain
from tests.conftest import read_golden

D2R = math.pi / 180.0


def rand_wcs(rng, dec0=None, ra0=None, n=512):
    rot = rng.uniform(-180, 180)
    scale = S.PIXSCALE * rng.uniform(0.5, 20.0)
    w = S.make_wcs(n, n, rng.uniform(0, 360) if ra0 is None else ra0,
                   rng.uniform(-85, 85) if dec0 is None else dec0, rot, scale)
    # general (skewed) CD, not just a rotation
    cd = np.array(w.cd).reshape(2, 2) @ np.array([[1.0, rng.uniform(-0.05, 0.05)],
                                                   [rng.uniform(-0.05, 0.05), rng.uniform(0.9, 1.1)]])
    w.cd = tuple(cd.ravel())
    w.crpix = (rng.uniform(1, n), rng.uniform(1, n))
    return w


def angdiff(a, b):
    return np.abs((np.asarray(a) - np.asarray(b) + 180.0) % 360.0 - 180.0)


# ---------------------------------------------------------------- P1
@pytest.mark.parametrize("dec0", [2.0, -35.5, 89.9, -90.0, 90.0, 0.0])
def test_p1_crpix_maps_to_crval(dec0):
    rng = np.random.default_rng(11)
    w = rand_wcs(rng, dec0=dec0, ra0=359.99999)
    S.add_sip(w, 3, 256.0, rng, amp=1e-3)
    ra, dec = oracle.pix2world(w, [w.crpix[0] - 1], [w.crpix[1] - 1])
    assert abs(dec[0] - dec0) < 1e-12
    if abs(dec0) < 90:
        assert angdiff(ra[0], 359.99999) < 1e-12


# ---------------------------------------------------------------- P2
def triad(ra_deg, dec_deg):
    a, d = ra_deg * D2R, dec_deg * D2R
    e = np.array([-math.sin(a), math.cos(a), 0.0])
    n = np.array([-math.sin(d) * math.cos(a), -math.sin(d) * math.sin(a), math.cos(d)])
    k = np.array([math.cos(d) * math.cos(a), math.cos(d) * math.sin(a), math.sin(d)])
    return e, n, k


@pytest.mark.parametrize("dec0,ra0", [(2.0, 150.0), (89.999, 10.0), (-90.0, 0.0), (90.0, 200.0),
                                      (45.0, 0.0001), (-60.0, 359.9999)])
def test_p2_literal_equals_closed_form_and_homography(dec0, ra0):
    rng = np.random.default_rng(int(abs(dec0) * 100 + ra0))
    t = rand_wcs(rng, dec0=dec0, ra0=ra0)
    x = rng.uniform(-50, 600, 400)
    y = rng.uniform(-50, 600, 400)
    # form (i): the oracle's literal chain
    ra, dec = oracle.pix2world(t, x, y)
    # form (ii): textbook gnomonic on intermediate world coordinates
    cd = np.array(t.cd).reshape(2, 2)
    uv = np.stack([x - (t.crpix[0] - 1), y - (t.crpix[1] - 1)])
    up, vp = cd @ uv
    ra2, dec2 = oracle.closed_iwc2sky(t.crval, up, vp)
    # asin near |dec| = 90 amplifies rounding by 1/cos(dec) (the literal form's own
    # conditioning), hence the second term
    assert np.all(np.abs(dec - dec2) < 1e-12 + 3e-14 / np.maximum(np.cos(dec * D2R), 1e-9))
    far = np.abs(dec) < 89.999
    assert np.max(angdiff(ra[far], ra2[far]) * np.cos(dec[far] * D2R)) < 1e-12
    # inverse: world2pix (literal) vs closed form + CD^-1
    s = rand_wcs(rng, dec0=float(np.clip(dec0 + rng.uniform(-0.3, 0.3), -90, 90)),
                 ra0=ra0 + rng.uniform(-0.2, 0.2))
    xs, ys = oracle.world2pix(s, ra, dec)
    ups, vps = oracle.closed_sky2iwc(s.crval, ra, dec)
    uvs = np.linalg.solve(np.array(s.cd).reshape(2, 2), np.stack([ups, vps]))
    ok = np.isfinite(xs)
    assert ok.all() == np.isfinite(ups).all()
    assert np.max(np.abs(uvs[0][ok] + s.crpix[0] - 1 - xs[ok])) < 1e-8
    assert np.max(np.abs(uvs[1][ok] + s.crpix[1] - 1 - ys[ok])) < 1e-8
    # form (iii): trig-free homography p = k_t + xi e_t + eta n_t
    et, nt, kt = triad(*t.crval)
    es, ns, ks = triad(*s.crval)
    p = kt[:, None] + (up * D2R)[None, :] * et[:, None] + (vp * D2R)[None, :] * nt[:, None]
    xi_s = (es @ p) / (ks @ p) / D2R
    eta_s = (ns @ p) / (ks @ p) / D2R
    uvh = np.linalg.solve(np.array(s.cd).reshape(2, 2), np.stack([xi_s, eta_s]))
    assert np.max(np.abs(uvh[0][ok] + s.crpix[0] - 1 - xs[ok])) < 1e-8
    assert np.max(np.abs(uvh[1][ok] + s.crpix[1] - 1 - ys[ok])) < 1e-8


# ---------------------------------------------------------------- P3
def test_p3_angular_separation_is_atan_r():
    rng = np.random.default_rng(3)
    for _ in range(5):
        w = rand_wcs(rng)
        x = rng.uniform(0, 512, 300)
        y = rng.uniform(0, 512, 300)
        ra, dec = oracle.pix2world(w, x, y)
        cd = np.array(w.cd).reshape(2, 2)
        up, vp = cd @ np.stack([x - (w.crpix[0] - 1), y - (w.crpix[1] - 1)])
        want = np.degrees(np.arctan(np.hypot(up, vp) * D2R))
        d1, d2 = dec * D2R, w.crval[1] * D2R
        dl = (ra - w.crval[0]) * D2R
        hav = np.sin((d1 - d2) / 2) ** 2 + np.cos(d1) * np.cos(d2) * np.sin(dl / 2) ** 2
        got = np.degrees(2 * np.arcsin(np.sqrt(hav)))
        assert np.max(np.abs(got - want)) < 1e-12


# ---------------------------------------------------------------- P4
def test_p4_pole_special_case():
    ra0, dec0, up, vp, ra_w, dec_w = read_golden("p4_pole.txt")[0]
    # CD = identity deg/px, crpix = 1 so that (x, y) = (u', v')
    w = S.WCS(crpix=(1.0, 1.0), crval=(ra0, dec0), cd=(1.0, 0.0, 0.0, 1.0))
    ra, dec = oracle.pix2world(w, [up], [vp])
    assert abs(ra[0] - ra_w) < 1e-11 and abs(dec[0] - dec_w) < 1e-11
    # the closed forms written in the fixture header
    assert abs(dec_w - math.degrees(math.atan2(1.0, 0.5 * D2R))) < 1e-12
    assert abs(ra_w - (10 + math.degrees(math.atan2(0.3, 0.4)))) < 1e-12
    # cardinal directions (sign/orientation pin): +v' is north, +u' is east
    w2 = S.WCS(crpix=(1.0, 1.0), crval=(100.0, 20.0), cd=(1.0, 0.0, 0.0, 1.0))
    ra, dec = oracle.pix2world(w2, [0.0, 0.01], [0.01, 0.0])
    assert abs(ra[0] - 100.0) < 1e-12 and abs(dec[0] - 20.01) < 1e-9
    assert ra[1] > 100.0 and abs((ra[1] - 100.0) * math.cos(20 * D2R) - 0.01) < 1e-6


# ---------------------------------------------------------------- P5
def test_p5_roundtrip_no_sip_and_fitted_sip():
    rng = np.random.default_rng(5)
    for _ in range(4):
        w = rand_wcs(rng)
        x = rng.uniform(0, 511, 500)
        y = rng.uniform(0, 511, 500)
        ra, dec = oracle.pix2world(w, x, y)
        xb, yb = oracle.world2pix(w, ra, dec)
        # theta = asin(s) is ill-conditioned near the tangent point:
        # 1 - s = r^2/2 is known to ~1e-16 absolute, so r carries
        # ~1e-16 / (r_px * scale_rad^2) px of rounding (DESIGN.md §3 "oracle conditioning")
        scale_rad = math.sqrt(abs(w.cd[0] * w.cd[3] - w.cd[1] * w.cd[2])) * D2R
        r_px = np.hypot(x - (w.crpix[0] - 1), y - (w.crpix[1] - 1))
        assert np.all(np.hypot(xb - x, yb - y) < 1e-9 + 4e-16 / (r_px * scale_rad ** 2))
    w = S.add_sip(S.make_wcs(2048, 2048, 150.0, 2.0, 0.0, S.PIXSCALE), 3, 1024.0, rng)
    resid = S.sip_roundtrip_residual(w, 1024.0, rng, 20000)
    assert resid < 1e-3                       # BASELINE.json acceptance
    x = rng.uniform(0, 2047, 2000)
    y = rng.uniform(0, 2047, 2000)
    ra, dec = oracle.pix2world(w, x, y)
    xb, yb = oracle.world2pix(w, ra, dec)
    scale_rad = S.PIXSCALE * D2R
    r_px = np.hypot(x - 1023.5, y - 1023.5)
    assert np.all(np.hypot(xb - x, yb - y) < resid + 1e-9 + 4e-16 / (r_px * scale_rad ** 2))


def test_world2pix_far_side_is_nan():
    w = S.make_wcs(64, 64, 10.0, 20.0, 0.0, S.PIXSCALE)
    x, y = oracle.world2pix(w, [190.0, 10.0], [-20.0, -75.0])     # antipode; >90 deg away
    assert np.isnan(x).all() and np.isnan(y).all()
    x, y = oracle.world2pix(w, [10.0 + 360.0], [20.0])            # periodic in RA (G11)
    assert abs(x[0] - 31.5) < 1e-9 and abs(y[0] - 31.5) < 1e-9


# ---------------------------------------------------------------- P14
def test_p14_sip_polynomial_index_order():
    """Every (p, q) gets a distinct strong coefficient; the inverse polynomial is
    isolated as x_sip - x_nosip and compared with a 50-digit power sum."""
    rng = np.random.default_rng(14)
    base = S.make_wcs(1024, 1024, 80.0, -30.0, 12.0, S.PIXSCALE)
    for order in (2, 3, 5, 9):
        w = base.copy()
        half = 512.0
        for p in range(order + 1):
            for q in range(order + 1 - p):
                w.ap[p, q] = rng.normal(0, 3e-3 * half ** (1 - p - q)) * (1 + p + 3 * q)
                w.bp[p, q] = rng.normal(0, 3e-3 * half ** (1 - p - q)) * (1 + 2 * p + q)
        w.ap_order, w.bp_order = order, order - 1 if order > 2 else order
        ra, dec = oracle.pix2world(base, rng.uniform(0, 1023, 50), rng.uniform(0, 1023, 50))
        x0, y0 = oracle.world2pix(base, ra, dec)
        x1, y1 = oracle.world2pix(w, ra, dec)
        for k in range(0, 50, 7):
            u, v = x0[k] - (base.crpix[0] - 1), y0[k] - (base.crpix[1] - 1)
            fa = float(mp_chain.sip_value(w.ap, w.ap_order, u, v))
            fb = float(mp_chain.sip_value(w.bp, w.bp_order, u, v))
            assert abs((x1[k] - x0[k]) - fa) < 1e-9
            assert abs((y1[k] - y0[k]) - fb) < 1e-9
    # forward polynomial, the hand-computed value quoted in p15_sip_example.txt
    a = np.zeros((10, 10))
    a[2, 0], a[1, 1], a[0, 3] = 2e-6, -1e-6, 3e-10
    u = v = -1023.5
    hand = 2e-6 * u * u - 1e-6 * u * v + 3e-10 * v ** 3
    assert abs(hand - 0.7259013316375) < 1e-12
    assert abs(float(mp_chain.sip_value(a, 3, u, v)) - 0.7259013316375) < 1e-12


# ---------------------------------------------------------------- P15
def cfg0_pair():
    w0 = S.config0()
    return w0.src_wcs[0], w0.tgt_wcs


def sip_example_wcs():
    w = S.make_wcs(2048, 2048, 210.25, -35.5, 0.5, S.PIXSCALE)
    w.a[2, 0], w.a[1, 1], w.a[0, 3] = 2e-6, -1e-6, 3e-10
    w.b[0, 2], w.b[2, 1] = -1.5e-6, 2e-10
    w.a_order = w.b_order = 3
    return w


def test_p15_golden_config0_pair():
    src, tgt = cfg0_pair()
    assert tgt.crpix == pytest.approx((131.9, 125.8), abs=1e-12)
    for tx, ty, ra_w, dec_w, sx_w, sy_w in read_golden("p15_config0_pair.txt"):
        ra, dec = oracle.pix2world(tgt, [tx], [ty])
        assert angdiff(ra[0], ra_w) < 1e-11 and abs(dec[0] - dec_w) < 1e-11
        mra, mdec = mp_chain.pix2world_deg(tgt, tx, ty)
        assert abs(float(mra) - ra_w) < 1e-11 and abs(float(mdec) - dec_w) < 1e-11
        if sx_w is not None:
            sx, sy = oracle.world2pix(src, ra, dec)
            # double chain: 1e-8 px (pin P16's bound; asin conditioning), mp chain: 1e-10
            assert abs(sx[0] - sx_w) < 1e-8 and abs(sy[0] - sy_w) < 1e-8
            mx, my = mp_chain.src_coord(tgt, src, tx, ty)
            assert abs(float(mx) - sx_w) < 1e-10 and abs(float(my) - sy_w) < 1e-10
    # and through the whole-grid entry point
    X, Y = oracle.src_coords(tgt, src, 256, 256)
    assert abs(X[37, 100] - 97.3673663940743) < 1e-8 and abs(Y[37, 100] - 39.433693208066) < 1e-8
    assert abs(X[255, 0] + 4.53121065098831) < 1e-8 and abs(Y[255, 0] - 256.552738886218) < 1e-8


def test_p15_golden_sip_example():
    w = sip_example_wcs()
    for x, y, ra_w, dec_w in read_golden("p15_sip_example.txt"):
        ra, dec = oracle.pix2world(w, [x], [y])
        assert angdiff(ra[0], ra_w) < 1e-11 and abs(dec[0] - dec_w) < 1e-11
        mra, mdec = mp_chain.pix2world_deg(w, x, y)
        assert abs(float(mra) - ra_w) < 1e-11 and abs(float(mdec) - dec_w) < 1e-11


# ---------------------------------------------------------------- P16
def test_p16_double_vs_50_digits_on_config3_geometry():
    w = S.config3(scale_down=8)          # images unused here; WCS built at reduced size ...
    # ... but the rounding test wants the full-size geometry: rebuild the WCS only
    rng = np.random.default_rng(3)
    rng.normal(100.0, 5.0, (8, 8))       # (not the config's stream; any SIP4 pair of that size)
    src = S.add_sip(S.make_wcs(6248, 4176, 150.0, 2.0, 0.0, S.PIXSCALE), 4, 3124.0, rng)
    tgt = S.add_sip(S.make_wcs(6400, 4400, 150.03, 2.03, 2.0, S.PIXSCALE), 4, 3200.0, rng)
    pts = [(0, 0), (6399, 0), (0, 4399), (6399, 4399), (3200, 2200), (17, 4001), (5555, 123)]
    rng2 = np.random.default_rng(16)
    pts += [(int(a), int(b)) for a, b in zip(rng2.integers(0, 6400, 40), rng2.integers(0, 4400, 40))]
    xs = np.array([p[0] for p in pts], dtype=float)
    ys = np.array([p[1] for p in pts], dtype=float)
    ra, dec = oracle.pix2world(tgt, xs, ys)
    X, Y = oracle.world2pix(src, ra, dec)     # goes through degrees: a slightly longer chain
    worst = 0.0
    for k, (i, j) in enumerate(pts):
        mx, my = mp_chain.src_coord(tgt, src, i, j)
        worst = max(worst, abs(float(mx) - X[k]), abs(float(my) - Y[k]))
    assert worst < 1e-8
    assert w.shape_out == (550, 800)


def test_pc_cdelt_composition():
    cd = oracle.cd_from_pc_cdelt([0.6, -0.8, 0.8, 0.6], [-2.0, 3.0])
    assert np.allclose(cd, [-1.2, 1.6, 2.4, 1.8], rtol=0, atol=1e-15)
