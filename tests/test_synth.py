"""The seeded input generators (dfr_synth) produce what BASELINE.json's configs and
DESIGN.md §5 say: shapes, seeds, SIP round-trip acceptance, expected NaN fractions."""
import numpy as np

import dfr_synth as S
import oracle


def test_config0_recipe():
    w = S.config0()
    assert w.images.shape == (1, 256, 256) and w.images.dtype == np.float32
    assert w.src_wcs[0].crpix == (128.5, 128.5) and w.src_wcs[0].a_order == 0
    assert abs(w.tgt_wcs.crpix[0] - 131.9) < 1e-12 and abs(w.tgt_wcs.crpix[1] - 125.8) < 1e-12
    again = S.config0()
    assert np.array_equal(w.images, again.images)               # seeded
    bg = np.median(w.images)
    assert 99 < bg < 101 and 400 < w.images.max() < 5200
    out = oracle.reproject(w.images, w.src_wcs, w.tgt_wcs, w.shape_out, 1)
    assert abs(np.isnan(out).mean() - 0.024) < 0.004              # 2.4 %


def test_sip_draw_scale_and_inverse_fit():
    rng = np.random.default_rng(1)
    w = S.add_sip(S.make_wcs(2048, 2048, 150.0, 2.0, 0.0, S.PIXSCALE), 3, 1024.0, rng)
    assert w.a_order == w.bp_order == 3
    assert w.a[0, 0] == 0 and w.a[1, 0] == 0 and w.a[0, 1] == 0   # only 2 <= p+q <= 3 drawn
    assert w.a[2, 0] != 0 and w.b[0, 3] != 0 and w.a[2, 2] == 0
    assert abs(w.a[2, 0]) < 6e-6 / 1024 and abs(w.a[3, 0]) < 6e-6 / 1024 ** 2
    assert S.sip_roundtrip_residual(w, 1024.0, np.random.default_rng(2)) < 1e-3
    strong_s, strong_t = S.stress_sip_pair()
    # an order-3 inverse cannot undo a ~9 px order-3 distortion to 1e-3 px; the stress pair is
    # for coordinate parity only (both sides apply the same AP/BP), so only sanity-check it
    assert S.sip_roundtrip_residual(strong_s, 512.0, np.random.default_rng(3)) < 0.1
    # the stress pair really has pixel-scale distortion
    u = np.array([500.0]); v = np.array([-500.0])
    assert abs(S._poly_eval(strong_s.a, 3, u, v)[0]) + abs(S._poly_eval(strong_t.a, 3, u, v)[0]) > 0.3


def test_jittered_exposure_wcs_independent_of_image_flag():
    _, w1 = S.jittered_exposure([2, 5], 64, 64, 10)
    _, w2 = S.jittered_exposure([2, 5], 64, 64, 10, with_image=False)
    assert w1.crval == w2.crval and w1.cd == w2.cd and np.array_equal(w1.ap, w2.ap)
    _, w3 = S.jittered_exposure([4, 5], 64, 64, 10, fast_image=True)
    _, w4 = S.jittered_exposure([4, 5], 64, 64, 10, with_image=False, fast_image=True)
    assert w3.crval == w4.crval and np.array_equal(w3.b, w4.b)
    assert abs(w1.crval[0] - 150.0) <= 5 / 60 and abs(w1.crval[1] - 2.0) <= 5 / 60


def test_config3_reduced_nan_fraction():
    w = S.config3(scale_down=8)
    assert w.images.shape == (1, 522, 781) and w.shape_out == (550, 800) and w.orders == (0, 1, 3)
    X, Y = oracle.src_coords(w.tgt_wcs, w.src_wcs[0], *w.shape_out)
    inside = (X >= -0.5) & (X < 781 - 0.5) & (Y >= -0.5) & (Y < 522 - 0.5)
    assert abs((1 - inside.mean()) - 0.075) < 0.02               # "about 8 %" (BASELINE.json)
