"""FITS-keyword parsing of paper_2505_03932_b200.api (host only) and, -m gpu, the paper's
user-facing call against the oracle."""
import math

import numpy as np
import pytest

import dfr_synth as S
import oracle


def header_of(w, nx, ny, inverse=True, use_pc=False):
    h = {"NAXIS1": nx, "NAXIS2": ny, "CTYPE1": "RA---TAN-SIP" if w.a_order else "RA---TAN",
         "CTYPE2": "DEC--TAN-SIP" if w.a_order else "DEC--TAN",
         "CRPIX1": w.crpix[0], "CRPIX2": w.crpix[1], "CRVAL1": w.crval[0], "CRVAL2": w.crval[1]}
    if use_pc:
        cdelt = (-abs(w.cd[0]) * 1.5, abs(w.cd[3]) * 0.75)
        h.update({"CDELT1": cdelt[0], "CDELT2": cdelt[1], "PC1_1": w.cd[0] / cdelt[0], "PC1_2": w.cd[1] / cdelt[0],
                  "PC2_1": w.cd[2] / cdelt[1], "PC2_2": w.cd[3] / cdelt[1]})
    else:
        h.update({"CD1_1": w.cd[0], "CD1_2": w.cd[1], "CD2_1": w.cd[2], "CD2_2": w.cd[3]})
    keys = [("A", w.a, w.a_order), ("B", w.b, w.b_order)]
    if inverse:
        keys += [("AP", w.ap, w.ap_order), ("BP", w.bp, w.bp_order)]
    for key, arr, order in keys:
        if order:
            h[f"{key}_ORDER"] = order
            for p in range(order + 1):
                for q in range(order + 1 - p):
                    if arr[p][q] != 0.0:
                        h[f"{key}_{p}_{q}"] = float(arr[p][q])
    return h


@pytest.fixture(scope="module")
def A():
    from paper_2505_03932_b200 import api, build
    build.build()
    return api


def test_header_round_trip(A):
    rng = np.random.default_rng(3)
    w = S.add_sip(S.make_wcs(300, 200, 210.25, -35.5, 12.0, S.PIXSCALE), 4, 150.0, rng, amp=1e-4)
    for use_pc in (False, True):
        s = A.wcs_from_header(header_of(w, 300, 200, use_pc=use_pc))
        assert tuple(s.crpix) == tuple(w.crpix) and tuple(s.crval) == tuple(w.crval)
        assert np.allclose(list(s.cd), list(w.cd), rtol=1e-15, atol=0)
        assert (s.a_order, s.b_order, s.ap_order, s.bp_order) == (4, 4, 4, 4)
        for name in ("a", "b", "ap", "bp"):
            assert np.array_equal(np.array(getattr(s, name)[:]).reshape(10, 10), getattr(w, name))


def test_header_crota_and_defaults(A):
    h = {"CRPIX1": 10.0, "CRPIX2": 20.0, "CRVAL1": 5.0, "CRVAL2": -5.0, "CDELT1": -0.001, "CDELT2": 0.001, "CROTA2": 30.0}
    s = A.wcs_from_header(h)
    c, n = math.cos(math.radians(30)), math.sin(math.radians(30))
    # CD = [[cdelt1 cos, -cdelt2 sin], [cdelt1 sin, cdelt2 cos]] (AIPS CROTA2 convention)
    assert np.allclose(list(s.cd), [-0.001 * c, -0.001 * n, -0.001 * n, 0.001 * c], rtol=1e-14, atol=0)
    assert (s.a_order, s.ap_order) == (0, 0)
    with pytest.raises(A.HeaderError):
        A.wcs_from_header({**h, "CTYPE1": "RA---SIN"})
    with pytest.raises(A.HeaderError):
        A.wcs_from_header({**h, "LONPOLE": 90.0})
    with pytest.raises(A.HeaderError):
        A.wcs_from_header({k: v for k, v in h.items() if k != "CRVAL2"})


def test_missing_inverse_is_fitted(A):
    rng = np.random.default_rng(5)
    w = S.add_sip(S.make_wcs(512, 512, 150.0, 2.0, 0.0, S.PIXSCALE), 3, 256.0, rng, amp=1e-3)
    s = A.wcs_from_header(header_of(w, 512, 512, inverse=False))
    assert s.ap_order == 5 and s.bp_order == 5
    from oracle import sip_inverse as SI
    x, y = rng.uniform(0, 511, 5000), rng.uniform(0, 511, 5000)
    u, v = x - (w.crpix[0] - 1), y - (w.crpix[1] - 1)
    U, V = SI.forward(w, u, v)
    ap = np.array(s.ap[:]).reshape(10, 10)
    assert np.abs(U + SI.poly(ap, 5, U, V) - u).max() < 1e-4
    with pytest.raises(A.HeaderError):
        h = header_of(w, 512, 512, inverse=False)
        del h["NAXIS1"]
        A.wcs_from_header(h)
    # inverse_order="exact": no fit; the library inverts A/B itself (DFR_SIP_INVERSE_EXACT)
    e = A.wcs_from_header(header_of(w, 512, 512, inverse=False), inverse_order="exact")
    assert e.ap_order == -1 and e.bp_order == -1 and e.a_order == 3


@pytest.mark.gpu
def test_calculate_reprojection_against_oracle(A):
    torch = pytest.importorskip("torch")
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    from tests import parity as PR
    rng = np.random.default_rng(11)
    imgs = [S.make_image(240, 320, 40, rng) for _ in range(2)]
    srcs = [S.add_sip(S.make_wcs(320, 240, 150.0 + 1e-3 * k, 2.0, 4.0 * k, S.PIXSCALE), 3, 160.0, rng, amp=1e-4)
            for k in range(2)]
    tgt = S.make_wcs(300, 260, 150.0008, 2.0004, -3.0, S.PIXSCALE)

    class HDU:
        def __init__(self, data, header):
            self.data, self.header = data, header

    hdus = [HDU(im, header_of(w, 320, 240)) for im, w in zip(imgs, srcs)]
    out = A.calculate_reprojection(hdus, header_of(tgt, 300, 260, use_pc=True), shape_out=(260, 300), order="bicubic")
    assert out.shape == (2, 260, 300)
    for e in range(2):
        xo, yo = oracle.src_coords(tgt, srcs[e], 260, 300)
        ref = oracle.interp(imgs[e], xo.ravel(), yo.ravel(), 3).reshape(260, 300).astype(np.float32)
        PR.check_image(out[e], ref, xo, yo, imgs[e], 3)
    # single source, default shape_out = input shape, (array, header) pair
    one = A.calculate_reprojection((imgs[0], header_of(srcs[0], 320, 240)), header_of(tgt, 300, 260))
    assert one.shape == (240, 320)
    xo, yo = oracle.src_coords(tgt, srcs[0], 240, 320)
    ref = oracle.interp(imgs[0], xo.ravel(), yo.ravel(), 1).reshape(240, 320).astype(np.float32)
    PR.check_image(one, ref, xo, yo, imgs[0], 1)
    # sources of different shapes in one call: grouped by shape inside, order preserved
    small = imgs[1][:200, :280].copy()
    ws_small = srcs[1].copy()
    mixed = A.calculate_reprojection([hdus[0], HDU(small, header_of(ws_small, 280, 200)), hdus[1]],
                                     header_of(tgt, 300, 260), shape_out=(260, 300))
    assert mixed.shape == (3, 260, 300)
    ref_all = A.calculate_reprojection(hdus, header_of(tgt, 300, 260), shape_out=(260, 300))
    assert np.array_equal(np.nan_to_num(mixed[0], nan=-1), np.nan_to_num(ref_all[0], nan=-1))
    assert np.array_equal(np.nan_to_num(mixed[2], nan=-1), np.nan_to_num(ref_all[1], nan=-1))
    xo, yo = oracle.src_coords(tgt, ws_small, 260, 300)
    ref = oracle.interp(small, xo.ravel(), yo.ravel(), 1).reshape(260, 300).astype(np.float32)
    PR.check_image(mixed[1], ref, xo, yo, small, 1)
    mean, wsum = A.calculate_stack(hdus, header_of(tgt, 300, 260), shape_out=(260, 300))
    so, wo = oracle.stack(np.stack(imgs), srcs, tgt, (260, 300), 1)
    ok = wo == 2
    assert np.abs(mean[ok] - so[ok] / 2).max() < 1e-5 * PR.dyn_range(imgs[0]) * 2 and np.isnan(mean[wo == 0]).all()
