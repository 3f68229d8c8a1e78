"""Pins of the oracle's stacking routine (orc_stack, S1-S6). -m "not gpu".

The stack is defined from the per-exposure reprojection (already pinned by P1-P16), so
these pins fix what is new: which exposures contribute where, the weights, the
accumulation, and the two outputs."""
import numpy as np

import dfr_synth as S
import oracle


def _wcs(n=48, ra=150.0, dec=2.0, rot=0.0):
    return S.make_wcs(n, n, ra, dec, rot, S.PIXSCALE)


def test_s1_single_exposure_is_the_reprojection():
    """n = 1, weight 1: sum == reproject output where it is finite, 0 elsewhere; wsum is
    the 0/1 footprint."""
    rng = np.random.default_rng(1)
    img = S.make_image(48, 48, 5, rng)
    src, tgt = _wcs(), _wcs(ra=150.002, dec=2.001, rot=7.0)
    for order in (0, 1, 3):
        ref = oracle.reproject(img, [src], tgt, (40, 56), order)[0]
        s, w = oracle.stack(img, [src], tgt, (40, 56), order)
        m = np.isnan(ref)
        assert 0.02 < m.mean() < 0.9
        assert np.array_equal(w, (~m).astype(np.float32))
        assert np.array_equal(s[~m], ref[~m]) and np.all(s[m] == 0.0)


def test_s2_integer_shifts_brute_force():
    """Integer CRPIX shifts, nearest: the stack is the NaN-aware sum of shifted copies,
    computed here with numpy slicing (exact in float32 for integer-valued pixels)."""
    rng = np.random.default_rng(2)
    n = 32
    imgs = rng.integers(0, 1000, (3, n, n)).astype(np.float32)
    tgt = _wcs(n)
    shifts = [(0, 0), (5, -3), (-7, 11)]
    wts = np.array([1.0, 2.0, 0.5])
    srcs = []
    for dx, dy in shifts:
        w = _wcs(n)
        w.crpix = (tgt.crpix[0] - dx, tgt.crpix[1] - dy)     # out[j][i] = src[j - dy][i - dx]
        srcs.append(w)
    s, wsum = oracle.stack(imgs, srcs, tgt, (n, n), 0, wts)
    es, ew = np.zeros((n, n)), np.zeros((n, n))
    for k, (dx, dy) in enumerate(shifts):
        for j in range(n):
            for i in range(n):
                jj, ii = j - dy, i - dx
                if 0 <= jj < n and 0 <= ii < n:
                    es[j, i] += wts[k] * imgs[k, jj, ii]
                    ew[j, i] += wts[k]
    assert np.array_equal(s, es.astype(np.float32)) and np.array_equal(wsum, ew.astype(np.float32))
    assert ew.min() == 1.0 and ew.max() == 3.5


def test_s3_constants_and_weights_closed_form():
    """Constant images c_e on any geometry: sum = sum_e w_e c_e [valid_e], wsum = sum_e w_e
    [valid_e], for every interpolation order (all three reproduce constants)."""
    n = 40
    c = np.array([3.0, -1.5, 10.0])
    wts = np.array([0.25, 4.0, 1.0])
    imgs = np.ones((3, n, n), dtype=np.float32) * c[:, None, None].astype(np.float32)
    srcs = [_wcs(n, 150.0, 2.0, 0.0), _wcs(n, 150.004, 2.0, 20.0), _wcs(n, 149.997, 2.003, -35.0)]
    tgt = _wcs(n, 150.001, 2.001, 3.0)
    for order in (0, 1, 3):
        s, w = oracle.stack(imgs, srcs, tgt, (n, n), order, wts)
        es, ew = np.zeros((n, n)), np.zeros((n, n))
        for e in range(3):
            x, y = oracle.src_coords(tgt, srcs[e], n, n)
            valid = (x >= -0.5) & (x < n - 0.5) & (y >= -0.5) & (y < n - 0.5)
            es += np.where(valid, wts[e] * c[e], 0.0)
            ew += np.where(valid, wts[e], 0.0)
        assert np.allclose(s, es, rtol=0, atol=1e-5) and np.array_equal(w, ew.astype(np.float32))
        assert len(np.unique(ew)) >= 4                      # several overlap depths occur


def test_s4_linearity_and_permutation():
    """stack(a . images) = a . stack(images); reordering exposures changes nothing beyond
    the last bit of the double accumulation; default weights are 1."""
    rng = np.random.default_rng(4)
    n = 36
    imgs = np.stack([S.make_image(n, n, 4, rng) for _ in range(4)])
    srcs = [_wcs(n, 150.0 + 1e-3 * k, 2.0 - 7e-4 * k, 5.0 * k) for k in range(4)]
    tgt = _wcs(n, 150.001, 2.0, 1.0)
    s, w = oracle.stack(imgs, srcs, tgt, (n, n), 1)
    s1, w1 = oracle.stack(imgs, srcs, tgt, (n, n), 1, np.ones(4))
    assert np.array_equal(s, s1) and np.array_equal(w, w1)
    perm = [2, 0, 3, 1]
    sp, wp = oracle.stack(imgs[perm], [srcs[k] for k in perm], tgt, (n, n), 1)
    assert np.array_equal(w, wp) and np.allclose(s, sp, rtol=3e-7, atol=0)
    s2, w2 = oracle.stack(imgs, srcs, tgt, (n, n), 1, 2.0 * np.ones(4))
    assert np.array_equal(s2, 2.0 * s) and np.array_equal(w2, 2.0 * w)   # powers of two: exact
    # additivity over a split of the exposure list
    sa, wa = oracle.stack(imgs[:2], srcs[:2], tgt, (n, n), 1)
    sb, wb = oracle.stack(imgs[2:], srcs[2:], tgt, (n, n), 1)
    assert np.array_equal(w, wa + wb) and np.allclose(s, sa.astype(np.float64) + sb, rtol=3e-7, atol=1e-4)


def test_s5_equals_sum_of_reprojections():
    """Independent route through the pinned per-exposure path: nansum over exposures of
    orc_reproject outputs (each rounded to float32, so equal only to ~n ulp)."""
    rng = np.random.default_rng(5)
    n = 40
    imgs = np.stack([S.make_image(n, n, 6, rng) for _ in range(5)])
    srcs = [S.add_sip(_wcs(n, 150.0 + 8e-4 * k, 2.0 + 5e-4 * k, 9.0 * k - 10), 3, n / 2.0, rng, amp=1e-4)
            for k in range(5)]
    tgt = _wcs(n, 150.0015, 2.001, 2.0)
    wts = rng.uniform(0.5, 2.0, 5)
    for order in (0, 1, 3):
        per = oracle.reproject(imgs, srcs, tgt, (n, n), order).astype(np.float64)
        valid = ~np.isnan(per)
        es = np.where(valid, per * wts[:, None, None], 0.0).sum(0)
        ew = (valid * wts[:, None, None]).sum(0)
        s, w = oracle.stack(imgs, srcs, tgt, (n, n), order, wts)
        assert np.allclose(w, ew, rtol=1e-6, atol=0)
        assert np.allclose(s, es, rtol=1e-6, atol=1e-3)


def test_s6_nan_source_pixels_do_not_contribute():
    """A NaN source pixel is skipped by the exposure that holds it and only there."""
    n = 24
    a = np.full((n, n), 5.0, dtype=np.float32)
    b = np.full((n, n), 7.0, dtype=np.float32)
    a[10, 13] = np.nan
    w = _wcs(n)
    s, ws = oracle.stack(np.stack([a, b]), [w, w], w, (n, n), 0)
    assert ws[10, 13] == 1.0 and s[10, 13] == 7.0
    ws[10, 13] = 2.0
    s[10, 13] = 12.0
    assert np.all(ws == 2.0) and np.all(s == 12.0)
    # bilinear at a half-pixel offset: the four output pixels whose taps include the NaN drop out
    t = _wcs(n)
    t.crpix = (w.crpix[0] + 0.5, w.crpix[1] + 0.5)
    s, ws = oracle.stack(np.stack([a, b]), [w, w], t, (n, n), 1)
    assert int((ws == 1.0).sum()) >= 4 and np.all(s[ws == 1.0] == 7.0)
    assert not np.isnan(s).any()
