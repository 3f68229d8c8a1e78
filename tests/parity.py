"""Parity rules GPU vs oracle (BASELINE.json north_star), written out
once so every -m gpu test applies the same bar.

  coordinates : |x_gpu - x_orc| <= COORD_TOL (+ the oracle's own conditioning term)
                wherever both are finite
  mask        : identical, except where the oracle coordinate lies within EDGE_BAND of
                a footprint edge (-0.5 or n-0.5)
  values      : |v_gpu - v_orc| <= VALUE_TOL * DR on pixels valid in both; for nearest,
                additionally excluding pixels within TIE_BAND of a half-integer
  NaN == NaN
"""
import math

import numpy as np

COORD_TOL = 1e-4        # px   (north_star)
VALUE_TOL = 1e-5        # x dynamic range (north_star)
EDGE_BAND = 1e-3        # px   (north_star)
TIE_BAND = 2e-4         # px   (G8/G9: 2 x COORD_TOL)
D2R = math.pi / 180.0


def dyn_range(img):
    f = img[np.isfinite(img)]
    return float(f.max() - f.min())


def oracle_conditioning(xo, yo, src_wcs):
    """Rounding of the oracle's literal theta = asin(s) near the source tangent point
    (PAPER.md:105): ~1e-16 / (r_px scale_rad^2) px (tests P5)."""
    scale_rad = math.sqrt(abs(src_wcs.cd[0] * src_wcs.cd[3] - src_wcs.cd[1] * src_wcs.cd[2])) * D2R
    r = np.hypot(xo - (src_wcs.crpix[0] - 1), yo - (src_wcs.crpix[1] - 1))
    return 4e-16 / (np.maximum(r, 1e-12) * scale_rad ** 2)


def check_coords(xg, yg, xo, yo, src_wcs, tol=COORD_TOL):
    both = np.isfinite(xg) & np.isfinite(yg) & np.isfinite(xo) & np.isfinite(yo)
    assert np.array_equal(np.isfinite(xg), np.isfinite(xo)), "finite-ness of coordinates differs"
    err = np.maximum(np.abs(xg - xo), np.abs(yg - yo))[both]
    lim = tol + oracle_conditioning(xo, yo, src_wcs)[both]
    stats = {"max": float(err.max()) if err.size else 0.0,
             "p9999": float(np.quantile(err, 0.9999)) if err.size else 0.0}
    assert np.all(err <= lim), f"coordinate parity: max {stats['max']:.3e} px"
    return stats


def edge_band(xo, yo, sny, snx, band=EDGE_BAND):
    return ((np.abs(xo + 0.5) < band) | (np.abs(xo - (snx - 0.5)) < band)
            | (np.abs(yo + 0.5) < band) | (np.abs(yo - (sny - 0.5)) < band))


def check_image(out_gpu, out_orc, xo, yo, src_img, order):
    """Mask + value parity for one exposure; xo, yo are the oracle's source coordinates."""
    sny, snx = src_img.shape
    mg, mo = np.isnan(out_gpu), np.isnan(out_orc)
    near_edge = edge_band(xo, yo, sny, snx) | ~np.isfinite(xo)
    bad_mask = (mg != mo) & ~near_edge
    assert not bad_mask.any(), f"{int(bad_mask.sum())} mask mismatches away from the footprint edge"
    valid = ~mg & ~mo
    if order == 0:
        tie = ((np.abs(xo - np.floor(xo) - 0.5) < TIE_BAND) | (np.abs(yo - np.floor(yo) - 0.5) < TIE_BAND))
        valid &= ~tie
    dr = dyn_range(src_img)
    err = np.abs(out_gpu[valid].astype(np.float64) - out_orc[valid].astype(np.float64))
    stats = {"max": float(err.max()) if err.size else 0.0,
             "p9999": float(np.quantile(err, 0.9999)) if err.size else 0.0,
             "dr": dr, "nan_frac": float(mo.mean()), "mask_diff_in_band": int((mg != mo).sum())}
    assert stats["max"] <= VALUE_TOL * dr, \
        f"value parity: max {stats['max']:.3e} > {VALUE_TOL * dr:.3e} (order {order})"
    return stats
