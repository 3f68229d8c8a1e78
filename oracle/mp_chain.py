"""50-digit (mpmath) statement of PAPER.md §3.2 — TEST INFRASTRUCTURE, part of
the oracle side. Used to pin the double-precision C oracle (pins P14-P16 of
DESIGN.md §4) and to regenerate tests/golden/ (tests/golden/make_golden.py).
Shares no code with orc.c or with the CUDA path; scalar, one point at a time.

Readings as in orc.c (SIP sign plus, both polynomials at the pre-update
(u, v), atan2(y, x) argument order, degrees for u', v').
"""
from __future__ import annotations

import mpmath as mp

mp.mp.dps = 50


def _poly(c, order, u, v):
    s = mp.mpf(0)
    if order <= 0:
        return s
    for p in range(order + 1):
        for q in range(order + 1 - p):
            cf = c[p][q]
            if cf != 0:
                s += mp.mpf(float(cf)) * u ** p * v ** q
    return s


def pix2sky(w, x, y):
    """PAPER.md:87-95. Returns (ra, dec) in radians (mpf)."""
    u = mp.mpf(x) - (mp.mpf(float(w.crpix[0])) - 1)
    v = mp.mpf(y) - (mp.mpf(float(w.crpix[1])) - 1)
    f = _poly(w.a, w.a_order, u, v)
    g = _poly(w.b, w.b_order, u, v)
    u, v = u + f, v + g
    cd = [mp.mpf(float(t)) for t in w.cd]
    up = cd[0] * u + cd[1] * v
    vp = cd[2] * u + cd[3] * v
    r = mp.sqrt(up * up + vp * vp)
    r0 = 180 / mp.pi
    phi = mp.atan2(-up, vp)
    theta = mp.atan2(r0, r)
    ra0 = mp.radians(mp.mpf(float(w.crval[0])))
    dec0 = mp.radians(mp.mpf(float(w.crval[1])))
    dec = mp.asin(mp.sin(theta) * mp.sin(dec0) + mp.cos(theta) * mp.cos(dec0) * mp.cos(phi))
    ra = ra0 + mp.atan2(-mp.cos(theta) * mp.sin(phi),
                        mp.sin(theta) * mp.cos(dec0) - mp.cos(theta) * mp.sin(dec0) * mp.cos(phi))
    return ra, dec


def sky2pix(w, ra, dec):
    """PAPER.md:101-121. (ra, dec) radians -> (x, y) pixels (mpf)."""
    ra0 = mp.radians(mp.mpf(float(w.crval[0])))
    dec0 = mp.radians(mp.mpf(float(w.crval[1])))
    dra = ra - ra0
    phi = mp.atan2(-mp.cos(dec) * mp.sin(dra),
                   mp.sin(dec) * mp.cos(dec0) - mp.cos(dec) * mp.sin(dec0) * mp.cos(dra))
    theta = mp.asin(mp.sin(dec) * mp.sin(dec0) + mp.cos(dec) * mp.cos(dec0) * mp.cos(dra))
    r = (180 / mp.pi) * mp.cos(theta) / mp.sin(theta)
    up = -r * mp.sin(phi)
    vp = r * mp.cos(phi)
    cd = [mp.mpf(float(t)) for t in w.cd]
    det = cd[0] * cd[3] - cd[1] * cd[2]
    u = (cd[3] * up - cd[1] * vp) / det
    v = (-cd[2] * up + cd[0] * vp) / det
    f = _poly(w.ap, w.ap_order, u, v)
    g = _poly(w.bp, w.bp_order, u, v)
    u, v = u + f, v + g
    return u + (mp.mpf(float(w.crpix[0])) - 1), v + (mp.mpf(float(w.crpix[1])) - 1)


def pix2world_deg(w, x, y):
    ra, dec = pix2sky(w, x, y)
    rd = mp.degrees(ra) % 360
    return rd, mp.degrees(dec)


def src_coord(tgt, src, i, j):
    ra, dec = pix2sky(tgt, i, j)
    return sky2pix(src, ra, dec)


def sip_value(c, order, u, v):
    return _poly(c, order, mp.mpf(u), mp.mpf(v))
