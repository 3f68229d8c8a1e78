"""Pins of the f4 oracle (oracle/sip_inverse.py) and, on the same inputs, the library's host
helper dfr_wcs_fit_inverse_sip (host-only C++: runs without a GPU). -m "not gpu"."""
import ctypes as C

import numpy as np
import pytest

import dfr_synth as S
from oracle import sip_inverse as SI


def _wcs(order, amp, seed, n=2048):
    rng = np.random.default_rng(seed)
    w = S.make_wcs(n, n, 150.0, 2.0, 0.0, S.PIXSCALE)
    w.a, w.b = S.draw_sip(order, n / 2.0, rng, amp)
    w.a_order = w.b_order = order
    return w


def test_i1_newton_inverse_is_the_inverse():
    w = _wcs(4, 3e-3, 1)
    rng = np.random.default_rng(2)
    u, v = rng.uniform(-1024, 1024, 5000), rng.uniform(-1024, 1024, 5000)
    U, V = SI.forward(w, u, v)
    assert np.abs(U - u).max() > 3.0                       # a real distortion (several px)
    ub, vb = SI.newton_inverse(w, U, V)
    assert np.abs(ub - u).max() < 1e-10 and np.abs(vb - v).max() < 1e-10


def test_i2_series_coefficients_of_a_1d_quadratic():
    """U = u + c u^2 has the series inverse u = U - c U^2 + 2 c^2 U^3 - 5 c^3 U^4 + ...:
    the fit must find AP_20 ~ -c, AP_30 ~ 2 c^2 and nothing in v (sign and index order)."""
    w = S.make_wcs(1024, 1024, 10.0, 20.0, 0.0, S.PIXSCALE)
    c = 2e-6
    w.a[2][0] = c
    w.a_order = w.b_order = 2
    ap, bp = SI.fit_inverse_sip(w, 5, 1024, 1024)
    assert abs(ap[2][0] / -c - 1.0) < 2e-3
    assert abs(ap[3][0] / (2 * c * c) - 1.0) < 2e-2
    assert np.abs(bp).max() < 1e-12 and abs(ap[0][2]) < 1e-12 and abs(ap[1][1]) < 1e-12


@pytest.mark.parametrize("amp,order,fit_order,bound", [(1e-6, 3, 3, 3e-8), (3e-3, 3, 3, 0.2), (3e-3, 3, 6, 5e-4),
                                                       (3e-3, 3, 9, 5e-7)])
def test_i3_fit_against_newton(amp, order, fit_order, bound):
    """The fitted polynomials against the exact inverse at random points: the residual is
    the truncation error of the chosen order and falls as the order grows."""
    w = _wcs(order, amp, 3)
    ap, bp = SI.fit_inverse_sip(w, fit_order, 2048, 2048)
    rng = np.random.default_rng(4)
    x, y = rng.uniform(0, 2047, 20000), rng.uniform(0, 2047, 20000)
    u, v = x - (w.crpix[0] - 1), y - (w.crpix[1] - 1)
    U, V = SI.forward(w, u, v)
    ue, ve = SI.newton_inverse(w, U, V)
    uf = U + SI.poly(ap, fit_order, U, V)
    vf = V + SI.poly(bp, fit_order, U, V)
    res = max(np.abs(uf - ue).max(), np.abs(vf - ve).max())
    assert res < bound, res


# ---------------------------------------------------------------- the library helper
@pytest.fixture(scope="module")
def P():
    import paper_2505_03932_b200 as pkg
    from paper_2505_03932_b200 import build
    build.build()
    pkg.lib()
    return pkg


@pytest.mark.parametrize("amp,order,fit_order", [(1e-6, 3, 3), (3e-3, 3, 6), (3e-3, 4, 9), (1e-4, 9, 9)])
def test_library_fit_matches_oracle(P, amp, order, fit_order):
    """Same least-squares problem, different solvers (Householder QR in C++ vs LAPACK): the
    fitted polynomials agree to 1e-9 px over the image, and the helper's reported residual
    is the oracle's residual against the exact inverse on the fit grid."""
    nx, ny = 2048, 1600
    w = _wcs(order, amp, 7)
    w.crpix = (1000.5, 801.25)
    s = P.pack_wcs(w)
    res = P.dfr_wcs_fit_inverse_sip(s, fit_order, nx, ny)
    assert s.ap_order == fit_order and s.bp_order == fit_order
    ap = np.array(s.ap[:]).reshape(10, 10)
    bp = np.array(s.bp[:]).reshape(10, 10)
    apo, bpo = SI.fit_inverse_sip(w, fit_order, nx, ny)
    rng = np.random.default_rng(8)
    x, y = rng.uniform(0, nx - 1, 20000), rng.uniform(0, ny - 1, 20000)
    u, v = x - (w.crpix[0] - 1), y - (w.crpix[1] - 1)
    U, V = SI.forward(w, u, v)
    d = max(np.abs(SI.poly(ap, fit_order, U, V) - SI.poly(apo, fit_order, U, V)).max(),
            np.abs(SI.poly(bp, fit_order, U, V) - SI.poly(bpo, fit_order, U, V)).max())
    assert d < 1e-9, d
    # reported residual = max over the fit grid of |u - (U + AP)|, |v - (V + BP)|
    g = SI.GRID
    xx, yy = np.meshgrid(np.linspace(0, nx - 1, g), np.linspace(0, ny - 1, g))
    ug, vg = xx.ravel() - (w.crpix[0] - 1), yy.ravel() - (w.crpix[1] - 1)
    Ug, Vg = SI.forward(w, ug, vg)
    ro = max(np.abs(Ug + SI.poly(apo, fit_order, Ug, Vg) - ug).max(), np.abs(Vg + SI.poly(bpo, fit_order, Ug, Vg) - vg).max())
    assert abs(res - ro) <= 1e-9 + 1e-6 * ro
    # entries outside the triangle are zero
    for p in range(10):
        for q in range(10):
            if p + q > fit_order:
                assert ap[p, q] == 0.0 and bp[p, q] == 0.0


def test_library_fit_errors(P):
    w = P.pack_wcs(_wcs(3, 1e-6, 9))
    for bad in (0, 10, -1):
        with pytest.raises(P.DfrError):
            P.dfr_wcs_fit_inverse_sip(w, bad, 100, 100)
    with pytest.raises(P.DfrError):
        P.dfr_wcs_fit_inverse_sip(w, 3, 0, 100)
    # no forward distortion: the inverse is the zero polynomial
    z = P.pack_wcs(S.make_wcs(64, 64, 1.0, 2.0, 0.0, S.PIXSCALE))
    r = P.dfr_wcs_fit_inverse_sip(z, 2, 64, 64)
    assert r == 0.0 and max(abs(t) for t in z.ap[:]) == 0.0
