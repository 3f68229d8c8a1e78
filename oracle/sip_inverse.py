"""Oracle for SURVEY.md §8(f) f4 — TEST INFRASTRUCTURE (see orc.h for the rules).

The paper assumes the inverse SIP polynomials exist ("SIP_INV_A / SIP_INV_B",
:115-117); headers often lack them. Two plain numpy routines, sharing nothing with the
library's C++ helper (dfr_wcs_fit_inverse_sip):

  newton_inverse   the DEFINITION of the inverse distortion: solve U = u + A(u,v),
                   V = v + B(u,v) for (u, v) by Newton iteration to ~1e-13 px;
  fit_inverse_sip  reading G18 of DESIGN.md: least-squares AP, BP of a given order on a
                   64 x 64 uniform grid of pixel centres over [0, nx-1] x [0, ny-1]
                   (numpy.linalg.lstsq, columns scaled to [-1, 1]).
Pins: tests/test_oracle_sip_inverse.py.
"""
import numpy as np

GRID = 64


def poly(c, order, u, v):
    """sum_{p+q<=order} c[p][q] u^p v^q, written out term by term."""
    r = np.zeros_like(u, dtype=np.float64)
    for p in range(order + 1):
        for q in range(order + 1 - p):
            r = r + c[p][q] * u ** p * v ** q
    return r


def dpoly(c, order, u, v):
    """(d/du, d/dv) of poly."""
    du = np.zeros_like(u, dtype=np.float64)
    dv = np.zeros_like(u, dtype=np.float64)
    for p in range(order + 1):
        for q in range(order + 1 - p):
            if p > 0:
                du = du + c[p][q] * p * u ** (p - 1) * v ** q
            if q > 0:
                dv = dv + c[p][q] * q * u ** p * v ** (q - 1)
    return du, dv


def forward(w, u, v):
    """PAPER.md:89 with the Shupe sign (G3): (U, V) = (u + A(u,v), v + B(u,v))."""
    return u + poly(w.a, w.a_order, u, v), v + poly(w.b, w.b_order, u, v)


def newton_inverse(w, U, V, iters=50):
    u, v = np.array(U, dtype=np.float64), np.array(V, dtype=np.float64)
    for _ in range(iters):
        fu, fv = forward(w, u, v)
        au, av = dpoly(w.a, w.a_order, u, v)
        bu, bv = dpoly(w.b, w.b_order, u, v)
        j11, j12, j21, j22 = 1.0 + au, av, bu, 1.0 + bv
        det = j11 * j22 - j12 * j21
        ru, rv = fu - U, fv - V
        u = u - (j22 * ru - j12 * rv) / det
        v = v - (-j21 * ru + j11 * rv) / det
    return u, v


def fit_inverse_sip(w, order, nx, ny):
    """(ap, bp) as (10, 10) arrays; u ~= U + AP(U, V), v ~= V + BP(U, V)."""
    x = np.linspace(0.0, nx - 1.0, GRID)
    y = np.linspace(0.0, ny - 1.0, GRID)
    xx, yy = np.meshgrid(x, y)
    u = xx.ravel() - (w.crpix[0] - 1.0)
    v = yy.ravel() - (w.crpix[1] - 1.0)
    U, V = forward(w, u, v)
    hx, hy = np.abs(U).max(), np.abs(V).max()
    terms = [(p, q) for p in range(order + 1) for q in range(order + 1 - p)]
    M = np.stack([(U / hx) ** p * (V / hy) ** q for p, q in terms], axis=1)
    ca = np.linalg.lstsq(M, u - U, rcond=None)[0]
    cb = np.linalg.lstsq(M, v - V, rcond=None)[0]
    ap, bp = np.zeros((10, 10)), np.zeros((10, 10))
    for (p, q), ka, kb in zip(terms, ca, cb):
        ap[p, q] = ka / (hx ** p * hy ** q)
        bp[p, q] = kb / (hx ** p * hy ** q)
    return ap, bp
