"""Seeded synthetic inputs for the reprojection hot path.

This module serves BOTH the oracle-side tests and the CUDA-side tests/bench. It
holds none of the method's arithmetic: it only draws images and WCS *parameters*
(BASELINE.json `configs`); the one polynomial it evaluates is
the least-squares fit that BASELINE.json prescribes for producing the inverse
SIP coefficients of an input WCS. It imports neither `oracle` nor the CUDA
package.

The paper's workloads are synthetic FITS frames "sized 256x256 to 4000x6000"
with and without SIP; these generators stand in for them.
"""
from __future__ import annotations

import math
from dataclasses import dataclass, field

import numpy as np

SIP_DIM = 10                      # orders 0..9
ARCSEC = 1.0 / 3600.0
PIXSCALE = 2.85 * ARCSEC          # deg / px (BASELINE.json configs[0])


@dataclass
class WCS:
    """Plain description of a TAN(-SIP) WCS; angles in degrees, CRPIX FITS 1-based.

    a, b, ap, bp are (10, 10) float64 arrays indexed [p][q] (coefficient of
    u^p v^q); an order of 0 means the polynomial is absent.
    """
    crpix: tuple
    crval: tuple
    cd: tuple                     # (cd11, cd12, cd21, cd22)
    a_order: int = 0
    b_order: int = 0
    ap_order: int = 0
    bp_order: int = 0
    a: np.ndarray = field(default_factory=lambda: np.zeros((SIP_DIM, SIP_DIM)))
    b: np.ndarray = field(default_factory=lambda: np.zeros((SIP_DIM, SIP_DIM)))
    ap: np.ndarray = field(default_factory=lambda: np.zeros((SIP_DIM, SIP_DIM)))
    bp: np.ndarray = field(default_factory=lambda: np.zeros((SIP_DIM, SIP_DIM)))

    def copy(self) -> "WCS":
        return WCS(tuple(self.crpix), tuple(self.crval), tuple(self.cd),
                   self.a_order, self.b_order, self.ap_order, self.bp_order,
                   self.a.copy(), self.b.copy(), self.ap.copy(), self.bp.copy())


# --------------------------------------------------------------------------- images

def make_image(ny: int, nx: int, nstars: int, rng: np.random.Generator) -> np.ndarray:
    """Sky background N(100, 5^2) + circular Gaussian stars (sigma 1.5 px, peak
    U(500, 5000)) at uniform positions (BASELINE.json configs[0]). float32 [ny][nx].

    Draw order: background, xs, ys, peaks.
    """
    img = rng.normal(100.0, 5.0, (ny, nx))
    xs = rng.uniform(0.0, nx - 1.0, nstars)
    ys = rng.uniform(0.0, ny - 1.0, nstars)
    peak = rng.uniform(500.0, 5000.0, nstars)
    sig = 1.5
    for k in range(nstars):
        cx, cy = int(round(xs[k])), int(round(ys[k]))
        x0, x1 = max(cx - 8, 0), min(cx + 9, nx)
        y0, y1 = max(cy - 8, 0), min(cy + 9, ny)
        if x0 >= x1 or y0 >= y1:
            continue
        ii = np.arange(x0, x1)[None, :]
        jj = np.arange(y0, y1)[:, None]
        img[y0:y1, x0:x1] += peak[k] * np.exp(-((ii - xs[k]) ** 2 + (jj - ys[k]) ** 2)
                                              / (2.0 * sig * sig))
    return img.astype(np.float32)


def make_image_fast(ny: int, nx: int, nstars: int, rng: np.random.Generator) -> np.ndarray:
    """Same statistics as make_image, float32 draws (about 3x faster); used where
    gigabytes of exposures are needed (configs[4]) and only the GPU/oracle
    agreement on identical pixels matters."""
    img = rng.standard_normal((ny, nx), dtype=np.float32)
    img *= np.float32(5.0)
    img += np.float32(100.0)
    xs = rng.uniform(0.0, nx - 1.0, nstars)
    ys = rng.uniform(0.0, ny - 1.0, nstars)
    peak = rng.uniform(500.0, 5000.0, nstars)
    for k in range(nstars):
        cx, cy = int(round(xs[k])), int(round(ys[k]))
        x0, x1 = max(cx - 8, 0), min(cx + 9, nx)
        y0, y1 = max(cy - 8, 0), min(cy + 9, ny)
        if x0 >= x1 or y0 >= y1:
            continue
        ii = np.arange(x0, x1, dtype=np.float32)[None, :]
        jj = np.arange(y0, y1, dtype=np.float32)[:, None]
        img[y0:y1, x0:x1] += (peak[k] * np.exp(-((ii - xs[k]) ** 2 + (jj - ys[k]) ** 2)
                                               / 4.5)).astype(np.float32)
    return img


# --------------------------------------------------------------------------- WCS

def make_wcs(nx: int, ny: int, ra: float, dec: float, rot_deg: float, scale: float) -> WCS:
    """TAN WCS with CRPIX at the image centre ((n+1)/2, FITS 1-based) and
    CD = diag(-scale, +scale) . R(rot), R(r) = [[cos r, -sin r], [sin r, cos r]]."""
    c, s = math.cos(math.radians(rot_deg)), math.sin(math.radians(rot_deg))
    cd = (-scale * c, scale * s, scale * s, scale * c)
    return WCS(crpix=((nx + 1) / 2.0, (ny + 1) / 2.0), crval=(ra, dec), cd=cd)


def draw_sip(order: int, half: float, rng: np.random.Generator, amp: float = 1e-6):
    """Forward SIP coefficients A_pq, B_pq ~ N(0, amp * half^(1-p-q)) for
    2 <= p+q <= order (BASELINE.json configs[1]). Draw order: for total degree
    d = 2..order, for p = d..0 (q = d - p): A_pq then B_pq."""
    a = np.zeros((SIP_DIM, SIP_DIM))
    b = np.zeros((SIP_DIM, SIP_DIM))
    for d in range(2, order + 1):
        for p in range(d, -1, -1):
            q = d - p
            sd = amp * half ** (1 - p - q)
            a[p, q] = rng.normal(0.0, sd)
            b[p, q] = rng.normal(0.0, sd)
    return a, b


def _poly_eval(c: np.ndarray, order: int, u: np.ndarray, v: np.ndarray) -> np.ndarray:
    out = np.zeros_like(u)
    for p in range(order + 1):
        for q in range(order + 1 - p):
            if c[p, q] != 0.0:
                out = out + c[p, q] * u ** p * v ** q
    return out


def fit_inverse_sip(a: np.ndarray, b: np.ndarray, order: int, half: float, ngrid: int = 64):
    """Least-squares AP, BP on the full triangle 0 <= p+q <= order from an
    ngrid x ngrid uniform grid over [-half, half]^2 (BASELINE.json configs[1]):
    with (U, V) = (u + A(u,v), v + B(u,v)) find AP, BP with u ~= U + AP(U,V),
    v ~= V + BP(U,V). Columns are scaled by `half` for conditioning."""
    g = np.linspace(-half, half, ngrid)
    u, v = np.meshgrid(g, g)
    u, v = u.ravel(), v.ravel()
    U = u + _poly_eval(a, order, u, v)
    V = v + _poly_eval(b, order, u, v)
    terms = [(p, q) for p in range(order + 1) for q in range(order + 1 - p)]
    M = np.stack([(U / half) ** p * (V / half) ** q for p, q in terms], axis=1)
    ca, *_ = np.linalg.lstsq(M, u - U, rcond=None)
    cb, *_ = np.linalg.lstsq(M, v - V, rcond=None)
    ap = np.zeros((SIP_DIM, SIP_DIM))
    bp = np.zeros((SIP_DIM, SIP_DIM))
    for (p, q), ka, kb in zip(terms, ca, cb):
        ap[p, q] = ka / half ** (p + q)
        bp[p, q] = kb / half ** (p + q)
    return ap, bp


def add_sip(w: WCS, order: int, half: float, rng: np.random.Generator, amp: float = 1e-6) -> WCS:
    """Attach a drawn forward SIP and its fitted inverse to w (in place)."""
    a, b = draw_sip(order, half, rng, amp)
    ap, bp = fit_inverse_sip(a, b, order, half)
    w.a, w.b, w.ap, w.bp = a, b, ap, bp
    w.a_order = w.b_order = w.ap_order = w.bp_order = order
    return w


def sip_roundtrip_residual(w: WCS, half: float, rng: np.random.Generator, npts: int = 200000):
    """max |(u,v) - inverse(forward(u,v))| in px on random points (the <1e-3 px
    acceptance test of BASELINE.json configs[1])."""
    u = rng.uniform(-half, half, npts)
    v = rng.uniform(-half, half, npts)
    U = u + _poly_eval(w.a, w.a_order, u, v)
    V = v + _poly_eval(w.b, w.b_order, u, v)
    ub = U + _poly_eval(w.ap, w.ap_order, U, V)
    vb = V + _poly_eval(w.bp, w.bp_order, U, V)
    return float(np.max(np.hypot(ub - u, vb - v)))


def _offset_crval(ra: float, dec: float, sep_deg: float, pa_deg: float):
    """Small offset of `sep` at position angle `pa` (N through E):
    d_dec = sep cos pa, d_ra = sep sin pa / cos dec."""
    dd = sep_deg * math.cos(math.radians(pa_deg))
    dr = sep_deg * math.sin(math.radians(pa_deg)) / math.cos(math.radians(dec))
    return ra + dr, dec + dd


def jittered_exposure(seed_pair, ny: int = 2048, nx: int = 2048, nstars: int = 2000,
                      with_image: bool = True, fast_image: bool = False):
    """One exposure of configs[2]/[4]: rng = default_rng(seed_pair). Draw order:
    image, d_ra, d_dec (U(-5', 5') each), rot U(-1, 1) deg, scale factor
    1 + U(-1e-3, 1e-3), SIP3 forward draw. When with_image is False the image
    draws are still consumed (so the WCS is identical) but the stars are skipped."""
    rng = np.random.default_rng(seed_pair)
    if with_image:
        img = (make_image_fast if fast_image else make_image)(ny, nx, nstars, rng)
    else:
        img = None
        if fast_image:
            rng.standard_normal((ny, nx), dtype=np.float32)
        else:
            rng.normal(100.0, 5.0, (ny, nx))
        rng.uniform(0.0, nx - 1.0, nstars)
        rng.uniform(0.0, ny - 1.0, nstars)
        rng.uniform(500.0, 5000.0, nstars)
    dra = rng.uniform(-5.0 / 60.0, 5.0 / 60.0)
    ddec = rng.uniform(-5.0 / 60.0, 5.0 / 60.0)
    rot = rng.uniform(-1.0, 1.0)
    scl = PIXSCALE * (1.0 + rng.uniform(-1e-3, 1e-3))
    w = make_wcs(nx, ny, 150.0 + dra, 2.0 + ddec, rot, scl)
    add_sip(w, 3, nx / 2.0, rng)
    return img, w


# --------------------------------------------------------------------------- configs

@dataclass
class Workload:
    name: str
    images: np.ndarray            # float32 [n][ny][nx]
    src_wcs: list                 # n WCS
    tgt_wcs: WCS
    shape_out: tuple              # (ny, nx)
    orders: tuple                 # interpolation orders to run (0, 1, 3)


def config0() -> Workload:
    """configs[0]: 256^2, no SIP, target shifted (+3.4, -2.7) px and rotated 0.5 deg."""
    rng = np.random.default_rng(0)
    img = make_image(256, 256, 50, rng)
    src = make_wcs(256, 256, 150.0, 2.0, 0.0, PIXSCALE)
    tgt = make_wcs(256, 256, 150.0, 2.0, 0.5, PIXSCALE)
    tgt.crpix = (tgt.crpix[0] + 3.4, tgt.crpix[1] - 2.7)
    return Workload("C0", img[None], [src], tgt, (256, 256), (1,))


def config1(n: int = 2048, nstars: int = 2000) -> Workload:
    """configs[1]: one 2048^2 TAN-SIP3 exposure; target offset 30" at PA 45 deg,
    rotated 0.3 deg, own SIP3. Draw order (seed 1): image, source SIP, target SIP."""
    rng = np.random.default_rng(1)
    img = make_image(n, n, nstars, rng)
    src = add_sip(make_wcs(n, n, 150.0, 2.0, 0.0, PIXSCALE), 3, n / 2.0, rng)
    ra, dec = _offset_crval(150.0, 2.0, 30.0 * ARCSEC, 45.0)
    tgt = add_sip(make_wcs(n, n, ra, dec, 0.3, PIXSCALE), 3, n / 2.0, rng)
    return Workload("C1", img[None], [src], tgt, (n, n), (1,))


def config2_target(n: int = 2048) -> WCS:
    return add_sip(make_wcs(n, n, 150.0, 2.0, 0.0, PIXSCALE), 3, n / 2.0,
                   np.random.default_rng([2, 10 ** 6]))


def config2(batch: int = 32, n: int = 2048, nstars: int = 2000, fast_image: bool = False) -> Workload:
    """configs[2]: `batch` jittered 2048^2 TAN-SIP3 exposures onto one shared
    2048^2 TAN-SIP3 target. Exposure k uses default_rng([2, k])."""
    imgs = np.empty((batch, n, n), dtype=np.float32)
    ws = []
    for k in range(batch):
        img, w = jittered_exposure([2, k], n, n, nstars, fast_image=fast_image)
        imgs[k] = img
        ws.append(w)
    return Workload("C2", imgs, ws, config2_target(n), (n, n), (1,))


def config3(scale_down: int = 1) -> Workload:
    """configs[3]: 6248x4176 SIP4 exposure onto a 6400x4400 SIP4 target rotated
    2 deg with a 3' CRVAL offset at PA 45 deg; nearest, bilinear, bicubic.
    scale_down > 1 shrinks both grids (for CPU-side tests only)."""
    snx, sny = 6248 // scale_down, 4176 // scale_down
    tnx, tny = 6400 // scale_down, 4400 // scale_down
    rng = np.random.default_rng(3)
    img = make_image(sny, snx, 12000 // (scale_down * scale_down), rng)
    src = add_sip(make_wcs(snx, sny, 150.0, 2.0, 0.0, PIXSCALE), 4, snx / 2.0, rng)
    ra, dec = _offset_crval(150.0, 2.0, 3.0 / 60.0 / scale_down, 45.0)
    tgt = add_sip(make_wcs(tnx, tny, ra, dec, 2.0, PIXSCALE), 4, tnx / 2.0, rng)
    return Workload("C3", img[None], [src], tgt, (tny, tnx), (0, 1, 3))


def config4_target(n: int = 4096) -> WCS:
    return add_sip(make_wcs(n, n, 150.0, 2.0, 0.0, PIXSCALE), 3, n / 2.0,
                   np.random.default_rng([4, 10 ** 6]))


def config4(indices, n: int = 2048, nstars: int = 2000, mosaic: int = 4096) -> Workload:
    """configs[4] restricted to the exposures in `indices` (the full stream is
    range(1024)); exposure k uses default_rng([4, k]); float32 image draws."""
    indices = list(indices)
    imgs = np.empty((len(indices), n, n), dtype=np.float32)
    ws = []
    for t, k in enumerate(indices):
        img, w = jittered_exposure([4, k], n, n, nstars, fast_image=True)
        imgs[t] = img
        ws.append(w)
    return Workload("C4", imgs, ws, config4_target(mosaic), (mosaic, mosaic), (1,))


def stress_sip_pair(n: int = 1024, amp: float = 3e-3, order: int = 3, seed: int = 77):
    """Extra coordinate-parity case: strong SIP (~10 px) so a
    percent-level error in SIP evaluation is visible above 1e-4 px."""
    rng = np.random.default_rng(seed)
    src = add_sip(make_wcs(n, n, 150.0, 2.0, 0.0, PIXSCALE), order, n / 2.0, rng, amp)
    ra, dec = _offset_crval(150.0, 2.0, 60.0 * ARCSEC, 30.0)
    tgt = add_sip(make_wcs(n, n, ra, dec, 0.7, PIXSCALE), order, n / 2.0, rng, amp)
    return src, tgt
