"""Pins P6-P13: the oracle's interpolation / footprint rules and
whole-path special cases (oracle/orc.c steps O11-O13) against closed forms, brute
force, hand-computed values and independent library routines. CPU only."""
import math

import numpy as np
import pytest
import scipy.ndimage as ndi
import torch

import dfr_synth as S
import oracle


def dyn_range(img):
    f = img[np.isfinite(img)]
    return float(f.max() - f.min())


@pytest.fixture(scope="module")
def small():
    rng = np.random.default_rng(42)
    img = S.make_image(96, 80, 12, rng)          # ny = 96, nx = 80 (non-square on purpose)
    w = S.make_wcs(80, 96, 150.0, 2.0, 0.0, S.PIXSCALE)
    return img, w


# ---------------------------------------------------------------- P6
@pytest.mark.parametrize("order", [0, 1, 3])
def test_p6_identity_wcs_returns_source(small, order):
    img, w = small
    out = oracle.reproject(img, [w], w, img.shape, order)[0]
    assert not np.isnan(out).any()
    if order == 0:
        assert np.array_equal(out, img)
    else:
        assert np.max(np.abs(out - img)) < 1e-5 * dyn_range(img)


# ---------------------------------------------------------------- P7
@pytest.mark.parametrize("dx,dy", [(3, 0), (0, -5), (-7, 4), (80, 0), (11, 96)])
def test_p7_integer_crpix_shift(small, dx, dy):
    img, w = small
    t = w.copy()
    t.crpix = (w.crpix[0] + dx, w.crpix[1] + dy)
    out = oracle.reproject(img, [w], t, img.shape, 0)[0]
    ny, nx = img.shape
    want = np.full_like(img, np.nan)
    for j in range(ny):
        for i in range(nx):
            si, sj = i - dx, j - dy
            if 0 <= si < nx and 0 <= sj < ny:
                want[j, i] = img[sj, si]
    assert np.array_equal(np.isnan(out), np.isnan(want))
    assert np.array_equal(out[~np.isnan(want)], want[~np.isnan(want)])


# ---------------------------------------------------------------- P8
@pytest.mark.parametrize("k", [1, 2, 3])
def test_p8_quarter_turns(k):
    rng = np.random.default_rng(8)
    n = 33
    img = rng.normal(0, 1, (n, n)).astype(np.float32)
    s = S.make_wcs(n, n, 30.0, -10.0, 0.0, S.PIXSCALE)
    t = S.make_wcs(n, n, 30.0, -10.0, 90.0 * k, S.PIXSCALE)     # CD_t = CD_s . R(90k)
    out = oracle.reproject(img, [s], t, (n, n), 0)[0]
    c = (n - 1) / 2.0
    ck, sk = round(math.cos(math.radians(90 * k))), round(math.sin(math.radians(90 * k)))
    want = np.empty_like(img)
    for j in range(n):
        for i in range(n):
            ut, vt = i - c, j - c
            us, vs = ck * ut - sk * vt, sk * ut + ck * vt       # R(90k) (u, v)
            want[j, i] = img[int(round(vs + c)), int(round(us + c))]
    assert np.array_equal(out, want)
    # the same statement through numpy: out is a rot90 of src (direction fixed by R's sense)
    assert np.array_equal(out, np.rot90(img, k=k))


# ---------------------------------------------------------------- P9
def test_p9_half_pixel_shift_is_neighbour_mean(small):
    """The paper's own demo offset: 0.5 px."""
    img, w = small
    t = w.copy()
    t.crpix = (w.crpix[0] - 0.5, w.crpix[1])          # source x = i + 0.5
    out = oracle.reproject(img, [w], t, img.shape, 1)[0]
    want = 0.5 * (img[:, :-1].astype(np.float64) + img[:, 1:].astype(np.float64))
    assert np.max(np.abs(out[:, :-1] - want)) < 1e-6 * dyn_range(img)
    # last column: x = nx - 0.5 up to rounding, i.e. ON the footprint edge — either NaN
    # or the replicated last pixel (this is the 1e-3 px edge band parity excludes)
    last = out[:, -1]
    assert np.all(np.isnan(last) | (np.abs(last - img[:, -1]) < 1e-6 * dyn_range(img)))


# ---------------------------------------------------------------- P10
def test_p10_polynomial_reproduction():
    rng = np.random.default_rng(10)
    ny, nx = 24, 31
    jj, ii = np.mgrid[0:ny, 0:nx].astype(np.float64)
    x = rng.uniform(1.0, nx - 3.0, 500)
    y = rng.uniform(1.0, ny - 3.0, 500)
    # values exactly representable in float32 so the image itself is exact
    ramp = (2.0 + 0.5 * ii - 0.25 * jj).astype(np.float32)
    v = oracle.interp(ramp, x, y, 1)
    assert np.max(np.abs(v - (2.0 + 0.5 * x - 0.25 * y))) < 1e-12
    # bilinear on the whole pixel-centre hull incl. the borders
    xe = rng.uniform(0.0, nx - 1.0, 300)
    ye = rng.uniform(0.0, ny - 1.0, 300)
    assert np.max(np.abs(oracle.interp(ramp, xe, ye, 1) - (2.0 + 0.5 * xe - 0.25 * ye))) < 1e-12
    quad = (1.0 + 0.5 * ii + 0.25 * jj + 0.125 * ii * ii - 0.5 * ii * jj + 0.25 * jj * jj).astype(np.float32)
    want = 1.0 + 0.5 * x + 0.25 * y + 0.125 * x * x - 0.5 * x * y + 0.25 * y * y
    assert np.max(np.abs(oracle.interp(quad, x, y, 3, a=-0.5) - want)) < 1e-10
    # a = -0.75 (the default bicubic) does NOT reproduce ramps (G7) ...
    assert np.max(np.abs(oracle.interp(ramp, x, y, 3, a=-0.75) - (2.0 + 0.5 * x - 0.25 * y))) > 1e-3
    # ... but every a reproduces constants (weights sum to 1)
    const = np.full((ny, nx), 7.25, dtype=np.float32)
    for a in (-0.75, -0.5, -1.0):
        assert np.max(np.abs(oracle.interp(const, x, y, 3, a=a) - 7.25)) < 1e-12


# ---------------------------------------------------------------- P11
IMG4 = np.array([[1, 2, 4, 8], [3, 5, 7, 11], [13, 17, 19, 23], [29, 31, 37, 41]], dtype=np.float32)


@pytest.mark.parametrize("x,y,order,want", [
    (-0.25, 0.0, 1, 1.0),            # rim: taps -1 and 0 both replicate pixel 0
    (0.5, 0.5, 1, 2.75),             # (1+2+3+5)/4
    (3.0, 3.0, 1, 41.0),             # exact integer corner
    (1.25, 2.5, 1, 25.0),            # rows: .75*17+.25*19 = 17.5 ; .75*31+.25*37 = 32.5 ; mean
    (3.25, 1.0, 1, 11.0),            # right rim, tap 4 replicates pixel 3
    (-0.5, -0.5, 1, 1.0),            # footprint edge is inclusive on the low side
    (3.5, 0.0, 1, None),             # ... and exclusive on the high side
    (-0.500001, 1.0, 1, None),
    (1.0, 3.5, 1, None),
    (0.5, 0.0, 0, 1.0),              # nearest: rint(0.5) = 0 (half-even)
    (1.5, 0.0, 0, 4.0),              # rint(1.5) = 2
    (2.5, 3.0, 0, 37.0),             # rint(2.5) = 2
    (3.49, 3.49, 0, 41.0),
    (-0.5, 0.0, 0, 1.0),
    (2.0, 1.0, 3, 7.0),              # Keys kernel interpolates: integer -> pixel value
    (1.5, 1.0, 3, 5.8125),           # -3/32*3 + 19/32*5 + 19/32*7 - 3/32*11 (a = -0.75)
    (1.0, 1.5, 3, -3 / 32 * 2 + 19 / 32 * 5 + 19 / 32 * 17 - 3 / 32 * 31),
    (0.0, 0.5, 3, -3 / 32 * 1 + 19 / 32 * 1 + 19 / 32 * 3 - 3 / 32 * 13),   # tap -1 replicates row 0
])
def test_p11_hand_computed_4x4(x, y, order, want):
    v = oracle.interp(IMG4, [x], [y], order)[0]
    if want is None:
        assert math.isnan(v)
    else:
        assert v == pytest.approx(want, abs=1e-13)


def test_p11_keys_weights_at_half():
    # w(1.5) = a/8, w(0.5) = 1 - (a+3)/4 + (a+2)/8 ; a = -0.75 -> -3/32, 19/32
    a = -0.75
    assert a / 8 == -3 / 32 and 1 - (a + 3) / 4 + (a + 2) / 8 == 19 / 32


# ---------------------------------------------------------------- P12
@pytest.mark.parametrize("order,mode", [(0, "nearest"), (1, "bilinear"), (3, "bicubic")])
def test_p12_torch_grid_sample_float64(small, order, mode):
    img, _ = small
    ny, nx = img.shape
    rng = np.random.default_rng(12)
    x = rng.uniform(-0.5, nx - 0.5 - 1e-9, 4000)
    y = rng.uniform(-0.5, ny - 0.5 - 1e-9, 4000)
    # include exact integers and exact half-integers (nearest ties, G8)
    x[:50] = rng.integers(0, nx, 50)
    y[50:100] = rng.integers(0, ny, 50)
    x[100:150] = rng.integers(0, nx - 1, 50) + 0.5
    y[100:150] = rng.integers(0, ny - 1, 50) + 0.5
    got = oracle.interp(img, x, y, order)
    gx = 2.0 * x / (nx - 1) - 1.0
    gy = 2.0 * y / (ny - 1) - 1.0
    grid = torch.from_numpy(np.stack([gx, gy], axis=-1)).reshape(1, 1, -1, 2)
    inp = torch.from_numpy(img.astype(np.float64)).reshape(1, 1, ny, nx)
    ref = torch.nn.functional.grid_sample(inp, grid, mode=mode, padding_mode="border",
                                          align_corners=True).reshape(-1).numpy()
    if order == 0:
        # torch un-normalises g back to a pixel coordinate, which can move an exact tie
        # by an ulp; compare away from ties, and the ties against the rule itself
        tie = (np.abs(x - np.floor(x) - 0.5) < 1e-9) | (np.abs(y - np.floor(y) - 0.5) < 1e-9)
        assert np.array_equal(got[~tie], ref[~tie])
        xi = np.clip(np.rint(x[tie]).astype(int), 0, nx - 1)
        yi = np.clip(np.rint(y[tie]).astype(int), 0, ny - 1)
        assert np.array_equal(got[tie], img[yi, xi].astype(np.float64))
    else:
        assert np.max(np.abs(got - ref)) < 1e-12 * dyn_range(img) * 10


# ---------------------------------------------------------------- P13
def test_p13_scipy_map_coordinates(small):
    img, _ = small
    ny, nx = img.shape
    rng = np.random.default_rng(13)
    x = rng.uniform(-0.5, nx - 0.5 - 1e-9, 4000)
    y = rng.uniform(-0.5, ny - 0.5 - 1e-9, 4000)
    ref1 = ndi.map_coordinates(img.astype(np.float64), [y, x], order=1, mode="nearest")
    assert np.max(np.abs(oracle.interp(img, x, y, 1) - ref1)) < 1e-12 * dyn_range(img) * 10
    ref0 = ndi.map_coordinates(img.astype(np.float64), [y, x], order=0, mode="nearest")
    tie = (np.abs(x - np.floor(x) - 0.5) < 1e-6) | (np.abs(y - np.floor(y) - 0.5) < 1e-6)
    assert np.array_equal(oracle.interp(img, x, y, 0)[~tie], ref0[~tie])


# ---------------------------------------------------------------- G6
def test_g6_edge_replication_equals_footprint_normalisation(small):
    """zero-padded bilinear of the image divided by zero-padded bilinear
    of an all-ones 'footprint' equals edge-replicated bilinear wherever footprint > 0
    (checked on the rim, where the two could differ)."""
    img, _ = small
    ny, nx = img.shape
    rng = np.random.default_rng(6)
    n = 2000
    x = np.concatenate([rng.uniform(-0.5, 0.0, n), rng.uniform(nx - 1.0, nx - 0.5 - 1e-9, n)])
    y = np.concatenate([rng.uniform(-0.5, ny - 0.5 - 1e-9, n), rng.uniform(-0.5, 0.0, n)])
    img64 = img.astype(np.float64)
    num = ndi.map_coordinates(img64, [y, x], order=1, mode="grid-constant", cval=0.0)
    den = ndi.map_coordinates(np.ones_like(img64), [y, x], order=1, mode="grid-constant", cval=0.0)
    assert (den > 0).all()
    assert np.max(np.abs(num / den - oracle.interp(img, x, y, 1))) < 1e-11 * dyn_range(img)


def test_footprint_mask_is_order_independent_and_half_open(small):
    img, w = small
    t = w.copy()
    t.crpix = (w.crpix[0] + 10.25, w.crpix[1] - 3.5)
    t.cd = S.make_wcs(80, 96, 150.0, 2.0, 7.0, S.PIXSCALE).cd
    outs = [oracle.reproject(img, [w], t, (100, 90), o)[0] for o in (0, 1, 3)]
    m = np.isnan(outs[0])
    assert np.array_equal(m, np.isnan(outs[1])) and np.array_equal(m, np.isnan(outs[2]))
    X, Y = oracle.src_coords(t, w, 100, 90)
    inside = (X >= -0.5) & (X < 80 - 0.5) & (Y >= -0.5) & (Y < 96 - 0.5)
    assert np.array_equal(~m, inside)
    assert 0.05 < m.mean() < 0.6


def test_batch_uses_per_exposure_wcs(small):
    img, w = small
    w2 = w.copy()
    w2.crpix = (w.crpix[0] + 2, w.crpix[1])
    imgs = np.stack([img, img[::-1].copy()])
    out = oracle.reproject(imgs, [w, w2], w, img.shape, 0)
    assert np.array_equal(out[0], img)
    assert np.array_equal(out[1][:, :-2], img[::-1][:, 2:])       # x_s = i + 2
    assert np.isnan(out[1][:, -2:]).all()


# ------------------------------------------------- F1-F4: the paper's literal normalisation (G19)
def test_f1_paper_mode_equals_area_rule_inside_and_extends_half_a_pixel():
    """Bilinear: footprint > 0 exactly on (-1, n) x (-1, n); wherever the area rule is valid
    the two values agree (this is G6); in the extra half-pixel band the value is the edge
    replication the area rule would have produced had it been valid."""
    rng = np.random.default_rng(70)
    img = rng.normal(100, 20, (9, 13)).astype(np.float32)
    x = rng.uniform(-2.0, 14.0, 20000)
    y = rng.uniform(-2.0, 10.0, 20000)
    val, foot = oracle.interp_paper(img, x, y, 1)
    inside = (x > -1) & (x < 13) & (y > -1) & (y < 9)
    assert np.array_equal(foot > 0, inside) and np.array_equal(~np.isnan(val), inside)
    area = oracle.interp(img, x, y, 1)
    ok = ~np.isnan(area)
    assert ok.sum() > 5000 and np.abs(val[ok] - area[ok]).max() < 1e-10
    band = inside & ~ok
    xc, yc = np.clip(x[band], 0, 12), np.clip(y[band], 0, 8)
    assert band.sum() > 500 and np.abs(val[band] - oracle.interp(img, xc, yc, 1)).max() < 1e-10


def test_f2_paper_mode_hand_values():
    img = np.arange(16, dtype=np.float32).reshape(4, 4)
    x = np.array([-0.75, 3.9, 1.5, -1.0, 4.0, 0.25])
    y = np.array([2.0, -0.5, 3.999, 1.0, 1.0, 0.5])
    val, foot = oracle.interp_paper(img, x, y, 1)
    assert val[0] == 8.0 and abs(foot[0] - 0.25) < 1e-15            # only the tap (0, 2), weight 1/4
    assert abs(val[1] - 3.0) < 1e-12 and abs(foot[1] - 0.05) < 1e-12  # only (3, 0): 0.1 x 0.5
    assert abs(val[2] - 13.5) < 1e-12                                # bottom row only: mean of 13, 14
    assert np.isnan(val[3]) and np.isnan(val[4]) and foot[3] == 0.0  # x = -1 and x = n: nothing in bounds
    assert abs(val[5] - (0.25 + 0.5 * 4.0)) < 1e-12 and abs(foot[5] - 1.0) < 1e-15


def test_f3_paper_mode_is_zero_padded_grid_sample_ratio():
    """Library routine: torch-CPU float64 grid_sample(padding_mode='zeros', align_corners=True)
    of the image and of ones; their ratio is the paper's normalised frame."""
    torch = pytest.importorskip("torch")
    rng = np.random.default_rng(71)
    ny, nx = 11, 17
    img = rng.normal(0, 1, (ny, nx)).astype(np.float32)
    x = rng.uniform(-1.5, nx + 0.5, 5000)
    y = rng.uniform(-1.5, ny + 0.5, 5000)
    g = torch.from_numpy(np.stack([2 * x / (nx - 1) - 1, 2 * y / (ny - 1) - 1], -1))[None, None]
    for order, mode in ((1, "bilinear"), (0, "nearest")):
        t = torch.from_numpy(img.astype(np.float64))[None, None]
        num = torch.nn.functional.grid_sample(t, g, mode=mode, padding_mode="zeros", align_corners=True)[0, 0, 0].numpy()
        den = torch.nn.functional.grid_sample(torch.ones_like(t), g, mode=mode, padding_mode="zeros", align_corners=True)[0, 0, 0].numpy()
        val, foot = oracle.interp_paper(img, x, y, order)
        tie = (np.abs(x - np.floor(x) - 0.5) < 1e-9) | (np.abs(y - np.floor(y) - 0.5) < 1e-9)
        keep = ~tie if order == 0 else np.ones_like(tie)
        assert np.abs(foot[keep] - den[keep]).max() < 1e-12
        pos = keep & (den > 1e-9)
        assert np.abs(val[pos] - num[pos] / den[pos]).max() < 1e-9


def test_f4_paper_mode_rejects_bicubic_and_nearest_matches_area_rule():
    img = np.arange(30, dtype=np.float32).reshape(5, 6)
    with pytest.raises(ValueError):
        oracle.interp_paper(img, np.zeros(1), np.zeros(1), 3)
    rng = np.random.default_rng(72)
    x, y = rng.uniform(-1.5, 7.0, 5000), rng.uniform(-1.5, 6.0, 5000)
    val, _ = oracle.interp_paper(img, x, y, 0)
    area = oracle.interp(img, x, y, 0)
    assert np.array_equal(np.isnan(val), np.isnan(area)) and np.array_equal(np.nan_to_num(val), np.nan_to_num(area))


# ------------------------------------------------- G14: NaN source pixels under the 16 bicubic taps
def test_g14_bicubic_nan_reach_is_exactly_the_4x4_taps():
    """Reading G14: a NaN source pixel poisons a sample iff it lies under one of the
    taps read — for bicubic the edge-replicated 4x4 neighbourhood floor(x)-1 .. floor(x)+2, including
    taps whose Keys weight is zero (integer coordinates: IEEE 0 x NaN = NaN). Pinned twice:
    (i) against a hand-counted neighbourhood written as index logic only, on a lattice that contains
    every integer and quarter-integer coordinate; (ii) mask and finite values against torch-CPU
    float64 grid_sample(bicubic, border, align_corners=True) at generic coordinates (torch
    un-normalises the grid, which may move an exact integer by an ulp, so integers are left to (i))."""
    rng = np.random.default_rng(14)
    ny, nx = 12, 14
    img = rng.normal(100.0, 20.0, (ny, nx)).astype(np.float32)      # the oracle reads float32 images (G14)
    holes = [(5, 6), (0, 0), (11, 9), (7, 13)]                 # interior, corner, bottom edge, right edge
    for r, c in holes:
        img[r, c] = np.nan
    # (i) hand count
    xs = np.arange(-2, 4 * nx - 2 + 1) / 4.0                     # -0.5 .. nx - 0.5 in quarter steps
    ys = np.arange(-2, 4 * ny - 2 + 1) / 4.0
    xs, ys = xs[xs < nx - 0.5], ys[ys < ny - 0.5]
    X, Y = np.meshgrid(xs, ys)
    got = oracle.interp(img, X.ravel(), Y.ravel(), 3).reshape(X.shape)
    want = np.zeros(X.shape, dtype=bool)
    for j, y in enumerate(ys):
        rows = {min(max(int(math.floor(y)) + d, 0), ny - 1) for d in (-1, 0, 1, 2)}
        for i, x in enumerate(xs):
            cols = {min(max(int(math.floor(x)) + d, 0), nx - 1) for d in (-1, 0, 1, 2)}
            want[j, i] = any(r in rows and c in cols for r, c in holes)
    assert np.array_equal(np.isnan(got), want)
    # an interior hole is reached from exactly 4 x 4 unit cells: 16 quarter-lattice points each
    near = (X >= 4) & (X < 8) & (Y >= 3) & (Y < 7)               # cells whose taps include (5, 6)
    assert want[near].all() and int(near.sum()) == 16 * 16
    ring = (X >= 3) & (X < 9) & (Y >= 2) & (Y < 8) & ~near
    assert not want[ring].any()
    # at integer coordinates the taps at -1 and +2 have weight zero and still count
    k = np.argmin(np.abs(xs - 4.0)), np.argmin(np.abs(ys - 4.0))
    assert xs[k[0]] == 4.0 and ys[k[1]] == 4.0 and np.isnan(got[k[1], k[0]])      # (5, 6) is tap (+2, +1): weight 0 along x
    # (ii) torch float64 grid_sample at generic coordinates
    x = rng.uniform(-0.5, nx - 0.5 - 1e-9, 6000)
    y = rng.uniform(-0.5, ny - 0.5 - 1e-9, 6000)
    keep = (np.abs(x - np.rint(x)) > 1e-6) & (np.abs(y - np.rint(y)) > 1e-6)
    x, y = x[keep], y[keep]
    got = oracle.interp(img, x, y, 3)
    grid = torch.from_numpy(np.stack([2.0 * x / (nx - 1) - 1.0, 2.0 * y / (ny - 1) - 1.0], axis=-1)).reshape(1, 1, -1, 2)
    ref = torch.nn.functional.grid_sample(torch.from_numpy(img.astype(np.float64)).reshape(1, 1, ny, nx), grid, mode="bicubic",
                                          padding_mode="border", align_corners=True).reshape(-1).numpy()
    assert np.array_equal(np.isnan(got), np.isnan(ref))
    ok = ~np.isnan(ref)
    assert 0.2 < ok.mean() < 0.95
    assert np.max(np.abs(got[ok] - ref[ok])) < 1e-10
