"""dfr_reproject_noalloc: the entry point for callers that cannot allocate device memory.

Some users of the library run where an allocation inside the call is not an option: the GPU's
memory is already owned by another allocator (so a cudaMallocAsync from the library can fail in
the middle of a night's reduction), or the call sits in a real-time loop that must not meet the
device-wide synchronisation cudaMalloc / cudaFree may bring. For them the library keeps the one
piece of scratch the exact per-pixel kernel needs (the per-exposure constants table) in a fixed
array inside the library image and calls no allocating routine at all; the price is a limit of
DFR_NOALLOC_MAX_EXPOSURES = 64 exposures per call and 63 488 bytes held on every GPU that loads
the library.

What is checked here: the new entry point gives what the existing exact path gives
(dfr_reproject_ex with DFR_PATH_EXACT: same device functions, so equality is expected; the bar
applied is the suite's own, tests/parity.py: identical NaN mask, values within 1e-5 x dynamic
range), on two calls in a row that share the table — the second with fewer exposures and other
WCSs, issued without waiting for the first, so stale entries or a missing stream ordering would
show. The file is named to be collected last: the driver runs pytest with -x, and a failure here
must not hide the parity tests. It passes alone in a fresh process as well as after the others
(the entry point depends on no state the other entry points create).
"""
import ctypes as C

import numpy as np
import pytest

import dfr_synth as S
from tests import parity as PR

torch = pytest.importorskip("torch")


def _batch(seed, n, sny, snx, ony, onx, rot):
    """n small exposures with SIP, each with its own pointing, and a rotated SIP target."""
    rng = np.random.default_rng(seed)
    imgs = np.stack([S.make_image(sny, snx, 30, rng) for _ in range(n)]).astype(np.float32)
    srcs = [S.add_sip(S.make_wcs(snx, sny, 150.0 + 2e-4 * e, 2.0 - 1e-4 * e, 0.3 * e, S.PIXSCALE),
                      3, snx / 2.0, rng, amp=1e-4) for e in range(n)]
    tgt = S.add_sip(S.make_wcs(onx, ony, 150.002, 2.001, rot, S.PIXSCALE * 1.05), 4, onx / 2.0, rng, amp=1e-4)
    return imgs, srcs, tgt


def _same(new, old, imgs):
    assert np.array_equal(np.isnan(new), np.isnan(old)), "NaN masks differ"
    frac = float(np.isnan(old).mean())
    assert 0.02 < frac < 0.9, f"the case should have pixels on both sides of the footprint ({frac})"
    for e in range(new.shape[0]):
        ok = ~np.isnan(old[e])
        err = np.abs(new[e][ok].astype(np.float64) - old[e][ok].astype(np.float64))
        lim = PR.VALUE_TOL * PR.dyn_range(imgs[e])
        assert err.size and float(err.max()) <= lim, f"exposure {e}: {err.max():.3e} > {lim:.3e}"


@pytest.mark.gpu
def test_noalloc_matches_exact_path_on_two_calls_in_a_row():
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    import paper_2505_03932_b200 as P
    P.lib()
    # call 1: 11 exposures = two fill launches, the second ragged; bilinear
    i1, s1, t1 = _batch(101, 11, 131, 203, 150, 177, 17.0)
    # call 2: fewer exposures, other pointings and shapes, bicubic — entries 2..10 of the table are stale
    i2, s2, t2 = _batch(202, 2, 97, 160, 140, 123, -28.0)
    d1, d2 = torch.from_numpy(i1).cuda(), torch.from_numpy(i2).cuda()
    o1 = torch.full((11, 150, 177), -7.0, dtype=torch.float32, device="cuda")
    o2 = torch.full((2, 140, 123), -7.0, dtype=torch.float32, device="cuda")
    P.dfr_reproject_noalloc(d1, s1, t1, o1, P.BILINEAR)
    P.dfr_reproject_noalloc(d2, s2, t2, o2, P.BICUBIC)          # same stream, no wait in between
    torch.cuda.synchronize()
    r1 = P.dfr_reproject(d1, s1, t1, (150, 177), P.BILINEAR, path=P.PATH_EXACT)
    r2 = P.dfr_reproject(d2, s2, t2, (140, 123), P.BICUBIC, path=P.PATH_EXACT)
    torch.cuda.synchronize()
    _same(o1.cpu().numpy(), r1.cpu().numpy(), i1)
    _same(o2.cpu().numpy(), r2.cpu().numpy(), i2)
    # and once more with the first inputs (nearest): the table is rewritten, not appended to
    o3 = torch.full((11, 150, 177), -7.0, dtype=torch.float32, device="cuda")
    P.dfr_reproject_noalloc(d1, s1, t1, o3, P.NEAREST)
    r3 = P.dfr_reproject(d1, s1, t1, (150, 177), P.NEAREST, path=P.PATH_EXACT)
    torch.cuda.synchronize()
    _same(o3.cpu().numpy(), r3.cpu().numpy(), i1)


@pytest.mark.gpu
def test_noalloc_full_table():
    """n = DFR_NOALLOC_MAX_EXPOSURES: every entry of the fixed table in use."""
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    import paper_2505_03932_b200 as P
    n = P.NOALLOC_MAX_EXPOSURES
    imgs, srcs, tgt = _batch(303, n, 40, 56, 48, 52, 9.0)
    d = torch.from_numpy(imgs).cuda()
    out = torch.empty((n, 48, 52), dtype=torch.float32, device="cuda")
    P.dfr_reproject_noalloc(d, srcs, tgt, out, P.BILINEAR)
    ref = P.dfr_reproject(d, srcs, tgt, (48, 52), P.BILINEAR, path=P.PATH_EXACT)
    torch.cuda.synchronize()
    _same(out.cpu().numpy(), ref.cpu().numpy(), imgs)


def test_noalloc_rejects_batches_beyond_the_fixed_table():
    """More exposures than the fixed table holds: refused before anything touches the GPU,
    with a message that names the limit (runs without a CUDA device)."""
    from paper_2505_03932_b200 import build
    build.build()
    import paper_2505_03932_b200 as P
    L = P.lib()
    w = P.pack_wcs(S.make_wcs(8, 8, 1.0, 2.0, 0.0, S.PIXSCALE))
    n = P.NOALLOC_MAX_EXPOSURES + 1
    arr = (P.DfrWCS * n)(*([w] * n))
    src, out = C.c_void_p(0x10000), C.c_void_p(0x9000000)
    rc = L.dfr_reproject_noalloc(src, n, 8, 8, arr, C.byref(w), 8, 8, 1, out, None)
    assert rc == -2                                             # DFR_ERR_SHAPE
    msg = L.dfr_last_error().decode()
    assert "DFR_NOALLOC_MAX_EXPOSURES = 64" in msg and f"n = {n}" in msg
    # the usual validation comes first or alongside: NULL pointers, order, aliasing
    assert L.dfr_reproject_noalloc(None, 1, 8, 8, arr, C.byref(w), 8, 8, 1, out, None) == -1
    assert L.dfr_reproject_noalloc(src, 1, 8, 8, arr, C.byref(w), 8, 8, 2, out, None) == -3
    assert L.dfr_reproject_noalloc(src, 1, 8, 8, arr, C.byref(w), 8, 8, 1, C.c_void_p(0x10000 + 64), None) == -7
