"""-m "not gpu": libdfr.so builds, loads, exports every symbol include/dfr.h declares,
and rejects bad arguments before touching CUDA (no compute calls without a GPU)."""
import ctypes as C
import os
import re

import pytest

import dfr_synth as S

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def P():
    from paper_2505_03932_b200 import build
    build.build()
    import paper_2505_03932_b200 as pkg
    return pkg


def declared_functions():
    text = open(os.path.join(ROOT, "include", "dfr.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(dfr_[a-z0-9_]+)\s*\(", text)))


def test_every_declared_symbol_is_exported(P):
    names = declared_functions()
    assert "dfr_reproject" in names and "dfr_pix2world" in names and "dfr_world2pix" in names
    L = P.lib()
    for n in names:
        assert hasattr(L, n), f"{n} declared in dfr.h but not exported"
    assert sorted(P.EXPORTS) == names
    assert P.dfr_version() >= 100


def test_struct_layout_matches_header(P):
    assert C.sizeof(P.DfrWCS) == 3280
    assert P.DfrWCS.a_order.offset == 64 and P.DfrWCS.a.offset == 80
    assert P.DfrWCS.bp.offset == 80 + 3 * 800


def test_product_does_not_import_oracle():
    for dirpath, _, files in os.walk(os.path.join(ROOT, "paper_2505_03932_b200")):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h", ".cpp")):
                txt = open(os.path.join(dirpath, f)).read()
                assert "import oracle" not in txt and "from oracle" not in txt, f
                assert "orc.h" not in txt and "liboracle" not in txt, f


def test_validation_errors_without_gpu(P):
    L = P.lib()
    w = S.make_wcs(8, 8, 1.0, 2.0, 0.0, S.PIXSCALE)
    good = P.pack_wcs(w)
    arr = (P.DfrWCS * 1)(good)
    fake_src, fake_out = C.c_void_p(0x10000), C.c_void_p(0x90000)

    def call(src=fake_src, n=1, sny=8, snx=8, ws=arr, tw=good, ony=8, onx=8, order=1, out=fake_out, path=0):
        return L.dfr_reproject_ex(src, n, sny, snx, ws, C.byref(tw), ony, onx, order, out, None, path)

    assert call(src=None) == -1 and call(out=None) == -1                       # DFR_ERR_NULL
    assert call(n=0) == -2 and call(snx=0) == -2 and call(ony=-3) == -2         # DFR_ERR_SHAPE
    assert call(sny=65536, snx=65536) == -2                                     # ny*nx >= 2^31
    assert call(order=2) == -3 and call(order=4) == -3                          # DFR_ERR_ORDER
    assert call(path=7) == -3
    bad = P.pack_wcs(w); bad.ap_order = 10
    assert call(tw=bad) == -4                                                   # DFR_ERR_SIP_ORDER
    bad = P.pack_wcs(w); bad.cd[:] = [1.0, 2.0, 2.0, 4.0]
    assert call(tw=bad) == -5                                                   # DFR_ERR_SINGULAR_CD
    bad = P.pack_wcs(w); bad.crval[1] = float("nan")
    assert call(tw=bad) == -6                                                   # DFR_ERR_NONFINITE_WCS
    bad = P.pack_wcs(w); bad.a_order = 2; bad.a[2 * 10 + 0] = float("inf")
    assert call(ws=(P.DfrWCS * 1)(bad)) == -6
    bad = P.pack_wcs(w); bad.a_order = 2; bad.a[9 * 10 + 9] = float("inf")       # ignored: p+q > order
    assert call(ws=(P.DfrWCS * 1)(bad), out=C.c_void_p(0x10000 + 64)) == -7     # ... reaches DFR_ERR_ALIAS
    assert b"overlap" in L.dfr_last_error()
    assert L.dfr_strerror(-5) == b"singular CD matrix"
    # explicit footprint rule: unknown mode, and the paper's rule with bicubic, are refused
    def edge(order, mode):
        return L.dfr_reproject_edge(fake_src, 1, 8, 8, arr, C.byref(good), 8, 8, order, mode, fake_out, None)
    assert edge(1, 7) == -3 and edge(3, 1) == -3 and b"bicubic" in L.dfr_last_error()
    assert L.dfr_reproject_edge(None, 1, 8, 8, arr, C.byref(good), 8, 8, 1, 1, fake_out, None) == -1
    # sky entry points validate too
    assert L.dfr_pix2world(None, fake_src, fake_src, 1, fake_out, fake_out, None) == -1
    assert L.dfr_world2pix(C.byref(good), fake_src, fake_src, -1, fake_out, fake_out, None) == -2
    assert L.dfr_pix2world(C.byref(good), None, fake_src, 5, fake_out, fake_out, None) == -1


def test_stack_validation_errors_without_gpu(P):
    L = P.lib()
    w = S.make_wcs(8, 8, 1.0, 2.0, 0.0, S.PIXSCALE)
    good = P.pack_wcs(w)
    arr = (P.DfrWCS * 2)(good, good)
    src, a, b = C.c_void_p(0x10000), C.c_void_p(0x90000), C.c_void_p(0xA0000)
    wts = (C.c_float * 2)(1.0, 2.0)

    def call(src=src, n=2, order=1, weights=wts, s=a, c=b, tw=good):
        return L.dfr_reproject_stack(src, n, 8, 8, arr, C.byref(tw), 8, 8, order, weights, s, c, 0, None)

    assert call(src=None) == -1 and call(s=None) == -1 and call(c=None) == -1   # DFR_ERR_NULL
    assert call(n=0) == -2 and call(order=2) == -3
    assert call(s=C.c_void_p(0x10000 + 16)) == -7 and call(c=a) == -7            # overlap src / each other
    assert call(weights=(C.c_float * 2)(1.0, float("inf"))) == -9                # DFR_ERR_WEIGHT
    assert b"weights[1]" in L.dfr_last_error()
    # host-buffer form and finalize
    assert L.dfr_stack_host(None, 2, 8, 8, arr, C.byref(good), 8, 8, 1, None, a, b, 2) == -1
    assert L.dfr_stack_host(src, 2, 8, 8, arr, C.byref(good), 8, 8, 5, None, a, b, 2) == -3
    assert L.dfr_stack_finalize(a, b, -1, a, None) == -2
    assert L.dfr_stack_finalize(None, b, 4, a, None) == -1
    assert L.dfr_stack_finalize(None, None, 0, None, None) == 0                  # zero pixels is legal


def test_pc_cdelt_helper(P):
    s = P.pack_wcs(S.make_wcs(8, 8, 1.0, 2.0, 0.0, S.PIXSCALE))
    P.dfr_wcs_set_pc_cdelt(s, [0.6, -0.8, 0.8, 0.6], [-2.0, 3.0])
    assert list(s.cd) == pytest.approx([-1.2, 1.6, 2.4, 1.8], abs=1e-15)


def test_binding_refuses_cpu_tensors(P):
    import torch
    with pytest.raises(ValueError):
        P.dfr_reproject(torch.zeros(1, 8, 8), [S.make_wcs(8, 8, 1, 2, 0, S.PIXSCALE)],
                        S.make_wcs(8, 8, 1, 2, 0, S.PIXSCALE))


def test_footprint_and_multi_device_validation_without_gpu(P):
    L = P.lib()
    w = S.make_wcs(8, 8, 1.0, 2.0, 0.0, S.PIXSCALE)
    good = P.pack_wcs(w)
    arr = (P.DfrWCS * 2)(good, good)
    src, out, fp = C.c_void_p(0x10000), C.c_void_p(0x90000), C.c_void_p(0xA0000)

    def call_fp(order=1, mode=0, out=out, fp=fp):
        return L.dfr_reproject_fp(src, 2, 8, 8, arr, C.byref(good), 8, 8, order, mode, out, fp, None)

    assert call_fp(mode=3) == -3 and call_fp(order=3, mode=1) == -3
    assert call_fp(fp=C.c_void_p(0x90000 + 64)) == -7 and b"footprint" in L.dfr_last_error()   # overlaps out
    assert call_fp(fp=C.c_void_p(0x10000)) == -7                                                # overlaps src
    assert call_fp(out=None) == -1
    devs = (C.c_int32 * 2)(0, 0)
    assert L.dfr_reproject_host_multi(None, 2, 8, 8, arr, C.byref(good), 8, 8, 1, out, 2, devs, 2) == -1
    assert L.dfr_reproject_host_multi(src, 2, 8, 8, arr, C.byref(good), 8, 8, 1, out, 2, None, 2) == -1
    assert L.dfr_reproject_host_multi(src, 2, 8, 8, arr, C.byref(good), 8, 8, 1, out, 2, devs, 0) == -2
    assert L.dfr_stack_host_multi(src, 2, 8, 8, arr, C.byref(good), 8, 8, 2, None, out, fp, 2, devs, 2) == -3
    assert L.dfr_stack_host_multi(src, 2, 8, 8, arr, C.byref(good), 8, 8, 1, (C.c_float * 2)(1.0, float("nan")),
                                  out, fp, 2, devs, 2) == -9
    # the instruction-rate probes live in their own library, outside the product ABI
    assert not hasattr(L, "dfr_probe_rates")
    LP = P.probe_lib()
    assert LP.dfr_probe_rates(None, 12) == -1 and LP.dfr_probe_rates((C.c_double * 4)(), 4) == -2


def test_shard_range_is_a_partition_and_matches_the_python_rule(P):
    from paper_2505_03932_b200.shard import shard_range
    for n in (0, 1, 5, 32, 33, 1024, 1031):
        for parts in (1, 2, 3, 7, 8, 64):
            pieces = [P.dfr_shard_range(n, parts, k) for k in range(parts)]
            assert pieces[0][0] == 0 and pieces[-1][1] == n
            assert all(pieces[k][1] == pieces[k + 1][0] for k in range(parts - 1))       # contiguous, ordered
            sizes = [hi - lo for lo, hi in pieces]
            assert max(sizes) - min(sizes) <= 1 and sizes == sorted(sizes, reverse=True)
            for k in range(parts):
                r = shard_range(n, parts, k)
                assert (r.start, r.stop) == pieces[k]
    with pytest.raises(P.DfrError):
        P.dfr_shard_range(10, 0, 0)
    with pytest.raises(P.DfrError):
        P.dfr_shard_range(10, 4, 4)


def test_exact_inverse_sentinel_validation(P):
    """DFR_SIP_INVERSE_EXACT (-1) is accepted only for ap_order and bp_order together."""
    L = P.lib()
    w = S.make_wcs(8, 8, 1.0, 2.0, 0.0, S.PIXSCALE)
    src, out = C.c_void_p(0x10000), C.c_void_p(0x90000)

    def call(ap, bp, a=2):
        s = P.pack_wcs(w)
        s.a_order = s.b_order = a
        s.a[2 * 10 + 0] = 1e-6
        s.ap_order, s.bp_order = ap, bp
        arr = (P.DfrWCS * 1)(s)
        # an aliasing output stops the call after validation (no CUDA needed)
        return L.dfr_reproject_ex(src, 1, 8, 8, arr, C.byref(P.pack_wcs(w)), 8, 8, 1, C.c_void_p(0x10000 + 64), None, 0)

    assert call(-1, -1) == -7                      # valid WCS: reaches the alias check
    assert call(0, 0) == -7
    assert call(-1, 0) == -4 and call(3, -1) == -4 and call(-2, -2) == -4
