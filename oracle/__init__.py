"""ctypes front end of the oracle (oracle/orc.c) — TEST INFRASTRUCTURE.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
--impl reference legs may import this package. It never imports the CUDA
package and shares no code with it (see orc.h). `build()` compiles
liboracle.so with gcc; building the checker is not using it.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SO = os.path.join(_HERE, "liboracle.so")
_SRCS = ["orc.c", "orc_closed.c"]
SIP_DIM = 10
KEYS_A = -0.75          # reading G7

NEAREST, BILINEAR, BICUBIC = 0, 1, 3


class OrcWCS(C.Structure):
    _fields_ = [("crpix", C.c_double * 2), ("crval", C.c_double * 2), ("cd", C.c_double * 4),
                ("a_order", C.c_int32), ("b_order", C.c_int32),
                ("ap_order", C.c_int32), ("bp_order", C.c_int32),
                ("a", C.c_double * 100), ("b", C.c_double * 100),
                ("ap", C.c_double * 100), ("bp", C.c_double * 100)]


def build(force: bool = False) -> str:
    """gcc -O2 -fopenmp, strict IEEE (no fast-math, no FMA contraction)."""
    srcs = [os.path.join(_HERE, s) for s in _SRCS]
    deps = srcs + [os.path.join(_HERE, "orc.h")]
    if (not force and os.path.exists(_SO)
            and all(os.path.getmtime(_SO) >= os.path.getmtime(d) for d in deps)):
        return _SO
    cmd = ["gcc", "-std=c99", "-O2", "-fopenmp", "-ffp-contract=off", "-fPIC", "-shared",
           "-Wall", "-Wextra", "-o", _SO] + srcs + ["-lm"]
    subprocess.run(cmd, check=True, cwd=_HERE)
    return _SO


_lib = None


def lib():
    global _lib
    if _lib is None:
        _lib = C.CDLL(build())
        dp, fp = C.POINTER(C.c_double), C.POINTER(C.c_float)
        wp = C.POINTER(OrcWCS)
        _lib.orc_pix2world.argtypes = [wp, dp, dp, C.c_int64, dp, dp]
        _lib.orc_world2pix.argtypes = [wp, dp, dp, C.c_int64, dp, dp]
        _lib.orc_src_coords.argtypes = [wp, wp, C.c_int32, C.c_int32, dp, dp]
        _lib.orc_interp.argtypes = [fp, C.c_int32, C.c_int32, dp, dp, C.c_int64, C.c_int32,
                                    C.c_double, dp]
        _lib.orc_interp_paper.argtypes = [fp, C.c_int32, C.c_int32, dp, dp, C.c_int64, C.c_int32, dp, dp]
        _lib.orc_interp_paper.restype = C.c_int
        _lib.orc_reproject.argtypes = [fp, C.c_int32, C.c_int32, C.c_int32, wp, wp,
                                       C.c_int32, C.c_int32, C.c_int32, fp]
        _lib.orc_reproject.restype = C.c_int
        _lib.orc_stack.argtypes = [fp, C.c_int32, C.c_int32, C.c_int32, wp, wp,
                                   C.c_int32, C.c_int32, C.c_int32, dp, fp, fp]
        _lib.orc_stack.restype = C.c_int
        _lib.orc_cd_from_pc_cdelt.argtypes = [dp, dp, dp]
        _lib.orc_closed_iwc2sky.argtypes = [dp, dp, dp, C.c_int64, dp, dp]
        _lib.orc_closed_sky2iwc.argtypes = [dp, dp, dp, C.c_int64, dp, dp]
        _lib.orc_set_threads.argtypes = [C.c_int]
        _lib.orc_get_max_threads.restype = C.c_int
    return _lib


def pack(w) -> OrcWCS:
    """Pack any object with the WCS attribute names (e.g. dfr_synth.WCS)."""
    s = OrcWCS()
    s.crpix[:] = [float(v) for v in w.crpix]
    s.crval[:] = [float(v) for v in w.crval]
    s.cd[:] = [float(v) for v in w.cd]
    s.a_order, s.b_order = int(w.a_order), int(w.b_order)
    s.ap_order, s.bp_order = int(w.ap_order), int(w.bp_order)
    for name in ("a", "b", "ap", "bp"):
        arr = np.ascontiguousarray(getattr(w, name), dtype=np.float64).reshape(-1)
        assert arr.size == 100
        getattr(s, name)[:] = arr.tolist()
    return s


def _d(a):
    a = np.ascontiguousarray(a, dtype=np.float64)
    return a, a.ctypes.data_as(C.POINTER(C.c_double))


def pix2world(w, x, y):
    x, xp = _d(x)
    y, yp = _d(y)
    ra, dec = np.empty_like(x), np.empty_like(x)
    s = pack(w)
    lib().orc_pix2world(C.byref(s), xp, yp, x.size, _d(ra)[1], _d(dec)[1])
    return ra, dec


def world2pix(w, ra, dec):
    ra, rp = _d(ra)
    dec, dp_ = _d(dec)
    x, y = np.empty_like(ra), np.empty_like(ra)
    s = pack(w)
    lib().orc_world2pix(C.byref(s), rp, dp_, ra.size, _d(x)[1], _d(y)[1])
    return x, y


def src_coords(tgt, src, out_ny, out_nx):
    x = np.empty((out_ny, out_nx), dtype=np.float64)
    y = np.empty((out_ny, out_nx), dtype=np.float64)
    t, s = pack(tgt), pack(src)
    lib().orc_src_coords(C.byref(t), C.byref(s), out_ny, out_nx, _d(x)[1], _d(y)[1])
    return x, y


def interp(src, x, y, order, a=KEYS_A):
    src = np.ascontiguousarray(src, dtype=np.float32)
    assert src.ndim == 2
    x, xp = _d(x)
    y, yp = _d(y)
    val = np.empty(x.shape, dtype=np.float64)
    lib().orc_interp(src.ctypes.data_as(C.POINTER(C.c_float)), src.shape[0], src.shape[1],
                     xp, yp, x.size, int(order), float(a), _d(val)[1])
    return val


def interp_paper(src, x, y, order):
    """orc_interp_paper: (val, footprint) under the paper's literal normalisation (G19)."""
    src = np.ascontiguousarray(src, dtype=np.float32)
    assert src.ndim == 2
    x, xp = _d(x)
    y, yp = _d(y)
    val = np.empty(x.shape, dtype=np.float64)
    foot = np.empty(x.shape, dtype=np.float64)
    rc = lib().orc_interp_paper(src.ctypes.data_as(C.POINTER(C.c_float)), src.shape[0], src.shape[1],
                                xp, yp, x.size, int(order), _d(val)[1], _d(foot)[1])
    if rc != 0:
        raise ValueError("orc_interp_paper: defined for nearest and bilinear only")
    return val, foot


def reproject(images, src_wcs, tgt_wcs, shape_out, order):
    images = np.ascontiguousarray(images, dtype=np.float32)
    if images.ndim == 2:
        images = images[None]
    n, ny, nx = images.shape
    assert len(src_wcs) == n
    arr = (OrcWCS * n)(*[pack(w) for w in src_wcs])
    t = pack(tgt_wcs)
    out = np.empty((n, int(shape_out[0]), int(shape_out[1])), dtype=np.float32)
    rc = lib().orc_reproject(images.ctypes.data_as(C.POINTER(C.c_float)), n, ny, nx, arr,
                             C.byref(t), int(shape_out[0]), int(shape_out[1]), int(order),
                             out.ctypes.data_as(C.POINTER(C.c_float)))
    if rc != 0:
        raise ValueError("orc_reproject: bad order")
    return out


def stack(images, src_wcs, tgt_wcs, shape_out, order, weights=None):
    """orc_stack: (sum, wsum), float32 [ny][nx] each (orc.h; reading G17)."""
    images = np.ascontiguousarray(images, dtype=np.float32)
    if images.ndim == 2:
        images = images[None]
    n, ny, nx = images.shape
    assert len(src_wcs) == n
    arr = (OrcWCS * n)(*[pack(w) for w in src_wcs])
    t = pack(tgt_wcs)
    sum_ = np.empty((int(shape_out[0]), int(shape_out[1])), dtype=np.float32)
    wsum = np.empty_like(sum_)
    wp_ = None
    if weights is not None:
        weights, wp_ = _d(weights)
        assert weights.size == n
    rc = lib().orc_stack(images.ctypes.data_as(C.POINTER(C.c_float)), n, ny, nx, arr, C.byref(t),
                         int(shape_out[0]), int(shape_out[1]), int(order), wp_,
                         sum_.ctypes.data_as(C.POINTER(C.c_float)),
                         wsum.ctypes.data_as(C.POINTER(C.c_float)))
    if rc != 0:
        raise ValueError("orc_stack: bad order")
    return sum_, wsum


def cd_from_pc_cdelt(pc, cdelt):
    cd = np.empty(4)
    lib().orc_cd_from_pc_cdelt(_d(pc)[1], _d(cdelt)[1], _d(cd)[1])
    return cd


def closed_iwc2sky(crval, up, vp):
    up, a = _d(up)
    vp, b = _d(vp)
    ra, dec = np.empty_like(up), np.empty_like(up)
    lib().orc_closed_iwc2sky(_d(crval)[1], a, b, up.size, _d(ra)[1], _d(dec)[1])
    return ra, dec


def closed_sky2iwc(crval, ra, dec):
    ra, a = _d(ra)
    dec, b = _d(dec)
    up, vp = np.empty_like(ra), np.empty_like(ra)
    lib().orc_closed_sky2iwc(_d(crval)[1], a, b, ra.size, _d(up)[1], _d(vp)[1])
    return up, vp


def set_threads(n: int):
    lib().orc_set_threads(int(n))


def max_threads() -> int:
    return int(lib().orc_get_max_threads())
