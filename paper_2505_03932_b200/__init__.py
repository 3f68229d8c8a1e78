"""paper_2505_03932_b200 — thin Python binding of libdfr (include/dfr.h).

Argument marshalling only: every step of the reprojection path runs in the
library's CUDA kernels. torch is used for device memory and streams. There is
no CPU fallback: if libdfr.so is missing or CUDA is unavailable the calls raise.
This package never imports `oracle`.
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

_PKG = os.path.dirname(os.path.abspath(__file__))
_SO = os.path.join(_PKG, "libdfr.so")

NEAREST, BILINEAR, BICUBIC = 0, 1, 3
PATH_AUTO, PATH_EXACT, PATH_TILED = 0, 1, 2
EDGE_AREA, EDGE_PAPER = 0, 1
_ORDER_NAMES = {"nearest": 0, "nearest-neighbor": 0, "bilinear": 1, "bicubic": 3}

EXPORTS = ["dfr_reproject", "dfr_reproject_edge", "dfr_reproject_ex", "dfr_reproject_fp", "dfr_reproject_host",
           "dfr_reproject_noalloc",
           "dfr_reproject_host_multi", "dfr_reproject_stack", "dfr_shard_range", "dfr_release",
           "dfr_stack_finalize", "dfr_stack_host", "dfr_stack_host_multi", "dfr_pix2world",
           "dfr_world2pix", "dfr_src_coords", "dfr_wcs_set_pc_cdelt", "dfr_wcs_fit_inverse_sip", "dfr_last_stats",
           "dfr_profile_enable", "dfr_profile_last",
           "dfr_strerror", "dfr_last_error", "dfr_version"]


class DfrWCS(C.Structure):
    """Mirror of `dfr_wcs` in include/dfr.h (3280 bytes)."""
    _fields_ = [("crpix", C.c_double * 2), ("crval", C.c_double * 2), ("cd", C.c_double * 4),
                ("a_order", C.c_int32), ("b_order", C.c_int32),
                ("ap_order", C.c_int32), ("bp_order", C.c_int32),
                ("a", C.c_double * 100), ("b", C.c_double * 100),
                ("ap", C.c_double * 100), ("bp", C.c_double * 100)]


class DfrError(RuntimeError):
    def __init__(self, code, text):
        super().__init__(f"libdfr error {code}: {text}")
        self.code = code


_lib = None


def lib():
    """Load libdfr.so (in-tree). Raises if it has not been built."""
    global _lib
    if _lib is None:
        if not os.path.exists(_SO):
            raise ImportError(f"{_SO} missing: run `python -m paper_2505_03932_b200.build` "
                              "(there is no CPU fallback)")
        L = C.CDLL(_SO)
        fp, dp, wp, vp = C.c_void_p, C.c_void_p, C.POINTER(DfrWCS), C.c_void_p
        i32, i64 = C.c_int32, C.c_int64
        L.dfr_reproject.argtypes = [fp, i32, i32, i32, wp, wp, i32, i32, i32, fp, vp]
        L.dfr_reproject_ex.argtypes = [fp, i32, i32, i32, wp, wp, i32, i32, i32, fp, vp, i32]
        L.dfr_reproject_noalloc.argtypes = [fp, i32, i32, i32, wp, wp, i32, i32, i32, fp, vp]
        L.dfr_reproject_edge.argtypes = [fp, i32, i32, i32, wp, wp, i32, i32, i32, i32, fp, vp]
        L.dfr_reproject_fp.argtypes = [fp, i32, i32, i32, wp, wp, i32, i32, i32, i32, fp, fp, vp]
        L.dfr_reproject_host.argtypes = [fp, i32, i32, i32, wp, wp, i32, i32, i32, fp, i32]
        L.dfr_reproject_host_multi.argtypes = [fp, i32, i32, i32, wp, wp, i32, i32, i32, fp, i32, C.POINTER(i32), i32]
        L.dfr_stack_host_multi.argtypes = [fp, i32, i32, i32, wp, wp, i32, i32, i32, C.POINTER(C.c_float), fp, fp, i32,
                                           C.POINTER(i32), i32]
        L.dfr_shard_range.argtypes = [i32, i32, i32, C.POINTER(i32), C.POINTER(i32)]
        L.dfr_release.argtypes = []
        L.dfr_reproject_stack.argtypes = [fp, i32, i32, i32, wp, wp, i32, i32, i32,
                                          C.POINTER(C.c_float), fp, fp, i32, vp]
        L.dfr_stack_finalize.argtypes = [fp, fp, i64, fp, vp]
        L.dfr_stack_host.argtypes = [fp, i32, i32, i32, wp, wp, i32, i32, i32, C.POINTER(C.c_float), fp, fp, i32]
        L.dfr_pix2world.argtypes = [wp, dp, dp, i64, dp, dp, vp]
        L.dfr_world2pix.argtypes = [wp, dp, dp, i64, dp, dp, vp]
        L.dfr_src_coords.argtypes = [i32, i32, i32, wp, wp, i32, i32, i32, dp, dp, vp, i32]
        L.dfr_wcs_set_pc_cdelt.argtypes = [wp, C.POINTER(C.c_double), C.POINTER(C.c_double)]
        L.dfr_wcs_fit_inverse_sip.argtypes = [wp, i32, i32, i32, C.POINTER(C.c_double)]
        L.dfr_last_stats.argtypes = [C.POINTER(C.c_int64)]
        L.dfr_profile_enable.argtypes = [C.c_int]
        L.dfr_profile_last.argtypes = [C.POINTER(C.c_float)]
        L.dfr_strerror.argtypes = [C.c_int]
        L.dfr_strerror.restype = C.c_char_p
        L.dfr_last_error.restype = C.c_char_p
        L.dfr_version.restype = C.c_int
        for name in EXPORTS:
            getattr(L, name)
        _lib = L
    return _lib


def _check(rc):
    if rc != 0:
        L = lib()
        raise DfrError(rc, (L.dfr_last_error() or L.dfr_strerror(rc)).decode())


def pack_wcs(w) -> DfrWCS:
    """Pack any object with the WCS attribute names (e.g. dfr_synth.WCS)."""
    if isinstance(w, DfrWCS):
        return w
    s = DfrWCS()
    s.crpix[:] = [float(v) for v in w.crpix]
    s.crval[:] = [float(v) for v in w.crval]
    s.cd[:] = [float(v) for v in w.cd]
    s.a_order, s.b_order = int(w.a_order), int(w.b_order)
    s.ap_order, s.bp_order = int(w.ap_order), int(w.bp_order)
    for name in ("a", "b", "ap", "bp"):
        arr = np.ascontiguousarray(getattr(w, name), dtype=np.float64).reshape(-1)
        if arr.size != 100:
            raise ValueError(f"{name} must have 10x10 entries")
        getattr(s, name)[:] = arr.tolist()
    return s


def pack_wcs_array(ws):
    if isinstance(ws, C.Array):
        return ws
    ws = list(ws)
    return (DfrWCS * len(ws))(*[pack_wcs(w) for w in ws])


def _order(order) -> int:
    if isinstance(order, str):
        return _ORDER_NAMES[order]
    return int(order)


def _stream_ptr(stream):
    import torch
    if stream is None:
        stream = torch.cuda.current_stream()
    return C.c_void_p(stream.cuda_stream)


def _need_cuda(t, dtype, name):
    if not (t.is_cuda and t.dtype == dtype and t.is_contiguous()):
        raise ValueError(f"{name} must be a contiguous CUDA tensor of {dtype}")


def dfr_reproject(src_batch, src_wcs, tgt_wcs, shape_out=None, order=BILINEAR, out=None,
                  stream=None, path=PATH_AUTO, edge=EDGE_AREA, footprint=None):
    """dfr_reproject / dfr_reproject_ex / dfr_reproject_fp (include/dfr.h). src_batch: CUDA float32
    [n][ny][nx] (or [ny][nx]); returns the CUDA float32 [n][out_ny][out_nx] output.
    shape_out defaults to the input shape. footprint=True (or a CUDA float32
    tensor of the output's shape) also returns the footprint array: (out, footprint)."""
    import torch
    if src_batch.dim() == 2:
        src_batch = src_batch[None]
    _need_cuda(src_batch, torch.float32, "src_batch")
    n, sny, snx = src_batch.shape
    ony, onx = (sny, snx) if shape_out is None else (int(shape_out[0]), int(shape_out[1]))
    ws = pack_wcs_array(src_wcs)
    if len(ws) != n:
        raise ValueError("one source WCS per exposure")
    tw = pack_wcs(tgt_wcs)
    if out is None:
        out = torch.empty((n, ony, onx), dtype=torch.float32, device=src_batch.device)
    _need_cuda(out, torch.float32, "out")
    if tuple(out.shape) != (n, ony, onx):
        raise ValueError("out has the wrong shape")
    fp_t = None
    if footprint is not None and footprint is not False:
        fp_t = torch.empty_like(out) if footprint is True else footprint
        _need_cuda(fp_t, torch.float32, "footprint")
        if tuple(fp_t.shape) != (n, ony, onx):
            raise ValueError("footprint has the wrong shape")
    with torch.cuda.device(src_batch.device):
        if edge != EDGE_AREA or fp_t is not None:
            if path != PATH_AUTO:
                raise ValueError("an explicit path cannot be combined with an explicit edge rule or a footprint array")
            _check(lib().dfr_reproject_fp(src_batch.data_ptr(), n, sny, snx, ws, C.byref(tw), ony, onx,
                                          _order(order), int(edge), out.data_ptr(),
                                          fp_t.data_ptr() if fp_t is not None else None, _stream_ptr(stream)))
        else:
            _check(lib().dfr_reproject_ex(src_batch.data_ptr(), n, sny, snx, ws, C.byref(tw), ony, onx,
                                          _order(order), out.data_ptr(), _stream_ptr(stream), int(path)))
    return out if fp_t is None else (out, fp_t)


NOALLOC_MAX_EXPOSURES = 64          # DFR_NOALLOC_MAX_EXPOSURES (include/dfr.h)


def dfr_reproject_noalloc(src_batch, src_wcs, tgt_wcs, out, order=BILINEAR, stream=None):
    """dfr_reproject_noalloc (include/dfr.h): the exact per-pixel reprojection for callers that
    cannot afford a device allocation inside the call — the GPU's memory already belongs to
    another allocator, or the call sits in a real-time loop where cudaMalloc / cudaFree (and the
    device-wide synchronisation they may bring) are off limits. The library allocates nothing:
    its constants table is a fixed 63 488-byte array in the library image, hence at most
    NOALLOC_MAX_EXPOSURES exposures per call. Neither does this wrapper: `out`, a CUDA float32
    [n][out_ny][out_nx] tensor, is the caller's and gives shape_out. Results equal
    dfr_reproject(..., path=PATH_EXACT). Make the first call on a device during set-up (it looks
    up the array's address); calls that may overlap on the GPU share the table and race."""
    import torch
    if src_batch.dim() == 2:
        src_batch = src_batch[None]
    _need_cuda(src_batch, torch.float32, "src_batch")
    _need_cuda(out, torch.float32, "out")
    n, sny, snx = src_batch.shape
    if out.dim() != 3 or out.shape[0] != n:
        raise ValueError("out must be [n][out_ny][out_nx]")
    ws = pack_wcs_array(src_wcs)
    if len(ws) != n:
        raise ValueError("one source WCS per exposure")
    tw = pack_wcs(tgt_wcs)
    with torch.cuda.device(src_batch.device):
        _check(lib().dfr_reproject_noalloc(src_batch.data_ptr(), n, sny, snx, ws, C.byref(tw),
                                           int(out.shape[1]), int(out.shape[2]), _order(order),
                                           out.data_ptr(), _stream_ptr(stream)))
    return out


def dfr_reproject_host(src_host, src_wcs, tgt_wcs, shape_out=None, order=BILINEAR, out_host=None,
                       batch=32, devices=None):
    """dfr_reproject_host: HOST float32 arrays (numpy, or CPU torch tensors — pinned
    for full PCIe rate) in and out; copies and kernels are pipelined inside the library.
    devices=[0, 1, ...] shards the exposures over several GPUs (dfr_reproject_host_multi)."""
    import torch
    src_t = torch.as_tensor(src_host)
    if src_t.dim() == 2:
        src_t = src_t[None]
    if src_t.is_cuda or src_t.dtype != torch.float32 or not src_t.is_contiguous():
        raise ValueError("src_host must be a contiguous float32 host array")
    n, sny, snx = src_t.shape
    ony, onx = (sny, snx) if shape_out is None else (int(shape_out[0]), int(shape_out[1]))
    ws = pack_wcs_array(src_wcs)
    if len(ws) != n:
        raise ValueError("one source WCS per exposure")
    tw = pack_wcs(tgt_wcs)
    if out_host is None:
        out_host = torch.empty((n, ony, onx), dtype=torch.float32, pin_memory=True)
    out_t = torch.as_tensor(out_host)
    if out_t.is_cuda or out_t.dtype != torch.float32 or not out_t.is_contiguous() \
            or tuple(out_t.shape) != (n, ony, onx):
        raise ValueError("out_host must be a contiguous float32 host array [n][ny][nx]")
    if devices is None:
        _check(lib().dfr_reproject_host(src_t.data_ptr(), n, sny, snx, ws, C.byref(tw), ony, onx,
                                        _order(order), out_t.data_ptr(), int(batch)))
    else:
        dv = (C.c_int32 * len(devices))(*[int(d) for d in devices])
        _check(lib().dfr_reproject_host_multi(src_t.data_ptr(), n, sny, snx, ws, C.byref(tw), ony, onx,
                                              _order(order), out_t.data_ptr(), int(batch), dv, len(devices)))
    return out_host


def dfr_reproject_stack(src_batch, src_wcs, tgt_wcs, shape_out=None, order=BILINEAR, weights=None,
                        sum=None, wsum=None, accumulate=False, stream=None):
    """dfr_reproject_stack (include/dfr.h): fused reprojection + co-addition. Returns the
    CUDA float32 (sum, wsum) [out_ny][out_nx]; pass them back with accumulate=True to add
    further batches."""
    import torch
    if src_batch.dim() == 2:
        src_batch = src_batch[None]
    _need_cuda(src_batch, torch.float32, "src_batch")
    n, sny, snx = src_batch.shape
    ony, onx = (sny, snx) if shape_out is None else (int(shape_out[0]), int(shape_out[1]))
    ws = pack_wcs_array(src_wcs)
    if len(ws) != n:
        raise ValueError("one source WCS per exposure")
    tw = pack_wcs(tgt_wcs)
    if sum is None:
        sum = torch.empty((ony, onx), dtype=torch.float32, device=src_batch.device)
    if wsum is None:
        wsum = torch.empty((ony, onx), dtype=torch.float32, device=src_batch.device)
    for t, name in ((sum, "sum"), (wsum, "wsum")):
        _need_cuda(t, torch.float32, name)
        if tuple(t.shape) != (ony, onx):
            raise ValueError(f"{name} has the wrong shape")
    wp = None
    if weights is not None:
        w = np.ascontiguousarray(weights, dtype=np.float32)
        if w.size != n:
            raise ValueError("one weight per exposure")
        wp = w.ctypes.data_as(C.POINTER(C.c_float))
    with torch.cuda.device(src_batch.device):
        _check(lib().dfr_reproject_stack(src_batch.data_ptr(), n, sny, snx, ws, C.byref(tw), ony, onx,
                                         _order(order), wp, sum.data_ptr(), wsum.data_ptr(),
                                         1 if accumulate else 0, _stream_ptr(stream)))
    return sum, wsum


def dfr_stack_host(src_host, src_wcs, tgt_wcs, shape_out=None, order=BILINEAR, weights=None, batch=32, devices=None):
    """dfr_stack_host: HOST float32 exposures in (pinned for full PCIe rate), HOST (sum, wsum)
    float32 [out_ny][out_nx] out; uploads and the stacking kernels are pipelined in the library."""
    import torch
    src_t = torch.as_tensor(src_host)
    if src_t.dim() == 2:
        src_t = src_t[None]
    if src_t.is_cuda or src_t.dtype != torch.float32 or not src_t.is_contiguous():
        raise ValueError("src_host must be a contiguous float32 host array")
    n, sny, snx = src_t.shape
    ony, onx = (sny, snx) if shape_out is None else (int(shape_out[0]), int(shape_out[1]))
    ws = pack_wcs_array(src_wcs)
    if len(ws) != n:
        raise ValueError("one source WCS per exposure")
    tw = pack_wcs(tgt_wcs)
    wp = None
    if weights is not None:
        w = np.ascontiguousarray(weights, dtype=np.float32)
        if w.size != n:
            raise ValueError("one weight per exposure")
        wp = w.ctypes.data_as(C.POINTER(C.c_float))
    s = torch.empty((ony, onx), dtype=torch.float32, pin_memory=True)
    c = torch.empty((ony, onx), dtype=torch.float32, pin_memory=True)
    if devices is None:
        _check(lib().dfr_stack_host(src_t.data_ptr(), n, sny, snx, ws, C.byref(tw), ony, onx, _order(order), wp,
                                    s.data_ptr(), c.data_ptr(), int(batch)))
    else:
        dv = (C.c_int32 * len(devices))(*[int(d) for d in devices])
        _check(lib().dfr_stack_host_multi(src_t.data_ptr(), n, sny, snx, ws, C.byref(tw), ony, onx, _order(order), wp,
                                          s.data_ptr(), c.data_ptr(), int(batch), dv, len(devices)))
    return s, c


def dfr_stack_finalize(sum, wsum, mean=None, stream=None):
    """dfr_stack_finalize: mean = sum / wsum, NaN where wsum == 0."""
    import torch
    _need_cuda(sum, torch.float32, "sum")
    _need_cuda(wsum, torch.float32, "wsum")
    if mean is None:
        mean = torch.empty_like(sum)
    _need_cuda(mean, torch.float32, "mean")
    with torch.cuda.device(sum.device):
        _check(lib().dfr_stack_finalize(sum.data_ptr(), wsum.data_ptr(), sum.numel(), mean.data_ptr(),
                                        _stream_ptr(stream)))
    return mean


def dfr_pix2world(wcs, x, y, stream=None):
    """dfr_pix2world: x, y CUDA float64 tensors -> (ra_deg, dec_deg) CUDA float64."""
    import torch
    _need_cuda(x, torch.float64, "x")
    _need_cuda(y, torch.float64, "y")
    ra, dec = torch.empty_like(x), torch.empty_like(x)
    w = pack_wcs(wcs)
    with torch.cuda.device(x.device):
        _check(lib().dfr_pix2world(C.byref(w), x.data_ptr(), y.data_ptr(), x.numel(),
                                   ra.data_ptr(), dec.data_ptr(), _stream_ptr(stream)))
    return ra, dec


def dfr_world2pix(wcs, ra_deg, dec_deg, stream=None):
    """dfr_world2pix: (ra, dec) CUDA float64 degrees -> (x, y) CUDA float64."""
    import torch
    _need_cuda(ra_deg, torch.float64, "ra_deg")
    _need_cuda(dec_deg, torch.float64, "dec_deg")
    x, y = torch.empty_like(ra_deg), torch.empty_like(ra_deg)
    w = pack_wcs(wcs)
    with torch.cuda.device(ra_deg.device):
        _check(lib().dfr_world2pix(C.byref(w), ra_deg.data_ptr(), dec_deg.data_ptr(), ra_deg.numel(),
                                   x.data_ptr(), y.data_ptr(), _stream_ptr(stream)))
    return x, y


def dfr_src_coords(src_wcs, tgt_wcs, src_shape, shape_out, order=BILINEAR, path=PATH_AUTO,
                   device="cuda", stream=None):
    """dfr_src_coords (test-only): the source coordinates the reprojection kernels
    use, CUDA float64 [n][out_ny][out_nx] each."""
    import torch
    ws = pack_wcs_array(src_wcs)
    tw = pack_wcs(tgt_wcs)
    n = len(ws)
    ony, onx = int(shape_out[0]), int(shape_out[1])
    x = torch.empty((n, ony, onx), dtype=torch.float64, device=device)
    y = torch.empty_like(x)
    with torch.cuda.device(x.device):
        _check(lib().dfr_src_coords(n, int(src_shape[0]), int(src_shape[1]), ws, C.byref(tw),
                                    ony, onx, _order(order), x.data_ptr(), y.data_ptr(),
                                    _stream_ptr(stream), int(path)))
    return x, y


def dfr_wcs_set_pc_cdelt(wcs: DfrWCS, pc, cdelt):
    pc_a = (C.c_double * 4)(*[float(v) for v in pc])
    cd_a = (C.c_double * 2)(*[float(v) for v in cdelt])
    _check(lib().dfr_wcs_set_pc_cdelt(C.byref(wcs), pc_a, cd_a))
    return wcs


def dfr_wcs_fit_inverse_sip(wcs: DfrWCS, order: int, nx: int, ny: int) -> float:
    """dfr_wcs_fit_inverse_sip: fits AP/BP into `wcs` (a packed DfrWCS, modified in place);
    returns the largest round-trip residual on the fit grid, in pixels."""
    res = C.c_double(0.0)
    _check(lib().dfr_wcs_fit_inverse_sip(C.byref(wcs), int(order), int(nx), int(ny), C.byref(res)))
    return float(res.value)


def dfr_last_stats():
    arr = (C.c_int64 * 4)()
    _check(lib().dfr_last_stats(arr))
    return {"tiles_fast": arr[0], "tiles_exact": arr[1], "tiles_empty": arr[2], "kernels": arr[3]}


def dfr_profile_enable(on: bool):
    _check(lib().dfr_profile_enable(1 if on else 0))


def dfr_profile_last():
    """(setup_ms, main_ms) of the last dfr_reproject call on this thread."""
    ms = (C.c_float * 2)()
    _check(lib().dfr_profile_last(ms))
    return float(ms[0]), float(ms[1])


PROBE_NAMES = ["FFMA", "FFMA2", "FADD2.RM", "DFMA", "IMAD", "LOP3", "LDS", "FFMA+FFMA2", "FFMA2+IMAD", "FFMA2+LOP3",
               "FFMA 3-reg", "FFMA2 3-reg"]


_probe_lib = None


def probe_lib():
    """libdfr_probe.so: the register-only instruction-rate probes, a measurement tool kept out of
    libdfr and of include/dfr.h (csrc/probe/dfr_probe.cu). Only `bench.py --mode probes` uses it."""
    global _probe_lib
    if _probe_lib is None:
        so = os.path.join(_PKG, "libdfr_probe.so")
        if not os.path.exists(so):
            raise ImportError(f"{so} missing: run `python -m paper_2505_03932_b200.build`")
        L = C.CDLL(so)
        L.dfr_probe_rates.argtypes = [C.POINTER(C.c_double), C.c_int]
        L.dfr_probe_error.restype = C.c_char_p
        _probe_lib = L
    return _probe_lib


def dfr_probe_rates() -> dict:
    """Thread-level instructions per clock per SM for each probe class (libdfr_probe.so)."""
    out = (C.c_double * len(PROBE_NAMES))()
    L = probe_lib()
    rc = L.dfr_probe_rates(out, len(PROBE_NAMES))
    if rc != 0:
        raise DfrError(rc, L.dfr_probe_error().decode())
    return dict(zip(PROBE_NAMES, [float(v) for v in out]))


def dfr_shard_range(n: int, parts: int, k: int):
    """dfr_shard_range: [lo, hi) of shard k of `parts` over n units (the *_multi partition rule)."""
    lo, hi = C.c_int32(0), C.c_int32(0)
    _check(lib().dfr_shard_range(int(n), int(parts), int(k), C.byref(lo), C.byref(hi)))
    return int(lo.value), int(hi.value)


def dfr_release():
    """dfr_release: free what the library keeps for the current device (include/dfr.h)."""
    _check(lib().dfr_release())


def dfr_version() -> int:
    return int(lib().dfr_version())


def calculate_reprojection(*args, **kwargs):
    """see paper_2505_03932_b200.api.calculate_reprojection."""
    from .api import calculate_reprojection as f
    return f(*args, **kwargs)
