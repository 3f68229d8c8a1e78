"""The paper's user-facing call on top of libdfr.

    calculate_reprojection(source_hdus, target_wcs, shape_out=None, order="bilinear")

is the signature the paper gives as a drop-in for `reproject.reproject_interp`. astropy is
not a dependency (the paper uses it "only for convenience ... to read the header
information"): headers are any mapping of FITS keywords (a dict, or an
astropy Header if the caller has one), HDUs are anything with `.data` and `.header`, or
`(array, header)` pairs. This module only parses keywords and marshals arguments; every
step of the reprojection runs in the library's CUDA kernels.
"""
from __future__ import annotations

import numpy as np

from . import (BILINEAR, DfrWCS, dfr_reproject, dfr_reproject_stack, dfr_stack_finalize,
               dfr_wcs_fit_inverse_sip, dfr_wcs_set_pc_cdelt, pack_wcs)

_SIP = (("A", "a"), ("B", "b"), ("AP", "ap"), ("BP", "bp"))


class HeaderError(ValueError):
    pass


def _get(h, key, default=None):
    try:
        return h[key]
    except (KeyError, IndexError):
        return default


def wcs_from_header(header, shape=None, inverse_order=None) -> DfrWCS:
    """FITS keywords -> packed `dfr_wcs`.

    Understood: CTYPEi = RA---TAN / DEC--TAN with or without -SIP ("Gnomonic");
    CRPIXi, CRVALi; CDi_j, or PCi_j (default identity) with CDELTi, or CDELTi
    with CROTA2; A_ORDER/A_p_q, B_, AP_, BP_. If forward SIP terms are present
    without AP/BP, the inverse is fitted by dfr_wcs_fit_inverse_sip over `shape` (ny, nx)
    (default NAXIS2, NAXIS1) at `inverse_order` (default min(9, A_ORDER + 2));
    inverse_order="exact" marks the WCS DFR_SIP_INVERSE_EXACT instead: the library then inverts
    A/B itself by iteration (no fit, no truncation error).
    Rejected: any other projection, LONPOLE != 180, transposed axes."""
    c1, c2 = str(_get(header, "CTYPE1", "RA---TAN")).strip(), str(_get(header, "CTYPE2", "DEC--TAN")).strip()
    if not (c1 in ("RA---TAN", "RA---TAN-SIP") and c2 in ("DEC--TAN", "DEC--TAN-SIP")):
        raise HeaderError(f"only RA---TAN / DEC--TAN (with or without -SIP) is supported, got {c1!r}, {c2!r}")
    lonpole = _get(header, "LONPOLE")
    if lonpole is not None and abs(float(lonpole) - 180.0) > 1e-9:
        raise HeaderError("LONPOLE != 180 is outside the paper's formulas (PAPER.md:91-95)")
    w = DfrWCS()
    for k in (1, 2):
        for name, arr in (("CRPIX", w.crpix), ("CRVAL", w.crval)):
            v = _get(header, f"{name}{k}")
            if v is None:
                raise HeaderError(f"{name}{k} is missing")
            arr[k - 1] = float(v)
    if _get(header, "CD1_1") is not None or _get(header, "CD2_2") is not None:
        w.cd[:] = [float(_get(header, f"CD{i}_{j}", 0.0)) for i in (1, 2) for j in (1, 2)]
    else:
        cdelt = [float(_get(header, f"CDELT{i}", 1.0)) for i in (1, 2)]
        if _get(header, "PC1_1") is None and _get(header, "CROTA2") is not None:
            r = np.deg2rad(float(header["CROTA2"]))          # legacy AIPS convention
            pc = [np.cos(r), -np.sin(r) * cdelt[1] / cdelt[0], np.sin(r) * cdelt[0] / cdelt[1], np.cos(r)]
        else:
            pc = [float(_get(header, f"PC{i}_{j}", 1.0 if i == j else 0.0)) for i in (1, 2) for j in (1, 2)]
        dfr_wcs_set_pc_cdelt(w, pc, cdelt)
    for key, field in _SIP:
        order = int(_get(header, f"{key}_ORDER", 0) or 0)
        if not 0 <= order <= 9:
            raise HeaderError(f"{key}_ORDER = {order} outside [0, 9]")
        setattr(w, f"{field}_order", order)
        arr = getattr(w, field)
        for p in range(order + 1):
            for q in range(order + 1 - p):
                arr[p * 10 + q] = float(_get(header, f"{key}_{p}_{q}", 0.0))
    if (w.a_order or w.b_order) and not (w.ap_order or w.bp_order) and inverse_order == "exact":
        w.ap_order = w.bp_order = -1                            # DFR_SIP_INVERSE_EXACT
    elif (w.a_order or w.b_order) and not (w.ap_order or w.bp_order):
        ny, nx = shape if shape is not None else (_get(header, "NAXIS2"), _get(header, "NAXIS1"))
        if ny is None or nx is None:
            raise HeaderError("forward SIP without AP/BP: the image shape is needed to fit the inverse")
        order = inverse_order or min(9, max(w.a_order, w.b_order) + 2)
        dfr_wcs_fit_inverse_sip(w, order, int(nx), int(ny))
    return w


def _as_wcs(obj, shape=None):
    if isinstance(obj, DfrWCS):
        return obj
    if hasattr(obj, "crpix") and hasattr(obj, "cd"):
        return pack_wcs(obj)
    if hasattr(obj, "to_header"):                               # e.g. an astropy.wcs.WCS
        obj = obj.to_header(relax=True)
    return wcs_from_header(obj, shape)


def _split(hdu):
    if isinstance(hdu, (tuple, list)) and len(hdu) == 2:
        return hdu[0], hdu[1]
    if hasattr(hdu, "data") and hasattr(hdu, "header"):
        return hdu.data, hdu.header
    raise TypeError("a source must be an HDU-like object (.data, .header) or an (array, header) pair")


def _gather(source_hdus):
    """-> (single, [float32 2-D arrays], [DfrWCS])."""
    single = not isinstance(source_hdus, (list, tuple)) or (
        len(source_hdus) == 2 and not isinstance(source_hdus[0], (list, tuple)) and not hasattr(source_hdus[0], "header")
        and hasattr(source_hdus[0], "shape"))
    items = [source_hdus] if single else list(source_hdus)
    arrays, wcs = [], []
    for it in items:
        data, hdr = _split(it)
        a = np.ascontiguousarray(data, dtype=np.float32)
        if a.ndim != 2:
            raise ValueError("source images must be 2-D")
        arrays.append(a)
        wcs.append(_as_wcs(hdr, a.shape))
    return single, arrays, wcs


def _groups(arrays):
    """Indices of the sources grouped by image shape (one library call per shape)."""
    by_shape = {}
    for k, a in enumerate(arrays):
        by_shape.setdefault(a.shape, []).append(k)
    return list(by_shape.values())


def calculate_reprojection(source_hdus, target_wcs, shape_out=None, order="bilinear", device="cuda",
                           return_torch=False, return_footprint=False, paper_footprint=False):
    """PAPER.md:30-36. source_hdus: one HDU-like / (array, header) pair, or a list of them
    (each with its own WCS); target_wcs: header mapping, WCS-like object or
    DfrWCS; shape_out defaults to the input shape; order: 'nearest',
    'bilinear', 'bicubic'. Returns [ny][nx] for one source, [n][ny][nx] for a list; pixels
    outside a source's footprint are NaN. return_footprint=True returns (array, footprint)
    like reproject_interp: 1 inside the footprint, 0 outside; with
    paper_footprint=True (nearest / bilinear) the footprint rule is the paper's literal one
    (the projected identity, valid on (-1, n)) and the array is that identity."""
    import torch
    from . import EDGE_AREA, EDGE_PAPER
    single, arrays, wcs = _gather(source_hdus)
    shape_out = tuple(arrays[0].shape) if shape_out is None else (int(shape_out[0]), int(shape_out[1]))
    tgt = _as_wcs(target_wcs, shape_out)
    edge = EDGE_PAPER if paper_footprint else EDGE_AREA
    out = torch.empty((len(arrays),) + shape_out, dtype=torch.float32, device=device)
    foot = torch.empty_like(out) if return_footprint else None
    for idx in _groups(arrays):                     # sources may differ in shape
        src = torch.from_numpy(np.stack([arrays[k] for k in idx])).to(device)
        res = dfr_reproject(src, [wcs[k] for k in idx], tgt, shape_out, order, edge=edge,
                            footprint=True if return_footprint else None)
        res, fp = res if return_footprint else (res, None)
        if len(idx) == len(arrays):
            out, foot = res, fp
        else:
            sel = torch.as_tensor(idx, device=device)
            out[sel] = res
            if return_footprint:
                foot[sel] = fp
    if single:
        out = out[0]
        foot = foot[0] if return_footprint else None
    if not return_torch:
        out = out.cpu().numpy()
        foot = foot.cpu().numpy() if return_footprint else None
    return (out, foot) if return_footprint else out


def calculate_stack(source_hdus, target_wcs, shape_out=None, order="bilinear", weights=None, device="cuda",
                    return_torch=False):
    """The co-added mean of the sources on the target grid and its weight map (the stated
    purpose of reprojection): (mean, wsum), NaN where no source covers a pixel."""
    import torch
    _, arrays, wcs = _gather(source_hdus)
    shape_out = tuple(arrays[0].shape) if shape_out is None else (int(shape_out[0]), int(shape_out[1]))
    tgt = _as_wcs(target_wcs, shape_out)
    weights = None if weights is None else np.asarray(weights, dtype=np.float32)
    s = w = None
    for idx in _groups(arrays):                     # one fused call per source shape, accumulated
        src = torch.from_numpy(np.stack([arrays[k] for k in idx])).to(device)
        s, w = dfr_reproject_stack(src, [wcs[k] for k in idx], tgt, shape_out, order,
                                   weights=None if weights is None else weights[idx],
                                   sum=s, wsum=w, accumulate=s is not None)
    mean = dfr_stack_finalize(s, w)
    return (mean, w) if return_torch else (mean.cpu().numpy(), w.cpu().numpy())
