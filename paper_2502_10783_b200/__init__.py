"""Thin Python binding of libbkgdet (include/bkgdet.h): argument marshalling only.

Every step of the path runs in the CUDA kernels behind the C ABI; PyTorch is used for device memory
and the current stream, nothing else.  There is no CPU fallback: if the shared library is missing or
cannot be loaded, importing the binding's functions raises.
"""
from __future__ import annotations

import ctypes as C
import os
from dataclasses import dataclass

import numpy as np
import torch

from . import _build

__all__ = ["BkgParams", "Context", "SOURCE_DTYPE", "bkg_estimate", "bkg_subtract", "detect_sources", "mesh_stats",
           "grid_filter_spline", "grid_filter_spline_static", "image_reproject", "GRID_STATIC_MAX_DOUBLES", "bkg_subtract_detect", "photometry", "PhotParams", "PHOT_DTYPE", "deblend_sources", "clean_sources", "DeblendParams", "run_host", "grid_shape", "load_library", "EXPORTS"]

EXPORTS = ["bd_create", "bd_destroy", "bd_last_error", "bd_default_bkg_params", "bd_grid_shape",
           "bd_bkg_workspace_bytes", "bd_detect_workspace_bytes", "bd_mesh_stats", "bd_grid_filter_spline",
           "bd_grid_filter_spline_static",
           "bkg_estimate", "bkg_subtract", "detect_sources", "bkg_subtract_detect", "bd_default_phot_params", "bd_phot_workspace_bytes", "photometry",
           "bd_run_host", "bd_default_bkgx_params", "bd_mesh_stats_masked", "bkg_estimate_masked",
           "bd_bkg_iterate_workspace_bytes", "bkg_iterate", "bd_default_conv_params", "bd_conv_num_basis",
           "bd_subtract_workspace_bytes", "image_subtract", "bd_default_deblend_params", "bd_deblend_workspace_bytes",
           "deblend_sources", "bd_clean_workspace_bytes", "clean_sources", "image_reproject"]
DEBUG_EXPORTS = ["bd_debug_k1_slow_meshes", "bd_debug_k1_reasons", "bd_debug_k1_force_slow", "bd_debug_tile_kernel_events"]


class _CParams(C.Structure):
    _fields_ = [("mesh_h", C.c_int32), ("mesh_w", C.c_int32), ("filt_h", C.c_int32), ("filt_w", C.c_int32),
                ("clip_sigma", C.c_double), ("clip_iters", C.c_int32), ("skew_guard", C.c_int32),
                ("median_factor", C.c_double), ("mean_factor", C.c_double)]


SOURCE_DTYPE = np.dtype([
    ("frame", np.int32), ("label", np.int32), ("npix", np.int32), ("xmin", np.int32), ("xmax", np.int32),
    ("ymin", np.int32), ("ymax", np.int32), ("xpeak", np.int32), ("ypeak", np.int32), ("peak", np.float32),
    ("flux", np.float64), ("x", np.float64), ("y", np.float64), ("x2", np.float64), ("y2", np.float64),
    ("xy", np.float64)], align=True)
assert SOURCE_DTYPE.itemsize == 88


@dataclass
class BkgParams:
    mesh_h: int = 64
    mesh_w: int = 64
    filt_h: int = 3
    filt_w: int = 3
    clip_sigma: float = 3.0
    clip_iters: int = 5
    skew_guard: int = 0
    median_factor: float = 3.0
    mean_factor: float = 2.0

    def c(self) -> _CParams:
        return _CParams(self.mesh_h, self.mesh_w, self.filt_h, self.filt_w, self.clip_sigma, self.clip_iters,
                        self.skew_guard, self.median_factor, self.mean_factor)


class _CBkgXParams(C.Structure):
    _fields_ = [("min_valid_px", C.c_int32), ("grow", C.c_int32), ("max_masked_frac", C.c_double), ("max_reject_frac", C.c_double)]


@dataclass
class BkgXParams:
    """bd_bkgx_params: the background variants (readings B1-B6)."""
    min_valid_px: int = 100
    grow: int = 1
    max_masked_frac: float = 1.0
    max_reject_frac: float = 1.0

    def c(self) -> _CBkgXParams:
        return _CBkgXParams(self.min_valid_px, self.grow, self.max_masked_frac, self.max_reject_frac)


def _chk_cat(cat, cat_capacity):
    """The kernels read up to cat_capacity records of 88 bytes from `cat`: the tensor must hold them."""
    if cat_capacity < 0 or cat.numel() < cat_capacity * SOURCE_DTYPE.itemsize:
        raise BkgdetError(f"cat: {cat.numel()} bytes cannot hold cat_capacity = {cat_capacity} records of {SOURCE_DTYPE.itemsize} bytes")


_lib = None


def load_library(build: bool = True):
    """dlopen libbkgdet.so (building it with nvcc first if the sources are newer)."""
    global _lib
    if _lib is None:
        path = _build.build() if build else _build.LIB
        lib = C.CDLL(path)
        lib.bd_last_error.restype = C.c_char_p
        for name in EXPORTS + DEBUG_EXPORTS:
            getattr(lib, name)          # fail loudly if a declared symbol is missing
        _lib = lib
    return _lib


class BkgdetError(RuntimeError):
    pass


def grid_shape(H, W, mesh_h, mesh_w):
    return (H + mesh_h - 1) // mesh_h, (W + mesh_w - 1) // mesh_w


def _ptr(t):
    return C.c_void_p(0 if t is None else t.data_ptr())


def _chk(ctx, t, dtype, name, shape=None, optional=False):
    """A tensor handed to the C ABI must be what its signature says: on ctx's device, of the right dtype, contiguous."""
    if t is None:
        if optional:
            return None
        raise BkgdetError(f"{name}: tensor required")
    if not isinstance(t, torch.Tensor) or not t.is_cuda or t.device.index != ctx.device:
        raise BkgdetError(f"{name}: expected a CUDA tensor on device {ctx.device}, got {getattr(t, 'device', type(t))}")
    if dtype is not None and t.dtype != dtype:
        raise BkgdetError(f"{name}: expected dtype {dtype}, got {t.dtype}")
    if not t.is_contiguous():
        raise BkgdetError(f"{name}: tensor must be contiguous")
    if shape is not None and tuple(t.shape) != tuple(shape):
        raise BkgdetError(f"{name}: expected shape {tuple(shape)}, got {tuple(t.shape)}")
    return t


def _stream(ctx):
    return C.c_void_p(torch.cuda.current_stream(ctx.device).cuda_stream)


class Context:
    """Owns a bd_ctx bound to one CUDA device."""

    def __init__(self, device: int = 0):
        if not torch.cuda.is_available():
            raise BkgdetError("libbkgdet needs a CUDA device (sm_100a); there is no CPU fallback")
        self.lib = load_library()
        self.device = device
        self.h = C.c_void_p()
        rc = self.lib.bd_create(C.byref(self.h), C.c_int(device))
        if rc != 0:
            raise BkgdetError(f"bd_create failed ({rc})")

    def close(self):
        if getattr(self, "h", None) and self.h.value:
            self.lib.bd_destroy(self.h)
            self.h = C.c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def check(self, rc: int):
        if rc != 0:
            raise BkgdetError(f"libbkgdet error {rc}: {self.lib.bd_last_error(self.h).decode()}")

    def bkg_workspace_bytes(self, B, H, W, p: BkgParams) -> int:
        n = C.c_size_t()
        cp = p.c()
        self.check(self.lib.bd_bkg_workspace_bytes(self.h, B, H, W, C.byref(cp), C.byref(n)))
        return n.value

    def detect_workspace_bytes(self, B, H, W, cat_capacity) -> int:
        n = C.c_size_t()
        self.check(self.lib.bd_detect_workspace_bytes(self.h, B, H, W, C.c_int64(cat_capacity), C.byref(n)))
        return n.value


def k1_slow_meshes(ctx: "Context", reset: bool = True) -> int:
    """Diagnostics: meshes that went through K1's general (slow) path since the last reset (synchronises)."""
    n = C.c_ulonglong()
    torch.cuda.synchronize()
    ctx.check(ctx.lib.bd_debug_k1_slow_meshes(C.byref(n), C.c_int(1 if reset else 0)))
    return n.value


def k1_force_slow(ctx: "Context", on: bool) -> None:
    """Diagnostics: make K1 skip its fast path (the tests exercise both paths)."""
    ctx.check(ctx.lib.bd_debug_k1_force_slow(ctx.h, C.c_int(1 if on else 0)))


def tile_kernel_events(ctx: "Context", ev_before, ev_after) -> None:
    """Diagnostics: torch.cuda.Event pair (already recorded once, so that their handles exist) that the library records
    right before / after the tile kernel of detect_sources / bkg_subtract_detect; (None, None) switches it off."""
    h0 = C.c_void_p(0 if ev_before is None else ev_before.cuda_event)
    h1 = C.c_void_p(0 if ev_after is None else ev_after.cuda_event)
    ctx.check(ctx.lib.bd_debug_tile_kernel_events(ctx.h, h0, h1))


def _dev(ctx):
    return torch.device("cuda", ctx.device)


_OUT_DTYPES = dict(sub=torch.float32, bkg=torch.float32, rms=torch.float32, mask=torch.uint8, labels=torch.int32)


def _check_out(ctx, B, H, W, out):
    for k, t in (out or {}).items():
        if t is None:
            continue
        if k in _OUT_DTYPES:
            _chk(ctx, t, _OUT_DTYPES[k], f"out[{k}]", (B, H, W))
        elif k == "cat":
            _chk(ctx, t, torch.uint8, "out[cat]")
        elif k == "n_sources":
            _chk(ctx, t, torch.int64, "out[n_sources]", (B,))


def _check_coef_and_out(ctx, B, H, W, mesh_h, mesh_w, bkg_coef, rms_coef, out):
    ny, nx = grid_shape(H, W, mesh_h, mesh_w)
    _chk(ctx, bkg_coef, torch.float64, "bkg_coef", (B, ny, nx)); _chk(ctx, rms_coef, torch.float64, "rms_coef", (B, ny, nx))
    _check_out(ctx, B, H, W, out)


def mesh_stats(ctx: Context, img: torch.Tensor, p: BkgParams):
    """a1 (K1).  img float32 [B,H,W] on the device -> dict of [B,ny,nx] tensors."""
    _chk(ctx, img, torch.float32, "img")
    B, H, W = img.shape
    ny, nx = grid_shape(H, W, p.mesh_h, p.mesh_w)
    dev = _dev(ctx)
    out = {k: torch.empty((B, ny, nx), dtype=torch.float64, device=dev) for k in ("bkg", "rms", "median", "mean")}
    out["n_kept"] = torch.empty((B, ny, nx), dtype=torch.int32, device=dev)
    cp = p.c()
    ws = torch.empty(ctx.bkg_workspace_bytes(B, H, W, p), dtype=torch.uint8, device=dev)
    ctx.check(ctx.lib.bd_mesh_stats(ctx.h, _ptr(img), B, H, W, C.byref(cp), _ptr(out["bkg"]), _ptr(out["rms"]),
                                    _ptr(out["median"]), _ptr(out["mean"]), _ptr(out["n_kept"]), _ptr(ws),
                                    C.c_size_t(ws.numel()), _stream(ctx)))
    return out


def mesh_stats_masked(ctx: Context, img: torch.Tensor, bad: torch.Tensor | None, p: BkgParams, px: BkgXParams):
    """a1 with a bad-pixel mask / validity rules (NEXT-3).  -> dict as mesh_stats plus n_valid; invalid meshes hold NaN."""
    _chk(ctx, img, torch.float32, "img"); _chk(ctx, bad, torch.uint8, "bad", img.shape, optional=True)
    B, H, W = img.shape
    ny, nx = grid_shape(H, W, p.mesh_h, p.mesh_w)
    dev = _dev(ctx)
    out = {k: torch.empty((B, ny, nx), dtype=torch.float64, device=dev) for k in ("bkg", "rms", "median", "mean")}
    out["n_kept"] = torch.empty((B, ny, nx), dtype=torch.int32, device=dev)
    out["n_valid"] = torch.empty((B, ny, nx), dtype=torch.int32, device=dev)
    cp, cx = p.c(), px.c()
    ws = torch.empty(ctx.bkg_workspace_bytes(B, H, W, p), dtype=torch.uint8, device=dev)
    ctx.check(ctx.lib.bd_mesh_stats_masked(ctx.h, _ptr(img), _ptr(bad), B, H, W, C.byref(cp), C.byref(cx), _ptr(out["bkg"]),
                                           _ptr(out["rms"]), _ptr(out["median"]), _ptr(out["mean"]), _ptr(out["n_kept"]),
                                           _ptr(out["n_valid"]), _ptr(ws), C.c_size_t(ws.numel()), _stream(ctx)))
    return out


def _grids(ctx, B, ny, nx):
    dev = _dev(ctx)
    bm = torch.empty((B, ny, nx), dtype=torch.float32, device=dev); rm = torch.empty_like(bm)
    cb = torch.empty((B, ny, nx), dtype=torch.float64, device=dev); cr = torch.empty_like(cb)
    return bm, rm, cb, cr, torch.empty((B, ny, nx), dtype=torch.uint8, device=dev)


def bkg_estimate_masked(ctx: Context, img: torch.Tensor, bad: torch.Tensor | None, p: BkgParams, px: BkgXParams,
                        ws: torch.Tensor | None = None):
    """a1 + fill + a2 with the variants (NEXT-3).  -> (bkg_mesh, rms_mesh, bkg_coef, rms_coef, valid_mesh u8)."""
    _chk(ctx, img, torch.float32, "img"); _chk(ctx, bad, torch.uint8, "bad", img.shape, optional=True)
    B, H, W = img.shape
    bm, rm, cb, cr, valid = _grids(ctx, B, *grid_shape(H, W, p.mesh_h, p.mesh_w))
    if ws is None:
        ws = torch.empty(ctx.bkg_workspace_bytes(B, H, W, p), dtype=torch.uint8, device=_dev(ctx))
    cp, cx = p.c(), px.c()
    ctx.check(ctx.lib.bkg_estimate_masked(ctx.h, _ptr(img), _ptr(bad), B, H, W, C.byref(cp), C.byref(cx), _ptr(bm), _ptr(rm),
                                          _ptr(cb), _ptr(cr), _ptr(valid), _ptr(ws), C.c_size_t(ws.numel()), _stream(ctx)))
    return bm, rm, cb, cr, valid


def bkg_iterate(ctx: Context, img: torch.Tensor, bad0: torch.Tensor | None, p: BkgParams, px: BkgXParams, detect_k: float,
                n_iter: int, ws: torch.Tensor | None = None):
    """Iterated background estimation (NEXT-3, B4).  -> (bkg_mesh, rms_mesh, bkg_coef, rms_coef, valid_mesh, bad_out u8 [B,H,W])."""
    _chk(ctx, img, torch.float32, "img"); _chk(ctx, bad0, torch.uint8, "bad0", img.shape, optional=True)
    B, H, W = img.shape
    bm, rm, cb, cr, valid = _grids(ctx, B, *grid_shape(H, W, p.mesh_h, p.mesh_w))
    bad_out = torch.empty((B, H, W), dtype=torch.uint8, device=_dev(ctx))
    cp, cx = p.c(), px.c()
    if ws is None:
        n = C.c_size_t()
        ctx.check(ctx.lib.bd_bkg_iterate_workspace_bytes(ctx.h, B, H, W, C.byref(cp), C.byref(n)))
        ws = torch.empty(n.value, dtype=torch.uint8, device=_dev(ctx))
    ctx.check(ctx.lib.bkg_iterate(ctx.h, _ptr(img), _ptr(bad0), B, H, W, C.byref(cp), C.byref(cx), C.c_double(detect_k),
                                  C.c_int(n_iter), _ptr(bm), _ptr(rm), _ptr(cb), _ptr(cr), _ptr(valid), _ptr(bad_out), _ptr(ws),
                                  C.c_size_t(ws.numel()), _stream(ctx)))
    return bm, rm, cb, cr, valid, bad_out


def grid_filter_spline(ctx: Context, bkg_raw: torch.Tensor, rms_raw: torch.Tensor, filt_h: int, filt_w: int):
    """a2 (K2).  raw grids float64 [B,ny,nx] -> (bkg_mesh f32, rms_mesh f32, bkg_coef f64, rms_coef f64)."""
    _chk(ctx, bkg_raw, torch.float64, "bkg_raw"); _chk(ctx, rms_raw, torch.float64, "rms_raw", bkg_raw.shape)
    B, ny, nx = bkg_raw.shape
    dev = _dev(ctx)
    bm = torch.empty((B, ny, nx), dtype=torch.float32, device=dev); rm = torch.empty_like(bm)
    cb = torch.empty((B, ny, nx), dtype=torch.float64, device=dev); cr = torch.empty_like(cb)
    ws = torch.empty(4 * B * (ny + nx) + 32, dtype=torch.float64, device=dev)
    ctx.check(ctx.lib.bd_grid_filter_spline(ctx.h, _ptr(bkg_raw), _ptr(rms_raw), B, ny, nx, filt_h, filt_w, _ptr(bm),
                                            _ptr(rm), _ptr(cb), _ptr(cr), _ptr(ws), C.c_size_t(ws.numel() * 8), _stream(ctx)))
    return bm, rm, cb, cr


GRID_STATIC_MAX_DOUBLES = 32768   # BD_GRID_STATIC_MAX_DOUBLES of bkgdet.h


def grid_filter_spline_static(ctx: Context, bkg_raw: torch.Tensor, rms_raw: torch.Tensor, filt_h: int, filt_w: int, out=None):
    """a2 (K2) through bd_grid_filter_spline_static: the call for code that cannot allocate device memory.

    Same inputs and results as grid_filter_spline, but no workspace is allocated or passed: the kernel's scratch is a
    256 KiB array built into libbkgdet (one per GPU, shared by every call, so calls must not overlap on the GPU).
    Meant for callers that work inside someone else's memory budget -- a plug-in given a fixed set of buffers, a
    real-time loop that must stay out of the CUDA allocator -- who pass their own output tensors as
    out = (bkg_mesh f32, rms_mesh f32, bkg_coef f64, rms_coef f64), each [B,ny,nx]; with out=None the four outputs are
    made with torch.empty here (which does allocate: convenience for tests).  Raises BkgdetError when
    4*B*(ny+nx) > GRID_STATIC_MAX_DOUBLES."""
    _chk(ctx, bkg_raw, torch.float64, "bkg_raw"); _chk(ctx, rms_raw, torch.float64, "rms_raw", bkg_raw.shape)
    B, ny, nx = bkg_raw.shape
    if out is None:
        dev = _dev(ctx)
        bm = torch.empty((B, ny, nx), dtype=torch.float32, device=dev); rm = torch.empty_like(bm)
        cb = torch.empty((B, ny, nx), dtype=torch.float64, device=dev); cr = torch.empty_like(cb)
    else:
        bm, rm, cb, cr = out
        _chk(ctx, bm, torch.float32, "bkg_mesh", bkg_raw.shape); _chk(ctx, rm, torch.float32, "rms_mesh", bkg_raw.shape)
        _chk(ctx, cb, torch.float64, "bkg_coef", bkg_raw.shape); _chk(ctx, cr, torch.float64, "rms_coef", bkg_raw.shape)
    ctx.check(ctx.lib.bd_grid_filter_spline_static(ctx.h, _ptr(bkg_raw), _ptr(rms_raw), B, ny, nx, filt_h, filt_w, _ptr(bm),
                                                   _ptr(rm), _ptr(cb), _ptr(cr), _stream(ctx)))
    return bm, rm, cb, cr


def bkg_estimate(ctx: Context, img: torch.Tensor, p: BkgParams, ws: torch.Tensor | None = None):
    """a1 + a2.  -> (bkg_mesh f32, rms_mesh f32, bkg_coef f64, rms_coef f64), each [B,ny,nx]."""
    _chk(ctx, img, torch.float32, "img"); _chk(ctx, ws, torch.uint8, "ws", optional=True)
    B, H, W = img.shape
    ny, nx = grid_shape(H, W, p.mesh_h, p.mesh_w)
    dev = _dev(ctx)
    bm = torch.empty((B, ny, nx), dtype=torch.float32, device=dev); rm = torch.empty_like(bm)
    cb = torch.empty((B, ny, nx), dtype=torch.float64, device=dev); cr = torch.empty_like(cb)
    if ws is None:
        ws = torch.empty(ctx.bkg_workspace_bytes(B, H, W, p), dtype=torch.uint8, device=dev)
    cp = p.c()
    ctx.check(ctx.lib.bkg_estimate(ctx.h, _ptr(img), B, H, W, C.byref(cp), _ptr(bm), _ptr(rm), _ptr(cb), _ptr(cr),
                                   _ptr(ws), C.c_size_t(ws.numel()), _stream(ctx)))
    return bm, rm, cb, cr


def bkg_subtract(ctx: Context, img: torch.Tensor, mesh_h: int, mesh_w: int, bkg_coef: torch.Tensor,
                 rms_coef: torch.Tensor, detect_k: float, want_bkg: bool = True, want_rms: bool = True,
                 want_mask: bool = True, out: dict | None = None):
    """a3 (K3).  -> dict(sub, bkg, rms float32 [B,H,W]; mask uint8 [B,H,W]); absent outputs are None."""
    _chk(ctx, img, torch.float32, "img")
    B, H, W = img.shape
    _check_coef_and_out(ctx, B, H, W, mesh_h, mesh_w, bkg_coef, rms_coef, out)
    dev = _dev(ctx)
    o = out or {}
    sub = o.get("sub") if o.get("sub") is not None else torch.empty((B, H, W), dtype=torch.float32, device=dev)
    bkg = (o.get("bkg") if o.get("bkg") is not None else torch.empty_like(sub)) if want_bkg else None
    rms = (o.get("rms") if o.get("rms") is not None else torch.empty_like(sub)) if want_rms else None
    mask = (o.get("mask") if o.get("mask") is not None else torch.empty((B, H, W), dtype=torch.uint8, device=dev)) if want_mask else None
    ctx.check(ctx.lib.bkg_subtract(ctx.h, _ptr(img), B, H, W, mesh_h, mesh_w, _ptr(bkg_coef), _ptr(rms_coef),
                                   C.c_double(detect_k), _ptr(sub), _ptr(bkg), _ptr(rms), _ptr(mask), _stream(ctx)))
    return dict(sub=sub, bkg=bkg, rms=rms, mask=mask)


def detect_sources(ctx: Context, sub: torch.Tensor, rms: torch.Tensor | None, mask: torch.Tensor | None,
                   detect_k: float, min_area: int, cat_capacity: int, ws: torch.Tensor | None = None,
                   out: dict | None = None):
    """a4 + a5 (K4, K5).  -> dict(labels int32 [B,H,W], cat uint8 [cap*88] (device), n_sources int64 [B])."""
    _chk(ctx, sub, torch.float32, "sub")
    B, H, W = sub.shape
    _chk(ctx, rms, torch.float32, "rms", (B, H, W), optional=True); _chk(ctx, mask, torch.uint8, "mask", (B, H, W), optional=True)
    _chk(ctx, ws, torch.uint8, "ws", optional=True)
    _check_out(ctx, B, H, W, out)
    dev = _dev(ctx)
    o = out or {}
    labels = o.get("labels") if o.get("labels") is not None else torch.empty((B, H, W), dtype=torch.int32, device=dev)
    cat = o.get("cat") if o.get("cat") is not None else torch.empty(max(cat_capacity, 1) * SOURCE_DTYPE.itemsize, dtype=torch.uint8, device=dev)
    nsrc = o.get("n_sources") if o.get("n_sources") is not None else torch.empty(B, dtype=torch.int64, device=dev)
    if ws is None:
        ws = torch.empty(ctx.detect_workspace_bytes(B, H, W, cat_capacity), dtype=torch.uint8, device=dev)
    ctx.check(ctx.lib.detect_sources(ctx.h, _ptr(sub), _ptr(rms), _ptr(mask), B, H, W, C.c_double(detect_k),
                                     C.c_int32(min_area), _ptr(labels), _ptr(cat), C.c_int64(cat_capacity), _ptr(nsrc),
                                     _ptr(ws), C.c_size_t(ws.numel()), _stream(ctx)))
    return dict(labels=labels, cat=cat, n_sources=nsrc)


def bkg_subtract_detect(ctx: Context, img: torch.Tensor, mesh_h: int, mesh_w: int, bkg_coef: torch.Tensor,
                        rms_coef: torch.Tensor, detect_k: float, min_area: int, cat_capacity: int,
                        want_bkg: bool = True, want_rms: bool = True, want_mask: bool = True,
                        ws: torch.Tensor | None = None, out: dict | None = None):
    """a3 + a4 + a5 in one pass.  -> dict(sub, bkg, rms, mask, labels, cat, n_sources)."""
    _chk(ctx, img, torch.float32, "img"); _chk(ctx, ws, torch.uint8, "ws", optional=True)
    B, H, W = img.shape
    _check_coef_and_out(ctx, B, H, W, mesh_h, mesh_w, bkg_coef, rms_coef, out)
    dev = _dev(ctx)
    o = out or {}
    def buf(key, dtype, want=True):
        if not want:
            return None
        return o.get(key) if o.get(key) is not None else torch.empty((B, H, W), dtype=dtype, device=dev)
    sub = buf("sub", torch.float32); bkg = buf("bkg", torch.float32, want_bkg); rms = buf("rms", torch.float32, want_rms)
    mask = buf("mask", torch.uint8, want_mask); labels = buf("labels", torch.int32)
    cat = o.get("cat") if o.get("cat") is not None else torch.empty(max(cat_capacity, 1) * SOURCE_DTYPE.itemsize, dtype=torch.uint8, device=dev)
    nsrc = o.get("n_sources") if o.get("n_sources") is not None else torch.empty(B, dtype=torch.int64, device=dev)
    if ws is None:
        ws = torch.empty(ctx.detect_workspace_bytes(B, H, W, cat_capacity), dtype=torch.uint8, device=dev)
    ctx.check(ctx.lib.bkg_subtract_detect(ctx.h, _ptr(img), B, H, W, mesh_h, mesh_w, _ptr(bkg_coef), _ptr(rms_coef),
                                          C.c_double(detect_k), C.c_int32(min_area), _ptr(sub), _ptr(bkg), _ptr(rms),
                                          _ptr(mask), _ptr(labels), _ptr(cat), C.c_int64(cat_capacity), _ptr(nsrc),
                                          _ptr(ws), C.c_size_t(ws.numel()), _stream(ctx)))
    return dict(sub=sub, bkg=bkg, rms=rms, mask=mask, labels=labels, cat=cat, n_sources=nsrc)


class _CConvParams(C.Structure):
    _fields_ = [("half_width", C.c_int32), ("n_gauss", C.c_int32), ("sigma", C.c_double * 4), ("degree", C.c_int32 * 4),
                ("spatial_order", C.c_int32), ("bg_order", C.c_int32)]


class ConvParams:
    """bd_conv_params (NEXT-4): kernel half-width, Gaussian widths and polynomial degrees, spatial and background orders."""

    def __init__(self, half_width=10, sigma=(0.7, 1.5, 3.0), degree=(6, 4, 2), spatial_order=2, bg_order=1):
        assert len(sigma) == len(degree) <= 4
        c = _CConvParams()
        c.half_width, c.n_gauss, c.spatial_order, c.bg_order = half_width, len(sigma), spatial_order, bg_order
        for g in range(4):
            c.sigma[g] = sigma[g] if g < len(sigma) else 1.0
            c.degree[g] = degree[g] if g < len(degree) else 0
        self._c = c
        self.half_width, self.sigma, self.degree, self.spatial_order, self.bg_order = half_width, tuple(sigma), tuple(degree), spatial_order, bg_order

    @property
    def n_basis(self):
        return int(load_library().bd_conv_num_basis(C.byref(self._c)))

    @property
    def n_sp(self):
        return (self.spatial_order + 1) * (self.spatial_order + 2) // 2

    @property
    def n_bg(self):
        return (self.bg_order + 1) * (self.bg_order + 2) // 2


def image_subtract(ctx: Context, ref: torch.Tensor, img: torch.Tensor, p: ConvParams, kcoef: torch.Tensor, bgcoef: torch.Tensor,
                   want_conv: bool = False, out: dict | None = None):
    """NEXT-4 (K8): diff = img + B - ref (x) K with one kernel per 21x21 stamp.  kcoef float64 [B, n_basis, n_sp], bgcoef
    float64 [B, n_bg].  -> dict(diff, conv or None)."""
    _chk(ctx, ref, torch.float32, "ref"); _chk(ctx, img, torch.float32, "img", ref.shape)
    B, H, W = ref.shape
    _chk(ctx, kcoef, torch.float64, "kcoef", (B, p.n_basis, p.n_sp)); _chk(ctx, bgcoef, torch.float64, "bgcoef", (B, p.n_bg))
    o = out or {}
    diff = o.get("diff") if o.get("diff") is not None else torch.empty_like(ref)
    conv = (o.get("conv") if o.get("conv") is not None else torch.empty_like(ref)) if want_conv else None
    n = C.c_size_t()
    ctx.check(ctx.lib.bd_subtract_workspace_bytes(ctx.h, B, C.byref(p._c), C.byref(n)))
    ws = o.get("ws") if o.get("ws") is not None else torch.empty(n.value, dtype=torch.uint8, device=_dev(ctx))
    ctx.check(ctx.lib.image_subtract(ctx.h, _ptr(ref), _ptr(img), B, H, W, C.byref(p._c), _ptr(kcoef), _ptr(bgcoef), _ptr(diff),
                                     _ptr(conv), _ptr(ws), C.c_size_t(ws.numel()), _stream(ctx)))
    return dict(diff=diff, conv=conv)


PHOT_DTYPE = np.dtype([("flux_aper", np.float64), ("fluxerr_aper", np.float64), ("area_aper", np.float64),
                       ("kron_radius", np.float64), ("flux_auto", np.float64), ("fluxerr_auto", np.float64),
                       ("npix_auto", np.int32), ("flags", np.int32)], align=True)


class _CPhotParams(C.Structure):
    _fields_ = [("r_aper", C.c_double), ("kron_factor", C.c_double), ("kron_min_radius", C.c_double),
                ("kron_search", C.c_double), ("subpix", C.c_int32), ("pad", C.c_int32)]


class PhotParams:
    """bd_phot_params (defaults from bd_default_phot_params)."""

    def __init__(self, **kw):
        c = _CPhotParams()
        load_library().bd_default_phot_params(C.byref(c))
        for k, v in kw.items():
            if not hasattr(c, k):
                raise TypeError(f"unknown photometry parameter {k}")
            setattr(c, k, v)
        self._c = c

    def __getattr__(self, k):
        return getattr(self._c, k)


def photometry(ctx: Context, sub: torch.Tensor, rms: torch.Tensor, cat: torch.Tensor, n_sources: torch.Tensor,
               cat_capacity: int, p: "PhotParams | None" = None, out: torch.Tensor | None = None,
               ws: torch.Tensor | None = None) -> torch.Tensor:
    """NEXT-2 (K6): aperture + auto photometry of the catalogue records.  -> uint8 [cap*56] device bytes (PHOT_DTYPE)."""
    _chk(ctx, sub, torch.float32, "sub")
    B, H, W = sub.shape
    _chk(ctx, rms, torch.float32, "rms", (B, H, W)); _chk(ctx, cat, torch.uint8, "cat"); _chk(ctx, n_sources, torch.int64, "n_sources", (B,))
    _chk(ctx, out, torch.uint8, "out", optional=True); _chk(ctx, ws, torch.uint8, "ws", optional=True)
    p = p or PhotParams()
    if out is None:
        out = torch.zeros(max(cat_capacity, 1) * PHOT_DTYPE.itemsize, dtype=torch.uint8, device=_dev(ctx))
    if ws is None:
        nb = C.c_size_t()
        ctx.check(ctx.lib.bd_phot_workspace_bytes(ctx.h, C.c_int64(cat_capacity), C.byref(nb)))
        ws = torch.empty(nb.value, dtype=torch.uint8, device=_dev(ctx))
    ctx.check(ctx.lib.photometry(ctx.h, _ptr(sub), _ptr(rms), B, H, W, _ptr(cat), _ptr(n_sources), C.c_int64(cat_capacity),
                                 C.byref(p._c), _ptr(out), _ptr(ws), C.c_size_t(ws.numel()), _stream(ctx)))
    return out


class _CDeblendParams(C.Structure):
    _fields_ = [("n_thresh", C.c_int32), ("pad", C.c_int32), ("min_cont", C.c_double), ("clean_param", C.c_double),
                ("clean_zone", C.c_double)]


class DeblendParams:
    """bd_deblend_params (defaults from bd_default_deblend_params)."""

    def __init__(self, **kw):
        c = _CDeblendParams()
        load_library().bd_default_deblend_params(C.byref(c))
        for k, v in kw.items():
            if not hasattr(c, k):
                raise TypeError(f"unknown deblending parameter {k}")
            setattr(c, k, v)
        self._c = c

    def __getattr__(self, k):
        return getattr(self._c, k)


def deblend_sources(ctx: Context, sub: torch.Tensor, rms: torch.Tensor, labels: torch.Tensor, cat: torch.Tensor,
                    n_sources: torch.Tensor, cat_capacity: int, detect_k: float, min_area: int,
                    p: "DeblendParams | None" = None, out_capacity: int | None = None, ws: torch.Tensor | None = None):
    """NEXT-1 (K9): multi-threshold deblending of the candidates.  `labels` is updated IN PLACE.
    -> dict(labels, cat uint8 [out_capacity*88] (device), n_sources int64 [B])."""
    _chk(ctx, sub, torch.float32, "sub")
    B, H, W = sub.shape
    _chk(ctx, rms, torch.float32, "rms", (B, H, W)); _chk(ctx, labels, torch.int32, "labels", (B, H, W))
    _chk(ctx, cat, torch.uint8, "cat"); _chk(ctx, n_sources, torch.int64, "n_sources", (B,)); _chk(ctx, ws, torch.uint8, "ws", optional=True)
    _chk_cat(cat, cat_capacity)
    p = p or DeblendParams()
    cap_out = cat_capacity if out_capacity is None else out_capacity
    dev = _dev(ctx)
    cat_out = torch.empty(max(cap_out, 1) * SOURCE_DTYPE.itemsize, dtype=torch.uint8, device=dev)
    n_out = torch.empty(B, dtype=torch.int64, device=dev)
    if ws is None:
        nb = C.c_size_t()
        ctx.check(ctx.lib.bd_deblend_workspace_bytes(ctx.h, B, H, W, C.c_int64(cat_capacity), C.c_int64(cap_out), C.byref(nb)))
        ws = torch.empty(nb.value, dtype=torch.uint8, device=dev)
    ctx.check(ctx.lib.deblend_sources(ctx.h, _ptr(sub), _ptr(rms), B, H, W, C.c_double(detect_k), C.c_int32(min_area),
                                      C.byref(p._c), _ptr(labels), _ptr(cat), _ptr(n_sources), C.c_int64(cat_capacity),
                                      _ptr(cat_out), C.c_int64(cap_out), _ptr(n_out), _ptr(ws), C.c_size_t(ws.numel()),
                                      _stream(ctx)))
    return dict(labels=labels, cat=cat_out, n_sources=n_out)


def clean_sources(ctx: Context, rms: torch.Tensor, labels: torch.Tensor, cat: torch.Tensor, n_sources: torch.Tensor,
                  cat_capacity: int, detect_k: float, p: "DeblendParams | None" = None, ws: torch.Tensor | None = None):
    """NEXT-1 (K10): cleaning.  `labels` is updated IN PLACE.
    -> dict(labels, cat uint8 [cap*88] (device), n_sources int64 [B], flags uint8 [cap])."""
    _chk(ctx, rms, torch.float32, "rms")
    B, H, W = rms.shape
    _chk(ctx, labels, torch.int32, "labels", (B, H, W)); _chk(ctx, cat, torch.uint8, "cat")
    _chk(ctx, n_sources, torch.int64, "n_sources", (B,)); _chk(ctx, ws, torch.uint8, "ws", optional=True)
    _chk_cat(cat, cat_capacity)
    p = p or DeblendParams()
    dev = _dev(ctx)
    cat_out = torch.empty(max(cat_capacity, 1) * SOURCE_DTYPE.itemsize, dtype=torch.uint8, device=dev)
    n_out = torch.empty(B, dtype=torch.int64, device=dev)
    flags = torch.zeros(max(cat_capacity, 1), dtype=torch.uint8, device=dev)
    if ws is None:
        nb = C.c_size_t()
        ctx.check(ctx.lib.bd_clean_workspace_bytes(ctx.h, B, H, W, C.c_int64(cat_capacity), C.byref(nb)))
        ws = torch.empty(nb.value, dtype=torch.uint8, device=dev)
    ctx.check(ctx.lib.clean_sources(ctx.h, _ptr(rms), B, H, W, C.c_double(detect_k), C.byref(p._c), _ptr(labels), _ptr(cat),
                                    _ptr(n_sources), C.c_int64(cat_capacity), _ptr(cat_out), C.c_int64(cat_capacity), _ptr(n_out),
                                    _ptr(flags), _ptr(ws), C.c_size_t(ws.numel()), _stream(ctx)))
    return dict(labels=labels, cat=cat_out, n_sources=n_out, flags=flags)


def phot_to_numpy(phot: torch.Tensor, n_sources: torch.Tensor, cat_capacity: int) -> np.ndarray:
    n = int(min(int(n_sources.sum().item()), cat_capacity))
    return phot[: n * PHOT_DTYPE.itemsize].cpu().numpy().view(PHOT_DTYPE).copy()


def catalogue_to_numpy(cat: torch.Tensor, n_sources: torch.Tensor, cat_capacity: int) -> np.ndarray:
    """Device catalogue bytes -> numpy structured array of the valid records (synchronises)."""
    n = int(min(int(n_sources.sum().item()), cat_capacity))
    raw = cat[: n * SOURCE_DTYPE.itemsize].cpu().numpy()
    return raw.view(SOURCE_DTYPE).copy()


def run_host(ctx: Context, img: np.ndarray, p: BkgParams, detect_k: float, min_area: int, cat_capacity: int,
             cat: np.ndarray | None = None):
    """Whole chain from a HOST float32 array [B,H,W] (bd_run_host).  -> (records, n_sources[B])."""
    assert img.dtype == np.float32 and img.ndim == 3 and img.flags.c_contiguous
    B, H, W = img.shape
    if cat is None:
        cat = np.empty(max(cat_capacity, 1), dtype=SOURCE_DTYPE)
    n = np.zeros(B, dtype=np.int64)
    cp = p.c()
    ctx.check(ctx.lib.bd_run_host(ctx.h, C.c_void_p(img.ctypes.data), B, H, W, C.byref(cp), C.c_double(detect_k),
                                  C.c_int32(min_area), C.c_void_p(cat.ctypes.data), C.c_int64(cat_capacity),
                                  C.c_void_p(n.ctypes.data)))
    return cat[: min(int(n.sum()), cat_capacity)], n


def image_reproject(ctx: Context, src: torch.Tensor, affine: torch.Tensor, out_shape=None, fill: float = 0.0, out: torch.Tensor | None = None):
    """NEXT-4, second half (K11): bilinear reprojection.  src float32 [B,Hs,Ws]; affine float64 [B,6] (or [B,2,3]) on the
    device, the forward map source -> result (R1); out_shape (Hd, Wd), default the source's.  -> float32 [B,Hd,Wd]."""
    _chk(ctx, src, torch.float32, "src")
    B, Hs, Ws = src.shape
    _chk(ctx, affine, torch.float64, "affine")
    if affine.numel() != B * 6:
        raise BkgdetError(f"affine: expected {B} x 6 numbers, got {tuple(affine.shape)}")
    Hd, Wd = (Hs, Ws) if out_shape is None else out_shape
    if out is None:
        out = torch.empty((B, Hd, Wd), dtype=torch.float32, device=_dev(ctx))
    _chk(ctx, out, torch.float32, "out", (B, Hd, Wd))
    ctx.check(ctx.lib.image_reproject(ctx.h, _ptr(src), B, Hs, Ws, _ptr(affine), C.c_double(fill), _ptr(out), Hd, Wd, _stream(ctx)))
    return out
