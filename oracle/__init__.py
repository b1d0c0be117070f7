"""CPU oracle for the background + detection hot path (TEST INFRASTRUCTURE).

Plain float64 C (``oracle.c``) behind a ctypes wrapper.  Only ``tests/``,
``__graft_entry__.smoke()`` and ``bench.py``'s ``cpu_baseline`` / ``--impl reference`` legs may import
this package.  It shares no code with ``paper_2502_10783_b200`` and never imports it.

Steps O1..O6 follow PAPER.md:67-80 and :153-159 with the readings A1..A22 listed in DESIGN.md.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess
from dataclasses import dataclass

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "oracle.c")
_LIB = os.path.join(_HERE, "liboracle.so")


def build(force: bool = False) -> str:
    """Compile oracle.c with gcc (plain C11, -O2, OpenMP over independent outer loops)."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        subprocess.check_call(["gcc", "-std=c11", "-O2", "-fopenmp", "-shared", "-fPIC", _SRC,
                               "-o", _LIB, "-lm"])
    return _LIB


_lib = None


def lib():
    global _lib
    if _lib is None:
        _lib = C.CDLL(build())
        _lib.o6_reduce.restype = C.c_int64
        _lib.o6_source_size.restype = C.c_int
    return _lib


SOURCE_DTYPE = np.dtype([
    ("label", np.int32), ("npix", np.int32), ("xmin", np.int32), ("xmax", np.int32),
    ("ymin", np.int32), ("ymax", np.int32), ("xpeak", np.int32), ("ypeak", np.int32),
    ("peak", np.float64), ("flux", np.float64), ("x", np.float64), ("y", np.float64),
    ("x2", np.float64), ("y2", np.float64), ("xy", np.float64)], align=True)


def _p(a):
    return a.ctypes.data_as(C.c_void_p)


@dataclass
class BkgParams:
    mesh_h: int = 64
    mesh_w: int = 64
    filt_h: int = 3
    filt_w: int = 3
    clip_sigma: float = 3.0
    clip_iters: int = 5
    median_factor: float = 3.0
    mean_factor: float = 2.0
    skew_guard: int = 0


def grid_shape(H, W, mh, mw):
    return (H + mh - 1) // mh, (W + mw - 1) // mw


def mesh_stats(img: np.ndarray, p: BkgParams):
    """O1.  img float32 [H,W] -> dict of [ny,nx] arrays (bkg, rms float64; n_kept int32; median, mean, rounds)."""
    img = np.ascontiguousarray(img, dtype=np.float32)
    H, W = img.shape
    ny, nx = grid_shape(H, W, p.mesh_h, p.mesh_w)
    bkg = np.empty((ny, nx)); rms = np.empty((ny, nx)); med = np.empty((ny, nx)); mean = np.empty((ny, nx))
    nk = np.empty((ny, nx), dtype=np.int32); rounds = np.empty((ny, nx), dtype=np.int32)
    lib().o1_mesh_stats(_p(img), C.c_int(H), C.c_int(W), C.c_int(p.mesh_h), C.c_int(p.mesh_w),
                        C.c_double(p.clip_sigma), C.c_int(p.clip_iters), C.c_double(p.median_factor),
                        C.c_double(p.mean_factor), C.c_int(p.skew_guard), _p(bkg), _p(rms), _p(nk),
                        _p(med), _p(mean), _p(rounds))
    return dict(bkg=bkg, rms=rms, n_kept=nk, median=med, mean=mean, rounds=rounds)


@dataclass
class BkgXParams:
    """Background variants (readings B1-B6): PAPER.md:67 (mask-defined regions, >= 100 pixels), :181 (iteration)."""
    min_valid_px: int = 100          # B2: a mesh with fewer unmasked pixels is invalid
    grow: int = 1                    # B5: Chebyshev radius by which detections are grown before they are masked
    max_masked_frac: float = 1.0     # B2: invalid if more than this fraction of the mesh is masked (1 = never)
    max_reject_frac: float = 1.0     # B6: invalid if the clipping rejected more than this fraction (1 = never)


def mesh_stats_masked(img: np.ndarray, bad: np.ndarray | None, p: BkgParams, xp: BkgXParams):
    """O1 with a bad-pixel mask and the validity rules B1, B2, B6.  Invalid meshes hold NaN (n_kept 0)."""
    img = np.ascontiguousarray(img, dtype=np.float32)
    H, W = img.shape
    if bad is not None:
        bad = np.ascontiguousarray(bad, dtype=np.uint8)
        assert bad.shape == img.shape
    ny, nx = grid_shape(H, W, p.mesh_h, p.mesh_w)
    bkg = np.empty((ny, nx)); rms = np.empty((ny, nx)); med = np.empty((ny, nx)); mean = np.empty((ny, nx))
    nk = np.empty((ny, nx), dtype=np.int32); rounds = np.empty((ny, nx), dtype=np.int32); nv = np.empty((ny, nx), dtype=np.int32)
    lib().o1_mesh_stats_masked(_p(img), _p(bad) if bad is not None else None, C.c_int(H), C.c_int(W), C.c_int(p.mesh_h),
                               C.c_int(p.mesh_w), C.c_double(p.clip_sigma), C.c_int(p.clip_iters), C.c_double(p.median_factor),
                               C.c_double(p.mean_factor), C.c_int(p.skew_guard), C.c_int(xp.min_valid_px),
                               C.c_double(xp.max_masked_frac), C.c_double(xp.max_reject_frac), _p(bkg), _p(rms), _p(nk),
                               _p(med), _p(mean), _p(rounds), _p(nv))
    return dict(bkg=bkg, rms=rms, n_kept=nk, median=med, mean=mean, rounds=rounds, n_valid=nv)


def grid_median(grid: np.ndarray, fh: int, fw: int) -> np.ndarray:
    """O2."""
    grid = np.ascontiguousarray(grid, dtype=np.float64)
    out = np.empty_like(grid)
    lib().o2_grid_median(_p(grid), C.c_int(grid.shape[0]), C.c_int(grid.shape[1]), C.c_int(fh), C.c_int(fw), _p(out))
    return out


def spline_coeffs(grid: np.ndarray) -> np.ndarray:
    """O3, prefilter: cubic B-spline coefficients of the grid samples."""
    grid = np.ascontiguousarray(grid, dtype=np.float64)
    out = np.empty_like(grid)
    lib().o3_spline_coeffs(_p(grid), C.c_int(grid.shape[0]), C.c_int(grid.shape[1]), _p(out))
    return out


def spline_eval(coef: np.ndarray, H: int, W: int, mh: int, mw: int) -> np.ndarray:
    """O3, evaluation at every pixel centre -> float64 [H,W]."""
    coef = np.ascontiguousarray(coef, dtype=np.float64)
    out = np.empty((H, W))
    lib().o3_spline_eval(_p(coef), C.c_int(coef.shape[0]), C.c_int(coef.shape[1]), C.c_int(H), C.c_int(W),
                         C.c_int(mh), C.c_int(mw), _p(out))
    return out


def subtract_threshold(img, bkg64, rms64, k_d):
    """O3b/O4 -> (sub64, sub32, mask u8, fragile u8)."""
    img = np.ascontiguousarray(img, dtype=np.float32)
    H, W = img.shape
    sub64 = np.empty((H, W)); sub32 = np.empty((H, W), dtype=np.float32)
    mask = np.empty((H, W), dtype=np.uint8); frag = np.empty((H, W), dtype=np.uint8)
    lib().o4_subtract_threshold(_p(img), _p(np.ascontiguousarray(bkg64)), _p(np.ascontiguousarray(rms64)),
                                C.c_int(H), C.c_int(W), C.c_double(k_d), _p(sub64), _p(sub32), _p(mask), _p(frag))
    return sub64, sub32, mask, frag


def label(mask: np.ndarray) -> np.ndarray:
    """O5.  mask u8 [H,W] -> int32 labels, 1 + minimum raster index of the 8-connected component."""
    mask = np.ascontiguousarray(mask, dtype=np.uint8)
    H, W = mask.shape
    out = np.empty((H, W), dtype=np.int32)
    lib().o5_label(_p(mask), C.c_int(H), C.c_int(W), _p(out))
    return out


def reduce_sources(labels: np.ndarray, sub: np.ndarray, min_area: int) -> np.ndarray:
    """O6.  -> structured array (SOURCE_DTYPE), ascending label, npix >= min_area."""
    labels = np.ascontiguousarray(labels, dtype=np.int32)
    sub = np.ascontiguousarray(sub, dtype=np.float32)
    H, W = labels.shape
    assert lib().o6_source_size() == SOURCE_DTYPE.itemsize
    cap = int(np.count_nonzero(labels.reshape(-1) == np.arange(1, H * W + 1, dtype=np.int64))) + 1
    out = np.zeros(cap, dtype=SOURCE_DTYPE)
    n = lib().o6_reduce(_p(labels), _p(sub), C.c_int(H), C.c_int(W), C.c_int(min_area), _p(out), C.c_int64(cap))
    return out[:n]


def background(img: np.ndarray, p: BkgParams):
    """O1 -> O2 -> O3 for one frame.  Returns dict with mesh grids, filtered grids, coefficients, maps."""
    H, W = img.shape
    st = mesh_stats(img, p)
    bkg_f = grid_median(st["bkg"], p.filt_h, p.filt_w)
    rms_f = grid_median(st["rms"], p.filt_h, p.filt_w)
    cb, cr = spline_coeffs(bkg_f), spline_coeffs(rms_f)
    return dict(stats=st, bkg_grid=bkg_f, rms_grid=rms_f, bkg_coef=cb, rms_coef=cr,
                bkg=spline_eval(cb, H, W, p.mesh_h, p.mesh_w), rms=spline_eval(cr, H, W, p.mesh_h, p.mesh_w))


def chain(img: np.ndarray, p: BkgParams, detect_k: float, min_area: int):
    """Whole hot path on one frame: O1..O6."""
    b = background(img, p)
    sub64, sub32, mask, frag = subtract_threshold(img, b["bkg"], b["rms"], detect_k)
    lab = label(mask)
    cat = reduce_sources(lab, sub32, min_area)
    b.update(sub64=sub64, sub=sub32, mask=mask, fragile=frag, labels=lab, cat=cat)
    return b
