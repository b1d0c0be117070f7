"""Comparison rules between the CUDA path and the oracle (BASELINE.json north_star).

Tolerances, written out:
  * mesh statistics: n_kept and the survivor-defined median bit-exact; mean/std/bkg 1e-10 relative
    (float64 on both sides, only the summation order differs);
  * bkg / rms maps: |d| <= 1e-4 * |oracle|  (north_star: "within 1e-4 relative (float32 vs float64)");
  * sub: |d| <= 1e-4 * |bkg_oracle| (a relative test on a zero-mean quantity is meaningless);
  * mask: may differ only where the oracle's |sub - k*rms| <= 1e-5 * rms ("fragile" pixels);
  * labels: bit-exact against the oracle's labelling of the SAME mask;
  * catalogue: 1:1 on (frame, label); npix, bbox exact.  STAGE comparison (both sides reduce the same float32 sub map,
    `peak_pos_exact=True`): peak position and peak value bit-exact.  CHAIN comparison (each side reduces its own sub map;
    the two maps agree to ~1e-6 ADU): peak value 1e-6 relative, peak position may move between pixels that are equal to
    the last bit (<= 1 % of the records).  flux, x, y 1e-4 relative (the absolute centroid error is reported);
    x2, y2, xy 1e-3 relative to max(|moment|, 1e-3*(x2+y2) + 1e-9)  (derivation in DESIGN.md section 8).
"""
from __future__ import annotations

import numpy as np

import oracle

REL_MAP = 1e-4
REL_CAT = 1e-4
REL_MOM = 1e-3
REL_PEAK = 1e-6


def to_oracle_params(p):
    return oracle.BkgParams(mesh_h=p.mesh_h, mesh_w=p.mesh_w, filt_h=p.filt_h, filt_w=p.filt_w,
                            clip_sigma=p.clip_sigma, clip_iters=p.clip_iters, median_factor=p.median_factor,
                            mean_factor=p.mean_factor, skew_guard=p.skew_guard)


def assert_maps_close(got, want64, name, rel=REL_MAP, scale=None):
    got = np.asarray(got, dtype=np.float64)
    ref = np.abs(want64) if scale is None else np.abs(scale)
    err = np.abs(got - want64)
    bad = err > rel * ref + 1e-30
    assert not bad.any(), f"{name}: {bad.sum()} px beyond {rel} relative; worst {np.max(err / np.maximum(ref, 1e-300)):.3e}"
    return float(np.max(err / np.maximum(ref, 1e-300)))


def assert_mask_parity(mask_gpu, mask_or, fragile):
    diff = (mask_gpu != 0) != (mask_or != 0)
    assert not (diff & (fragile == 0)).any(), f"{(diff & (fragile == 0)).sum()} mask mismatches outside the fragile set"
    return int(diff.sum())


def assert_catalogue_equal(got, want, frame=None, exempt_labels=(), peak_pos_exact=True):
    """got: GPU records (bd_source dtype) of one frame; want: oracle records of the same labels/sub."""
    if frame is not None:
        got = got[got["frame"] == frame]
    ex = set(int(v) for v in exempt_labels)
    if ex:
        got = got[~np.isin(got["label"], list(ex))]
        want = want[~np.isin(want["label"], list(ex))]
    assert len(got) == len(want), f"catalogue length {len(got)} != oracle {len(want)}"
    if len(want) == 0:
        return dict(n=0)
    assert np.array_equal(got["label"], want["label"]), "labels / order differ"
    for k in ("npix", "xmin", "xmax", "ymin", "ymax"):
        assert np.array_equal(got[k], want[k]), f"{k} differs at {np.flatnonzero(got[k] != want[k])[:5]}"
    moved = (got["xpeak"] != want["xpeak"]) | (got["ypeak"] != want["ypeak"])
    if peak_pos_exact:
        # same sub map on both sides: the peak pixel (ties -> smallest raster index) is unique
        assert not moved.any(), f"peak position differs at {np.flatnonzero(moved)[:5]}"
    else:
        # each side takes the maximum of its OWN float32 sub map; the maps agree to ~1e-6 ADU, so where two
        # pixels of a component are equal to the last bit (adjacent saturated / hot pixels) the winner may
        # differ.  The peak VALUE is still compared below; such near-ties must stay rare.
        assert moved.sum() <= max(2, len(want) // 100), f"{moved.sum()} of {len(want)} peak positions differ"
    if peak_pos_exact:
        # stage comparison: the peak is an element of the one float32 sub map both sides read
        assert np.array_equal(got["peak"].astype(np.float64), want["peak"]), "peak value differs (must be bit-exact)"
    else:
        # chain comparison: each side rounds to float32 a value that agrees to ~1e-6 ADU, so the last bit may differ
        perr = np.abs(got["peak"].astype(np.float64) - want["peak"]) / np.maximum(np.abs(want["peak"]), 1e-300)
        assert np.all(perr <= REL_PEAK), f"peak: worst rel {perr.max():.3e}"
    worst = {}
    for k in ("flux", "x", "y"):
        err = np.abs(got[k] - want[k]) / np.maximum(np.abs(want[k]), 1e-300)
        assert np.all(err <= REL_CAT), f"{k}: worst rel {err.max():.3e}"
        worst[k] = float(err.max())
    worst["centroid_abs_px"] = float(max(np.abs(got["x"] - want["x"]).max(), np.abs(got["y"] - want["y"]).max()))
    for k in ("x2", "y2", "xy"):
        # a moment can be ~0 by symmetry (xy, or x2 of a one-column component): the error it inherits from a
        # relative perturbation eps of the pixel values is <= eps * (x2 + y2), so the scale has that floor
        # -- CHAIN comparison (each side reduces its own sub map, ~1e-6 ADU apart): floor 1e-3 (x2 + y2), DESIGN.md section 8.
        # -- STAGE comparison (peak_pos_exact: both sides read the SAME float32 sub; only the summation order differs):
        #    the tight floor 1e-6 (1 + x2 + y2), i.e. 1e-9 (1 + x2 + y2) absolute.
        floor = 1e-6 * (1.0 + want["x2"] + want["y2"]) if peak_pos_exact else 1e-3 * (want["x2"] + want["y2"]) + 1e-9
        scale = np.maximum(np.abs(want[k]), floor)
        err = np.abs(got[k] - want[k]) / scale
        assert np.all(err <= REL_MOM), f"{k}: worst rel {err.max():.3e}"
        worst[k] = float(err.max())
    worst["n"] = len(want)
    return worst


def fragile_touched_labels(labels_or, fragile):
    """Labels of oracle components that contain or 8-touch a fragile pixel (exempt from 1:1 matching)."""
    if not fragile.any():
        return np.zeros(0, dtype=np.int32)
    H, W = fragile.shape
    ys, xs = np.nonzero(fragile)
    out = set()
    for dy in (-1, 0, 1):
        for dx in (-1, 0, 1):
            yy, xx = np.clip(ys + dy, 0, H - 1), np.clip(xs + dx, 0, W - 1)
            out.update(int(v) for v in np.unique(labels_or[yy, xx]) if v)
    return np.array(sorted(out), dtype=np.int32)
