"""O7: aperture and auto (Kron-like) photometry per catalogue object -- CPU oracle (TEST INFRASTRUCTURE).

PAPER.md:159 ("we calculate the flux of each object using several established methods, such as: aperture photometry,
isophotal photometry and auto photometry ... Each GPU thread is assigned to measure a single object").  Isophotal
photometry is the `flux` of step O6.  The paper gives no constants and no formula for the other two; the readings below
(A23-A27 in DESIGN.md) follow the conventions of the method the paper adapts (SExtractor), and this file is
those definitions written out, one object at a time, in float64 with plain numpy.  It shares no code with the CUDA path.

A23  aperture: circle of radius r_aper (pixels) about the object's centroid (x, y) of O6, pixel centres at integer
     coordinates.  Weight of a pixel = 1 if its centre is closer than r - 0.75 to the centroid, 0 if farther than
     r + 0.75, otherwise the fraction of its subpix x subpix sub-pixel centres (offsets (i + 0.5)/subpix - 0.5) that
     lie within r.   flux_aper = sum w * sub,  area_aper = sum w,  fluxerr_aper = sqrt(sum w * rms^2)  (background noise
     only: the paper gives no gain).  Pixels outside the frame contribute nothing; flag bit 0 if one of them had w > 0.
A24  object shape: second moments x2, y2, xy of O6; if x2*y2 - xy^2 < 0.00694 (an object thinner than a pixel) 1/12 is
     added to x2 and y2.  Ellipse metric r^2 = cxx dx^2 + cyy dy^2 + cxy dx dy with cxx = y2/D, cyy = x2/D,
     cxy = -2 xy/D, D = x2 y2 - xy^2  (r = 1 is the 1-sigma ellipse).
A25  Kron radius: r1 = sum r * sub / sum sub over the pixels with r <= kron_search (6), pixel centres, no weights;
     kron_radius = max(kron_factor * r1, kron_min_radius)  (2.5, 3.5); if sum sub <= 0 or r1 is not positive,
     kron_radius = kron_min_radius.
A26  auto: flux_auto = sum of sub over the pixels with r <= kron_radius (hard edge, pixel centres), npix_auto their
     number, fluxerr_auto = sqrt(sum rms^2).  Flag bit 1: the bounding box of either ellipse leaves the frame (the sums
     then run over the part inside).
A27  no masking of neighbours (the measurement follows whatever catalogue it is given: raw, deblended or cleaned).
A28  a record whose centroid or moments are not finite, or whose (regularised) moments define no ellipse (D <= 0, x2 <= 0
     or y2 <= 0), is not measured: every output 0, flags = 4.
"""
from __future__ import annotations

from dataclasses import dataclass

import numpy as np

PHOT_DTYPE = np.dtype([("flux_aper", np.float64), ("fluxerr_aper", np.float64), ("area_aper", np.float64),
                       ("kron_radius", np.float64), ("flux_auto", np.float64), ("fluxerr_auto", np.float64),
                       ("npix_auto", np.int32), ("flags", np.int32)], align=True)


@dataclass
class PhotParams:
    r_aper: float = 5.0
    kron_factor: float = 2.5
    kron_min_radius: float = 3.5
    kron_search: float = 6.0
    subpix: int = 5


def ellipse_coefficients(x2: float, y2: float, xy: float):
    """A24."""
    if x2 * y2 - xy * xy < 0.00694:
        x2 = x2 + 1.0 / 12.0
        y2 = y2 + 1.0 / 12.0
    d = x2 * y2 - xy * xy
    return y2 / d, x2 / d, -2.0 * xy / d, x2, y2


def aperture_weights(xc: float, yc: float, r: float, xs: np.ndarray, ys: np.ndarray, subpix: int) -> np.ndarray:
    """A23: weights of the pixels (xs, ys) (integer arrays of the same shape)."""
    dx = xs.astype(np.float64) - xc
    dy = ys.astype(np.float64) - yc
    d = np.sqrt(dx * dx + dy * dy)
    w = np.where(d < r - 0.75, 1.0, 0.0)
    edge = (d >= r - 0.75) & (d <= r + 0.75)
    if edge.any():
        offs = (np.arange(subpix, dtype=np.float64) + 0.5) / subpix - 0.5
        ex, ey = dx[edge], dy[edge]
        cnt = np.zeros(ex.shape, dtype=np.int64)
        for oy in offs:
            for ox in offs:
                cnt += ((ex + ox) ** 2 + (ey + oy) ** 2 <= r * r)
        w[edge] = cnt / float(subpix * subpix)
    return w


def _box(c: float, half: float, n: int):
    lo = int(np.floor(c - half))
    hi = int(np.ceil(c + half))
    return lo, hi, (lo < 0) or (hi > n - 1)


def measure_one(sub: np.ndarray, rms: np.ndarray, src, p: PhotParams):
    H, W = sub.shape
    xc, yc = float(src["x"]), float(src["y"])
    flags = 0
    # ---- A28 degenerate record
    m = [xc, yc, float(src["x2"]), float(src["y2"]), float(src["xy"])]
    if not all(np.isfinite(v) for v in m):
        return 0.0, 0.0, 0.0, 0.0, 0.0, 0.0, 0, 4
    _x2, _y2 = (m[2] + 1.0 / 12.0, m[3] + 1.0 / 12.0) if m[2] * m[3] - m[4] * m[4] < 0.00694 else (m[2], m[3])
    if not (_x2 * _y2 - m[4] * m[4] > 0.0 and _x2 > 0.0 and _y2 > 0.0):
        return 0.0, 0.0, 0.0, 0.0, 0.0, 0.0, 0, 4
    # ---- A23 aperture
    x_lo, x_hi, cx = _box(xc, p.r_aper + 1.0, W)
    y_lo, y_hi, cy = _box(yc, p.r_aper + 1.0, H)
    ys, xs = np.mgrid[y_lo:y_hi + 1, x_lo:x_hi + 1]
    w = aperture_weights(xc, yc, p.r_aper, xs, ys, p.subpix)
    inside = (xs >= 0) & (xs < W) & (ys >= 0) & (ys < H)
    if (w[~inside] > 0).any():
        flags |= 1
    w = np.where(inside, w, 0.0)
    xi, yi = np.clip(xs, 0, W - 1), np.clip(ys, 0, H - 1)
    s = sub[yi, xi].astype(np.float64)
    v = rms[yi, xi].astype(np.float64) ** 2
    flux_aper = float((w * s).sum())
    area_aper = float(w.sum())
    err_aper = float(np.sqrt((w * v).sum()))
    # ---- A24 shape, A25 Kron radius
    cxx, cyy, cxy, x2, y2 = ellipse_coefficients(float(src["x2"]), float(src["y2"]), float(src["xy"]))

    def ellipse_pixels(R):
        hx, hy = R * np.sqrt(x2), R * np.sqrt(y2)
        xl, xh, tx = _box(xc, hx, W)
        yl, yh, ty = _box(yc, hy, H)
        yy, xx = np.mgrid[max(yl, 0):min(yh, H - 1) + 1, max(xl, 0):min(xh, W - 1) + 1]
        dx, dy = xx - xc, yy - yc
        r2 = cxx * dx * dx + cyy * dy * dy + cxy * dx * dy
        return yy, xx, np.sqrt(np.maximum(r2, 0.0)), (tx or ty)

    yy, xx, r, trunc = ellipse_pixels(p.kron_search)
    sel = r <= p.kron_search
    I = sub[yy, xx].astype(np.float64)
    s0 = float(I[sel].sum())
    s1 = float((r[sel] * I[sel]).sum())
    kron = p.kron_min_radius
    if s0 > 0.0 and s1 > 0.0:
        kron = max(p.kron_factor * s1 / s0, p.kron_min_radius)
    if trunc:
        flags |= 2
    # ---- A26 auto
    yy, xx, r, trunc = ellipse_pixels(kron)
    sel = r <= kron
    flux_auto = float(sub[yy, xx].astype(np.float64)[sel].sum())
    err_auto = float(np.sqrt((rms[yy, xx].astype(np.float64)[sel] ** 2).sum()))
    npix_auto = int(sel.sum())
    if trunc:
        flags |= 2
    return flux_aper, err_aper, area_aper, kron, flux_auto, err_auto, npix_auto, flags


def photometry(sub: np.ndarray, rms: np.ndarray, cat: np.ndarray, p: PhotParams) -> np.ndarray:
    """O7 for one frame: cat = records with fields x, y, x2, y2, xy (O6).  -> PHOT_DTYPE array, one per record."""
    sub = np.ascontiguousarray(sub, dtype=np.float32)
    rms = np.ascontiguousarray(rms, dtype=np.float32)
    out = np.zeros(len(cat), dtype=PHOT_DTYPE)
    for i, src in enumerate(cat):
        out[i] = measure_one(sub, rms, src, p)
    return out
