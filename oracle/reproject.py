"""O12: bilinear reprojection of a frame through an affine matrix -- CPU oracle (TEST INFRASTRUCTURE).

PAPER.md:114 (section 2.2.3): "we implement the estimation of the affine matrix using OpenCV's estimate AffinePartial2D
method ... and then perform image reprojection using the obtained affine matrix.  Specifically, we use the affine matrix to
obtain the coordinate mapping between the source image and the resulting image.  For each pixel in the source image, the
pixel value in the resulting image is calculated through bilinear interpolation based on the four neighboring pixels."
The FIT of the matrix (matched star lists) is out of scope; the matrix is an input.  Readings (R1-R5 in DESIGN.md):

R1  direction: the matrix A (2 x 3, row-major: x' = a0 x + a1 y + a2, y' = a3 x + a4 y + a5) is the FORWARD map the fit
    returns, source pixel (x, y) -> result pixel (x', y').  The result is formed by PULLING: for every result pixel
    (x', y') the source is sampled at (xs, ys) = A^-1 (x', y') -- the only way "bilinear interpolation based on the four
    neighbouring pixels" is defined for every pixel of the result, and what the OpenCV routine of that family does;
R2  coordinates: pixel centres at integers, x = column, y = row, 0-based (as in the catalogue);
R3  the four neighbours are (x0, y0), (x0+1, y0), (x0, y0+1), (x0+1, y0+1), x0 = floor(xs), y0 = floor(ys), with weights
    (1-fx)(1-fy), fx(1-fy), (1-fx)fy, fx fy, fx = xs - x0, fy = ys - y0;
R4  a neighbour outside the source frame has the value `fill` (default 0) and is interpolated like any other (constant
    border; a result pixel whose four neighbours are all outside is exactly `fill`);
R5  a matrix that cannot be inverted (det = a0 a4 - a1 a3 zero or not finite) gives a result frame of `fill`;
R6  arithmetic: float64 throughout here; the result frame may have a shape of its own (Hd, Wd).

One result pixel at a time in `reproject_pixel` (the definition); `reproject` is the same expression over whole index
arrays.  Shares no code with the CUDA path.
"""
from __future__ import annotations

import numpy as np


def invert_affine(A):
    """A: 6 numbers (R1).  -> the 6 numbers of A^-1 in float64, or None (R5)."""
    a0, a1, a2, a3, a4, a5 = (float(v) for v in np.asarray(A, dtype=np.float64).ravel())
    det = a0 * a4 - a1 * a3
    if not np.isfinite(det) or det == 0.0 or not all(np.isfinite(v) for v in (a2, a5)):
        return None
    i0, i1, i3, i4 = a4 / det, -a1 / det, -a3 / det, a0 / det
    return i0, i1, -(i0 * a2 + i1 * a5), i3, i4, -(i3 * a2 + i4 * a5)


def reproject_pixel(src: np.ndarray, inv, xd: int, yd: int, fill: float = 0.0) -> float:
    """R1-R4 for ONE result pixel (xd, yd); inv = invert_affine(A)."""
    H, W = src.shape
    xs = inv[0] * xd + inv[1] * yd + inv[2]
    ys = inv[3] * xd + inv[4] * yd + inv[5]
    x0, y0 = int(np.floor(xs)), int(np.floor(ys))
    fx, fy = xs - x0, ys - y0

    def px(x, y):
        return float(src[y, x]) if (0 <= x < W and 0 <= y < H) else float(fill)

    return ((1.0 - fx) * (1.0 - fy) * px(x0, y0) + fx * (1.0 - fy) * px(x0 + 1, y0)
            + (1.0 - fx) * fy * px(x0, y0 + 1) + fx * fy * px(x0 + 1, y0 + 1))


def reproject(src: np.ndarray, A, out_shape=None, fill: float = 0.0, only=None) -> np.ndarray:
    """O12 for one frame.  src [H, W]; A 6 numbers (R1); out_shape (Hd, Wd), default src.shape.  -> float64 [Hd, Wd], or,
    with only = (ys, xs) integer arrays, the values of those result pixels (sampling for full-size frames)."""
    src = np.asarray(src)
    H, W = src.shape
    Hd, Wd = src.shape if out_shape is None else out_shape
    if only is None:
        yd, xd = np.mgrid[:Hd, :Wd]
    else:
        yd, xd = (np.asarray(v, dtype=np.int64) for v in only)
    inv = invert_affine(A)
    if inv is None:
        return np.full(xd.shape, float(fill))
    xd = xd.astype(np.float64); yd = yd.astype(np.float64)
    xs = inv[0] * xd + inv[1] * yd + inv[2]
    ys = inv[3] * xd + inv[4] * yd + inv[5]
    # (coordinates far outside the frame, up to the overflow of a huge translation: all four neighbours are outside, R4;
    #  clamped to two pixels beyond the frame so that the integer cast below is defined -- the weights are then irrelevant)
    xs = np.clip(xs, -3.0, W + 2.0); ys = np.clip(ys, -3.0, H + 2.0)
    x0 = np.floor(xs); y0 = np.floor(ys)
    fx, fy = xs - x0, ys - y0
    x0 = x0.astype(np.int64); y0 = y0.astype(np.int64)

    def px(x, y):
        inside = (x >= 0) & (x < W) & (y >= 0) & (y < H)
        v = src[np.clip(y, 0, H - 1), np.clip(x, 0, W - 1)].astype(np.float64)
        return np.where(inside, v, float(fill))

    return ((1.0 - fx) * (1.0 - fy) * px(x0, y0) + fx * (1.0 - fy) * px(x0 + 1, y0)
            + (1.0 - fx) * fy * px(x0, y0 + 1) + fx * fy * px(x0 + 1, y0 + 1))
