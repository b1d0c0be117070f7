"""O9: stamp-wise spatially varying convolution of the template and image subtraction -- CPU oracle (TEST INFRASTRUCTURE).

PAPER.md:126-147 (section 2.2.4).  Eq. 8: K(u,v) = sum_n a_n(x,y) K_n(u,v); eq. 9: K_n(u,v) = exp(-(u^2+v^2)/(2 sigma_k^2)) u^i v^j
("Multiple Gaussians with different sigma_k can be chosen, each with a fixed spatial modulation order.  The values of i and j
and their sum do not exceed this order"); eq. 10: R (x) K = I + B.  "We then allocate a thread block for each stamp of the
convolution kernel size; by default, the size of the stamp is 21 x 21 pixels ... utilizing the preloaded convolution kernel
... Finally, by subtracting the convolved template image from the input image, we obtain the difference image."
Kernel FITTING (choosing stamps, solving for a_n) needs the science data of the method the paper adapts and is out of
scope; the coefficients are inputs here.  Readings (C1-C7 in DESIGN.md):

C1  basis order: Gaussians in the order given; inside Gaussian g the terms (i, j), i = 0..d_g, j = 0..d_g - i (i outer);
C2  a_n(x, y) = sum_{p+q<=ds} c[n, t(p,q)] xh^p yh^q with t enumerating p = 0..ds, q = 0..ds - p (p outer) and the
    normalised coordinates xh = (2x - (W-1))/W, yh = (2y - (H-1))/H (both in (-1, 1)); B(x, y) likewise with order db;
C3  the frame is cut into stamps of S x S pixels, S = 2 hw + 1 (the kernel size), from the top-left corner; partial
    stamps at the right / bottom edge; the kernel of a stamp is K evaluated ONCE at its nominal centre
    (x_c, y_c) = (sx S + hw, sy S + hw) ("the preloaded convolution kernel") and applied to every pixel of the stamp;
C4  convolution proper: conv(x, y) = sum_{u,v=-hw..hw} K(u, v) R(x - u, y - v), with R = 0 outside the frame;
C5  eq. 10 read literally: the model is R (x) K = I + B, so diff = I + B - R (x) K, B evaluated at the pixel;
C6  no kernel normalisation, no masking of saturated pixels, no noise image;
C7  arithmetic: float64 here.

One stamp at a time, one tap at a time: plain loops over the 441 taps with numpy slices.  Shares no code with the CUDA path.
"""
from __future__ import annotations

from dataclasses import dataclass, field

import numpy as np


@dataclass
class ConvParams:
    half_width: int = 10                                                   # 21 x 21
    sigma: tuple = (0.7, 1.5, 3.0)                                         # sigma_k of eq. 9
    degree: tuple = (6, 4, 2)                                              # order of u^i v^j per Gaussian
    spatial_order: int = 2                                                 # ds
    bg_order: int = 1                                                      # db


def n_poly(order: int) -> int:
    return (order + 1) * (order + 2) // 2


def n_basis(p: ConvParams) -> int:
    return sum(n_poly(d) for d in p.degree)


def poly_terms(order: int):
    return [(a, b) for a in range(order + 1) for b in range(order + 1 - a)]


def basis_kernels(p: ConvParams) -> np.ndarray:
    """Eq. 9 / C1.  -> float64 [N, S, S] indexed [n, v + hw, u + hw]."""
    hw = p.half_width
    u = np.arange(-hw, hw + 1, dtype=np.float64)[None, :]
    v = np.arange(-hw, hw + 1, dtype=np.float64)[:, None]
    out = []
    for s, d in zip(p.sigma, p.degree):
        g = np.exp(-(u * u + v * v) / (2.0 * s * s))
        for (i, j) in poly_terms(d):
            out.append(g * u ** i * v ** j)
    return np.stack(out)


def poly_eval(coef: np.ndarray, order: int, xh, yh):
    """C2: sum_t coef[..., t] xh^p yh^q."""
    acc = 0.0
    for t, (a, b) in enumerate(poly_terms(order)):
        acc = acc + coef[..., t] * xh ** a * yh ** b
    return acc


def stamp_kernel(p: ConvParams, kcoef: np.ndarray, H: int, W: int, sx: int, sy: int, basis=None) -> np.ndarray:
    """Eq. 8 at the stamp centre (C3).  kcoef float64 [N, n_poly(ds)] -> [S, S] indexed [v + hw, u + hw]."""
    basis = basis_kernels(p) if basis is None else basis
    S, hw = 2 * p.half_width + 1, p.half_width
    xh = (2.0 * (sx * S + hw) - (W - 1)) / W
    yh = (2.0 * (sy * S + hw) - (H - 1)) / H
    a = poly_eval(kcoef, p.spatial_order, xh, yh)            # [N]
    return np.tensordot(a, basis, axes=1)


def subtract(ref: np.ndarray, img: np.ndarray, p: ConvParams, kcoef: np.ndarray, bgcoef: np.ndarray, only=None):
    """O9 for one frame pair.  ref, img float32 [H, W]; kcoef [N, n_poly(ds)], bgcoef [n_poly(db)] float64.
    `only`: optional iterable of stamps (sy, sx); the other stamps are not computed (their pixels stay 0 in both outputs) --
    a sampling facility for full-size frames, the arithmetic of a computed stamp is the same.
    -> (diff float64 [H, W], conv float64 [H, W])."""
    ref = np.asarray(ref, dtype=np.float64) if only is None else ref
    img = np.asarray(img, dtype=np.float64) if only is None else img
    H, W = ref.shape
    hw = p.half_width
    S = 2 * hw + 1
    basis = basis_kernels(p)
    stamps = [(sy, sx) for sy in range((H + S - 1) // S) for sx in range((W + S - 1) // S)] if only is None else [(int(a), int(b)) for a, b in only]
    conv = np.zeros((H, W))
    diff = np.zeros((H, W))
    bgc = np.asarray(bgcoef, dtype=np.float64)
    for sy, sx in stamps:
        K = stamp_kernel(p, kcoef, H, W, sx, sy, basis)
        y0, y1, x0, x1 = sy * S, min((sy + 1) * S, H), sx * S, min((sx + 1) * S, W)
        # the template around the stamp, padded with zeros where it leaves the frame (C4: R = 0 outside the frame)
        pad = np.zeros((y1 - y0 + 2 * hw, x1 - x0 + 2 * hw))
        ya, yb, xa, xb = max(y0 - hw, 0), min(y1 + hw, H), max(x0 - hw, 0), min(x1 + hw, W)
        pad[ya - (y0 - hw):yb - (y0 - hw), xa - (x0 - hw):xb - (x0 - hw)] = ref[ya:yb, xa:xb]
        acc = np.zeros((y1 - y0, x1 - x0))
        for v in range(-hw, hw + 1):
            for u in range(-hw, hw + 1):
                # R(x - u, y - v) for the pixels of the stamp, in the coordinates of the padded patch
                acc += K[v + hw, u + hw] * pad[hw - v:hw - v + (y1 - y0), hw - u:hw - u + (x1 - x0)]
        conv[y0:y1, x0:x1] = acc
        yy, xx = np.mgrid[y0:y1, x0:x1].astype(np.float64)
        bg = poly_eval(bgc, p.bg_order, (2.0 * xx - (W - 1)) / W, (2.0 * yy - (H - 1)) / H)
        diff[y0:y1, x0:x1] = np.asarray(img[y0:y1, x0:x1], dtype=np.float64) + bg - acc
    return diff, conv
