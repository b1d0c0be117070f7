"""Pins for the oracle's stamp-wise convolution + subtraction O9 (eqs. 8-10; readings C1-C7).  CPU only.
Each pin is something other than the oracle: scipy.signal.convolve2d, an impulse response, closed forms, symmetry."""
import numpy as np
import pytest
from scipy.signal import convolve2d

from oracle import subtract as osub


def _coef_constant(p, a):
    """Spatially constant coefficients: only the (p, q) = (0, 0) term."""
    c = np.zeros((osub.n_basis(p), osub.n_poly(p.spatial_order)))
    c[:, 0] = a
    return c


def test_basis_count_and_values():
    p = osub.ConvParams()
    assert osub.n_basis(p) == 28 + 15 + 6 == 49 and osub.n_poly(2) == 6
    b = osub.basis_kernels(p)
    assert b.shape == (49, 21, 21)
    assert b[0, 10, 10] == 1.0 and b[0, 10, 11] == pytest.approx(np.exp(-1 / (2 * 0.49)))          # eq. 9, i = j = 0
    # C1: term 1 of Gaussian 0 is (i, j) = (0, 1): v^1, odd in v, even in u
    assert b[1, 12, 10] == pytest.approx(2 * np.exp(-4 / (2 * 0.49))) and b[1, 8, 10] == -b[1, 12, 10] and b[1, 10, 13] == 0.0
    # last term of Gaussian 0 is (6, 0): u^6
    assert b[27, 10, 12] == pytest.approx(64 * np.exp(-4 / (2 * 0.49)))
    assert b[28, 10, 10] == 1.0 and b[28, 10, 13] == pytest.approx(np.exp(-9 / (2 * 2.25)))     # Gaussian 1 starts at n = 28


def test_constant_kernel_is_scipy_convolve2d():
    """Spatially constant coefficients: every stamp has the same kernel, so the whole frame is one plain 2-D convolution
    (library routine, zero fill: C4), including partial stamps and the frame edge."""
    rng = np.random.default_rng(0)
    p = osub.ConvParams(half_width=3, sigma=(0.8, 1.7), degree=(2, 1), spatial_order=1, bg_order=0)
    ref = rng.normal(100, 10, size=(37, 45)).astype(np.float32)
    img = rng.normal(100, 10, size=(37, 45)).astype(np.float32)
    a = rng.normal(size=osub.n_basis(p))
    K = np.tensordot(a, osub.basis_kernels(p), axes=1)
    diff, conv = osub.subtract(ref, img, p, _coef_constant(p, a), np.array([2.5]))
    want = convolve2d(ref.astype(np.float64), K, mode="same", boundary="fill")
    assert np.max(np.abs(conv - want)) < 1e-9
    assert np.max(np.abs(diff - (img.astype(np.float64) + 2.5 - want))) < 1e-9                                        # C5


def test_impulse_response_gives_the_kernel_with_the_right_orientation():
    """R = delta at (y0, x0): conv(x, y) = K(x - x0, y - y0) (C4) -- catches a transposed kernel, a correlation instead of
    a convolution, or swapped i / j: the basis term u^1 must be positive to the RIGHT of the impulse."""
    p = osub.ConvParams(half_width=2, sigma=(1.0,), degree=(1,), spatial_order=0, bg_order=0)
    H = W = 5                                            # exactly one stamp
    ref = np.zeros((H, W), np.float32); ref[2, 2] = 1.0
    for n, (i, j) in enumerate(osub.poly_terms(1)):      # (0,0), (0,1), (1,0)
        c = np.zeros((3, 1)); c[n, 0] = 1.0
        _, conv = osub.subtract(ref, np.zeros_like(ref), p, c, np.array([0.0]))
        yy, xx = np.mgrid[:5, :5] - 2
        assert np.allclose(conv, np.exp(-(xx ** 2 + yy ** 2) / 2.0) * xx ** i * yy ** j, atol=1e-15), (i, j)


def test_each_stamp_uses_the_kernel_of_its_centre():
    """C3: with a spatially varying a_0 = 1 + xh the stamps are plain convolutions with differently scaled kernels; inside a
    stamp the kernel does not vary; the centre of stamp sx is x = sx S + hw."""
    p = osub.ConvParams(half_width=1, sigma=(0.9,), degree=(0,), spatial_order=1, bg_order=0)
    H, W = 7, 11
    rng = np.random.default_rng(1)
    ref = rng.uniform(1, 2, size=(H, W)).astype(np.float32)
    c = np.zeros((1, 3)); c[0, 0] = 1.0; c[0, 2] = 1.0   # terms (0,0), (0,1) = yh, (1,0) = xh  -> a = 1 + xh
    _, conv = osub.subtract(ref, np.zeros_like(ref), p, c, np.array([0.0]))
    g = osub.basis_kernels(p)[0]
    base = convolve2d(ref.astype(np.float64), g, mode="same", boundary="fill")
    for sx in range(4):
        xc = sx * 3 + 1
        scale = 1.0 + (2.0 * xc - (W - 1)) / W
        assert np.allclose(conv[:, sx * 3:sx * 3 + 3], scale * base[:, sx * 3:sx * 3 + 3], rtol=1e-13)


def test_background_polynomial_and_linearity():
    p = osub.ConvParams(half_width=2, sigma=(1.2,), degree=(2,), spatial_order=2, bg_order=2)
    rng = np.random.default_rng(2)
    H, W = 23, 19
    r1, r2 = (rng.integers(-50, 50, size=(H, W)).astype(np.float32) for _ in range(2))   # integers: 2 r1 - 3 r2 is exact in float32
    img = rng.normal(size=(H, W)).astype(np.float32)
    kc = rng.normal(size=(osub.n_basis(p), 6)); bc = rng.normal(size=6)
    zero = np.zeros_like(img)
    d0, _ = osub.subtract(zero, zero, p, kc, bc)          # pure background: C2 with t = (0,0),(0,1),(0,2),(1,0),(1,1),(2,0)
    yy, xx = np.mgrid[:H, :W]
    xh, yh = (2.0 * xx - (W - 1)) / W, (2.0 * yy - (H - 1)) / H
    assert np.allclose(d0, bc[0] + bc[1] * yh + bc[2] * yh ** 2 + bc[3] * xh + bc[4] * xh * yh + bc[5] * xh ** 2, atol=1e-14)
    _, c1 = osub.subtract(r1, img, p, kc, bc); _, c2 = osub.subtract(r2, img, p, kc, bc)
    _, c12 = osub.subtract((2 * r1 - 3 * r2).astype(np.float32), img, p, kc, bc)
    assert np.allclose(c12, 2 * c1 - 3 * c2, atol=1e-9)


def test_flat_template_closed_form():
    """R = const c away from the frame edge: conv = c * sum(K); the sum of a Gaussian x u^i v^j kernel vanishes for odd i or j."""
    p = osub.ConvParams(half_width=4, sigma=(1.5,), degree=(2,), spatial_order=0, bg_order=0)
    ref = np.full((27, 27), 3.0, np.float32)
    b = osub.basis_kernels(p)
    for n, (i, j) in enumerate(osub.poly_terms(2)):
        c = np.zeros((osub.n_basis(p), 1)); c[n, 0] = 1.0
        _, conv = osub.subtract(ref, ref, p, c, np.array([0.0]))
        want = 3.0 * b[n].sum()
        assert np.allclose(conv[4:-4, 4:-4], want, atol=1e-12)
        if i % 2 or j % 2:
            assert abs(want) < 1e-12
