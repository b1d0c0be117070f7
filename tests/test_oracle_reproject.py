"""CPU-only pins of the reprojection oracle (O12, readings R1-R6).  Each pin is something other than the
oracle's own formula: scipy's affine resampling (a different code base, (row, column) convention and matrix direction),
exact special cases (identity, integer and half-pixel shifts, a 90-degree rotation), and linearity (a bilinear
interpolant reproduces a plane exactly).  A swapped x/y, a forward instead of inverse map, a wrong neighbour or weight,
or a wrong border rule fails at least one."""
import numpy as np
import pytest
from scipy import ndimage

from oracle import reproject as rp


def frame(seed, H=37, W=52):
    return np.random.default_rng(seed).normal(100, 20, (H, W))


def test_identity_and_integer_shifts_are_exact():
    src = frame(1)
    assert np.array_equal(rp.reproject(src, [1, 0, 0, 0, 1, 0]), src)
    # forward map x' = x + 3, y' = y - 2: the source pixel (x, y) lands on (x + 3, y - 2); the uncovered part is `fill`
    out = rp.reproject(src, [1, 0, 3, 0, 1, -2], fill=-7.0)
    assert np.array_equal(out[:-2, 3:], src[2:, :-3])
    assert np.all(out[-2:, :] == -7.0) and np.all(out[:, :3] == -7.0)


def test_half_pixel_shift_is_the_mean_of_two_neighbours():
    src = frame(2)
    out = rp.reproject(src, [1, 0, 0.5, 0, 1, 0])      # result(x') = source(x' - 0.5)
    assert np.allclose(out[:, 1:], 0.5 * (src[:, :-1] + src[:, 1:]), rtol=0, atol=1e-12)
    assert np.allclose(out[:, 0], 0.5 * src[:, 0])     # R4: the neighbour at x = -1 is fill = 0 and is interpolated
    out = rp.reproject(src, [1, 0, 0, 0, 1, 0.25], fill=10.0)
    assert np.allclose(out[1:, :], 0.25 * src[:-1, :] + 0.75 * src[1:, :], atol=1e-12)
    assert np.allclose(out[0, :], 0.25 * 10.0 + 0.75 * src[0, :], atol=1e-12)


def test_rotation_by_90_degrees_is_a_transpose_with_a_flip():
    src = frame(3, 20, 20)
    # forward map (x, y) -> (19 - y, x): x' = -y + 19, y' = x
    out = rp.reproject(src, [0, -1, 19, 1, 0, 0])
    yy, xx = np.mgrid[:20, :20]
    want = np.empty_like(src); want[xx, 19 - yy] = src[yy, xx]      # push form of the same map
    assert np.allclose(out, want, atol=1e-10)


def test_a_plane_is_reproduced_exactly_inside_the_frame():
    yy, xx = np.mgrid[:60, :80].astype(np.float64)
    src = 3.0 + 0.5 * xx - 0.25 * yy
    th, s = 0.3, 1.07
    A = [s * np.cos(th), -s * np.sin(th), 4.2, s * np.sin(th), s * np.cos(th), -3.1]
    out = rp.reproject(src, A, out_shape=(70, 90), fill=np.nan)
    inv = rp.invert_affine(A)
    yd, xd = np.mgrid[:70, :90].astype(np.float64)
    xs, ys = inv[0] * xd + inv[1] * yd + inv[2], inv[3] * xd + inv[4] * yd + inv[5]
    inside = (xs >= 0) & (xs <= 79) & (ys >= 0) & (ys <= 59)
    assert inside.sum() > 2000
    # forward map of the sampled source point gives the result pixel back (R1: A is source -> result)
    assert np.allclose(A[0] * xs + A[1] * ys + A[2], xd, atol=1e-9) and np.allclose(A[3] * xs + A[4] * ys + A[5], yd, atol=1e-9)
    assert np.allclose(out[inside], (3.0 + 0.5 * xs - 0.25 * ys)[inside], rtol=0, atol=1e-10)
    assert np.isnan(out[(xs < -1) | (xs > 80) | (ys < -1) | (ys > 60)]).all()


@pytest.mark.parametrize("seed,th,s,sh,tx,ty,shape", [(4, 0.2, 1.0, 0.0, 2.3, -1.7, None), (5, -0.7, 0.9, 0.15, 10.0, 6.5, (45, 61)),
                                                      (6, 0.01, 1.002, 0.0, -0.37, 0.81, None), (7, 2.5, 1.3, -0.2, 30.0, 25.0, (30, 70))])
def test_against_scipy_affine_transform_and_map_coordinates(seed, th, s, sh, tx, ty, shape):
    """scipy.ndimage.affine_transform maps OUTPUT coordinates to INPUT coordinates, in (row, column) order: its matrix is
    A^-1 with x and y swapped.  mode='grid-constant' is the constant border that is interpolated (R4)."""
    src = frame(seed)
    A = np.array([[s * np.cos(th), -s * np.sin(th) + sh, tx], [s * np.sin(th), s * np.cos(th), ty]])
    out = rp.reproject(src, A.ravel(), out_shape=shape, fill=5.0)
    M = np.linalg.inv(np.vstack([A, [0, 0, 1]]))                 # result (x', y') -> source (x, y)
    M_rc = np.array([[M[1, 1], M[1, 0]], [M[0, 1], M[0, 0]]])    # the same in (row, column) order
    off_rc = np.array([M[1, 2], M[0, 2]])
    want = ndimage.affine_transform(src, M_rc, offset=off_rc, output_shape=shape or src.shape, order=1, mode="grid-constant", cval=5.0)
    assert np.allclose(out, want, rtol=0, atol=1e-9)
    Hd, Wd = shape or src.shape
    yd, xd = np.mgrid[:Hd, :Wd].astype(np.float64)
    coords = np.stack([M[1, 0] * xd + M[1, 1] * yd + M[1, 2], M[0, 0] * xd + M[0, 1] * yd + M[0, 2]])
    want2 = ndimage.map_coordinates(src, coords, order=1, mode="grid-constant", cval=5.0)
    assert np.allclose(out, want2, rtol=0, atol=1e-9)


def test_pixelwise_definition_equals_the_array_form_and_the_sampler():
    src = frame(8)
    A = [0.97, 0.26, -3.0, -0.25, 0.96, 4.5]
    out = rp.reproject(src, A, out_shape=(40, 50), fill=1.5)
    inv = rp.invert_affine(A)
    rng = np.random.default_rng(0)
    ys, xs = rng.integers(0, 40, 300), rng.integers(0, 50, 300)
    for y, x in zip(ys, xs):
        assert out[y, x] == pytest.approx(rp.reproject_pixel(src, inv, int(x), int(y), 1.5), rel=0, abs=1e-12)
    assert np.array_equal(rp.reproject(src, A, out_shape=(40, 50), fill=1.5, only=(ys, xs)), out[ys, xs])


def test_singular_or_non_finite_matrix_gives_fill():
    src = frame(9)
    for A in ([1, 2, 0, 2, 4, 0], [0, 0, 0, 0, 0, 0], [np.nan, 0, 0, 0, 1, 0], [1, 0, np.inf, 0, 1, 0]):
        assert np.all(rp.reproject(src, A, fill=2.5) == 2.5)
