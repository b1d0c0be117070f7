"""CPU-only pins of the photometry oracle (O7, readings A23-A27): closed forms of analytic sources and invariants,
chosen so that a dropped term, a wrong sign of cxy, swapped cxx/cyy, a wrong radius unit or a missing factor fails."""
import numpy as np
import pytest

from oracle import photometry as ph


def rec(x, y, x2, y2, xy):
    r = np.zeros(1, dtype=[("x", "f8"), ("y", "f8"), ("x2", "f8"), ("y2", "f8"), ("xy", "f8")])
    r[0] = (x, y, x2, y2, xy)
    return r


def gaussian(H, W, xc, yc, sx, sy, theta, flux):
    """Noise-free elliptical Gaussian sampled at pixel centres; returns image and its exact second moments."""
    yy, xx = np.mgrid[:H, :W].astype(np.float64)
    c, s = np.cos(theta), np.sin(theta)
    u = (xx - xc) * c + (yy - yc) * s
    v = -(xx - xc) * s + (yy - yc) * c
    img = flux / (2 * np.pi * sx * sy) * np.exp(-0.5 * (u * u / sx**2 + v * v / sy**2))
    x2 = sx**2 * c * c + sy**2 * s * s
    y2 = sx**2 * s * s + sy**2 * c * c
    xy = (sx**2 - sy**2) * s * c
    return img.astype(np.float32), x2, y2, xy


def test_constant_image_area_and_errors():
    sub = np.full((120, 120), 2.0, np.float32); rms = np.full((120, 120), 3.0, np.float32)
    for r in (3.0, 5.0, 8.5):
        o = ph.photometry(sub, rms, rec(60.3, 59.6, 4.0, 4.0, 0.0), ph.PhotParams(r_aper=r))[0]
        assert abs(o["area_aper"] / (np.pi * r * r) - 1) < 0.05 / r      # 5x5 sub-pixel sampling of the rim (0.2-px cells on a perimeter of 2 pi r)
        assert o["flux_aper"] == pytest.approx(2.0 * o["area_aper"], rel=1e-12)
        assert o["fluxerr_aper"] == pytest.approx(3.0 * np.sqrt(o["area_aper"]), rel=1e-12)
        assert o["flags"] == 0
    # flat image, circular 1-sigma radius 2 px: r1 = (2/3) * 6 = 4 -> kron 10 -> circle of 20 px
    o = ph.photometry(sub, rms, rec(60.0, 60.0, 4.0, 4.0, 0.0), ph.PhotParams())[0]
    assert o["kron_radius"] == pytest.approx(10.0, rel=2e-2)
    assert o["npix_auto"] == pytest.approx(np.pi * (2 * o["kron_radius"]) ** 2, rel=1e-2)
    assert o["flux_auto"] == pytest.approx(2.0 * o["npix_auto"], rel=1e-12)
    assert o["fluxerr_auto"] == pytest.approx(3.0 * np.sqrt(o["npix_auto"]), rel=1e-12)


@pytest.mark.parametrize("r", [3.0, 5.0, 8.0])
def test_gaussian_encircled_energy(r):
    F, sig = 1.0e4, 2.0
    sub, x2, y2, xy = gaussian(96, 96, 47.37, 48.81, sig, sig, 0.0, F)
    o = ph.photometry(sub, np.ones_like(sub), rec(47.37, 48.81, x2, y2, xy), ph.PhotParams(r_aper=r))[0]
    assert o["flux_aper"] == pytest.approx(F * (1 - np.exp(-r * r / (2 * sig * sig))), rel=0.05 / r + 2e-3)


@pytest.mark.parametrize("sx,sy,theta", [(2.0, 2.0, 0.0), (3.0, 1.5, np.pi / 6), (3.0, 1.5, -np.pi / 3), (1.2, 4.0, 0.4)])
def test_kron_radius_and_auto_flux_of_a_gaussian(sx, sy, theta):
    """In the normalised metric a Gaussian has r1 = sqrt(pi/2) whatever its shape and orientation; the auto aperture of
    2.5 r1 then holds 1 - exp(-(2.5 r1)^2 / 2) of the flux.  A wrong sign of cxy or swapped cxx/cyy misaligns the
    ellipse with the source and fails both."""
    F = 5.0e4
    sub, x2, y2, xy = gaussian(160, 160, 80.2, 79.7, sx, sy, theta, F)
    p = ph.PhotParams(kron_min_radius=0.1)
    o = ph.photometry(sub, np.ones_like(sub), rec(80.2, 79.7, x2, y2, xy), p)[0]
    r1 = np.sqrt(np.pi / 2)
    assert o["kron_radius"] == pytest.approx(2.5 * r1, rel=2e-2)
    assert o["flux_auto"] == pytest.approx(F * (1 - np.exp(-0.5 * (2.5 * r1) ** 2)), rel=5e-3)
    assert o["npix_auto"] == pytest.approx(np.pi * o["kron_radius"] ** 2 * sx * sy, rel=3e-2)
    # the minimum radius takes over when larger
    o2 = ph.photometry(sub, np.ones_like(sub), rec(80.2, 79.7, x2, y2, xy), ph.PhotParams(kron_min_radius=3.5))[0]
    assert o2["kron_radius"] == 3.5 and o2["flux_auto"] == pytest.approx(F * (1 - np.exp(-0.5 * 3.5**2)), rel=5e-3)


def test_invariants_translation_scaling_flags_degenerate():
    rng = np.random.default_rng(3)
    sub = rng.normal(0, 1, (90, 110)).astype(np.float32); rms = rng.uniform(1, 2, (90, 110)).astype(np.float32)
    g, x2, y2, xy = gaussian(90, 110, 40.4, 50.6, 2.5, 1.7, 0.7, 3000.0)
    sub = sub + g
    p = ph.PhotParams(r_aper=6.0)
    a = ph.photometry(sub, rms, rec(40.4, 50.6, x2, y2, xy), p)[0]
    # integer shift of image and centroid: identical sums
    sub2 = np.zeros((100, 130), np.float32); rms2 = np.ones((100, 130), np.float32)
    sub2[7:97, 13:123] = sub; rms2[7:97, 13:123] = rms
    b = ph.photometry(sub2, rms2, rec(40.4 + 13, 50.6 + 7, x2, y2, xy), p)[0]
    for k in ("flux_aper", "area_aper", "kron_radius", "flux_auto", "npix_auto"):
        assert a[k] == pytest.approx(b[k], rel=1e-12), k
    # scaling the image scales the fluxes and leaves radius, area and errors alone
    c = ph.photometry(2 * sub, rms, rec(40.4, 50.6, x2, y2, xy), p)[0]
    assert c["flux_aper"] == pytest.approx(2 * a["flux_aper"]) and c["flux_auto"] == pytest.approx(2 * a["flux_auto"])
    assert c["kron_radius"] == pytest.approx(a["kron_radius"]) and c["fluxerr_aper"] == pytest.approx(a["fluxerr_aper"])
    # larger aperture of a positive image holds more flux
    pos = np.abs(sub)
    f = [ph.photometry(pos, rms, rec(40.4, 50.6, x2, y2, xy), ph.PhotParams(r_aper=r))[0]["flux_aper"] for r in (2, 4, 6, 9)]
    assert all(f[i] < f[i + 1] for i in range(3))
    # frame edge: flags, and sums over the part inside
    e = ph.photometry(sub, rms, rec(2.0, 3.0, x2, y2, xy), p)[0]
    assert e["flags"] & 1 and e["flags"] & 2 and e["area_aper"] < np.pi * 36 * 0.8
    # degenerate moments get 1/12 added: a circle of sigma = sqrt(1/12)
    cxx, cyy, cxy, q2, r2 = ph.ellipse_coefficients(0.0, 0.0, 0.0)
    assert cxx == pytest.approx(12.0) and cyy == pytest.approx(12.0) and cxy == 0.0 and q2 == pytest.approx(1 / 12)
    spike = np.zeros((90, 110), np.float32); spike[50, 40] = 100.0       # all the flux at r = 0: r1 = 0 -> minimum radius
    d = ph.photometry(spike, rms, rec(40.0, 50.0, 0.0, 0.0, 0.0), ph.PhotParams())[0]
    assert d["kron_radius"] == 3.5 and d["npix_auto"] == 5     # radius 3.5 * 0.2887 = 1.01 px: the centre and its 4 neighbours
    assert d["flux_auto"] == 100.0
    # no positive flux: minimum radius
    z = ph.photometry(-np.abs(sub), rms, rec(40.4, 50.6, x2, y2, xy), ph.PhotParams())[0]
    assert z["kron_radius"] == 3.5


def test_aperture_weights_are_fractions():
    ys, xs = np.mgrid[-8:9, -8:9]
    w = ph.aperture_weights(0.0, 0.0, 5.0, xs, ys, 5)
    assert w.min() == 0.0 and w.max() == 1.0 and np.array_equal(w, w[::-1, ::-1]) and np.array_equal(w, w.T)
    assert w[8, 8] == 1.0 and w[8, 8 + 4] == 1.0 and w[8, 8 + 6] == 0.0 and 0.0 < w[8, 8 + 5] < 1.0
    assert w[8, 8 + 5] == pytest.approx(0.5, abs=0.11)     # the rim pixel on the axis is cut in half


def test_a28_records_without_an_ellipse_are_not_measured():
    """Reading A28 (PAPER.md:159 names the methods only): a record whose centroid or moments are not finite, or whose
    moments still define no ellipse after the 1/12 rule (A24), is not measured -- every sum 0, flags = 4 -- while the
    1/12 rule itself keeps measuring.  Expected values written out by hand: a spike of 100 at (40, 50) on zeros, rms = 1,
    so s1 = 0, the Kron radius is the minimum 3.5 and the auto ellipse is a circle of 3.5 sqrt(x2) pixels about (40, 50)."""
    sub = np.zeros((90, 110), np.float32); sub[50, 40] = 100.0
    rms = np.ones_like(sub)
    p = ph.PhotParams()
    zeros = (0.0, 0.0, 0.0, 0.0, 0.0, 0.0, 0, 4)
    nan, inf = float("nan"), float("inf")
    not_measured = [(nan, 50.0, 2.0, 2.0, 0.0), (40.0, nan, 2.0, 2.0, 0.0),        # centroid
                    (40.0, 50.0, inf, 2.0, 0.0), (40.0, 50.0, 2.0, -inf, 0.0), (40.0, 50.0, 2.0, 2.0, nan),   # moments
                    (40.0, 50.0, -3.0, -3.0, 0.0),      # D = 9 > 0 but both variances negative
                    (40.0, 50.0, -0.5, 2.0, 0.0),       # D = -1: the 1/12 rule gives (-0.4167, 2.0833), D still < 0
                    (40.0, 50.0, 1.0, 1.0, 1.5),        # |xy| > sqrt(x2 y2): D = -1.25, after 1/12: 1.1736 - 2.25 < 0
                    (40.0, 50.0, -1.0 / 12.0, 1.0, 0.0)]  # the rule lifts x2 to exactly 0: no ellipse
    for r in not_measured:
        o = ph.photometry(sub, rms, rec(*r), p)[0]
        assert tuple(o) == zeros, (r, tuple(o))
    # D = x2 y2 - xy^2 just BELOW 0.00694 (0.083^2 = 0.006889): 1/12 is added, radius 3.5 sqrt(0.083 + 1/12) = 1.427 px:
    # the centre, its 4 neighbours (1 px) and the 4 diagonals (1.414 px) = 9 pixels
    lo = ph.photometry(sub, rms, rec(40.0, 50.0, 0.083, 0.083, 0.0), p)[0]
    assert (lo["flags"], lo["npix_auto"], lo["kron_radius"], lo["flux_auto"]) == (0, 9, 3.5, 100.0)
    assert lo["fluxerr_auto"] == pytest.approx(3.0, rel=1e-12)
    # just ABOVE (0.0834^2 = 0.006956): measured as it stands, radius 3.5 sqrt(0.0834) = 1.011 px: centre + 4 neighbours
    hi = ph.photometry(sub, rms, rec(40.0, 50.0, 0.0834, 0.0834, 0.0), p)[0]
    assert (hi["flags"], hi["npix_auto"], hi["kron_radius"], hi["flux_auto"]) == (0, 5, 3.5, 100.0)
    assert hi["fluxerr_auto"] == pytest.approx(np.sqrt(5.0), rel=1e-12)
    # the aperture sums of a measured record do not depend on the moments: circle of r = 5 about the spike
    for o in (lo, hi):
        assert o["flux_aper"] == 100.0 and o["area_aper"] == pytest.approx(np.pi * 25.0, rel=0.01)
    # a degenerate record between two good ones leaves them alone (records are independent)
    cat = np.concatenate([rec(40.0, 50.0, 0.0834, 0.0834, 0.0), rec(nan, 50.0, 2.0, 2.0, 0.0), rec(40.0, 50.0, 0.083, 0.083, 0.0)])
    o3 = ph.photometry(sub, rms, cat, p)
    assert list(o3["flags"]) == [0, 4, 0] and list(o3["npix_auto"]) == [5, 0, 9]
