"""Pins for the oracle's background variants O8 (readings B1-B6).  CPU only.  Each pin is something other
than the oracle: numpy masked arrays, scipy.ndimage, hand-made grids, closed forms."""
import numpy as np
import pytest
import scipy.ndimage as ndi

import oracle
from oracle import BkgParams, BkgXParams
from oracle import bkg_variants as bv


def _brute_clip_masked(vals, bad, k, iters):
    """numpy masked arrays, no code shared with oracle.c: the caller's mask is simply the initial mask."""
    m = np.ma.masked_array(vals.astype(np.float64), mask=bad.astype(bool))
    for _ in range(iters):
        med, sd = np.ma.median(m), m.std()
        out = (m.data < med - k * sd) | (m.data > med + k * sd)
        newmask = m.mask | out
        if newmask.sum() == m.mask.sum() or newmask.all():
            break
        m = np.ma.masked_array(m.data, mask=newmask)
    return float(np.ma.median(m)), float(m.mean()), float(m.std()), int(m.count())


@pytest.mark.parametrize("seed", range(10))
def test_masked_mesh_is_numpy_masked_array(seed):
    """B1: a masked mesh has the statistics of np.ma on the same mask, with and without clipping, ties included."""
    rng = np.random.default_rng(seed)
    h, w = int(rng.integers(3, 12)), int(rng.integers(3, 12))
    v = (rng.integers(0, 7, size=(h, w)) if seed % 2 else rng.normal(50, 3, size=(h, w))).astype(np.float32)
    v.reshape(-1)[rng.integers(0, h * w, 2)] = 1.0e4
    bad = (rng.uniform(size=(h, w)) < 0.3).astype(np.uint8)
    bad.reshape(-1)[0] = 0
    for iters, k in ((0, 3.0), (5, 2.0)):
        st = oracle.mesh_stats_masked(v, bad, BkgParams(mesh_h=h, mesh_w=w, clip_sigma=k, clip_iters=iters), BkgXParams(min_valid_px=1))
        med, mean, sd, n = _brute_clip_masked(v.reshape(-1), bad.reshape(-1), k, iters)
        assert st["n_valid"][0, 0] == int((bad == 0).sum()) and st["n_kept"][0, 0] == n
        assert st["median"][0, 0] == pytest.approx(med, abs=1e-12)
        assert st["mean"][0, 0] == pytest.approx(mean, rel=1e-12, abs=1e-12)
        assert st["rms"][0, 0] == pytest.approx(sd, rel=1e-10, abs=1e-12)


def test_mask_of_zeros_is_the_unmasked_path_and_masked_values_do_not_matter():
    rng = np.random.default_rng(3)
    img = rng.normal(300, 10, size=(96, 160)).astype(np.float32)
    p = BkgParams(mesh_h=32, mesh_w=32)
    a = oracle.mesh_stats(img, p)
    b = oracle.mesh_stats_masked(img, np.zeros(img.shape, np.uint8), p, BkgXParams())
    for k in ("bkg", "rms", "median", "mean", "n_kept"):
        assert np.array_equal(a[k], b[k])
    bad = (rng.uniform(size=img.shape) < 0.2).astype(np.uint8)
    img2 = img.copy(); img2[bad != 0] = -7.0e7          # garbage under the mask
    c, d = (oracle.mesh_stats_masked(im, bad, p, BkgXParams()) for im in (img, img2))
    for k in ("bkg", "rms", "n_kept", "n_valid"):
        assert np.array_equal(c[k], d[k])
    assert np.all(c["n_valid"] == 1024 - np.add.reduceat(np.add.reduceat(bad.astype(int), np.arange(0, 96, 32), 0), np.arange(0, 160, 32), 1))


def test_validity_rules_by_hand():
    """B2 / B6: 100-pixel rule, masked-fraction rule, crowded-mesh rule."""
    img = np.random.default_rng(0).normal(100, 5, size=(32, 64)).astype(np.float32)
    bad = np.zeros((32, 64), np.uint8)
    bad[:, :32] = 1; bad[:9, :32] = 0; bad[9, :11] = 0           # left mesh keeps 9*32 + 11 = 299 px; right mesh all 1024
    p = BkgParams(mesh_h=32, mesh_w=32)
    st = oracle.mesh_stats_masked(img, bad, p, BkgXParams(min_valid_px=299))
    assert st["n_valid"].tolist() == [[299, 1024]] and not np.isnan(st["bkg"]).any()
    st = oracle.mesh_stats_masked(img, bad, p, BkgXParams(min_valid_px=300))
    assert np.isnan(st["bkg"][0, 0]) and np.isnan(st["rms"][0, 0]) and st["n_kept"][0, 0] == 0 and not np.isnan(st["bkg"][0, 1])
    st = oracle.mesh_stats_masked(img, bad, p, BkgXParams(min_valid_px=1, max_masked_frac=0.7))      # 725/1024 = 0.708 masked
    assert np.isnan(st["bkg"][0, 0])
    st = oracle.mesh_stats_masked(img, bad, p, BkgXParams(min_valid_px=1, max_masked_frac=0.71))
    assert not np.isnan(st["bkg"][0, 0])
    # crowded: 5 % of the right mesh are "source" pixels far above the noise (sd ~ 1.1e4, 3 sd < 5e4): clipped in round 1,
    # then the mesh is excluded because too many of its pixels were rejected
    img2 = img.copy(); img2[:, 32:][np.random.default_rng(1).uniform(size=(32, 32)) < 0.05] = 50000.0
    n_src = int((img2[:, 32:] == 50000.0).sum())
    assert n_src > 30
    st = oracle.mesh_stats_masked(img2, None, p, BkgXParams(max_reject_frac=(n_src - 1) / 1024))
    assert np.isnan(st["bkg"][0, 1]) and not np.isnan(st["bkg"][0, 0])
    st = oracle.mesh_stats_masked(img2, None, p, BkgXParams(max_reject_frac=0.5))
    assert not np.isnan(st["bkg"][0, 1]) and 1024 - st["n_kept"][0, 1] >= n_src


def test_fill_invalid_by_hand():
    """B3: centre of a 3x3 -> median of its 8 neighbours; a corner -> of its 3; two rings when the first is empty."""
    g = np.arange(9, dtype=np.float64).reshape(3, 3); g[1, 1] = np.nan
    assert bv.fill_invalid(g)[1, 1] == 0.5 * (3 + 5)                    # neighbours 0 1 2 3 5 6 7 8
    g = np.arange(9, dtype=np.float64).reshape(3, 3); g[0, 0] = np.nan
    assert bv.fill_invalid(g)[0, 0] == 3.0                              # neighbours 1 3 4
    g = np.full((5, 5), np.nan); g[0, 4] = 7.0; g[4, 4] = 9.0; g[4, 0] = 20.0
    f = bv.fill_invalid(g)
    assert f[2, 2] == 9.0 and f[1, 3] == 7.0 and f[0, 0] == 9.0         # r = 2: {7, 9, 20}; r = 1: {7}; r = 4: {7, 9, 20}
    assert f[3, 1] == 20.0 and f[4, 4] == 9.0
    assert np.all(bv.fill_invalid(np.full((2, 3), np.nan)) == 0.0)
    ok = np.random.default_rng(2).normal(size=(4, 6))
    assert np.array_equal(bv.fill_invalid(ok), ok)


def test_dilate_is_scipy_binary_dilation():
    rng = np.random.default_rng(5)
    m = (rng.uniform(size=(40, 57)) < 0.03).astype(np.uint8)
    for g in (0, 1, 2, 3):
        want = ndi.binary_dilation(m != 0, structure=np.ones((2 * g + 1, 2 * g + 1), bool)) if g else (m != 0)
        assert np.array_equal(bv.dilate(m, g) != 0, want)


def test_all_masked_mesh_is_filled_from_its_neighbours():
    """A frame with a linear ramp: the background of a fully masked mesh comes from its 8 neighbours (B3), and the map
    stays within the ramp's range there."""
    yy, xx = np.mgrid[:192, :192]
    img = (100.0 + 0.1 * xx + 0.05 * yy).astype(np.float32)
    bad = np.zeros(img.shape, np.uint8); bad[64:128, 64:128] = 1
    p = BkgParams(mesh_h=64, mesh_w=64, filt_h=1, filt_w=1)
    b = bv.background_masked(img, bad, p, BkgXParams())
    assert b["valid"].tolist() == [[1, 1, 1], [1, 0, 1], [1, 1, 1]]
    st = b["stats"]["bkg"]
    neigh = np.sort(np.delete(st.reshape(-1), 4))
    assert b["bkg_grid"][1, 1] == 0.5 * (neigh[3] + neigh[4])
    full = bv.background_masked(img, None, p, BkgXParams())
    assert abs(b["bkg_grid"][1, 1] - full["bkg_grid"][1, 1]) < 0.5       # the ramp's centre value, by symmetry


def test_iteration_constant_frame_is_a_fixed_point_and_stars_are_masked_out():
    """B4: (i) nothing is detected on a constant frame, so every iteration returns the same grids; (ii) flat sky c plus
    bright top-hat 'stars': once the stars are masked the background is exactly c and the rms exactly 0 (closed form),
    while the un-iterated estimate of the star meshes is not."""
    p = BkgParams(mesh_h=32, mesh_w=32, filt_h=1, filt_w=1, clip_iters=0)
    const = np.full((96, 96), 321.0, dtype=np.float32)
    b0, _ = bv.iterate(const, None, p, BkgXParams(), 1.5, 0)
    b2, bad = bv.iterate(const, None, p, BkgXParams(), 1.5, 2)
    assert np.array_equal(b0["bkg_grid"], b2["bkg_grid"]) and not bad.any()
    img = const.copy()
    for (y, x) in ((10, 12), (50, 50), (80, 20)):
        img[y - 2:y + 3, x - 2:x + 3] += 4000.0
    first, _ = bv.iterate(img, None, p, BkgXParams(grow=1), 1.5, 0)
    assert np.abs(first["stats"]["mean"] - 321.0).max() > 50.0 and first["stats"]["rms"].max() > 100.0
    last, bad = bv.iterate(img, None, p, BkgXParams(grow=1), 1.5, 1)
    assert np.all(last["stats"]["bkg"] == 321.0) and np.all(last["stats"]["rms"] == 0.0)
    assert bad[8:13, 10:15].all() and bad[7, 9] == 1 and bad.sum() >= 3 * 49
