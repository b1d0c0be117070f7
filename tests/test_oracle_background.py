"""Pins for the oracle's background steps O1-O3 (CPU only).  Each pin is something OTHER than the
oracle: a library routine on a special case, a closed form, a hand-made case, or brute force."""
import math
import os

import numpy as np
import pytest
import scipy.ndimage as ndi
from scipy.stats import norm

import oracle
from oracle import BkgParams
from synth import noise_frame

GOLDEN = os.path.join(os.path.dirname(__file__), "golden")


def P(mesh=64, **kw):
    return BkgParams(mesh_h=mesh, mesh_w=mesh, **kw)


# ---------------------------------------------------------------- O1
def test_o1_golden_eq1_4():
    """hand-worked eqs. 1-4 (tests/golden/estimators_eq1_4.txt)."""
    for line in open(os.path.join(GOLDEN, "estimators_eq1_4.txt")):
        if line.startswith("#") or not line.strip():
            continue
        _, vals, med, mean, eq3, eq4 = [s.strip() for s in line.split("|")]
        v = np.array([float(t) for t in vals.split()], dtype=np.float32)[None, :]
        for (a, b, want) in ((1, 0, med), (0, -1, mean), (2.5, 1.5, eq3), (3, 2, eq4)):   # eq2 = 0*med - (-1)*mean
            st = oracle.mesh_stats(v, BkgParams(mesh_h=1, mesh_w=v.shape[1], clip_iters=0,
                                                median_factor=a, mean_factor=b))
            assert st["bkg"][0, 0] == pytest.approx(float(want), abs=1e-12)


def test_o1_constant_mesh_exact():
    img = np.full((128, 192), 1234.5, dtype=np.float32)
    st = oracle.mesh_stats(img, P(64))
    assert np.all(st["bkg"] == 1234.5) and np.all(st["rms"] == 0.0)
    assert np.all(st["n_kept"] == 4096) and np.all(st["rounds"] == 0)


def test_o1_no_clipping_is_numpy():
    """clip_iters=0 reduces to np.median / np.mean / np.std on each mesh (library routine)."""
    rng = np.random.default_rng(5)
    img = rng.normal(500, 20, size=(100, 150)).astype(np.float32)      # partial edge meshes (A9)
    st = oracle.mesh_stats(img, BkgParams(mesh_h=32, mesh_w=64, clip_iters=0))
    for j in range(st["bkg"].shape[0]):
        for i in range(st["bkg"].shape[1]):
            t = img[j * 32:(j + 1) * 32, i * 64:(i + 1) * 64].astype(np.float64)
            assert st["median"][j, i] == np.median(t)
            assert st["mean"][j, i] == pytest.approx(np.mean(t), rel=1e-14)
            assert st["rms"][j, i] == pytest.approx(np.std(t), rel=1e-12)
            assert st["n_kept"][j, i] == t.size
            assert st["bkg"][j, i] == pytest.approx(3 * np.median(t) - 2 * np.mean(t), rel=1e-12)


def test_o1_outlier_mesh_by_hand():
    """4090 px at 100 + 6 px at 60000: round 1 has median 100, sd ~2291 -> bounds 100 +- 6874 drop
    exactly the 6; round 2 is constant (sd 0, inclusive bounds keep all) -> stable."""
    v = np.full(4096, 100.0, dtype=np.float32)
    v[[3, 500, 1000, 2000, 3000, 4095]] = 60000.0
    st = oracle.mesh_stats(v.reshape(64, 64), P(64))
    assert st["n_kept"][0, 0] == 4090 and st["rounds"][0, 0] == 1
    assert st["bkg"][0, 0] == 100.0 and st["rms"][0, 0] == 0.0


def _brute_clip(vals, k, iters):
    """Independent restatement with numpy masked arrays (no sorting code shared with oracle.c)."""
    m = np.ma.masked_array(vals.astype(np.float64), mask=np.zeros(vals.shape, bool))
    for _ in range(iters):
        med, sd = np.ma.median(m), m.std()
        bad = (m.data < med - k * sd) | (m.data > med + k * sd)
        newmask = m.mask | bad
        if newmask.sum() == m.mask.sum() or newmask.all():
            break
        m = np.ma.masked_array(m.data, mask=newmask)
    return float(np.ma.median(m)), float(m.mean()), float(m.std()), int(m.count())


@pytest.mark.parametrize("seed", range(12))
def test_o1_bruteforce_random_meshes(seed):
    rng = np.random.default_rng(seed)
    h, w = int(rng.integers(1, 9)), int(rng.integers(1, 9))
    if seed % 3 == 0:   # heavy ties (integer data)
        v = rng.integers(0, 6, size=(h, w)).astype(np.float32)
    elif seed % 3 == 1:  # outliers
        v = rng.normal(10, 1, size=(h, w)).astype(np.float32)
        v.reshape(-1)[rng.integers(0, h * w)] = 1e4
    else:
        v = rng.standard_cauchy(size=(h, w)).astype(np.float32)
    k = [3.0, 2.0, 1.0][seed % 3]
    st = oracle.mesh_stats(v, BkgParams(mesh_h=h, mesh_w=w, clip_sigma=k, clip_iters=5))
    med, mean, sd, n = _brute_clip(v.reshape(-1), k, 5)
    assert st["n_kept"][0, 0] == n
    assert st["median"][0, 0] == pytest.approx(med, abs=1e-12)
    assert st["mean"][0, 0] == pytest.approx(mean, rel=1e-12, abs=1e-12)
    assert st["rms"][0, 0] == pytest.approx(sd, rel=1e-10, abs=1e-12)


def _truncated_sigma_fixed_point(k, rounds):
    """s <- sqrt(1 - 2 a phi(a) / (2 Phi(a) - 1)), a = k*s: std of a Gaussian truncated at +-k*s."""
    s, out = 1.0, []
    for _ in range(rounds):
        a = k * s
        s = math.sqrt(1.0 - 2.0 * a * norm.pdf(a) / (2.0 * norm.cdf(a) - 1.0))
        out.append(s)
    return out


def test_o1_gaussian_noise_statistics():
    """Pure N(mu, sigma^2): bkg -> mu; rms/sigma lies between the 2-round and fixed-point values of the
    truncation recurrence (0.98505 .. 0.98485), within statistical error."""
    mu, sigma = 1000.0, 25.0
    img = noise_frame(11, 1024, 1024, mu, sigma)
    st = oracle.mesh_stats(img, P(256))           # 16 meshes of 65536 px
    seq = _truncated_sigma_fixed_point(3.0, 30)
    assert seq[0] == pytest.approx(0.98658, abs=2e-5) and seq[-1] == pytest.approx(0.98485, abs=2e-5)
    ratio = st["rms"].mean() / sigma
    assert seq[-1] - 1.5e-3 < ratio < seq[0] + 1.5e-3
    # mode estimator 3*med - 2*mean: var ~ (9*pi/2 + 4 - 12) sigma^2 / N for Gaussian data
    se = sigma * math.sqrt((9 * math.pi / 2 + 4 - 12) / 65536.0)
    assert np.all(np.abs(st["bkg"] - mu) < 5 * se)
    assert np.all(st["n_kept"] >= 0.98 * 65536) and np.all(st["rounds"] <= 5)


def test_o1_survivors_form_interval_and_nkept_monotone():
    rng = np.random.default_rng(3)
    v = np.concatenate([rng.normal(0, 1, 4000), rng.uniform(5, 50, 96)]).astype(np.float32).reshape(64, 64)
    prev = None
    for iters in range(6):
        st = oracle.mesh_stats(v, P(64, clip_iters=iters))
        n = int(st["n_kept"][0, 0])
        assert prev is None or n <= prev
        prev = n
        # survivors are exactly the n values of a contiguous run of the sorted data that contains the median
        s = np.sort(v.reshape(-1).astype(np.float64))
        best = min(abs(np.median(s[a:a + n]) - st["median"][0, 0]) for a in range(0, s.size - n + 1))
        assert best < 1e-12
        assert n >= 0.75 * 4096 ** 1 * (0.75 ** max(iters - 1, 0)) or n > 3000


def test_o1_skew_guard():
    v = np.array([[1, 2, 3, 4, 100]], dtype=np.float32)
    st = oracle.mesh_stats(v, BkgParams(mesh_h=1, mesh_w=5, clip_iters=0, skew_guard=1))
    assert st["bkg"][0, 0] == 3.0      # |mean-median|/sd = 19/39 >= 0.3 -> median
    c = np.full((1, 5), 9.0, dtype=np.float32)
    st = oracle.mesh_stats(c, BkgParams(mesh_h=1, mesh_w=5, clip_iters=0, skew_guard=1))
    assert st["bkg"][0, 0] == 9.0      # sd = 0 -> mean


# ---------------------------------------------------------------- O2
@pytest.mark.parametrize("shape,size", [((8, 8), 3), ((37, 36), 5), ((2, 3), 3), ((1, 5), 5), ((6, 4), 1),
                                        ((5, 9), (3, 5))])
def test_o2_equals_scipy_nanmedian_filter(shape, size):
    rng = np.random.default_rng(shape[0] * 100 + shape[1])
    g = rng.normal(100, 10, size=shape)
    fh, fw = (size, size) if isinstance(size, int) else size
    want = ndi.generic_filter(g, np.nanmedian, size=(fh, fw), mode="constant", cval=np.nan)
    got = oracle.grid_median(g, fh, fw)
    assert np.max(np.abs(got - want)) == 0.0


def test_o2_spike_removed_and_identity():
    g = np.full((7, 7), 5.0); g[3, 3] = 1e6
    assert np.all(oracle.grid_median(g, 3, 3) == 5.0)
    r = np.random.default_rng(0).normal(size=(4, 6))
    assert np.array_equal(oracle.grid_median(r, 1, 1), r)


# ---------------------------------------------------------------- O3
@pytest.mark.parametrize("shape,mesh", [((5, 7), (8, 8)), ((1, 6), (4, 6)), ((2, 2), (16, 16)), ((3, 3), (5, 7)),
                                        ((8, 8), (64, 64)), ((37, 36), (3, 3))])
def test_o3_equals_scipy_zoom(shape, mesh):
    rng = np.random.default_rng(shape[0] + 7 * shape[1])
    g = rng.normal(300, 30, size=shape)
    mh, mw = mesh
    want = ndi.zoom(g, (mh, mw), order=3, mode="reflect", grid_mode=True)
    got = oracle.spline_eval(oracle.spline_coeffs(g), shape[0] * mh, shape[1] * mw, mh, mw)
    assert np.max(np.abs(got - want)) < 5e-12 * 300


def test_o3_cropped_partial_mesh():
    """H, W not multiples of the mesh: the grid is uniform, the map is the crop of the full zoom."""
    rng = np.random.default_rng(9)
    g = rng.normal(size=(3, 4))
    full = ndi.zoom(g, (20, 16), order=3, mode="reflect", grid_mode=True)
    got = oracle.spline_eval(oracle.spline_coeffs(g), 45, 50, 20, 16)
    assert np.max(np.abs(got - full[:45, :50])) < 1e-12


def test_o3_constant_and_interpolation_property():
    g = np.full((4, 5), 17.25)
    out = oracle.spline_eval(oracle.spline_coeffs(g), 4 * 7, 5 * 9, 7, 9)
    assert np.max(np.abs(out - 17.25)) < 1e-13
    rng = np.random.default_rng(2)
    g = rng.normal(size=(6, 5))
    out = oracle.spline_eval(oracle.spline_coeffs(g), 6 * 5, 5 * 7, 5, 7)     # odd mesh: centres are pixels
    assert np.max(np.abs(out[2::5, 3::7] - g)) < 1e-13


def test_o3_cubic_reproduced_in_interior():
    ny, nx, m = 40, 40, 4
    jj, ii = np.meshgrid(np.arange(ny, dtype=float), np.arange(nx, dtype=float), indexing="ij")
    poly = lambda a, b: 1.0 + 0.3 * a - 0.02 * a * a + 1e-3 * a ** 3 + 0.1 * b + 5e-3 * a * b  # noqa: E731
    out = oracle.spline_eval(oracle.spline_coeffs(poly(jj, ii)), ny * m, nx * m, m, m)
    y = (np.arange(ny * m) + 0.5) / m - 0.5
    Y, X = np.meshgrid(y, y, indexing="ij")
    sl = slice(15 * m, 25 * m)
    assert np.max(np.abs(out[sl, sl] - poly(Y, X)[sl, sl])) < 1e-6


# ---------------------------------------------------------------- background end to end
def test_background_constant_frame():
    img = np.full((200, 264), 777.0, dtype=np.float32)
    b = oracle.background(img, P(64))
    assert np.max(np.abs(b["bkg"] - 777.0)) < 1e-10 and np.max(np.abs(b["rms"])) < 1e-12
