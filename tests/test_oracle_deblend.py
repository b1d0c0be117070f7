"""Pins for the deblending / cleaning oracle O10, O11 (CPU only, readings D1-D12)."""
import itertools
import math
import os

import numpy as np
import pytest
import scipy.ndimage as ndi

import oracle
from oracle import deblend as odb
from oracle.deblend import DeblendParams

GOLD = os.path.join(os.path.dirname(__file__), "golden", "deblend_two_peaks.txt")
EIGHT = np.ones((3, 3), dtype=int)


def gaussians(H, W, comps):
    """Noise-free sum of circular/elliptical Gaussians sampled at pixel centres: (amp, x, y, sx, sy)."""
    yy, xx = np.mgrid[:H, :W].astype(np.float64)
    img = np.zeros((H, W))
    for (a, x, y, sx, sy) in comps:
        img += a * np.exp(-0.5 * (((xx - x) / sx) ** 2 + ((yy - y) / sy) ** 2))
    return img.astype(np.float32)


def run(sub, t0=1.0, min_area=5, **kw):
    """Threshold at t0 (rms = t0, k = 1), label, reduce, deblend."""
    sub = np.asarray(sub, dtype=np.float32)
    rms = np.full(sub.shape, t0, dtype=np.float32)
    mask = (sub > t0).astype(np.uint8)
    lab = oracle.label(mask)
    cat = oracle.reduce_sources(lab, sub, min_area)
    prm = DeblendParams(**kw)
    lab2, nobj, frag = odb.deblend(sub, rms, lab, cat, 1.0, min_area, prm)
    return lab, cat, lab2, nobj, rms, prm


# ---------------------------------------------------------------- D2: thresholds
def test_thresholds_exact_powers_of_two_and_spacing():
    t = odb.thresholds(2.0 ** 32 * 3.0, 3.0, 32)              # q = 2 exactly: five exact square roots of 2^32
    assert np.array_equal(t, 3.0 * 2.0 ** np.arange(32))
    t = odb.thresholds(731.25, 1.7, 32)
    assert t[0] == 1.7 and np.all(np.diff(t) > 0)
    assert np.allclose(t[1:] / t[:-1], (731.25 / 1.7) ** (1 / 32), rtol=1e-14)
    assert abs(t[-1] * (731.25 / 1.7) ** (1 / 32) - 731.25) < 1e-9       # the level after the last one would be the peak
    with pytest.raises(AssertionError):
        odb.thresholds(10.0, 1.0, 24)


def test_candidate_threshold_is_the_float32_product():
    rms = np.full((3, 3), np.float32(2.1), dtype=np.float32)
    assert odb.candidate_threshold(1.3, rms, 1, 1) == float(np.float64(np.float32(1.3)) * np.float64(np.float32(2.1)))


# ---------------------------------------------------------------- golden: hand-worked strip
def test_golden_two_peaks_strip():
    sub, thr, cases = None, None, []
    for line in open(GOLD):
        w = line.split()
        if not w or w[0].startswith("#"):
            continue
        if w[0] == "sub":
            sub = np.array([[float(v) for v in w[1:]]], dtype=np.float32)
        elif w[0] == "thresholds":
            thr = [float(v) for v in w[1:]]
        elif w[0] == "case":
            kv = dict(s.split("=") for s in w[1:3])
            cases.append((float(kv["min_cont"]), int(kv["min_area"]), [int(v) for v in w[4:]]))
    assert np.array_equal(odb.thresholds(16.0, 1.0, 4), thr)
    assert len(cases) == 4
    for min_cont, min_area, want in cases:
        _, _, lab2, nobj, _, _ = run(sub, t0=1.0, min_area=min_area, n_thresh=4, min_cont=min_cont)
        assert lab2.tolist() == [want], (min_cont, min_area)
        assert list(nobj.values()) == [len(set(want))]


# ---------------------------------------------------------------- closed forms on analytic Gaussians
@pytest.mark.parametrize("amp,sx,sy,x,y", [(1000.0, 2.0, 2.0, 20.0, 20.0), (50.0, 1.3, 1.3, 20.4, 19.7),
                                           (3e5, 3.0, 1.5, 31.5, 30.0), (7.0, 2.5, 2.5, 25.0, 25.5)])
def test_single_gaussian_never_splits(amp, sx, sy, x, y):
    """A unimodal profile has one component above every level: the tree is a chain."""
    sub = gaussians(64, 64, [(amp, x, y, sx, sy)])
    lab, cat, lab2, nobj, _, _ = run(sub, t0=1.0, min_area=3)
    assert len(cat) == 1 and list(nobj.values()) == [1]
    assert np.array_equal(lab, lab2)


def test_two_equal_gaussians_split_symmetrically():
    """d = 5 sigma: saddle 2A exp(-d^2/8 s^2) = 0.088 A is far below the peaks, several levels lie between them -> two
    objects; the frame is mirror symmetric about x = 19.5, so are the objects, and each holds half the flux."""
    s, A = 2.0, 1000.0
    sub = gaussians(40, 40, [(A, 19.5 - 2.5 * s, 20.0, s, s), (A, 19.5 + 2.5 * s, 20.0, s, s)])
    assert np.array_equal(sub, sub[:, ::-1])
    lab, cat, lab2, nobj, _, _ = run(sub, t0=1.0, min_area=5)
    assert len(cat) == 1 and list(nobj.values()) == [2]
    ids = np.unique(lab2[lab2 > 0])
    assert len(ids) == 2
    a, b = lab2 == ids[0], lab2 == ids[1]
    assert np.array_equal(a, b[:, ::-1])
    assert a[:, :20].sum() == a.sum() and b[:, 20:].sum() == b.sum()        # split along the midline
    assert abs(sub[a].astype(np.float64).sum() - sub[b].astype(np.float64).sum()) < 1e-9 * sub.sum()
    assert np.array_equal(lab2 > 0, lab > 0)


def test_unimodal_pair_does_not_split():
    """Two equal Gaussians closer than 2 sigma add up to a single-peaked profile."""
    s = 2.5
    sub = gaussians(48, 48, [(500.0, 24.0 - 0.75 * s, 24.0, s, s), (500.0, 24.0 + 0.75 * s, 24.0, s, s)])
    lab, cat, lab2, nobj, _, _ = run(sub, t0=1.0, min_area=5)
    assert list(nobj.values()) == [1] and np.array_equal(lab, lab2)


def test_contrast_criterion_on_a_faint_companion():
    """Companion with 2 % of the primary's amplitude, 5 sigma away: its branch above the saddle (~9 ADU) holds
    ~20 * 2 pi s^2 * (1 - 9/20) = 1.1 % of the total flux: split at min_cont 0.005, not at 0.05."""
    s, A = 2.0, 1000.0
    sub = gaussians(48, 64, [(A, 24.0, 24.0, s, s), (0.02 * A, 24.0 + 5 * s, 24.0, s, s)])
    _, cat, lab2, nobj, _, _ = run(sub, t0=1.0, min_area=5, min_cont=0.005)
    assert len(cat) == 1 and list(nobj.values()) == [2]
    comp = oracle.reduce_sources(lab2, sub, 5)
    assert len(comp) == 2
    faint = comp[np.argmin(comp["flux"])]
    assert abs(faint["x"] - 34.0) < 0.7 and abs(faint["y"] - 24.0) < 0.2
    assert 0.005 < faint["flux"] / cat[0]["flux"] < 0.03
    _, _, lab3, nobj3, _, _ = run(sub, t0=1.0, min_area=5, min_cont=0.05)
    assert list(nobj3.values()) == [1]


def test_three_in_a_row_and_nested_split():
    """Three sources: the two close ones separate at a higher level than the far one -> a split below a split (D5)."""
    s = 1.8
    sub = gaussians(48, 96, [(2000.0, 20.0, 24.0, s, s), (1500.0, 20.0 + 4.2 * s, 24.0, s, s), (800.0, 70.0, 24.0, 2 * s, 2 * s)])
    sub += gaussians(48, 96, [(3.0, 45.0, 24.0, 20.0, 3.0)])                  # a faint bridge keeps them one candidate
    _, cat, lab2, nobj, _, _ = run(sub, t0=1.0, min_area=5)
    assert len(cat) == 1 and list(nobj.values()) == [3]
    comp = oracle.reduce_sources(lab2, sub, 5)
    assert sorted(np.round(comp["xpeak"]).astype(int).tolist()) == [20, 28, 70]


# ---------------------------------------------------------------- brute force on tiny images
def brute_force(sub, member, t, min_area, min_cont):
    """Independent statement of D3-D7: nodes as pixel sets (scipy.ndimage.label per level), pruning by the set-based
    characterisation 'an object is a significant node without two disjoint significant nodes inside it whose parent
    does have two', growth pixel by pixel with dictionaries."""
    h, w = sub.shape
    sub = sub.astype(np.float64)
    levels = [[frozenset(map(tuple, np.argwhere(member)))]]
    for i in range(1, len(t)):
        lab, n = ndi.label(member & (sub > t[i]), structure=EIGHT)
        levels.append([frozenset(map(tuple, np.argwhere(lab == k))) for k in range(1, n + 1) if (lab == k).sum() >= min_area])
    nodes = [(i, s) for i, lv in enumerate(levels) for s in lv]
    flux = {nd: sum(sub[p] for p in nd[1]) for nd in nodes}
    limit = min_cont * flux[nodes[0]]
    heavy = [nd for nd in nodes if nd[0] >= 1 and flux[nd] > limit]

    def simple(nd):                                   # no two disjoint significant nodes strictly inside nd
        inside = [h_ for h_ in heavy if h_[0] > nd[0] and h_[1] <= nd[1]]
        return not any(a[1].isdisjoint(b[1]) for a, b in itertools.combinations(inside, 2))

    def parent(nd):
        return next(p for p in nodes if p[0] == nd[0] - 1 and nd[1] <= p[1])

    root = nodes[0]
    if simple(root):
        return [root[1]]
    objs = [nd for nd in heavy if simple(nd) and not simple(parent(nd))]
    owner = {}
    for nd in objs:
        for p in nd[1]:
            assert p not in owner
            owner[p] = min(nd[1])                     # first pixel of the node in raster order
    todo = set(root[1]) - set(owner)
    while todo:
        new = {}
        for (y, x) in todo:
            best = None
            for dy in (-1, 0, 1):
                for dx in (-1, 0, 1):
                    q = (y + dy, x + dx)
                    if q != (y, x) and q in owner:
                        key = (-sub[q], owner[q])
                        if best is None or key < best[0]:
                            best = (key, owner[q])
            if best is not None:
                new[(y, x)] = best[1]
        assert new
        owner.update(new)
        todo -= set(new)
    out = {}
    for p, o in owner.items():
        out.setdefault(o, set()).add(p)
    return [frozenset(v) for v in out.values()]


@pytest.mark.parametrize("seed", range(40))
def test_brute_force_tiny_images(seed):
    rng = np.random.default_rng(1000 + seed)
    h, w = int(rng.integers(6, 13)), int(rng.integers(6, 13))
    nb = int(rng.integers(1, 5))
    comps = [(float(10 ** rng.uniform(1, 3)), float(rng.uniform(1, w - 2)), float(rng.uniform(1, h - 2)),
              float(rng.uniform(0.7, 1.8)), float(rng.uniform(0.7, 1.8))) for _ in range(nb)]
    sub = gaussians(h, w, comps).astype(np.float64) + rng.normal(0, 0.4, (h, w)) + 1.2
    if seed % 3 == 0:
        sub = np.round(sub)                           # ties
    sub = sub.astype(np.float32)
    min_area = int(rng.integers(1, 4))
    prm = DeblendParams(n_thresh=int(rng.choice([4, 8, 16])), min_cont=float(rng.choice([0.005, 0.03, 0.1, 0.25])))
    rms = np.full((h, w), 1.0, dtype=np.float32)
    lab = oracle.label((sub > 1.0).astype(np.uint8))
    cat = oracle.reduce_sources(lab, sub, min_area)
    lab2, nobj, _ = odb.deblend(sub, rms, lab, cat, 1.0, min_area, prm)
    for r in cat:
        member = lab == r["label"]
        t = odb.thresholds(float(r["peak"]), 1.0, prm.n_thresh)
        want = brute_force(sub, member, t, min_area, prm.min_cont)
        got = [frozenset(map(tuple, np.argwhere(lab2 == k))) for k in np.unique(lab2[member])]
        assert sorted(map(sorted, got)) == sorted(map(sorted, want))
        assert nobj[int(r["label"])] == len(want)


# ---------------------------------------------------------------- invariants on a realistic frame
def test_invariants_on_a_crowded_frame():
    rng = np.random.default_rng(5)
    H = W = 192
    n = 70
    comps = [(float(10 ** rng.uniform(1.2, 3.5)), float(rng.uniform(4, W - 4)), float(rng.uniform(4, H - 4)), 1.3, 1.3) for _ in range(n)]
    sub = (gaussians(H, W, comps).astype(np.float64) + rng.normal(0, 1.0, (H, W))).astype(np.float32)
    min_area = 5
    lab, cat, lab2, nobj, rms, prm = run(sub, t0=1.5, min_area=min_area)
    assert sum(v > 1 for v in nobj.values()) >= 3                     # the frame does have blends
    assert np.array_equal(lab2 > 0, lab > 0)                          # deblending only re-partitions candidates
    cat2 = oracle.reduce_sources(lab2, sub, min_area)
    assert len(cat2) == sum(nobj.values())
    small = ~np.isin(lab, cat["label"])
    assert np.array_equal(lab2[small], lab[small])                    # components below min_area are untouched (D1)
    for r in cat:
        member = lab == r["label"]
        ids = np.unique(lab2[member])
        assert len(ids) == nobj[int(r["label"])]
        assert np.all(np.isin(lab2[member], ids)) and not np.any(np.isin(lab2[~member], ids))
        tot = 0.0
        for k in ids:
            sel = lab2 == k
            assert ndi.label(sel, structure=EIGHT)[1] == 1            # every object is 8-connected
            assert sel.sum() >= min_area
            assert k == 1 + np.flatnonzero(sel.reshape(-1))[0]        # D8
            tot += float(sub[sel].astype(np.float64).sum())
        assert abs(tot - r["flux"]) <= 1e-9 * abs(r["flux"])          # flux is conserved over the children


# ---------------------------------------------------------------- cleaning
def make_cat(rows):
    """rows: dict(label, npix, flux, x, y, x2, y2, xy) -> O6-shaped records (peak pixel = rounded centroid)."""
    cat = np.zeros(len(rows), dtype=oracle.SOURCE_DTYPE)
    for k, r in enumerate(rows):
        for f, v in r.items():
            cat[k][f] = v
        cat[k]["xpeak"], cat[k]["ypeak"] = int(round(r["x"])), int(round(r["y"]))
    return cat


def test_clean_profile_crosses_the_threshold_on_the_isophote():
    """Circular neighbour j (x2 = y2 = s^2): I_j = t_j exactly at r^2 = rho_j^2, i.e. at distance s * rho_j.  An object
    sitting there is a false detection iff its mean surface brightness m satisfies m - t_j <= t_i, here m <= 2."""
    rms = np.ones((200, 200), dtype=np.float32)
    s2, npix, F = 4.0, 400, 1e5
    rho = math.sqrt(npix / (math.pi * s2))
    d = math.sqrt(s2) * rho
    prm = DeblendParams()
    for m, want in [(1.9, 1), (2.1, 0)]:
        cat = make_cat([dict(label=1, npix=npix, flux=F, x=100.0, y=100.0, x2=s2, y2=s2, xy=0.0),
                        dict(label=2, npix=10, flux=10 * m, x=100.0 + d, y=100.0, x2=1.0, y2=1.0, xy=0.0)])
        flag, frag = odb.clean_flags(cat, rms, 1.0, prm)
        assert flag.tolist() == [0, want] and frag.tolist() == [0, 0]
    # at the neighbour's centre the profile is its central amplitude F / (2 pi s^2): flagged iff m <= 1 + A
    A = F / (2 * math.pi * s2)
    for m, want in [(A + 0.9, 1), (A + 1.1, 0)]:
        cat = make_cat([dict(label=1, npix=npix, flux=F, x=100.0, y=100.0, x2=s2, y2=s2, xy=0.0),
                        dict(label=2, npix=10, flux=10 * m, x=100.0, y=100.0, x2=1.0, y2=1.0, xy=0.0)])
        assert odb.clean_flags(cat, rms, 1.0, prm)[0].tolist() == [0, want]


def test_clean_zone_brightness_order_and_orientation():
    rms = np.ones((400, 400), dtype=np.float32)
    prm = DeblendParams(clean_zone=3.0)
    big = dict(label=1, npix=300, flux=5e4, x=200.0, y=200.0, x2=9.0, y2=9.0, xy=0.0)
    rho = math.sqrt(300 / (math.pi * 9.0))
    faint = lambda lab, x, y: dict(label=lab, npix=10, flux=10.0, x=x, y=y, x2=4.0, y2=4.0, xy=0.0)   # mean sb = t: always
    # flagged when a brighter neighbour's zone holds it (lhs = 1 - I_j < 1), never outside the zone
    cat = make_cat([big, faint(2, 200.0 + 3 * rho * 3.0 * 0.99, 200.0), faint(3, 200.0 + 3 * rho * 3.0 * 1.01, 200.0)])
    assert odb.clean_flags(cat, rms, 1.0, prm)[0].tolist() == [0, 1, 0]
    # the brighter object is never flagged by a fainter one; equal fluxes: the smaller label is the brighter
    cat = make_cat([faint(1, 50.0, 50.0), faint(2, 51.0, 50.0)])
    cat["flux"] = 200.0; cat["npix"] = 200
    assert odb.clean_flags(cat, rms, 1.0, prm)[0].tolist() == [0, 1]
    # elongated neighbour along x (x2 >> y2): the same distance is inside the zone along x, outside along y
    lng = dict(label=1, npix=300, flux=5e4, x=200.0, y=200.0, x2=36.0, y2=2.25, xy=0.0)
    rho = math.sqrt(300 / (math.pi * math.sqrt(36.0 * 2.25)))
    d = 0.5 * (6.0 + 1.5) * 3 * rho                      # between the zone's semi-axes 3 rho * 1.5 and 3 rho * 6
    cat = make_cat([lng, faint(2, 200.0 + d, 200.0), faint(3, 200.0, 200.0 + d)])
    assert odb.clean_flags(cat, rms, 1.0, prm)[0].tolist() == [0, 1, 0]
    # the same ellipse rotated by +45 degrees (major axis along x = y): xy = (36 - 2.25) / 2 > 0
    rot = dict(label=1, npix=300, flux=5e4, x=200.0, y=200.0, x2=19.125, y2=19.125, xy=16.875)
    e = d / math.sqrt(2.0)
    cat = make_cat([rot, faint(2, 200.0 + e, 200.0 + e), faint(3, 200.0 + e, 200.0 - e)])
    assert odb.clean_flags(cat, rms, 1.0, prm)[0].tolist() == [0, 1, 0]
    # a neighbour whose central amplitude is below its threshold influences nobody
    weak = dict(label=1, npix=300, flux=50.0, x=200.0, y=200.0, x2=9.0, y2=9.0, xy=0.0)
    cat = make_cat([weak, faint(2, 201.0, 200.0)])
    assert odb.clean_flags(cat, rms, 1.0, prm)[0].tolist() == [0, 0]


def test_clean_removes_pixels_and_records():
    """A bright star with a detached noise bump in its wing: the bump is removed (D12), the star and a far object stay."""
    sub = gaussians(96, 160, [(4000.0, 40.0, 48.0, 2.0, 2.0), (30.0, 130.0, 48.0, 1.5, 1.5)])
    sub[47:50, 51:54] += 1.4       # 9-px bump 12 px (6 sigma) from the star, detached from it: I_j there = 4000 / (1 + 242 * 36) = 0.46
    sub = sub.astype(np.float32)
    lab, cat, lab2, nobj, rms, prm = run(sub, t0=1.0, min_area=5)
    cat2 = oracle.reduce_sources(lab2, sub, 5)
    assert len(cat2) == 3
    lab3, cat3, flag, frag = odb.clean(lab2, cat2, rms, 1.0, prm)
    bump = int(np.argmin(np.abs(cat2["x"] - 52.0)))
    assert flag.tolist() == [1 if k == bump else 0 for k in range(3)]
    assert len(cat3) == 2 and np.all(lab3[lab2 == cat2[bump]["label"]] == 0)
    keep = lab2 != cat2[bump]["label"]
    assert np.array_equal(lab3[keep], lab2[keep])
    out = odb.deblend_clean(sub, rms, lab, cat, 1.0, 5, prm)
    assert np.array_equal(out["labels"], lab3) and np.array_equal(out["cat"], cat3)
