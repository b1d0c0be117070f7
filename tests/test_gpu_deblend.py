"""GPU parity tests of NEXT-1: deblend_sources (K9) and clean_sources (K10) against oracle/deblend.py (O10, O11)
on the same inputs (stage parity: the oracle is fed the maps, labels and catalogue the GPU chain produced).
PAPER.md:155-157; readings D1-D12.  Run with `python -m pytest tests -m gpu` on a B200."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")

import oracle  # noqa: E402
from oracle import deblend as odb  # noqa: E402
from parity_util import assert_catalogue_equal  # noqa: E402
from synth import CONFIGS, make_frames, small  # noqa: E402


@pytest.fixture(scope="module")
def bd():
    import paper_2502_10783_b200 as m
    return m


@pytest.fixture(scope="module")
def ctx(bd):
    c = bd.Context(0)
    yield c
    c.close()


def dev(a):
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


def cat_to_dev(bd, cat, cap):
    raw = np.zeros(max(cap, 1), dtype=bd.SOURCE_DTYPE)
    for k in bd.SOURCE_DTYPE.names:
        raw[k][: len(cat)] = cat[k]
    return torch.from_numpy(raw.view(np.uint8)).cuda()


def gaussians(H, W, comps):
    yy, xx = np.mgrid[0:H, 0:W].astype(np.float64)
    img = np.zeros((H, W))
    for amp, x, y, sx, sy in comps:
        img += amp * np.exp(-0.5 * (((xx - x) / sx) ** 2 + ((yy - y) / sy) ** 2))
    return img.astype(np.float32)


def check_deblend(bd, ctx, sub, rms, labels, cat, detect_k, min_area, prm_kw=None, frame_of=None):
    """sub, rms float32 [B,H,W]; labels int32 [B,H,W]; cat: bd_source records (frame, label ascending).
    Runs K9 and O10 on the same inputs; labels bit-exact outside fragile candidates; records at the a5 tolerances."""
    prm_kw = prm_kw or {}
    B, H, W = sub.shape
    cap = max(len(cat), 1)
    n_in = np.array([(cat["frame"] == f).sum() for f in range(B)], dtype=np.int64)
    d_lab = dev(labels.copy())
    cap_out = 4 * cap + 64
    out = bd.deblend_sources(ctx, dev(sub), dev(rms), d_lab, cat_to_dev(bd, cat, cap), dev(n_in), cap, detect_k, min_area,
                             bd.DeblendParams(**prm_kw), out_capacity=cap_out)
    torch.cuda.synchronize()
    lab_g = out["labels"].cpu().numpy()
    n_out = out["n_sources"].cpu().numpy()
    cat_g = bd.catalogue_to_numpy(out["cat"], out["n_sources"], cap_out)
    oprm = odb.DeblendParams(**{k: v for k, v in prm_kw.items() if k in ("n_thresh", "min_cont")})
    stats = dict(n_split=0, n_objects=0, fragile=0)
    for f in range(B):
        cf = cat[cat["frame"] == f]
        lab_o, nobj, frag = odb.deblend(sub[f], rms[f], labels[f], cf, detect_k, min_area, oprm)
        cat_o = oracle.reduce_sources(lab_o, sub[f], min_area)
        ok = ~np.isin(labels[f], frag) if frag else np.ones((H, W), bool)
        assert np.array_equal(lab_g[f][ok], lab_o[ok]), f"frame {f}: {(lab_g[f][ok] != lab_o[ok]).sum()} label mismatches"
        exempt = set()
        for L in frag:
            exempt.update(int(v) for v in np.unique(lab_o[labels[f] == L]))
            exempt.update(int(v) for v in np.unique(lab_g[f][labels[f] == L]))
        got = cat_g[cat_g["frame"] == f]
        if not frag:
            assert n_out[f] == len(cat_o), (n_out[f], len(cat_o))
        assert_catalogue_equal(got, cat_o, exempt_labels=exempt)
        stats["n_split"] += sum(v > 1 for v in nobj.values())
        stats["n_objects"] += len(cat_o)
        stats["fragile"] += len(frag)
    return stats, lab_g, cat_g, n_out


def labelled(sub, rms, detect_k, min_area):
    """O4-O6 of a given (sub, rms): mask by the float32 rule, labels, records with the frame field."""
    B = sub.shape[0]
    labs, cats = [], []
    for f in range(B):
        mask = ((rms[f] > 0) & (sub[f] > np.float32(detect_k) * rms[f])).astype(np.uint8)
        lab = oracle.label(mask)
        c = oracle.reduce_sources(lab, sub[f], min_area)
        labs.append(lab)
        cats.append(as_sources(c, f))
    return np.stack(labs), np.concatenate(cats)


def as_sources(c, frame):
    import paper_2502_10783_b200 as m
    out = np.zeros(len(c), dtype=m.SOURCE_DTYPE)
    for k in m.SOURCE_DTYPE.names:
        if k == "frame":
            out[k] = frame
        else:
            out[k] = c[k]
    return out


# ------------------------------------------------------------------------------------------- analytic scenes, every tier
@pytest.mark.parametrize("scale,name", [(1.0, "warp"), (2.2, "mid"), (4.5, "big"), (9.0, "global")])
def test_k9_gaussian_scenes_every_tier(bd, ctx, scale, name):
    """Pairs, a triple, a faint companion and an isolated source, scaled so that the candidates' bounding boxes fall into
    each of the four tiers of K9 (<= 256, <= 1536, <= 5120 pixels, larger)."""
    s = 1.6 * scale
    H = W = int(64 * scale) * 4
    u = 64 * scale
    comps = [(200.0, 0.5 * u, 0.5 * u, s, s), (200.0, 0.5 * u + 3.2 * s, 0.5 * u, s, s),                  # equal pair
             (300.0, 1.5 * u, 0.5 * u, s, s), (3.0, 1.5 * u + 3.5 * s, 0.5 * u + s, s, s),                # faint companion
             (150.0, 2.5 * u, 0.5 * u, s, 1.4 * s),                                                       # alone
             (120.0, 0.6 * u, 1.6 * u, s, s), (90.0, 0.6 * u + 3.4 * s, 1.6 * u, s, s), (60.0, 0.6 * u + 6.8 * s, 1.6 * u, s, s),
             (250.0, 2.2 * u, 2.2 * u, s, s), (220.0, 2.2 * u + 2.4 * s, 2.2 * u + 2.4 * s, s, s),        # diagonal pair
             (80.0, 3.3 * u, 3.3 * u, s, s), (80.0, 3.3 * u + 1.5 * s, 3.3 * u, s, s)]                    # unimodal pair
    rng = np.random.default_rng(int(scale * 10))
    sub = (gaussians(H, W, comps).astype(np.float64) + rng.normal(0, 0.2, (H, W))).astype(np.float32)[None]
    rms = np.full_like(sub, 1.0)
    labels, cat = labelled(sub, rms, 1.5, 5)
    areas = (cat["xmax"] - cat["xmin"] + 1) * (cat["ymax"] - cat["ymin"] + 1)
    lo, hi = dict(warp=(0, 256), mid=(257, 1536), big=(1537, 5120), **{"global": (5121, 1 << 30)})[name]
    assert ((areas >= lo) & (areas <= hi)).sum() >= 3, (name, sorted(areas)[-8:])
    stats, lab_g, cat_g, _ = check_deblend(bd, ctx, sub, rms, labels, cat, 1.5, 5)
    assert stats["n_split"] >= 3 and stats["fragile"] == 0


def test_k9_parameters_and_degenerate_candidates(bd, ctx):
    """n_thresh 2..64, min_cont 0 and 1, min_area 1; a candidate whose peak does not exceed t_0; plateaus (ties)."""
    H = W = 96
    comps = [(50.0, 20, 20, 2.0, 2.0), (45.0, 27, 20, 2.0, 2.0), (30.0, 60, 60, 1.5, 3.0), (28.0, 60, 70, 1.5, 3.0), (6.0, 80, 15, 1.2, 1.2)]
    sub = gaussians(H, W, comps)[None].copy()
    sub[0, 40:44, 8:20] = 12.0          # a plateau: every pixel enters at the same level, ties in the growth
    sub[0, 40:44, 13] = 3.0
    rms = np.ones_like(sub)
    rms[0, 78:83, 13:18] = 4.5          # the faint source's peak pixel sits on a high-rms patch: peak <= t0 there
    for kw, min_area in ((dict(n_thresh=2), 5), (dict(n_thresh=8), 3), (dict(n_thresh=64), 5), (dict(min_cont=0.0), 5),
                         (dict(min_cont=1.0), 5), (dict(min_cont=0.05), 1)):
        labels, cat = labelled(sub, rms, 1.5, min_area)
        stats, *_ = check_deblend(bd, ctx, sub, rms, labels, cat, 1.5, min_area, kw)
        if kw.get("min_cont") == 1.0:
            assert stats["n_split"] == 0


@pytest.mark.parametrize("cfgn,S", [(1, 512), (2, 640), (3, 768), (5, 768)])
def test_k9_k10_config_crops(bd, ctx, cfgn, S):
    """The GPU chain on a crop of every config, then K9 / K10 against O10 / O11 fed with the GPU's own maps, labels and
    catalogue.  Config 5 (crowded, saturated stars) is the case the deblender exists for."""
    cfg = CONFIGS[cfgn]
    img = make_frames(small(cfg, S, S, B=1))
    p = bd.BkgParams(mesh_h=cfg.mesh, mesh_w=cfg.mesh, filt_h=cfg.filt, filt_w=cfg.filt)
    cap = 1 << 17
    d_img = dev(img)
    _, _, cb, cr = bd.bkg_estimate(ctx, d_img, p)
    fz = bd.bkg_subtract_detect(ctx, d_img, p.mesh_h, p.mesh_w, cb, cr, cfg.detect_k, cfg.min_area, cap)
    torch.cuda.synchronize()
    sub, rms, labels = fz["sub"].cpu().numpy(), fz["rms"].cpu().numpy(), fz["labels"].cpu().numpy()
    cat = bd.catalogue_to_numpy(fz["cat"], fz["n_sources"], cap)
    assert len(cat) < cap
    stats, lab_g, cat_g, n_out = check_deblend(bd, ctx, sub, rms, labels, cat, cfg.detect_k, cfg.min_area)
    if cfgn in (3, 5):
        assert stats["n_split"] > 10
    # ---- cleaning of the GPU's deblended catalogue
    check_clean(bd, ctx, rms, lab_g, cat_g, cfg.detect_k)


def check_clean(bd, ctx, rms, labels, cat, detect_k, prm_kw=None):
    prm_kw = prm_kw or {}
    B, H, W = rms.shape
    cap = max(len(cat), 1)
    n_in = np.array([(cat["frame"] == f).sum() for f in range(B)], dtype=np.int64)
    out = bd.clean_sources(ctx, dev(rms), dev(labels.copy()), cat_to_dev(bd, cat, cap), dev(n_in), cap, detect_k, bd.DeblendParams(**prm_kw))
    torch.cuda.synchronize()
    flags_g = out["flags"].cpu().numpy()[: len(cat)]
    lab_g = out["labels"].cpu().numpy()
    cat_g = bd.catalogue_to_numpy(out["cat"], out["n_sources"], cap)
    n_out = out["n_sources"].cpu().numpy()
    oprm = odb.DeblendParams(**{k: v for k, v in prm_kw.items() if k in ("clean_param", "clean_zone")})
    nflag = 0
    off = 0
    for f in range(B):
        cf = cat[cat["frame"] == f]
        lab_o, cat_o, flag_o, frag_o = odb.clean(labels[f], as_oracle(cf), rms[f], detect_k, oprm)
        fg = flags_g[off: off + len(cf)]
        off += len(cf)
        solid = frag_o == 0
        assert np.array_equal(fg[solid], flag_o[solid]), f"{(fg[solid] != flag_o[solid]).sum()} clean flags differ"
        nflag += int(flag_o.sum())
        if solid.all():
            assert np.array_equal(lab_g[f], lab_o)
            got = cat_g[cat_g["frame"] == f]
            assert n_out[f] == len(cat_o) == len(got)
            for k in got.dtype.names:
                if k != "frame":
                    assert np.array_equal(got[k], cat_o[k]), k      # survivors are copied, bit for bit
        else:
            # the label map may differ only on the objects whose decision is fragile
            amb = np.isin(labels[f], cf["label"][~solid])
            assert np.array_equal(lab_g[f][~amb], lab_o[~amb])
    return nflag


def as_oracle(c):
    """bd_source records -> the oracle's record dtype (same field names, no frame)."""
    ref = oracle.reduce_sources(np.zeros((1, 4), np.int32), np.zeros((1, 4), np.float32), 1)
    out = np.zeros(len(c), dtype=ref.dtype)
    for k in ref.dtype.names:
        out[k] = c[k]
    return out


def test_k10_clean_synthetic_catalogue(bd, ctx):
    """A bright elongated object and faint ones around it (inside and outside the zone, along and across the major axis),
    equal-flux ties, a degenerate (point-like) record; several beta / zone values."""
    H = W = 256
    comps = [(5000.0, 128, 128, 6.0, 2.0)]
    for ang in range(0, 360, 20):
        for rad, amp in ((14, 12.0), (30, 25.0), (60, 8.0)):
            if rad == 14 and 50 < ang % 180 < 130:
                continue                                   # (room for the faint objects off the short axis)
            comps.append((amp, 128 + rad * np.cos(np.deg2rad(ang)), 128 + rad * np.sin(np.deg2rad(ang)), 1.3, 1.3))
    # faint objects just off the short axis of the bright one: the Moffat-like wing extrapolated from its isophote
    # (D10) exceeds what they stand above their own threshold, so they are false detections (D11)
    comps += [(2.8, 128, 139, 1.3, 1.3), (2.8, 118, 140, 1.3, 1.3), (3.0, 140, 116, 1.3, 1.3), (2.6, 128, 117, 1.3, 1.3)]
    sub = gaussians(H, W, comps)[None]
    sub[0, 10, 10] = 40.0
    sub[0, 10, 11] = 40.0                                # a two-pixel object: degenerate moments
    sub[0, 200:203, 20:23] = 9.0
    sub[0, 200:203, 30:33] = 9.0                         # two objects with equal flux: the label breaks the tie
    rms = np.ones_like(sub)
    labels, cat = labelled(sub, rms, 1.5, 2)
    d = bd.deblend_sources(ctx, dev(sub), dev(rms), dev(labels.copy()), cat_to_dev(bd, cat, len(cat)), dev(np.array([len(cat)], np.int64)),
                           len(cat), 1.5, 2, bd.DeblendParams(min_cont=1e-5), out_capacity=8 * len(cat))
    torch.cuda.synchronize()
    lab2 = d["labels"].cpu().numpy()
    cat2 = bd.catalogue_to_numpy(d["cat"], d["n_sources"], 8 * len(cat))
    assert len(cat2) > len(cat)
    total = 0
    for kw in ({}, dict(clean_param=1.5), dict(clean_param=0.7, clean_zone=8.0), dict(clean_zone=1.0)):
        total += check_clean(bd, ctx, rms, lab2, cat2, 1.5, kw)
    assert total > 0


def test_k9_batch_and_capacity(bd, ctx):
    """B = 3 frames in one call (per-frame counts, frame-major order); an output capacity that is too small still gives the
    new label map and the true counts."""
    H = W = 160
    subs = []
    for f in range(3):
        rng = np.random.default_rng(100 + f)
        comps = [(float(10 ** rng.uniform(1.3, 2.8)), float(rng.uniform(6, W - 6)), float(rng.uniform(6, H - 6)), 1.5, 1.5) for _ in range(60)]
        subs.append((gaussians(H, W, comps).astype(np.float64) + rng.normal(0, 0.5, (H, W))).astype(np.float32))
    sub = np.stack(subs)
    rms = np.full_like(sub, 0.5)
    labels, cat = labelled(sub, rms, 1.5, 5)
    stats, lab_g, cat_g, n_out = check_deblend(bd, ctx, sub, rms, labels, cat, 1.5, 5)
    assert stats["n_split"] >= 6 and (n_out > 0).all()
    n_in = np.array([(cat["frame"] == f).sum() for f in range(3)], dtype=np.int64)
    tiny = bd.deblend_sources(ctx, dev(sub), dev(rms), dev(labels.copy()), cat_to_dev(bd, cat, len(cat)), dev(n_in), len(cat), 1.5, 5,
                              out_capacity=4)
    torch.cuda.synchronize()
    assert np.array_equal(tiny["labels"].cpu().numpy(), lab_g)
    assert np.array_equal(tiny["n_sources"].cpu().numpy(), n_out)


# ------------------------------------------------------------------------------------------- full-size frames, sampled
def _reach_bound(c, zone):
    """A generous upper bound of the distance at which record j can satisfy the zone test of D11 (test-side selection
    only: r_j^2 >= |d|^2 / (x2 + y2), so |d|^2 <= zone^2 rho^2 (x2 + y2) with rho^2 = npix / (pi sqrt(D)))."""
    x2, y2 = c["x2"] + 1.0 / 12.0, c["y2"] + 1.0 / 12.0
    D = np.maximum(c["x2"] * c["y2"] - c["xy"] ** 2, 1e-3)
    return 1.05 * zone * np.sqrt(c["npix"] / (np.pi * np.sqrt(D)) * (x2 + y2)) + 2.0


@pytest.mark.parametrize("cfgn", [3, 5])
def test_k9_k10_full_size_sampled(bd, ctx, cfgn):
    """BASELINE.json's full configs 3 and 5 in the launch configuration the bench uses: K9 on the whole frame; O10 on a
    sample of the candidates (the 12 largest, which take the workspace tier, and 400 seeded random ones): their pixels and
    records must agree.  K10 on the whole catalogue; O11 on the objects of a 768 x 768 window plus every object that can
    reach into it."""
    cfg = CONFIGS[cfgn]
    img = make_frames(cfg)
    B, H, W = img.shape
    p = bd.BkgParams(mesh_h=cfg.mesh, mesh_w=cfg.mesh, filt_h=cfg.filt, filt_w=cfg.filt)
    cap = 1 << 20
    d_img = dev(img)
    _, _, cb, cr = bd.bkg_estimate(ctx, d_img, p)
    fz = bd.bkg_subtract_detect(ctx, d_img, p.mesh_h, p.mesh_w, cb, cr, cfg.detect_k, cfg.min_area, cap)
    torch.cuda.synchronize()
    sub, rms, labels = fz["sub"][0].cpu().numpy(), fz["rms"][0].cpu().numpy(), fz["labels"][0].cpu().numpy()
    cat = bd.catalogue_to_numpy(fz["cat"], fz["n_sources"], cap)
    assert len(cat) < cap
    lab_d = fz["labels"].clone()
    out = bd.deblend_sources(ctx, fz["sub"], fz["rms"], lab_d, fz["cat"], fz["n_sources"], cap, cfg.detect_k, cfg.min_area)
    torch.cuda.synchronize()
    lab_g = lab_d[0].cpu().numpy()
    cat_g = bd.catalogue_to_numpy(out["cat"], out["n_sources"], cap)
    assert len(cat_g) < cap and np.all(np.diff(cat_g["label"].astype(np.int64)) > 0)
    assert np.array_equal(lab_g > 0, labels > 0)
    rng = np.random.default_rng(cfgn)
    big = np.argsort(cat["npix"])[-12:]
    pick = np.unique(np.concatenate([big, rng.choice(len(cat), 400, replace=False)]))
    only = cat["label"][pick]
    lab_o, nobj, frag = odb.deblend(sub, rms, labels, as_oracle(cat), cfg.detect_k, cfg.min_area, odb.DeblendParams(), only=only)
    solid = np.setdiff1d(only, frag)
    sel = np.isin(labels, solid)
    assert np.array_equal(lab_g[sel], lab_o[sel]), f"{(lab_g[sel] != lab_o[sel]).sum()} label mismatches"
    assert sum(v > 1 for v in nobj.values()) >= 5
    new_labels = np.unique(lab_o[sel])
    cat_o = oracle.reduce_sources(lab_o, sub, cfg.min_area)
    want = cat_o[np.isin(cat_o["label"], new_labels)]
    got = cat_g[np.isin(cat_g["label"], new_labels)]
    assert_catalogue_equal(got, want)
    # untouched by K9: everything that is not a candidate's pixel
    small_px = ~np.isin(labels, cat["label"])
    assert np.array_equal(lab_g[small_px], labels[small_px])

    # ---- K10 on the whole deblended catalogue; O11 on a window
    lab_c = lab_d.clone()
    cl = bd.clean_sources(ctx, fz["rms"], lab_c, out["cat"], out["n_sources"], cap, cfg.detect_k)
    torch.cuda.synchronize()
    flags_g = cl["flags"].cpu().numpy()[: len(cat_g)]
    x0, y0, S = W // 2 - 384, H // 2 - 384, 768
    inner = (cat_g["x"] >= x0) & (cat_g["x"] < x0 + S) & (cat_g["y"] >= y0) & (cat_g["y"] < y0 + S)
    reach = _reach_bound(cat_g, 4.0)
    dx = np.maximum(np.maximum(x0 - cat_g["x"], cat_g["x"] - (x0 + S)), 0.0)
    dy = np.maximum(np.maximum(y0 - cat_g["y"], cat_g["y"] - (y0 + S)), 0.0)
    near = np.hypot(dx, dy) <= reach
    idx = np.flatnonzero(inner | near)
    sub_cat = as_oracle(cat_g[idx])
    flag_o, frag_o = odb.clean_flags(sub_cat, rms, cfg.detect_k, odb.DeblendParams())
    chk = inner[idx] & (frag_o == 0)
    assert np.array_equal(flags_g[idx][chk], flag_o[chk]), f"{(flags_g[idx][chk] != flag_o[chk]).sum()} clean flags differ"
    assert flag_o[chk].sum() > 0
    # survivors: order kept, records copied; erased pixels are exactly those of the flagged records
    cat_c = bd.catalogue_to_numpy(cl["cat"], cl["n_sources"], cap)
    assert np.array_equal(cat_c["label"], cat_g["label"][flags_g == 0])
    lab_cg = lab_c[0].cpu().numpy()
    gone = np.isin(lab_g, cat_g["label"][flags_g != 0])
    assert not lab_cg[gone].any() and np.array_equal(lab_cg[~gone], lab_g[~gone])


def test_k9_workspace_tier_in_a_batch_and_reproducibility(bd, ctx):
    """Candidates of every tier (the largest take the frame-coordinate workspace arrays) in the SECOND frame of a batch;
    two runs give bit-identical label maps, counts and record keys (labels never depend on atomic order)."""
    scale = 9.0
    s = 1.6 * scale
    H = W = int(64 * scale) * 2
    u = 64 * scale
    big = [(200.0, 0.5 * u, 0.5 * u, s, s), (200.0, 0.5 * u + 3.2 * s, 0.5 * u, s, s),
           (120.0, 0.6 * u, 1.5 * u, s, s), (90.0, 0.6 * u + 3.4 * s, 1.5 * u, s, s)]
    small_ = [(60.0, 40 + 30 * k, 60 + 25 * (k % 3), 1.5, 1.5) for k in range(12)] + [(55.0, 44 + 30 * k, 61 + 25 * (k % 3), 1.5, 1.5) for k in range(12)]
    rng = np.random.default_rng(3)
    f0 = (gaussians(H, W, small_).astype(np.float64) + rng.normal(0, 0.2, (H, W))).astype(np.float32)
    f1 = (gaussians(H, W, big + [(c[0], c[1] + 600, c[2] + 700, c[3], c[4]) for c in small_]).astype(np.float64)
          + rng.normal(0, 0.2, (H, W))).astype(np.float32)
    sub = np.stack([f0, f1])
    rms = np.ones_like(sub)
    labels, cat = labelled(sub, rms, 1.5, 5)
    areas = (cat["xmax"] - cat["xmin"] + 1) * (cat["ymax"] - cat["ymin"] + 1)
    assert (areas[cat["frame"] == 1] > 5120).sum() >= 2
    stats, lab_a, cat_a, n_a = check_deblend(bd, ctx, sub, rms, labels, cat, 1.5, 5)
    assert stats["n_split"] >= 6
    _, lab_b, cat_b, n_b = check_deblend(bd, ctx, sub, rms, labels, cat, 1.5, 5)
    assert np.array_equal(lab_a, lab_b) and np.array_equal(n_a, n_b)
    for k in ("frame", "label", "npix", "xmin", "xmax", "ymin", "ymax", "xpeak", "ypeak", "peak"):
        assert np.array_equal(cat_a[k], cat_b[k]), k


def test_k9_k10_empty_and_tiny_inputs(bd, ctx):
    """Degenerate inputs: an empty catalogue (nothing detected), a zero capacity, a frame of one tile row; labels untouched,
    zero counts, no fault."""
    H, W = 32, 64
    sub = np.zeros((2, H, W), np.float32)
    rms = np.ones_like(sub)
    labels = np.zeros((2, H, W), np.int32)
    cat = np.zeros(0, dtype=bd.SOURCE_DTYPE)
    n0 = dev(np.zeros(2, np.int64))
    for cap in (0, 16):
        d_lab = dev(labels.copy())
        out = bd.deblend_sources(ctx, dev(sub), dev(rms), d_lab, cat_to_dev(bd, cat, cap), n0, cap, 1.5, 5, out_capacity=cap)
        cl = bd.clean_sources(ctx, dev(rms), d_lab, out["cat"], out["n_sources"], cap, 1.5)
        ph = bd.photometry(ctx, dev(sub), dev(rms), cl["cat"], cl["n_sources"], cap)
        torch.cuda.synchronize()
        assert out["n_sources"].sum().item() == 0 and cl["n_sources"].sum().item() == 0
        assert not d_lab.any().item() and ph is not None
    # one small candidate that cannot split (fewer than 2 * min_area pixels) next to one that can
    sub[1, 10:12, 10:13] = 9.0
    sub[1, 20:23, 30:40] = 9.0
    sub[1, 20:23, 34:36] = 2.0
    labels2, cat2 = labelled(sub, rms, 1.5, 5)
    stats, lab_g, cat_g, n_out = check_deblend(bd, ctx, sub, rms, labels2, cat2, 1.5, 5)
    assert n_out[0] == 0 and n_out[1] == 3 and stats["n_split"] == 1
