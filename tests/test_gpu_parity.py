"""GPU parity tests: the CUDA path (through the C ABI) against the CPU oracle on the same seeded inputs.
Run with `python -m pytest tests -m gpu` on a B200."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")

import oracle  # noqa: E402
from parity_util import (assert_catalogue_equal, assert_maps_close, assert_mask_parity, fragile_touched_labels,  # noqa: E402
                         to_oracle_params)
from synth import CONFIGS, make_frame, make_frames, noise_frame  # noqa: E402


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


def params_for(bd, cfg, **kw):
    d = dict(mesh_h=cfg.mesh, mesh_w=cfg.mesh, filt_h=cfg.filt, filt_w=cfg.filt, clip_sigma=cfg.clip_sigma,
             clip_iters=cfg.clip_iters)
    d.update(kw)
    return bd.BkgParams(**d)


# ------------------------------------------------------------------------------------------- K1
def check_mesh_stats(bd, ctx, img, p):
    """img float32 [B,H,W] numpy.  Both the fast path (where it applies) and the forced general path."""
    for force_slow in (False, True):
        bd.k1_force_slow(ctx, force_slow)
        try:
            out = bd.mesh_stats(ctx, dev(img), p)
            torch.cuda.synchronize()
        finally:
            bd.k1_force_slow(ctx, False)
        _compare_mesh_stats(out, img, p)


def _compare_mesh_stats(out, img, p):
    op = to_oracle_params(p)
    for f in range(img.shape[0]):
        st = oracle.mesh_stats(img[f], op)
        assert np.array_equal(out["n_kept"][f].cpu().numpy(), st["n_kept"]), "n_kept differs"
        assert np.array_equal(out["median"][f].cpu().numpy(), st["median"]), "median differs"
        for k, ok in (("mean", "mean"), ("rms", "rms"), ("bkg", "bkg")):
            g, w = out[k][f].cpu().numpy(), st[ok]
            tol = 1e-10 * np.maximum(np.abs(w), np.abs(st["median"])) + 1e-300
            if k == "rms":
                tol = 1e-9 * np.maximum(np.abs(w), 1e-6 * np.abs(st["median"])) + 1e-300
            assert np.all(np.abs(g - w) <= tol), f"{k}: worst {np.max(np.abs(g - w) / tol)} x tol"


@pytest.mark.parametrize("cid,H,W", [(1, 512, 512), (2, 512, 640), (3, 528, 768), (4, 256, 320), (5, 384, 512)])
def test_k1_mesh_stats_configs(bd, ctx, cid, H, W):
    """Each config's frame recipe at a reduced size (several meshes + a ragged last mesh row for cfg 3)."""
    cfg = CONFIGS[cid]
    img = make_frames(cfg, H=H, W=W, B=2 if cid == 4 else 1)
    check_mesh_stats(bd, ctx, img, params_for(bd, cfg))


@pytest.mark.parametrize("mh,mw", [(64, 64), (32, 48), (50, 36), (17, 23), (128, 128), (256, 256), (100, 300), (7, 5), (1, 4)])
def test_k1_mesh_shapes(bd, ctx, mh, mw):
    """TMA and plain loaders, cluster sizes 1/2/4, partial meshes on both edges."""
    rng = np.random.default_rng(mh * 1000 + mw)
    img = rng.normal(500, 20, size=(1, 300, 340)).astype(np.float32)
    img[0, rng.integers(0, 300, 200), rng.integers(0, 340, 200)] = 60000.0
    check_mesh_stats(bd, ctx, img, bd.BkgParams(mesh_h=mh, mesh_w=mw))


def test_k1_degenerate_inputs(bd, ctx):
    const = np.full((1, 128, 128), 1234.5, dtype=np.float32)
    check_mesh_stats(bd, ctx, const, bd.BkgParams())
    ties = np.random.default_rng(1).integers(0, 4, size=(1, 128, 192)).astype(np.float32)     # heavy ties
    check_mesh_stats(bd, ctx, ties, bd.BkgParams())
    neg = np.random.default_rng(2).normal(0, 1, size=(1, 64, 128)).astype(np.float32)        # both signs
    check_mesh_stats(bd, ctx, neg, bd.BkgParams(clip_sigma=1.0))
    check_mesh_stats(bd, ctx, neg, bd.BkgParams(clip_iters=0))
    check_mesh_stats(bd, ctx, neg, bd.BkgParams(median_factor=2.5, mean_factor=1.5, skew_guard=1))
    outl = np.full((1, 64, 64), 100.0, dtype=np.float32)
    outl[0, 3, 5] = outl[0, 60, 60] = 60000.0
    check_mesh_stats(bd, ctx, outl, bd.BkgParams())
    cauchy = np.random.default_rng(3).standard_cauchy(size=(1, 64, 128)).astype(np.float32)
    check_mesh_stats(bd, ctx, cauchy, bd.BkgParams(clip_sigma=2.0))
    # meshes large enough for the fast path, built so that it gives up half-way (a clipping bound enters the
    # core interval; the median rank leaves the candidate window) and the general path takes over
    big = np.random.default_rng(4).normal(0, 1, size=(1, 256, 384)).astype(np.float32)
    for mesh in (128, 256):
        check_mesh_stats(bd, ctx, big, bd.BkgParams(mesh_h=mesh, mesh_w=mesh, clip_sigma=1.0))
        check_mesh_stats(bd, ctx, big, bd.BkgParams(mesh_h=mesh, mesh_w=mesh, clip_sigma=2.0, clip_iters=20))
    bigc = np.random.default_rng(5).standard_cauchy(size=(1, 256, 384)).astype(np.float32)
    skew = np.random.default_rng(6).exponential(50.0, size=(1, 256, 384)).astype(np.float32) + 100.0
    tie2 = np.random.default_rng(7).integers(0, 4, size=(1, 256, 384)).astype(np.float32)
    for mesh in (128, 256):
        for im in (bigc, skew, tie2):
            check_mesh_stats(bd, ctx, im, bd.BkgParams(mesh_h=mesh, mesh_w=mesh))


# ------------------------------------------------------------------------------------------- K2
@pytest.mark.parametrize("ny,nx,fh,fw", [(8, 8, 3, 3), (37, 36, 5, 5), (2, 3, 3, 3), (1, 5, 5, 1), (96, 96, 3, 3),
                                         (1, 1, 3, 3), (5, 9, 1, 1), (40, 300, 11, 7), (144, 143, 3, 5), (150, 100, 3, 3), (161, 40, 3, 3)])
def test_k2_filter_and_prefilter(bd, ctx, ny, nx, fh, fw):
    rng = np.random.default_rng(ny * 100 + nx)
    B = 3
    raw_b = rng.normal(1000, 30, size=(B, ny, nx)); raw_r = rng.uniform(5, 40, size=(B, ny, nx))
    bm, rm, cb, cr = bd.grid_filter_spline(ctx, dev(raw_b), dev(raw_r), fh, fw)
    torch.cuda.synchronize()
    for f in range(B):
        for raw, m, c in ((raw_b, bm, cb), (raw_r, rm, cr)):
            filt = oracle.grid_median(raw[f], fh, fw)
            assert np.array_equal(m[f].cpu().numpy(), filt.astype(np.float32))
            want = oracle.spline_coeffs(filt)
            assert np.max(np.abs(c[f].cpu().numpy() - want)) <= 1e-11 * np.max(np.abs(want))


# ------------------------------------------------------------------------------------------- K3
@pytest.mark.parametrize("H,W,mh,mw", [(256, 512, 64, 64), (300, 1028, 64, 64), (528, 2048, 256, 256), (97, 132, 50, 36),
                                       (64, 64, 64, 64), (40, 1024, 7, 5)])
@pytest.mark.parametrize("k_d", [1.5, 1.3, 2.7])
def test_k3_maps_and_mask(bd, ctx, H, W, mh, mw, k_d):
    """detect_k = 1.3, 2.7 are not representable in float32: the library compares sub > (float)k * rms in float32
    (bkgdet.h), the oracle in float64; they may differ on the oracle's fragile set only (A15)."""
    rng = np.random.default_rng(H + W)
    ny, nx = oracle.grid_shape(H, W, mh, mw)
    B = 2
    img = rng.normal(1000, 30, size=(B, H, W)).astype(np.float32)
    gb = 1000 + 50 * rng.normal(size=(B, ny, nx)); gr = rng.uniform(20, 40, size=(B, ny, nx))
    cb = np.stack([oracle.spline_coeffs(g) for g in gb]); cr = np.stack([oracle.spline_coeffs(g) for g in gr])
    out = bd.bkg_subtract(ctx, dev(img), mh, mw, dev(cb), dev(cr), k_d)
    torch.cuda.synchronize()
    # the library's own rule, restated on its float32 outputs: one rounded float32 product, float32 compare
    s32, r32 = out["sub"].cpu().numpy(), out["rms"].cpu().numpy()
    assert np.array_equal(out["mask"].cpu().numpy() != 0, (r32 > 0) & (s32 > np.float32(k_d) * r32))
    # the mask-less route of detect_sources applies the same rule: same labels as with bkg_subtract's mask
    cap = 1 << 14
    d1 = bd.detect_sources(ctx, out["sub"], out["rms"], None, k_d, 5, cap)
    d2 = bd.detect_sources(ctx, out["sub"], out["rms"], out["mask"], k_d, 5, cap)
    torch.cuda.synchronize()
    assert torch.equal(d1["labels"], d2["labels"]) and torch.equal(d1["n_sources"], d2["n_sources"])
    for f in range(B):
        bkg64 = oracle.spline_eval(cb[f], H, W, mh, mw); rms64 = oracle.spline_eval(cr[f], H, W, mh, mw)
        sub64, _, mask, frag = oracle.subtract_threshold(img[f], bkg64, rms64, k_d)
        assert_maps_close(out["bkg"][f].cpu().numpy(), bkg64, "bkg")
        assert_maps_close(out["rms"][f].cpu().numpy(), rms64, "rms")
        assert_maps_close(out["sub"][f].cpu().numpy(), sub64, "sub", scale=bkg64)
        assert_mask_parity(out["mask"][f].cpu().numpy(), mask, frag)
        # tighter than the bar: float32 rounding of a float64 evaluation
        assert np.max(np.abs(out["bkg"][f].cpu().numpy() - bkg64) / np.abs(bkg64)) < 1e-7
    o2 = bd.bkg_subtract(ctx, dev(img), mh, mw, dev(cb), dev(cr), k_d, want_bkg=False, want_rms=False, want_mask=False)
    torch.cuda.synchronize()
    assert o2["bkg"] is None and torch.equal(o2["sub"], out["sub"])


# ------------------------------------------------------------------------------------------- K4 / K5
def run_detect(bd, ctx, sub, mask, min_area, cap=None, rms=None, k=1.5):
    B, H, W = sub.shape
    cap = cap if cap is not None else B * ((H + 1) // 2) * ((W + 1) // 2) + 1
    out = bd.detect_sources(ctx, dev(sub), None if rms is None else dev(rms), None if mask is None else dev(mask), k, min_area, cap)
    torch.cuda.synchronize()
    n = out["n_sources"].cpu().numpy()
    cat = bd.catalogue_to_numpy(out["cat"], out["n_sources"], cap)
    return out["labels"].cpu().numpy(), cat, n


def check_detect(bd, ctx, sub, mask, min_area):
    labels, cat, n = run_detect(bd, ctx, sub, mask, min_area)
    worst = {}
    for f in range(sub.shape[0]):
        want_lab = oracle.label(mask[f])
        assert np.array_equal(labels[f], want_lab), f"labels differ in frame {f}: {np.count_nonzero(labels[f] != want_lab)} px"
        want_cat = oracle.reduce_sources(want_lab, sub[f], min_area)
        assert n[f] == len(want_cat)
        worst = assert_catalogue_equal(cat, want_cat, frame=f)
    return worst


@pytest.mark.parametrize("density", [0.02, 0.07, 0.16, 0.32, 0.41, 0.6, 0.95])
@pytest.mark.parametrize("H,W", [(211, 172), (64, 256), (33, 132), (300, 516)])
def test_k45_random_masks(bd, ctx, density, H, W):
    rng = np.random.default_rng(int(density * 100) + H)
    B = 2
    mask = (rng.uniform(size=(B, H, W)) < density).astype(np.uint8)
    sub = rng.uniform(0.5, 50.0, size=(B, H, W)).astype(np.float32)
    check_detect(bd, ctx, sub, mask, 1)
    check_detect(bd, ctx, sub, mask, 5)


def test_k45_structured_masks(bd, ctx):
    H, W = 97, 388
    yy, xx = np.mgrid[:H, :W]
    cases = [np.eye(H, W, dtype=np.uint8), np.fliplr(np.eye(H, W, dtype=np.uint8)),
             ((yy + xx) % 2 == 0).astype(np.uint8), np.ones((H, W), np.uint8), np.zeros((H, W), np.uint8),
             (yy % 2 == 0).astype(np.uint8), (xx % 2 == 0).astype(np.uint8),
             ((yy % 4 == 0) | ((xx % 6 == 0) & (yy % 8 < 5))).astype(np.uint8),           # comb across tile seams
             (((yy // 3 + xx // 5) % 2 == 0) & (yy % 7 != 0)).astype(np.uint8)]
    spiral = np.zeros((H, W), np.uint8)
    for k in range(0, 40, 4):   # nested rectangles joined into one long snake crossing every seam
        spiral[k, k:W - k] = 1; spiral[H - 1 - k, k:W - k] = 1; spiral[k:H - k, k] = 1; spiral[k:H - k, W - 1 - k] = 1
        spiral[k + 1:k + 4, k + 2] = 0 if k % 8 else 1
    cases.append(spiral)
    mask = np.stack(cases)
    sub = np.random.default_rng(0).uniform(1, 2, size=mask.shape).astype(np.float32)
    check_detect(bd, ctx, sub, mask, 1)


def test_k45_exhaustive_4x4(bd, ctx):
    """All 65536 masks of a 4x4 frame, as batches of 4096 frames (also exercises B > 1 bookkeeping)."""
    P = 16
    allm = ((np.arange(2 ** P)[:, None] >> np.arange(P)[None, :]) & 1).astype(np.uint8).reshape(-1, 4, 4)
    sub = np.random.default_rng(4).uniform(1, 9, size=(4096, 4, 4)).astype(np.float32)
    for c in range(0, 65536, 4096):              # all 16 batches: every one of the 65536 masks
        m = allm[c:c + 4096]
        labels, cat, n = run_detect(bd, ctx, sub, m, 2)
        for f in range(0, 4096):
            want = oracle.label(m[f])
            assert np.array_equal(labels[f], want)
        f_check = [0, 1, 777, 4095]
        for f in f_check:
            assert_catalogue_equal(cat, oracle.reduce_sources(oracle.label(m[f]), sub[f], 2), frame=f)
        assert n.sum() == len(cat)


@pytest.mark.parametrize("k_d", [1.0, 1.3, 2.7])
def test_k45_mask_from_sub_rms_and_overflow(bd, ctx, k_d):
    """No mask given: the threshold is taken on the float32 inputs with the library's float32 rule (bkgdet.h; both sides
    of this comparison decide in that precision).  With rms a multiple of 0.1 and sub drawn on a 0.01 grid, ties and
    near-ties of sub against k*rms occur, so a float64 product would give a different mask for k = 1.3, 2.7."""
    rng = np.random.default_rng(12)
    B, H, W = 1, 130, 260
    sub = (np.round(rng.normal(0, 10, size=(B, H, W)), 2)).astype(np.float32)
    rms = (np.round(rng.uniform(5, 15, size=(B, H, W)), 1)).astype(np.float32); rms[0, :5] = 0.0
    labels, cat, n = run_detect(bd, ctx, sub, None, 3, rms=rms, k=k_d)
    mask = ((rms > 0) & (sub > np.float32(k_d) * rms)).astype(np.uint8)
    want_lab = oracle.label(mask[0])
    assert np.array_equal(labels[0], want_lab)
    want = oracle.reduce_sources(want_lab, sub[0], 3)
    assert_catalogue_equal(cat, want, frame=0)
    # capacity smaller than the catalogue: counts stay true, the first `cap` records are valid
    assert len(want) >= 2
    cap = min(7, len(want) - 1)
    _, cat2, n2 = run_detect(bd, ctx, sub, mask, 3, cap=cap)
    assert n2[0] == len(want) and len(cat2) == cap
    assert_catalogue_equal(cat2, want[:cap], frame=0)


# ------------------------------------------------------------------------------------------- whole chain
def run_chain(bd, ctx, img, p, k, min_area, cap):
    d_img = dev(img)
    bm, rm, cb, cr = bd.bkg_estimate(ctx, d_img, p)
    o = bd.bkg_subtract(ctx, d_img, p.mesh_h, p.mesh_w, cb, cr, k)
    det = bd.detect_sources(ctx, o["sub"], o["rms"], o["mask"], k, min_area, cap)
    torch.cuda.synchronize()
    return bm, rm, o, det


def check_chain(bd, ctx, img, p, k, min_area, frames=None):
    B, H, W = img.shape
    cap = 1 << 20
    bm, rm, o, det = run_chain(bd, ctx, img, p, k, min_area, cap)
    cat = bd.catalogue_to_numpy(det["cat"], det["n_sources"], cap)
    n = det["n_sources"].cpu().numpy()
    fz = bd.bkg_subtract_detect(ctx, dev(img), p.mesh_h, p.mesh_w, *bd.bkg_estimate(ctx, dev(img), p)[2:], k, min_area, cap)
    torch.cuda.synchronize()
    for key in ("sub", "bkg", "rms", "mask"):
        assert torch.equal(fz[key], o[key]), f"fused {key} differs from bkg_subtract"
    assert torch.equal(fz["labels"], det["labels"]) and torch.equal(fz["n_sources"], det["n_sources"])
    del fz
    report = {}
    for f in (range(B) if frames is None else frames):
        r = oracle.chain(img[f], to_oracle_params(p), k, min_area)
        assert np.array_equal(bm[f].cpu().numpy(), r["bkg_grid"].astype(np.float32)) or \
            np.max(np.abs(bm[f].cpu().numpy() - r["bkg_grid"]) / np.abs(r["bkg_grid"])) < 1e-6
        assert_maps_close(o["bkg"][f].cpu().numpy(), r["bkg"], "bkg")
        assert_maps_close(o["rms"][f].cpu().numpy(), r["rms"], "rms")
        assert_maps_close(o["sub"][f].cpu().numpy(), r["sub64"], "sub", scale=r["bkg"])
        mask_g = o["mask"][f].cpu().numpy()
        ndiff = assert_mask_parity(mask_g, r["mask"], r["fragile"])
        # labels: bit-exact given the same mask
        lab_g = det["labels"][f].cpu().numpy()
        assert np.array_equal(lab_g, oracle.label(mask_g))
        # catalogue from the GPU's own labels/sub: exact stage parity
        sub_g = o["sub"][f].cpu().numpy()
        stage = oracle.reduce_sources(lab_g, sub_g, min_area)
        assert n[f] == len(stage)
        worst = assert_catalogue_equal(cat, stage, frame=f)
        # catalogue against the oracle's own chain: 1:1 outside components touching fragile pixels
        exempt = fragile_touched_labels(r["labels"], r["fragile"]) if ndiff else ()
        if ndiff:
            exempt = np.union1d(exempt, fragile_touched_labels(lab_g, r["fragile"]))
        worst2 = assert_catalogue_equal(cat, r["cat"], frame=f, exempt_labels=exempt, peak_pos_exact=False)
        report[f] = dict(mask_diff=ndiff, n_sources=int(n[f]), fragile=int(r["fragile"].sum()), stage=worst, chain=worst2,
                         exempt=len(exempt))
    return report


@pytest.mark.parametrize("cid,H,W,B", [(1, 512, 512, 1), (2, 1024, 1024, 1), (3, 1040, 1024, 1), (4, 512, 512, 3), (5, 768, 768, 1)])
def test_chain_configs_reduced(bd, ctx, cid, H, W, B):
    """configs[0] at full size; the others at a size the oracle finishes in seconds (several tiles, ragged tail)."""
    cfg = CONFIGS[cid]
    img = make_frames(cfg, H=H, W=W, B=B)
    rep = check_chain(bd, ctx, img, params_for(bd, cfg), cfg.detect_k, cfg.min_area)
    assert all(v["n_sources"] > 0 for v in rep.values())


@pytest.mark.parametrize("cid,H,W,B,mesh", [(1, 512, 512, 1, 64), (3, 528, 768, 1, 256), (5, 300, 388, 2, 64), (2, 200, 260, 1, 50),
                                            (1, 97, 132, 1, 36), (1, 64, 64, 1, 20)])
def test_fused_subtract_detect_equals_two_passes(bd, ctx, cid, H, W, B, mesh):
    """bkg_subtract_detect (fused tile kernel) against bkg_subtract + detect_sources: maps, mask and labels bit-identical,
    catalogue equal up to the order of the float64 atomics.  mesh 36/50: four columns of a thread straddle grid cells;
    mesh 20: the documented fallback to the two passes; ragged tiles and frame edges in all of them."""
    cfg = CONFIGS[cid]
    img = make_frames(cfg, H=H, W=W, B=B)
    p = params_for(bd, cfg, mesh_h=mesh, mesh_w=mesh)
    d_img = dev(img)
    bm, rm, cb, cr = bd.bkg_estimate(ctx, d_img, p)
    cap = 1 << 16
    o = bd.bkg_subtract(ctx, d_img, p.mesh_h, p.mesh_w, cb, cr, cfg.detect_k)
    det = bd.detect_sources(ctx, o["sub"], o["rms"], o["mask"], cfg.detect_k, cfg.min_area, cap)
    f = bd.bkg_subtract_detect(ctx, d_img, p.mesh_h, p.mesh_w, cb, cr, cfg.detect_k, cfg.min_area, cap)
    torch.cuda.synchronize()
    for k in ("sub", "bkg", "rms", "mask"):
        assert torch.equal(f[k], o[k]), k
    assert torch.equal(f["labels"], det["labels"]) and torch.equal(f["n_sources"], det["n_sources"])
    c1 = bd.catalogue_to_numpy(det["cat"], det["n_sources"], cap); c2 = bd.catalogue_to_numpy(f["cat"], f["n_sources"], cap)
    assert len(c1) == len(c2) and len(c1) > 0
    for k in ("frame", "label", "npix", "xmin", "xmax", "ymin", "ymax", "xpeak", "ypeak", "peak"):
        assert np.array_equal(c1[k], c2[k]), k
    for k in ("flux", "x", "y", "x2", "y2", "xy"):
        assert np.allclose(c1[k], c2[k], rtol=1e-9, atol=1e-9), k
    # without the optional outputs
    f2 = bd.bkg_subtract_detect(ctx, d_img, p.mesh_h, p.mesh_w, cb, cr, cfg.detect_k, cfg.min_area, cap, want_bkg=False,
                                want_rms=False, want_mask=False)
    torch.cuda.synchronize()
    assert f2["bkg"] is None and torch.equal(f2["labels"], det["labels"]) and torch.equal(f2["sub"], o["sub"])


@pytest.mark.parametrize("H,W,B,mesh", [(97, 132, 2, 36), (130, 260, 1, 64), (64, 128, 3, 64), (200, 516, 1, 128)])
def test_no_writes_outside_the_outputs(bd, ctx, H, W, B, mesh):
    """Guard bands around every output buffer of both detection paths stay untouched (ragged tiles, frame edges, TMA
    label-tile stores clipped at the frame edge)."""
    cfg = CONFIGS[1]
    img = make_frames(cfg, H=H, W=W, B=B)
    p = params_for(bd, cfg, mesh_h=mesh, mesh_w=mesh)
    d_img = dev(img)
    bm, rm, cb, cr = bd.bkg_estimate(ctx, d_img, p)
    G, P, cap = 4096, B * H * W, 512
    def guarded(dtype, n, fill):
        flat = torch.full((n + 2 * G,), fill, dtype=dtype, device="cuda")
        return flat, flat[G:G + n]
    for fused in (True, False):
        bufs = {k: guarded(torch.float32, P, -777.0) for k in ("sub", "bkg", "rms")}
        bufs["mask"] = guarded(torch.uint8, P, 0xAB)
        bufs["labels"] = guarded(torch.int32, P, -5)
        bufs["cat"] = guarded(torch.uint8, cap * bd.SOURCE_DTYPE.itemsize, 0xCD)
        bufs["n_sources"] = guarded(torch.int64, B, -9)
        out = {k: (v[1].view(B, H, W) if k in ("sub", "bkg", "rms", "mask", "labels") else v[1]) for k, v in bufs.items()}
        if fused:
            bd.bkg_subtract_detect(ctx, d_img, p.mesh_h, p.mesh_w, cb, cr, cfg.detect_k, cfg.min_area, cap, out=out)
        else:
            bd.bkg_subtract(ctx, d_img, p.mesh_h, p.mesh_w, cb, cr, cfg.detect_k, out=out)
            bd.detect_sources(ctx, out["sub"], out["rms"], out["mask"], cfg.detect_k, cfg.min_area, cap, out=out)
        torch.cuda.synchronize()
        for k, (flat, view) in bufs.items():
            n = view.numel()
            fill = flat[0].item()
            assert bool((flat[:G] == fill).all()) and bool((flat[G + n:] == fill).all()), f"{k}: guard band overwritten (fused={fused})"
        assert int(out["labels"].min()) >= 0 and int(out["n_sources"].min()) >= 0


def test_chain_constant_frame(bd, ctx):
    img = np.full((1, 256, 320), 4321.0, dtype=np.float32)
    p = bd.BkgParams()
    bm, rm, o, det = run_chain(bd, ctx, img, p, 1.5, 5, 16)
    assert torch.all(o["bkg"] == 4321.0) and torch.all(o["rms"].abs() < 1e-9)
    assert int(o["mask"].sum()) == 0 and int(det["n_sources"].sum()) == 0 and int(det["labels"].abs().sum()) == 0


@pytest.mark.parametrize("cid", [2, 3, 5])
def test_chain_full_size(bd, ctx, cid):
    """BASELINE.json full sizes, in the launch configuration bench.py times."""
    cfg = CONFIGS[cid]
    img = make_frames(cfg)
    rep = check_chain(bd, ctx, img, params_for(bd, cfg), cfg.detect_k, cfg.min_area)
    print(cfg.name, rep)


def test_chain_config4_batch(bd, ctx):
    """64 x 2048^2 in one call.  Frames 0, 31 and 63 go through the whole oracle chain (maps, mask, labels, catalogue).
    EVERY one of the 64 frames is checked against the oracle for a4 + a5: the oracle's flood fill of the frame's GPU mask
    must equal the GPU labels bit for bit, and the oracle's reduction of (those labels, the frame's GPU sub map) must equal
    the frame's slice of the catalogue (stage parity: exact npix / bbox / peak, sums at the a5 tolerances) and its
    n_sources; the mesh grids of every frame are compared with the oracle's O1 + O2 as well (PAPER.md:43 pipeline mode)."""
    cfg = CONFIGS[4]
    img = make_frames(cfg)
    p = params_for(bd, cfg)
    rep = check_chain(bd, ctx, img, p, cfg.detect_k, cfg.min_area, frames=[0, 31, 63])
    print(cfg.name, rep)
    cap = 1 << 20
    d_img = dev(img)
    bm, rm, cb, cr = bd.bkg_estimate(ctx, d_img, p)
    fz = bd.bkg_subtract_detect(ctx, d_img, p.mesh_h, p.mesh_w, cb, cr, cfg.detect_k, cfg.min_area, cap)
    torch.cuda.synchronize()
    cat = bd.catalogue_to_numpy(fz["cat"], fz["n_sources"], cap)
    n = fz["n_sources"].cpu().numpy()
    assert n.sum() == len(cat) and np.all(np.diff(cat["frame"]) >= 0)
    op = to_oracle_params(p)
    for f in range(img.shape[0]):
        b = oracle.background(img[f], op) if f % 8 == 0 else None
        st = oracle.mesh_stats(img[f], op)
        want_b = oracle.grid_median(st["bkg"], p.filt_h, p.filt_w); want_r = oracle.grid_median(st["rms"], p.filt_h, p.filt_w)
        assert np.max(np.abs(bm[f].cpu().numpy() - want_b) / np.abs(want_b)) < 1e-6, f"bkg grid of frame {f}"
        assert np.max(np.abs(rm[f].cpu().numpy() - want_r) / np.abs(want_r)) < 1e-6, f"rms grid of frame {f}"
        if b is not None:
            assert_maps_close(fz["bkg"][f].cpu().numpy(), b["bkg"], f"bkg map of frame {f}")
        mask_g = fz["mask"][f].cpu().numpy(); lab_g = fz["labels"][f].cpu().numpy(); sub_g = fz["sub"][f].cpu().numpy()
        assert np.array_equal(lab_g, oracle.label(mask_g)), f"labels of frame {f}"
        stage = oracle.reduce_sources(lab_g, sub_g, cfg.min_area)
        assert n[f] == len(stage), f"n_sources of frame {f}"
        assert_catalogue_equal(cat, stage, frame=f)


@pytest.mark.parametrize("cid,H,W,B", [(1, 512, 512, 1), (3, 1100, 768, 1), (4, 256, 256, 11), (5, 200, 260, 2)])
def test_run_host_matches_device_path(bd, ctx, cid, H, W, B):
    """bd_run_host copies the frame in chunks (strips of mesh rows, or frames of a batch) and runs K1 per chunk: the same
    catalogue as the device calls; a partial last mesh row, more frames than chunks, fewer mesh rows than chunks; called
    twice (cached buffers)."""
    cfg = CONFIGS[cid]
    img = make_frames(cfg, H=H, W=W, B=B)
    p = params_for(bd, cfg)
    bm, rm, o, det = run_chain(bd, ctx, img, p, cfg.detect_k, cfg.min_area, 1 << 15)
    cat_d = bd.catalogue_to_numpy(det["cat"], det["n_sources"], 1 << 15)
    for _ in range(2):
        cat_h, n_h = bd.run_host(ctx, img, p, cfg.detect_k, cfg.min_area, 1 << 15)
        assert np.array_equal(n_h, det["n_sources"].cpu().numpy())
        for k in ("frame", "label", "npix", "xpeak", "ypeak"):
            assert np.array_equal(cat_h[k], cat_d[k])
        assert np.allclose(cat_h["flux"], cat_d["flux"], rtol=1e-12)


# ------------------------------------------------------------------------------------------- NEXT-2: photometry (K6)
from oracle import photometry as oph  # noqa: E402


@pytest.mark.parametrize("cid,H,W,B,kw", [(1, 512, 512, 1, {}), (3, 528, 768, 1, dict(r_aper=3.0, subpix=7)),
                                           (5, 300, 388, 2, dict(r_aper=8.5, kron_min_radius=0.5)),
                                           (2, 260, 260, 1, dict(r_aper=12.0, kron_factor=2.0, kron_search=4.0, subpix=1))])
def test_k6_photometry_against_oracle(bd, ctx, cid, H, W, B, kw):
    """Stage parity: the oracle measures the GPU's own sub / rms maps and catalogue.  Pixel membership (npix_auto, flags)
    exact; sums to 1e-9 relative (float64 on both sides, only the summation order differs)."""
    cfg = CONFIGS[cid]
    img = make_frames(cfg, H=H, W=W, B=B)
    p = params_for(bd, cfg)
    cap = 1 << 15
    bm, rm, o, det = run_chain(bd, ctx, img, p, cfg.detect_k, cfg.min_area, cap)
    pp = bd.PhotParams(**kw)
    ph = bd.photometry(ctx, o["sub"], o["rms"], det["cat"], det["n_sources"], cap, pp)
    ph2 = bd.photometry(ctx, o["sub"], o["rms"], det["cat"], det["n_sources"], cap, pp)
    torch.cuda.synchronize()
    assert torch.equal(ph, ph2), "photometry is not bit-reproducible"
    cat = bd.catalogue_to_numpy(det["cat"], det["n_sources"], cap)
    got = bd.phot_to_numpy(ph, det["n_sources"], cap)
    assert len(got) == len(cat) > 0
    op = oph.PhotParams(r_aper=pp.r_aper, kron_factor=pp.kron_factor, kron_min_radius=pp.kron_min_radius,
                        kron_search=pp.kron_search, subpix=pp.subpix)
    for f in range(B):
        sel = cat["frame"] == f
        want = oph.photometry(o["sub"][f].cpu().numpy(), o["rms"][f].cpu().numpy(), cat[sel], op)
        g = got[sel]
        assert np.array_equal(g["npix_auto"], want["npix_auto"]) and np.array_equal(g["flags"], want["flags"])
        assert np.allclose(g["kron_radius"], want["kron_radius"], rtol=1e-12, atol=0)
        for k in ("flux_aper", "fluxerr_aper", "area_aper", "flux_auto", "fluxerr_auto"):
            assert np.allclose(g[k], want[k], rtol=1e-9, atol=1e-6), f"{k}: worst {np.max(np.abs(g[k] - want[k]))}"
        assert (want["flags"] != 0).any() or cid == 1          # the reduced frames have sources at their edges


def _k6_compare(bd, got, cat, sub, rms, idx, op):
    want = oph.photometry(sub, rms, cat[idx], op)
    g = got[idx]
    assert np.array_equal(g["npix_auto"], want["npix_auto"]) and np.array_equal(g["flags"], want["flags"])
    assert np.allclose(g["kron_radius"], want["kron_radius"], rtol=1e-12, atol=0)
    for k in ("flux_aper", "fluxerr_aper", "area_aper", "flux_auto", "fluxerr_auto"):
        assert np.allclose(g[k], want[k], rtol=1e-9, atol=1e-6), f"{k}: worst {np.max(np.abs(g[k] - want[k]))}"
    return want


def test_k6_full_size_config3_sampled(bd, ctx):
    """K6 at BASELINE.json's full size (9216x9232, ~174 k records), in the launch configuration a user runs: every record is
    measured on the GPU; the oracle (one object at a time, pure numpy) re-measures a seeded sample of 1500 records plus
    the 64 records with the largest second moments (the ones that go through the large-object path) -- same membership,
    sums to 1e-9.  PAPER.md:159."""
    cfg = CONFIGS[3]
    img = make_frames(cfg)
    p = params_for(bd, cfg)
    cap = 1 << 19
    d_img = dev(img)
    bm, rm, cb, cr = bd.bkg_estimate(ctx, d_img, p)
    fz = bd.bkg_subtract_detect(ctx, d_img, p.mesh_h, p.mesh_w, cb, cr, cfg.detect_k, cfg.min_area, cap, want_bkg=False, want_mask=False)
    ph = bd.photometry(ctx, fz["sub"], fz["rms"], fz["cat"], fz["n_sources"], cap)
    torch.cuda.synchronize()
    cat = bd.catalogue_to_numpy(fz["cat"], fz["n_sources"], cap)
    got = bd.phot_to_numpy(ph, fz["n_sources"], cap)
    assert len(got) == len(cat) > 100000
    rng = np.random.default_rng(33)
    idx = np.union1d(rng.choice(len(cat), 1500, replace=False), np.argsort(cat["x2"] + cat["y2"])[-64:])
    want = _k6_compare(bd, got, cat, fz["sub"][0].cpu().numpy(), fz["rms"][0].cpu().numpy(), idx, oph.PhotParams())
    assert want["npix_auto"].max() > 300
    assert np.all(np.isfinite(got["flux_auto"])) and np.all(got["flags"] < 4)


def test_k6_config5_crop_with_saturated_stars(bd, ctx):
    """A 1024x1024 frame of the config-5 recipe (crowded, 6 saturated stars whose blended regions give search ellipses of
    many thousand pixels: the large-object path at real scale), every record against the oracle."""
    cfg = CONFIGS[5]
    img = make_frames(cfg, H=1024, W=1024)
    assert (img >= 65535.0).sum() > 20
    p = params_for(bd, cfg)
    cap = 1 << 16
    bm, rm, o, det = run_chain(bd, ctx, img, p, cfg.detect_k, cfg.min_area, cap)
    ph = bd.photometry(ctx, o["sub"], o["rms"], det["cat"], det["n_sources"], cap)
    torch.cuda.synchronize()
    cat = bd.catalogue_to_numpy(det["cat"], det["n_sources"], cap)
    got = bd.phot_to_numpy(ph, det["n_sources"], cap)
    want = _k6_compare(bd, got, cat, o["sub"][0].cpu().numpy(), o["rms"][0].cpu().numpy(), np.arange(len(cat)), oph.PhotParams())
    assert want["npix_auto"].max() > 4096, want["npix_auto"].max()


def test_k6_degenerate_records(bd, ctx):
    """A28: records with non-finite or ellipse-less moments are not measured (zeros, flags = 4); their neighbours are."""
    rng = np.random.default_rng(2)
    sub = rng.normal(5, 1, (1, 64, 96)).astype(np.float32); rms = np.ones_like(sub)
    cat = np.zeros(5, dtype=bd.SOURCE_DTYPE)
    cat["x"], cat["y"], cat["x2"], cat["y2"], cat["xy"] = 40.0, 30.0, 2.0, 2.0, 0.0
    cat["x"][1] = np.nan; cat["y2"][2] = np.inf; cat["x2"][3] = -3.0; cat["y2"][3] = -3.0
    n = torch.tensor([5], dtype=torch.int64, device="cuda")
    ph = bd.photometry(ctx, dev(sub), dev(rms), torch.from_numpy(cat.view(np.uint8)).cuda(), n, 8)
    torch.cuda.synchronize()
    got = bd.phot_to_numpy(ph, n, 8)
    want = oph.photometry(sub[0], rms[0], cat, oph.PhotParams())
    assert list(got["flags"]) == [0, 4, 4, 4, 0] == list(want["flags"])
    for k in got.dtype.names:
        assert np.allclose(got[k], want[k], rtol=1e-9, atol=1e-9), k
    with pytest.raises(bd.BkgdetError):
        bd.photometry(ctx, dev(sub), dev(rms), torch.from_numpy(cat.view(np.uint8)).cuda(), n, 8, bd.PhotParams(r_aper=1.0e5))


def test_k6_large_objects_take_the_block_path(bd, ctx):
    """Objects whose search ellipse covers more than 4096 px are queued and measured by one thread block each: same
    membership and sums as the oracle, mixed with small objects, at the frame edge, in the second frame of a batch."""
    rng = np.random.default_rng(11)
    B, H, W = 2, 300, 420
    sub = rng.normal(0, 1, (B, H, W)).astype(np.float32); rms = rng.uniform(0.8, 1.3, (B, H, W)).astype(np.float32)
    yy, xx = np.mgrid[:H, :W].astype(np.float64)
    objs = [(0, 150.3, 140.7, 15.0, 9.0, 0.5), (0, 30.2, 25.5, 2.0, 1.5, 0.1), (1, 400.6, 10.2, 20.0, 20.0, 0.0),
            (1, 200.1, 150.9, 40.0, 3.0, -0.7), (1, 100.0, 250.0, 1.2, 1.2, 0.0), (0, 300.5, 200.5, 11.0, 10.5, 1.2)]
    cat = np.zeros(len(objs), dtype=bd.SOURCE_DTYPE)
    objs.sort(key=lambda o: o[0])
    for i, (f, xc, yc, sx, sy, th) in enumerate(objs):
        c, s_ = np.cos(th), np.sin(th)
        u = (xx - xc) * c + (yy - yc) * s_; v = -(xx - xc) * s_ + (yy - yc) * c
        sub[f] += (5e4 / (2 * np.pi * sx * sy) * np.exp(-0.5 * (u * u / sx**2 + v * v / sy**2))).astype(np.float32)
        cat[i]["frame"], cat[i]["x"], cat[i]["y"] = f, xc, yc
        cat[i]["x2"] = sx**2 * c * c + sy**2 * s_ * s_; cat[i]["y2"] = sx**2 * s_ * s_ + sy**2 * c * c
        cat[i]["xy"] = (sx**2 - sy**2) * s_ * c
    n = torch.tensor([sum(o[0] == 0 for o in objs), sum(o[0] == 1 for o in objs)], dtype=torch.int64, device="cuda")
    d_cat = torch.from_numpy(cat.view(np.uint8)).cuda()
    ph = bd.photometry(ctx, dev(sub), dev(rms), d_cat, n, 16)
    ph2 = bd.photometry(ctx, dev(sub), dev(rms), d_cat, n, 16)
    torch.cuda.synchronize()
    assert torch.equal(ph, ph2)
    got = bd.phot_to_numpy(ph, n, 16)
    for f in range(B):
        sel = cat["frame"] == f
        want = oph.photometry(sub[f], rms[f], cat[sel], oph.PhotParams())
        g = got[sel]
        assert np.array_equal(g["npix_auto"], want["npix_auto"]) and np.array_equal(g["flags"], want["flags"])
        assert want["npix_auto"].max() > 4096
        for k in ("flux_aper", "fluxerr_aper", "area_aper", "kron_radius", "flux_auto", "fluxerr_auto"):
            assert np.allclose(g[k], want[k], rtol=1e-9, atol=1e-6), k


def test_k6_huge_objects_take_the_grid_path(bd, ctx):
    """Objects whose search box exceeds 2^18 pixels are cut into chunks that all CTAs share (k6h_*): same membership and
    sums as the oracle; elongated and rotated, cut by the frame edge, in the second frame of a batch, next to small and
    block-path objects; bit-reproducible run to run."""
    rng = np.random.default_rng(12)
    B, H, W = 2, 1100, 1500
    sub = rng.normal(0, 1, (B, H, W)).astype(np.float32); rms = rng.uniform(0.8, 1.3, (B, H, W)).astype(np.float32)
    yy, xx = np.mgrid[:H, :W].astype(np.float64)
    objs = [(0, 700.3, 540.7, 60.0, 42.0, 0.4), (0, 30.2, 25.5, 2.0, 1.5, 0.1), (0, 1300.5, 200.5, 11.0, 10.5, 1.2),
            (1, 1450.6, 60.2, 70.0, 55.0, 0.0), (1, 600.1, 550.9, 150.0, 16.0, -0.7), (1, 100.0, 250.0, 1.2, 1.2, 0.0)]
    cat = np.zeros(len(objs), dtype=bd.SOURCE_DTYPE)
    for i, (f, xc, yc, sx, sy, th) in enumerate(objs):
        c, s_ = np.cos(th), np.sin(th)
        u = (xx - xc) * c + (yy - yc) * s_; v = -(xx - xc) * s_ + (yy - yc) * c
        sub[f] += (5e5 / (2 * np.pi * sx * sy) * np.exp(-0.5 * (u * u / sx**2 + v * v / sy**2))).astype(np.float32)
        cat[i]["frame"], cat[i]["x"], cat[i]["y"] = f, xc, yc
        cat[i]["x2"] = sx**2 * c * c + sy**2 * s_ * s_; cat[i]["y2"] = sx**2 * s_ * s_ + sy**2 * c * c
        cat[i]["xy"] = (sx**2 - sy**2) * s_ * c
    n = torch.tensor([3, 3], dtype=torch.int64, device="cuda")
    d_cat = torch.from_numpy(cat.view(np.uint8)).cuda()
    ph = bd.photometry(ctx, dev(sub), dev(rms), d_cat, n, 16)
    ph2 = bd.photometry(ctx, dev(sub), dev(rms), d_cat, n, 16)
    torch.cuda.synchronize()
    assert torch.equal(ph, ph2)
    got = bd.phot_to_numpy(ph, n, 16)
    for f in range(B):
        sel = cat["frame"] == f
        want = oph.photometry(sub[f], rms[f], cat[sel], oph.PhotParams())
        g = got[sel]
        assert np.array_equal(g["npix_auto"], want["npix_auto"]) and np.array_equal(g["flags"], want["flags"])
        assert want["npix_auto"].max() > (1 << 16)
        for k in ("flux_aper", "fluxerr_aper", "area_aper", "kron_radius", "flux_auto", "fluxerr_auto"):
            assert np.allclose(g[k], want[k], rtol=1e-9, atol=1e-6), k


def test_k6_full_size_config5_sampled(bd, ctx):
    """Config 5 at full size (6144 x 6144, crowded, 200 saturated stars whose Kron ellipses cover megapixels: the grid-wide
    path at real scale): the 10 records with the largest second moments and 400 seeded random ones against the oracle."""
    cfg = CONFIGS[5]
    img = make_frames(cfg)
    p = params_for(bd, cfg)
    cap = 1 << 20
    d_img = dev(img)
    bm, rm, cb, cr = bd.bkg_estimate(ctx, d_img, p)
    fz = bd.bkg_subtract_detect(ctx, d_img, p.mesh_h, p.mesh_w, cb, cr, cfg.detect_k, cfg.min_area, cap, want_bkg=False, want_mask=False)
    ph = bd.photometry(ctx, fz["sub"], fz["rms"], fz["cat"], fz["n_sources"], cap)
    torch.cuda.synchronize()
    cat = bd.catalogue_to_numpy(fz["cat"], fz["n_sources"], cap)
    got = bd.phot_to_numpy(ph, fz["n_sources"], cap)
    rng = np.random.default_rng(35)
    idx = np.union1d(rng.choice(len(cat), 400, replace=False), np.argsort(cat["x2"] + cat["y2"])[-10:])
    # ... and the records with the largest Kron ellipses (A25 has no upper limit: a faint object whose flux sum inside the
    # search ellipse is nearly zero gets an ellipse that can cover the frame)
    idx = np.union1d(idx, np.argsort(got["npix_auto"])[-6:])
    want = _k6_compare(bd, got, cat, fz["sub"][0].cpu().numpy(), fz["rms"][0].cpu().numpy(), idx, oph.PhotParams())
    assert want["npix_auto"].max() > (1 << 18)


def test_k6_isolated_gaussian_and_errors(bd, ctx):
    """An analytic source through the GPU path alone: encircled energy and the Kron radius of a Gaussian."""
    H = W = 128
    yy, xx = np.mgrid[:H, :W].astype(np.float64)
    F, sig, xc, yc = 2.0e4, 2.0, 63.3, 64.6
    sub = (F / (2 * np.pi * sig**2) * np.exp(-0.5 * ((xx - xc) ** 2 + (yy - yc) ** 2) / sig**2)).astype(np.float32)[None]
    rms = np.ones_like(sub)
    cat = np.zeros(1, dtype=bd.SOURCE_DTYPE)
    cat["x"], cat["y"], cat["x2"], cat["y2"], cat["xy"] = xc, yc, sig**2, sig**2, 0.0
    d_cat = torch.from_numpy(cat.view(np.uint8)).cuda(); n = torch.tensor([1], dtype=torch.int64, device="cuda")
    ph = bd.photometry(ctx, dev(sub), dev(rms), d_cat, n, 4, bd.PhotParams(r_aper=5.0, kron_min_radius=0.1))
    torch.cuda.synchronize()
    g = bd.phot_to_numpy(ph, n, 4)[0]
    assert g["flux_aper"] == pytest.approx(F * (1 - np.exp(-25 / (2 * sig**2))), rel=1.2e-2)
    assert g["kron_radius"] == pytest.approx(2.5 * np.sqrt(np.pi / 2), rel=2e-2)
    assert g["flux_auto"] == pytest.approx(F * (1 - np.exp(-0.5 * g["kron_radius"] ** 2)), rel=5e-3) and g["flags"] == 0
    with pytest.raises(bd.BkgdetError):
        bd.photometry(ctx, dev(sub), dev(rms), d_cat, n, 4, bd.PhotParams(r_aper=-1.0))
    with pytest.raises(bd.BkgdetError):
        bd.photometry(ctx, dev(sub), dev(rms), d_cat, n, 4, bd.PhotParams(subpix=0))


# ------------------------------------------------------------------------------------------- NEXT-3: background variants
from oracle import bkg_variants as obv  # noqa: E402


def _bad_mask(rng, shape, frac, blobs=3):
    bad = (rng.uniform(size=shape) < frac).astype(np.uint8) * 255         # any non-zero value masks
    for _ in range(blobs):
        y, x = int(rng.integers(0, shape[-2] - 40)), int(rng.integers(0, shape[-1] - 40))
        bad[..., y:y + int(rng.integers(8, 80)), x:x + int(rng.integers(8, 80))] = 1
    return bad


def _cmp_masked_stats(out, st, f):
    inv = np.isnan(st["bkg"])
    assert np.array_equal(out["n_valid"][f].cpu().numpy(), st["n_valid"]) and np.array_equal(out["n_kept"][f].cpu().numpy(), st["n_kept"])
    for k in ("bkg", "rms", "median", "mean"):
        g = out[k][f].cpu().numpy()
        assert np.array_equal(np.isnan(g), inv), f"{k}: invalid meshes differ"
    assert np.array_equal(out["median"][f].cpu().numpy()[~inv], st["median"][~inv])
    for k in ("mean", "rms", "bkg"):
        g, w = out[k][f].cpu().numpy()[~inv], st[k][~inv]
        tol = 1e-9 * np.maximum(np.abs(w), np.abs(st["median"][~inv])) + 1e-300
        assert np.all(np.abs(g - w) <= tol), k
    return int(inv.sum())


@pytest.mark.parametrize("cid,H,W,mesh,frac", [(1, 512, 512, 64, 0.05), (3, 528, 768, 256, 0.2), (5, 384, 512, 64, 0.6), (2, 300, 340, 50, 0.1),
                                                (4, 256, 320, 32, 0.3), (2, 384, 384, 128, 0.02)])
def test_k1_masked_mesh_stats(bd, ctx, cid, H, W, mesh, frac):
    """NEXT-3, B1/B2/B6: sigma-clipped statistics under a bad-pixel mask against the oracle: n_valid, n_kept, median and the
    set of invalid meshes exact, sums 1e-9.  Slab, stream and cluster configurations of K1."""
    cfg = CONFIGS[cid]
    rng = np.random.default_rng(cid * 7 + mesh)
    B = 2 if cid == 4 else 1
    img = make_frames(cfg, H=H, W=W, B=B)
    bad = _bad_mask(rng, img.shape, frac)
    p = params_for(bd, cfg, mesh_h=mesh, mesh_w=mesh)
    n_inv = 0
    for kw in (dict(), dict(min_valid_px=int(0.5 * mesh * mesh)), dict(min_valid_px=1, max_masked_frac=0.3), dict(max_reject_frac=0.02)):
        out = bd.mesh_stats_masked(ctx, dev(img), dev(bad), p, bd.BkgXParams(**kw))
        torch.cuda.synchronize()
        for f in range(B):
            n_inv += _cmp_masked_stats(out, oracle.mesh_stats_masked(img[f], bad[f], to_oracle_params(p), oracle.BkgXParams(**kw)), f)
    assert n_inv > 0 or frac < 0.05
    # no mask, rules only: the fast paths stay on
    out = bd.mesh_stats_masked(ctx, dev(img), None, p, bd.BkgXParams(max_reject_frac=0.01))
    torch.cuda.synchronize()
    for f in range(B):
        _cmp_masked_stats(out, oracle.mesh_stats_masked(img[f], None, to_oracle_params(p), oracle.BkgXParams(max_reject_frac=0.01)), f)


@pytest.mark.parametrize("cid,H,W,mesh", [(1, 512, 512, 64), (3, 1040, 1024, 256), (5, 512, 512, 32)])
def test_bkg_estimate_masked_and_fill(bd, ctx, cid, H, W, mesh):
    """NEXT-3, B3: whole meshes masked out -> filled from their valid neighbours, then the ordinary filter and spline."""
    cfg = CONFIGS[cid]
    rng = np.random.default_rng(cid)
    img = make_frames(cfg, H=H, W=W, B=1)
    bad = _bad_mask(rng, img.shape, 0.02, blobs=0)
    bad[0, mesh:3 * mesh, mesh:2 * mesh] = 1            # two whole meshes, one above the other
    bad[0, :mesh, -mesh:] = 1                           # a corner mesh
    p = params_for(bd, cfg, mesh_h=mesh, mesh_w=mesh)
    px = bd.BkgXParams()
    bm, rm, cb, cr, valid = bd.bkg_estimate_masked(ctx, dev(img), dev(bad), p, px)
    torch.cuda.synchronize()
    b = obv.background_masked(img[0], bad[0], to_oracle_params(p), oracle.BkgXParams())
    assert np.array_equal(valid[0].cpu().numpy(), b["valid"]) and (b["valid"] == 0).sum() >= 3
    assert np.max(np.abs(bm[0].cpu().numpy() - b["bkg_grid"]) / np.abs(b["bkg_grid"])) < 1e-6
    assert np.max(np.abs(rm[0].cpu().numpy() - b["rms_grid"]) / np.abs(b["rms_grid"])) < 1e-6
    assert np.max(np.abs(cb[0].cpu().numpy() - b["bkg_coef"])) <= 1e-9 * np.max(np.abs(b["bkg_coef"]))
    assert np.max(np.abs(cr[0].cpu().numpy() - b["rms_coef"])) <= 1e-9 * np.max(np.abs(b["rms_coef"]))
    # everything masked: no valid cell, the grids are 0
    allbad = np.ones_like(bad)
    bm, rm, cb, cr, valid = bd.bkg_estimate_masked(ctx, dev(img), dev(allbad), p, px)
    torch.cuda.synchronize()
    assert int(valid.sum()) == 0 and float(bm.abs().max()) == 0.0 and float(cb.abs().max()) == 0.0


def _time_ms(fn, reps=3):
    fn(); torch.cuda.synchronize()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record()
    for _ in range(reps):
        fn()
    e1.record(); torch.cuda.synchronize()
    return e0.elapsed_time(e1) / reps


@pytest.mark.parametrize("keep", ["5%", "one corner cell", "all but a right strip", "none"])
def test_k2f_mostly_invalid_grid_of_config3_size(bd, ctx, keep):
    """B3 on a 144 x 145 mesh grid (the grid of config 3; 8 x 8 meshes keep the frame small) of which almost every cell is
    invalid: the fill scans rings, not whole windows, and a frame without a valid cell is written as 0 at once, so the
    stage stays in milliseconds where rescanning windows took seconds (about cells x grid loads).  Parity with O8's
    fill on every cell, plus a time bound for the whole masked estimate."""
    mesh, ny, nx = 8, 144, 145
    H, W = ny * mesh, nx * mesh
    rng = np.random.default_rng(31)
    img = rng.normal(500, 10, size=(1, H, W)).astype(np.float32)
    img[0] += np.linspace(0, 80, W, dtype=np.float32)[None, :]
    good = np.zeros((ny, nx), bool)
    if keep == "5%":
        good = rng.uniform(size=(ny, nx)) < 0.05
    elif keep == "one corner cell":
        good[ny - 1, 0] = True
    elif keep == "all but a right strip":      # rings that hold many valid cells
        good[:, : nx - 12] = True
    bad = np.repeat(np.repeat((~good).astype(np.uint8), mesh, axis=0), mesh, axis=1)[None]
    p = bd.BkgParams(mesh_h=mesh, mesh_w=mesh)
    px = bd.BkgXParams(min_valid_px=32)
    d_img, d_bad = dev(img), dev(bad)
    bm, rm, cb, cr, valid = bd.bkg_estimate_masked(ctx, d_img, d_bad, p, px)
    torch.cuda.synchronize()
    assert np.array_equal(valid[0].cpu().numpy() != 0, good)
    if keep == "none":
        assert float(bm.abs().max()) == 0.0 and float(rm.abs().max()) == 0.0 and float(cb.abs().max()) == 0.0
    else:
        st = oracle.mesh_stats_masked(img[0], bad[0], to_oracle_params(p), oracle.BkgXParams(min_valid_px=32))
        assert np.array_equal(~np.isnan(st["bkg"]), good)
        for raw, got in ((st["bkg"], bm), (st["rms"], rm)):
            if keep == "one corner cell":   # every window that holds a valid cell holds exactly this one: B3 gives its value
                filled = np.full((ny, nx), raw[ny - 1, 0])   # (O8's loop would sort ~2e6 windows here)
            else:
                filled = obv.fill_invalid(raw)
            want = oracle.grid_median(filled, p.filt_h, p.filt_w)
            assert np.max(np.abs(got[0].cpu().numpy() - want) / np.abs(want)) < 1e-6
    ms = _time_ms(lambda: bd.bkg_estimate_masked(ctx, d_img, d_bad, p, px))
    assert ms < 50.0, f"masked estimate with a {keep} valid grid took {ms:.1f} ms"


def test_k7_frame_taller_than_the_grid_limit(bd, ctx):
    """bkg_iterate on a frame of more than 65 535 rows: the dilation kernel folds the rows into its y blocks."""
    H, W = 65600, 8
    rng = np.random.default_rng(9)
    img = rng.normal(100, 1, size=(1, H, W)).astype(np.float32)
    img[0, 65590:65593, 2:5] += 50.0                       # a detection in the rows beyond the limit
    bad0 = (rng.uniform(size=img.shape) < 0.05).astype(np.uint8) * 3
    p = bd.BkgParams(mesh_h=64, mesh_w=8)
    px = bd.BkgXParams(min_valid_px=100, grow=1)
    out = bd.bkg_iterate(ctx, dev(img), dev(bad0), p, px, 1.5, 0)
    torch.cuda.synchronize()
    assert np.array_equal(out[5].cpu().numpy(), (bad0 != 0).astype(np.uint8))
    # one iteration: the exclusion mask is the dilated mask of the first estimate, OR bad0 (stage check, as in
    # test_bkg_iterate_stage_parity (i))
    first = bd.bkg_estimate_masked(ctx, dev(img), dev((bad0 != 0).astype(np.uint8)), p, px)
    m0 = bd.bkg_subtract(ctx, dev(img), p.mesh_h, p.mesh_w, first[2], first[3], 1.5)["mask"][0].cpu().numpy()
    out = bd.bkg_iterate(ctx, dev(img), dev(bad0), p, px, 1.5, 1)
    torch.cuda.synchronize()
    got = out[5][0].cpu().numpy()
    assert np.array_equal(got, obv.dilate(m0, 1) | (bad0[0] != 0))
    assert got[65589:65594, 1:6].all()


def test_k7_dilate_or_exhaustive_window(bd, ctx):
    """B5 through bkg_iterate's exclusion mask with n_iter = 0 / the dilation kernel against scipy-pinned oracle dilation:
    every grow, frame edges, bad0 with arbitrary non-zero bytes."""
    rng = np.random.default_rng(8)
    img = rng.normal(100, 1, size=(2, 64, 96)).astype(np.float32)
    bad0 = (rng.uniform(size=img.shape) < 0.05).astype(np.uint8) * 7
    p = bd.BkgParams(mesh_h=32, mesh_w=32)
    out = bd.bkg_iterate(ctx, dev(img), dev(bad0), p, bd.BkgXParams(min_valid_px=1), 1.5, 0)
    torch.cuda.synchronize()
    assert np.array_equal(out[5].cpu().numpy(), (bad0 != 0).astype(np.uint8))
    out = bd.bkg_iterate(ctx, dev(img), None, p, bd.BkgXParams(), 1.5, 0)
    assert int(out[5].sum()) == 0


@pytest.mark.parametrize("cid,H,W,mesh,grow,n_iter", [(1, 512, 512, 64, 1, 1), (3, 528, 768, 256, 2, 2), (5, 384, 512, 64, 0, 1), (2, 300, 340, 50, 3, 1)])
def test_bkg_iterate_stage_parity(bd, ctx, cid, H, W, mesh, grow, n_iter):
    """NEXT-3, B4.  The threshold inside the iteration is the library's float32 rule, the oracle's is float64:
    masks may differ on fragile pixels, so the comparison is stage-wise and exact, EVERY round k = 1..n_iter:
    (i) the library's detection mask of round k (its estimate under its exclusion mask of round k - 1, thresholded by
    bkg_subtract) equals the oracle's threshold of the oracle's masked estimate under that SAME exclusion mask, except on
    the oracle's fragile set of that round; (ii) the exclusion mask of round k is oracle.dilate(that library mask) | bad0, bit
    for bit, and the last one is what bkg_iterate returns; (iii) the final grids equal the oracle's masked estimate under the
    library's final exclusion mask.  (iv) Against the oracle's own free-running iteration: with one round every differing
    pixel lies within `grow` of a fragile pixel; from the second round on a pixel that differed in round 1 moves a mesh's
    statistics by ~1e-4 sigma, more than the fragile band, so there the difference is bounded by count."""
    cfg = CONFIGS[cid]
    rng = np.random.default_rng(cid + 40)
    img = make_frames(cfg, H=H, W=W, B=1)
    bad0 = _bad_mask(rng, img.shape, 0.01, blobs=1)
    p = params_for(bd, cfg, mesh_h=mesh, mesh_w=mesh)
    px, opx = bd.BkgXParams(grow=grow), oracle.BkgXParams(grow=grow)
    d_img = dev(img)
    bm, rm, cb, cr, valid, bad_out = bd.bkg_iterate(ctx, d_img, dev(bad0), p, px, cfg.detect_k, n_iter)
    torch.cuda.synchronize()
    bad_g = bad_out[0].cpu().numpy()
    assert set(np.unique(bad_g)) <= {0, 1}
    bad_k = (bad0[0] != 0).astype(np.uint8)
    frag1 = None
    for k in range(1, n_iter + 1):
        _, _, cbk, crk, _ = bd.bkg_estimate_masked(ctx, d_img, dev(bad_k[None]), p, px)
        m_k = bd.bkg_subtract(ctx, d_img, p.mesh_h, p.mesh_w, cbk, crk, cfg.detect_k)["mask"][0].cpu().numpy()
        ok = obv.background_masked(img[0], bad_k, to_oracle_params(p), opx)
        _, _, det_k, frag_k = oracle.subtract_threshold(img[0], ok["bkg"], ok["rms"], cfg.detect_k)
        assert_mask_parity(m_k, det_k, frag_k)                                   # (i)
        frag1 = frag_k if k == 1 else frag1
        bad_k = (obv.dilate(m_k, grow) | (bad0[0] != 0)).astype(np.uint8)        # (ii)
    assert np.array_equal(bad_g, bad_k)
    b = obv.background_masked(img[0], bad_g, to_oracle_params(p), opx)           # (iii)
    assert np.array_equal(valid[0].cpu().numpy(), b["valid"])
    assert np.max(np.abs(bm[0].cpu().numpy() - b["bkg_grid"]) / np.abs(b["bkg_grid"])) < 1e-6
    assert np.max(np.abs(cb[0].cpu().numpy() - b["bkg_coef"])) <= 1e-9 * np.max(np.abs(b["bkg_coef"]))
    assert np.max(np.abs(cr[0].cpu().numpy() - b["rms_coef"])) <= 1e-9 * np.max(np.abs(b["rms_coef"]))
    ob, obad = obv.iterate(img[0], bad0[0], to_oracle_params(p), opx, cfg.detect_k, n_iter)   # (iv)
    diff = obad != bad_g
    if n_iter == 1:
        assert not (diff & ~(obv.dilate(frag1.astype(np.uint8), grow) != 0)).any()
    assert diff.sum() <= 1e-4 * bad_g.size
    assert np.max(np.abs(bm[0].cpu().numpy() - ob["bkg_grid"]) / np.abs(ob["bkg_grid"])) < 1e-4


def test_bkg_iterate_full_size_config3(bd, ctx):
    """NEXT-3 at BASELINE.json's full size (9216 x 9232, mesh 256, filter 5 x 5) with a bad-pixel mask (1 % random pixels and
    blobs): one re-estimation.  (i) the exclusion mask equals oracle.dilate(the library's own first mask) | bad0, bit for bit;
    (ii) validity flags, filtered grids and spline coefficients equal the oracle's masked estimate under that mask."""
    cfg = CONFIGS[3]
    rng = np.random.default_rng(43)
    img = make_frames(cfg)
    bad0 = _bad_mask(rng, img.shape, 0.01, blobs=6)
    p = params_for(bd, cfg)
    px, opx = bd.BkgXParams(grow=1), oracle.BkgXParams(grow=1)
    d_img, d_bad = dev(img), dev(bad0)
    bm, rm, cb, cr, valid, bad_out = bd.bkg_iterate(ctx, d_img, d_bad, p, px, cfg.detect_k, 1)
    _, _, cb0, cr0, _ = bd.bkg_estimate_masked(ctx, d_img, d_bad, p, px)
    m0 = bd.bkg_subtract(ctx, d_img, p.mesh_h, p.mesh_w, cb0, cr0, cfg.detect_k, want_bkg=False)["mask"][0].cpu().numpy()
    torch.cuda.synchronize()
    bad_g = bad_out[0].cpu().numpy()
    assert np.array_equal(bad_g, obv.dilate(m0, 1) | (bad0[0] != 0))
    b = obv.background_masked(img[0], bad_g, to_oracle_params(p), opx)
    assert np.array_equal(valid[0].cpu().numpy(), b["valid"])
    assert np.max(np.abs(bm[0].cpu().numpy() - b["bkg_grid"]) / np.abs(b["bkg_grid"])) < 1e-6
    assert np.max(np.abs(rm[0].cpu().numpy() - b["rms_grid"]) / np.abs(b["rms_grid"])) < 1e-6
    assert np.max(np.abs(cb[0].cpu().numpy() - b["bkg_coef"])) <= 1e-9 * np.max(np.abs(b["bkg_coef"]))
    assert np.max(np.abs(cr[0].cpu().numpy() - b["rms_coef"])) <= 1e-9 * np.max(np.abs(b["rms_coef"]))


# ------------------------------------------------------------------------------------------- NEXT-4: stamp convolution (K8)
from oracle import subtract as osub  # noqa: E402


def _conv_case(rng, B, H, W, p):
    """Template / science frames shaped like a survey frame (sky + noise + a few stars) and kernel coefficients of the size a
    fit returns: a_0 ~ 1 on the narrow Gaussian, small higher-order and spatially varying terms."""
    ref = rng.normal(500, 12, size=(B, H, W)).astype(np.float32)
    for _ in range(max(4, H * W // 4000)):
        f, y, x = int(rng.integers(0, B)), int(rng.integers(0, H)), int(rng.integers(0, W))
        yy, xx = np.mgrid[max(0, y - 6):min(H, y + 7), max(0, x - 6):min(W, x + 7)]
        ref[f, yy, xx] += (rng.uniform(200, 5000) * np.exp(-0.5 * ((yy - y) ** 2 + (xx - x) ** 2) / 1.5 ** 2)).astype(np.float32)
    img = (ref * 1.03 + rng.normal(20, 12, size=ref.shape)).astype(np.float32)
    kc = rng.normal(0, 0.02, size=(B, p.n_basis, p.n_sp))
    kc[:, 0, 0] += 0.6
    bc = rng.normal(0, 5, size=(B, p.n_bg))
    return ref, img, kc, bc


@pytest.mark.parametrize("H,W,B,kw", [(100, 132, 2, {}), (42, 128, 1, {}), (64, 64, 1, dict(spatial_order=0, bg_order=0)),
                                      (75, 88, 2, dict(half_width=3, sigma=(0.8, 1.7), degree=(2, 1), spatial_order=1, bg_order=2)),
                                      (40, 52, 1, dict(half_width=15, sigma=(2.0,), degree=(3,), spatial_order=3, bg_order=0))])
def test_k8_stamp_convolution_against_oracle(bd, ctx, H, W, B, kw):
    """NEXT-4: conv and diff of every pixel against the float64 oracle.  Tolerance: the taps are float32
    roundings of float64 values and the 441-term sum is float32 FMA, so |d conv| <= eps32 * S^2/2 * sum|K| * max|R| in the
    worst case; 3e-6 * sum|K| * max|R| is asserted (observed: a few 1e-7).  Partial stamps, frame edges (zero fill),
    several frames with their own coefficients, the generic kernel for other half-widths."""
    p = bd.ConvParams(**kw)
    op = osub.ConvParams(half_width=p.half_width, sigma=p.sigma, degree=p.degree, spatial_order=p.spatial_order, bg_order=p.bg_order)
    assert p.n_basis == osub.n_basis(op)
    rng = np.random.default_rng(H * W + B)
    ref, img, kc, bc = _conv_case(rng, B, H, W, p)
    out = bd.image_subtract(ctx, dev(ref), dev(img), p, dev(kc), dev(bc), want_conv=True)
    torch.cuda.synchronize()
    S = 2 * p.half_width + 1
    for f in range(B):
        diff, conv = osub.subtract(ref[f], img[f], op, kc[f], bc[f])
        tol = np.empty((H, W))
        for sy in range((H + S - 1) // S):
            for sx in range((W + S - 1) // S):
                tol[sy * S:(sy + 1) * S, sx * S:(sx + 1) * S] = 3e-6 * np.abs(osub.stamp_kernel(op, kc[f], H, W, sx, sy)).sum() * np.abs(ref[f]).max()
        e1 = np.abs(out["conv"][f].cpu().numpy() - conv)
        e2 = np.abs(out["diff"][f].cpu().numpy() - diff)
        assert np.all(e1 <= tol), f"conv: worst {np.max(e1 / tol):.2f} x tol"
        assert np.all(e2 <= tol + 1e-6 * np.abs(diff) + 1e-4), f"diff: worst {np.max(e2 / (tol + 1e-4)):.2f} x tol"
    o2 = bd.image_subtract(ctx, dev(ref), dev(img), p, dev(kc), dev(bc))
    torch.cuda.synchronize()
    assert o2["conv"] is None and torch.equal(o2["diff"], out["diff"])


def test_k8_full_size_config3_sampled(bd, ctx):
    """K8 on the full 9216 x 9232 frame of config 3 (the launch configuration bench.py times, default 21 x 21 stamps with
    spatially varying kernels): 60 seeded stamps plus the four corner stamps, the last (partial) stamp row and column, against
    the oracle computed for those stamps only."""
    cfg = CONFIGS[3]
    ref = make_frames(cfg)
    B, H, W = ref.shape
    p = bd.ConvParams()
    op = osub.ConvParams()
    rng = np.random.default_rng(77)
    img = (ref * np.float32(1.02) + rng.normal(5, 3, size=ref.shape).astype(np.float32)).astype(np.float32)
    kc = rng.normal(0, 0.01, size=(B, p.n_basis, p.n_sp))
    kc[:, 0, 0] += 0.7
    bc = rng.normal(0, 3, size=(B, p.n_bg))
    out = bd.image_subtract(ctx, dev(ref), dev(img), p, dev(kc), dev(bc), want_conv=True)
    torch.cuda.synchronize()
    S = 2 * p.half_width + 1
    nsy, nsx = (H + S - 1) // S, (W + S - 1) // S
    stamps = {(0, 0), (0, nsx - 1), (nsy - 1, 0), (nsy - 1, nsx - 1), (nsy - 1, nsx // 2), (nsy // 2, nsx - 1)}
    stamps |= {(int(a), int(b)) for a, b in zip(rng.integers(0, nsy, 60), rng.integers(0, nsx, 60))}
    diff, conv = osub.subtract(ref[0], img[0], op, kc[0], bc[0], only=sorted(stamps))
    g_conv, g_diff = out["conv"][0].cpu().numpy(), out["diff"][0].cpu().numpy()
    rmax = float(np.abs(ref[0]).max())
    for sy, sx in sorted(stamps):
        sl = (slice(sy * S, min((sy + 1) * S, H)), slice(sx * S, min((sx + 1) * S, W)))
        tol = 3e-6 * np.abs(osub.stamp_kernel(op, kc[0], H, W, sx, sy)).sum() * rmax
        e1, e2 = np.abs(g_conv[sl] - conv[sl]), np.abs(g_diff[sl] - diff[sl])
        assert np.all(e1 <= tol), f"stamp {(sy, sx)} conv: worst {e1.max() / tol:.2f} x tol"
        assert np.all(e2 <= tol + 1e-6 * np.abs(diff[sl]) + 1e-4), f"stamp {(sy, sx)} diff"


def test_k8_impulse_and_identity(bd, ctx):
    """Properties through the GPU path alone: a delta template returns the stamp's kernel (orientation: convolution, not
    correlation); a delta KERNEL (a_0 = 1 on a very narrow Gaussian) returns the template, so diff = I + B - R exactly."""
    p = bd.ConvParams(sigma=(0.05,), degree=(1,), spatial_order=0, bg_order=0)          # exp(-1/(2*0.0025)) = 0: a delta
    H = W = 64
    rng = np.random.default_rng(3)
    ref = rng.normal(100, 5, size=(1, H, W)).astype(np.float32); img = rng.normal(100, 5, size=(1, H, W)).astype(np.float32)
    kc = np.zeros((1, 3, 1)); kc[0, 0, 0] = 1.0
    out = bd.image_subtract(ctx, dev(ref), dev(img), p, dev(kc), dev(np.array([[2.0]])), want_conv=True)
    torch.cuda.synchronize()
    assert np.array_equal(out["conv"][0].cpu().numpy(), ref[0])
    assert np.array_equal(out["diff"][0].cpu().numpy(), ((img[0].astype(np.float64) + 2.0) - ref[0].astype(np.float64)).astype(np.float32))
    p = bd.ConvParams(sigma=(2.0,), degree=(1,), spatial_order=0, bg_order=0)
    ref = np.zeros((1, H, W), np.float32); ref[0, 31, 31] = 1.0                               # centre of the middle stamp
    for n, (i, j) in enumerate(osub.poly_terms(1)):
        kc = np.zeros((1, 3, 1)); kc[0, n, 0] = 1.0
        conv = bd.image_subtract(ctx, dev(ref), dev(ref), p, dev(kc), dev(np.zeros((1, 1))), want_conv=True)["conv"][0].cpu().numpy()
        yy, xx = np.mgrid[21:42, 21:42] - 31
        want = np.exp(-(xx ** 2 + yy ** 2) / 8.0) * xx ** i * yy ** j
        assert np.allclose(conv[21:42, 21:42], want, rtol=2e-7, atol=1e-12), (i, j)


def test_k8_errors(bd, ctx):
    p = bd.ConvParams()
    ref = torch.zeros((1, 64, 64), dtype=torch.float32, device="cuda")
    with pytest.raises(bd.BkgdetError):
        bd.image_subtract(ctx, ref, ref, p, torch.zeros((1, 48, 6), dtype=torch.float64, device="cuda"), torch.zeros((1, 3), dtype=torch.float64, device="cuda"))
    with pytest.raises((bd.BkgdetError, AssertionError)):
        bd.image_subtract(ctx, ref, ref, bd.ConvParams(half_width=20), torch.zeros((1, 49, 6), dtype=torch.float64, device="cuda"),
                          torch.zeros((1, 3), dtype=torch.float64, device="cuda"))


# ------------------------------------------------------------------------------------------- errors
def test_binding_rejects_bad_tensors(bd, ctx):
    """The binding marshals only what the C signatures describe: CUDA, right dtype, contiguous, right shape."""
    good = torch.zeros((1, 64, 64), dtype=torch.float32, device="cuda")
    for bad in (torch.zeros((1, 64, 64), dtype=torch.float32), torch.zeros((1, 64, 64), dtype=torch.float64, device="cuda"),
                torch.zeros((1, 64, 128), dtype=torch.float32, device="cuda")[:, :, ::2]):
        with pytest.raises(bd.BkgdetError):
            bd.mesh_stats(ctx, bad, bd.BkgParams())
        with pytest.raises(bd.BkgdetError):
            bd.bkg_estimate(ctx, bad, bd.BkgParams())
    bm, rm, cb, cr = bd.bkg_estimate(ctx, good, bd.BkgParams())
    with pytest.raises(bd.BkgdetError):
        bd.bkg_subtract(ctx, good, 64, 64, cb.float(), cr, 1.5)
    with pytest.raises(bd.BkgdetError):
        bd.bkg_subtract(ctx, good, 32, 32, cb, cr, 1.5)          # coefficient grid of another mesh size
    with pytest.raises(bd.BkgdetError):
        bd.detect_sources(ctx, good, good, torch.zeros((1, 64, 64), dtype=torch.int32, device="cuda"), 1.5, 5, 16)


def test_error_codes(bd, ctx):
    img = torch.zeros((1, 64, 66), dtype=torch.float32, device="cuda")     # W % 4 != 0
    with pytest.raises(bd.BkgdetError):
        bd.mesh_stats(ctx, img, bd.BkgParams())
    img = torch.zeros((1, 64, 64), dtype=torch.float32, device="cuda")
    with pytest.raises(bd.BkgdetError):
        bd.mesh_stats(ctx, img, bd.BkgParams(filt_h=4))
    with pytest.raises(bd.BkgdetError):
        bd.bkg_estimate(ctx, img, bd.BkgParams(), ws=torch.empty(8, dtype=torch.uint8, device="cuda"))
    with pytest.raises(bd.BkgdetError):
        bd.detect_sources(ctx, img, None, None, 1.5, 5, 16)                   # no mask and no rms
    with pytest.raises(bd.BkgdetError):
        bd.mesh_stats(ctx, torch.zeros((1, 4096, 4096), dtype=torch.float32, device="cuda"), bd.BkgParams(mesh_h=2048, mesh_w=2048))
