"""O10 / O11: multi-threshold deblending and cleaning of the source candidates -- CPU oracle (TEST INFRASTRUCTURE).

PAPER.md:153 ("The source detection algorithm adapted in this paper is based on the approach proposed in SExtractor
(Bertin & Arnouts 1996) ... pixel detection, source deblending, cleaning, and photometry"), :155 ("calculate multi-level
deblending thresholds.  At each threshold level, the algorithm re-evaluates objects and splits them as necessary,
constructing a binary tree structure rooted in the original source candidate ... traversed from bottom to top ... pruning
... based on rigorous intensity and spatial criteria"), :157 ("determine if the current object can be merged with any
adjacent objects based on predefined criteria.  If the analysis indicates that merging is appropriate, the current object
is flagged as a false detection ... a parallel operation to remove the marked pixels").
The paper gives no constants and no formulas; the readings (D1-D12 in DESIGN.md) restate the published method it adapts:

D1  candidates = the components of O5 that O6 keeps (npix >= min_area); smaller components are left alone;
D2  levels of a candidate: t_0 = k_d * rms[peak pixel], t_i = t_(i-1) * q, q = (peak / t_0)^(1 / n_thresh) (exponential
    spacing between the detection threshold and the peak), i = 1 .. n_thresh - 1.  n_thresh is a power of two and q is
    taken by repeated square roots, every product rounded once in float64, so that both sides get the same t_i bit for
    bit; k_d enters as the float32 the mask used.  peak <= t_0: the candidate is not deblended;
D3  node of level 0 = the whole candidate; nodes of level i >= 1 = the 8-connected components of
    {p in candidate : sub[p] > t_i} (float64 compare) that have at least min_area pixels ("spatial criterion");
    the parent of a node is the node of the previous level that contains it;
D4  a node is significant when its flux (sum of sub over its pixels) exceeds min_cont * (flux of the candidate)
    ("intensity criterion");
D5  pruning, bottom to top: S(n) = the objects node n resolves into.  With split = the children c with |S(c)| >= 2 and
    sig = the children with |S(c)| = 1 that are significant: |split| + |sig| >= 2 -> S(n) = union of S(c), c in split,
    plus the nodes of sig; otherwise |split| = 1 -> S(n) = S(that child); otherwise S(n) = {n};
D6  |S(root)| = 1: the candidate is unchanged;
D7  pixels of a node of S(root) belong to that object; the other pixels of the candidate are handed out by synchronous
    growth: in every round each still unassigned pixel with at least one assigned 8-neighbour (as of the previous round)
    joins the object of its brightest assigned neighbour (largest sub; ties: the object whose node starts first in
    raster order); rounds until no pixel is left;
D8  label of an object = 1 + the minimum raster index of its pixels; the catalogue is O6 on the new label map;
D9  cleaning looks at the catalogue: shape of object j = ellipse of its second moments, Dj = x2 y2 - xy^2 (1/12 added to
    x2 and y2 when Dj < 0.00694, as in A24), r_j^2(dx, dy) = (y2 dx^2 + x2 dy^2 - 2 xy dx dy) / Dj;
D10 profile of a neighbour j: I_j(r^2) = A_j (1 + alpha_j r^2)^(-beta), A_j = flux_j / (2 pi sqrt(Dj)), alpha_j such that
    I_j = t_j (its threshold, D2) on the ellipse whose area is npix_j: rho_j^2 = npix_j / (pi sqrt(Dj)),
    alpha_j = ((A_j / t_j)^(1 / beta) - 1) / rho_j^2; A_j <= t_j: j influences nobody;
D11 object i is a false detection when some j with flux_j > flux_i (ties: the smaller label counts as brighter) and
    r_j^2(centroid_i - centroid_j) <= clean_zone^2 rho_j^2 has flux_i / npix_i - I_j(r_j^2) <= t_i; every decision is
    taken on the input catalogue (one simultaneous pass);
D12 the pixels of false detections become 0 in the label map and their records leave the catalogue.

Plain numpy, one candidate at a time; the labelling of each level is O5 (oracle.label).  Shares no code with the CUDA path.
"""
from __future__ import annotations

import math
from dataclasses import dataclass

import numpy as np

from . import label, reduce_sources


@dataclass
class DeblendParams:
    n_thresh: int = 32               # D2: number of levels (power of two)
    min_cont: float = 0.005          # D4: minimum contrast
    clean_param: float = 1.0         # D10: beta
    clean_zone: float = 4.0          # D11: zone, in isophotal radii of the neighbour


def thresholds(peak: float, t0: float, n_thresh: int) -> np.ndarray:
    """D2.  -> float64 [n_thresh] with t[0] = t0."""
    m = int(round(math.log2(n_thresh)))
    assert n_thresh >= 2 and 2 ** m == n_thresh, "n_thresh must be a power of two"
    q = np.float64(peak) / np.float64(t0)
    for _ in range(m):
        q = np.sqrt(q)
    t = np.empty(n_thresh, dtype=np.float64)
    t[0] = t0
    for i in range(1, n_thresh):
        t[i] = t[i - 1] * q
    return t


def candidate_threshold(detect_k: float, rms: np.ndarray, ypeak: int, xpeak: int) -> float:
    """D2: t_0 of a candidate (exact float64 product of two float32)."""
    return float(np.float64(np.float32(detect_k)) * np.float64(np.float32(rms[ypeak, xpeak])))


def build_tree(sub_box: np.ndarray, member: np.ndarray, t: np.ndarray, min_area: int):
    """D3.  sub_box float64, member bool [h, w] -> (nodes, level label maps).
    nodes: dict (level, label) -> dict(npix, flux, parent, children); level 0 holds the single root (0, first-pixel label)."""
    h, w = member.shape
    lab0 = np.where(member, int(np.flatnonzero(member.reshape(-1))[0]) + 1, 0).astype(np.int32)
    labs = [lab0]
    nodes = {}
    root = (0, int(lab0.max()))
    nodes[root] = dict(npix=int(member.sum()), flux=float(sub_box[member].sum()), parent=None, children=[])
    for i in range(1, len(t)):
        on = member & (sub_box > t[i])
        li = label(on.astype(np.uint8))
        labs.append(li)
        for L in np.unique(li[li > 0]):
            sel = li == L
            npix = int(sel.sum())
            if npix < min_area:
                continue
            first = int(L) - 1                                   # the node's first pixel in raster order
            parent = (i - 1, int(labs[i - 1].reshape(-1)[first]))
            assert parent in nodes                               # it contains the child, so it is at least as large
            nodes[(i, int(L))] = dict(npix=npix, flux=float(sub_box[sel].sum()), parent=parent, children=[])
            nodes[parent]["children"].append((i, int(L)))
    return nodes, labs, root


def resolve(nodes, n, min_flux: float):
    """D4 + D5.  -> list of node keys node n resolves into."""
    split, sig = [], []
    for c in nodes[n]["children"]:
        sc = resolve(nodes, c, min_flux)
        if len(sc) >= 2:
            split.append(sc)
        elif nodes[c]["flux"] > min_flux:
            sig.append(c)
    if len(split) + len(sig) >= 2:
        out = [k for sc in split for k in sc] + sig
        return sorted(out, key=lambda k: k[1])
    if len(split) == 1:
        return split[0]
    return [n]


def grow(obj: np.ndarray, member: np.ndarray, sub_box: np.ndarray) -> np.ndarray:
    """D7.  obj int64 [h, w]: object key (first pixel of its node + 1) on assigned pixels, 0 elsewhere."""
    h, w = obj.shape
    obj = obj.copy()
    while True:
        todo = member & (obj == 0)
        if not todo.any():
            return obj
        best_sub = np.full((h, w), -np.inf)
        best_obj = np.zeros((h, w), dtype=np.int64)
        for dy in (-1, 0, 1):
            for dx in (-1, 0, 1):
                if dy == 0 and dx == 0:
                    continue
                # neighbour q = p + (dy, dx): shifted views, zero (unassigned) outside the box
                q_obj = np.zeros((h, w), dtype=np.int64)
                q_sub = np.full((h, w), -np.inf)
                ys0, ys1, xs0, xs1 = max(0, -dy), min(h, h - dy), max(0, -dx), min(w, w - dx)
                q_obj[ys0:ys1, xs0:xs1] = obj[ys0 + dy:ys1 + dy, xs0 + dx:xs1 + dx]
                q_sub[ys0:ys1, xs0:xs1] = sub_box[ys0 + dy:ys1 + dy, xs0 + dx:xs1 + dx]
                better = (q_obj > 0) & ((q_sub > best_sub) | ((q_sub == best_sub) & (q_obj < best_obj)))
                best_sub = np.where(better, q_sub, best_sub)
                best_obj = np.where(better, q_obj, best_obj)
        new = todo & (best_obj > 0)
        assert new.any(), "candidate is not 8-connected"
        obj[new] = best_obj[new]


def deblend_candidate(sub_box: np.ndarray, member: np.ndarray, peak: float, t0: float, min_area: int, prm: DeblendParams):
    """One candidate inside its bounding box.  sub_box float32/64 [h, w], member bool [h, w].
    -> (obj int64 [h, w]: 0 outside the candidate, else 1 + box-raster index of the first pixel of the object's node;
        n_objects; fragile: True when some node's flux is within 1e-9 relative of the contrast limit)."""
    sub_box = np.asarray(sub_box, dtype=np.float64)
    first = int(np.flatnonzero(member.reshape(-1))[0]) + 1
    whole = np.where(member, first, 0).astype(np.int64)
    if not (peak > t0):
        return whole, 1, False
    t = thresholds(peak, t0, prm.n_thresh)
    nodes, labs, root = build_tree(sub_box, member, t, min_area)
    min_flux = prm.min_cont * nodes[root]["flux"]
    fragile = any(abs(v["flux"] - min_flux) <= 1e-9 * abs(min_flux) for v in nodes.values())
    objs = resolve(nodes, root, min_flux)
    if len(objs) == 1:
        return whole, 1, fragile
    obj = np.zeros(member.shape, dtype=np.int64)
    for (lev, L) in objs:
        obj[labs[lev] == L] = L
    return grow(obj, member, sub_box), len(objs), fragile


def deblend(sub: np.ndarray, rms: np.ndarray, labels: np.ndarray, cat: np.ndarray, detect_k: float, min_area: int,
            prm: DeblendParams, only=None):
    """O10 on one frame.  sub, rms float32 [H, W]; labels int32 (O5); cat = O6 records of the candidates.
    `only`: optional iterable of candidate labels to process (the others are left as they are).
    -> (new labels int32, n_objects per processed candidate {label: n}, fragile candidate labels)."""
    H, W = labels.shape
    out = labels.copy()
    nobj, frag = {}, []
    want = None if only is None else set(int(v) for v in only)
    for r in cat:
        L = int(r["label"])
        if want is not None and L not in want:
            continue
        y0, y1, x0, x1 = int(r["ymin"]), int(r["ymax"]) + 1, int(r["xmin"]), int(r["xmax"]) + 1
        member = labels[y0:y1, x0:x1] == L
        t0 = candidate_threshold(detect_k, rms, int(r["ypeak"]), int(r["xpeak"]))
        obj, n, fr = deblend_candidate(sub[y0:y1, x0:x1], member, float(np.float32(r["peak"])), t0, min_area, prm)
        nobj[L] = n
        if fr:
            frag.append(L)
        if n == 1:
            continue
        w = x1 - x0
        box = out[y0:y1, x0:x1]
        for key in np.unique(obj[obj > 0]):
            sel = obj == key
            ys, xs = np.nonzero(sel)
            box[sel] = 1 + (y0 + int(ys[0])) * W + (x0 + int(xs[0]))       # D8: first pixel in raster order = minimum index
    return out, nobj, frag


# ------------------------------------------------------------------------------------------------ cleaning
def _shape(r):
    """D9: (x2, y2, xy, D) with the degenerate-moment rule of A24."""
    x2, y2, xy = float(r["x2"]), float(r["y2"]), float(r["xy"])
    D = x2 * y2 - xy * xy
    if D < 0.00694:
        x2 += 1.0 / 12.0
        y2 += 1.0 / 12.0
        D = x2 * y2 - xy * xy
    return x2, y2, xy, D


def clean_flags(cat: np.ndarray, rms: np.ndarray, detect_k: float, prm: DeblendParams):
    """D9-D11.  -> (false-detection flags uint8 [n], fragile uint8 [n]: some deciding comparison within 1e-9 relative)."""
    n = len(cat)
    flag = np.zeros(n, dtype=np.uint8)
    fragile = np.zeros(n, dtype=np.uint8)
    beta = float(prm.clean_param)
    t = np.array([candidate_threshold(detect_k, rms, int(r["ypeak"]), int(r["xpeak"])) for r in cat], dtype=np.float64)
    flux, npix, lab = cat["flux"].astype(np.float64), cat["npix"].astype(np.float64), cat["label"].astype(np.int64)
    xs, ys = cat["x"].astype(np.float64), cat["y"].astype(np.float64)
    for j in range(n):                                   # the neighbour j, against every i at once
        x2, y2, xy, D = _shape(cat[j])
        if not (D > 0.0) or not (t[j] > 0.0):
            continue
        sD = math.sqrt(D)
        A = flux[j] / (2.0 * math.pi * sD)
        if not (A > t[j]):
            continue
        rho2 = npix[j] / (math.pi * sD)
        alpha = ((A / t[j]) ** (1.0 / beta) - 1.0) / rho2
        brighter = (flux[j] > flux) | ((flux[j] == flux) & (lab[j] < lab))
        dx, dy = xs - xs[j], ys - ys[j]
        r2 = (y2 * dx * dx + x2 * dy * dy - 2.0 * xy * dx * dy) / D
        zone = r2 <= prm.clean_zone * prm.clean_zone * rho2
        Ij = A * (1.0 + alpha * r2) ** (-beta)
        lhs = flux / npix - Ij
        pair = brighter & zone
        pair[j] = False
        flag[pair & (lhs <= t)] = 1
        fragile[pair & (np.abs(lhs - t) <= 1e-9 * np.abs(t))] = 1
    return flag, fragile


def clean(labels: np.ndarray, cat: np.ndarray, rms: np.ndarray, detect_k: float, prm: DeblendParams):
    """O11 on one frame.  -> (labels with the false detections removed, kept records, flags, fragile)."""
    flag, fragile = clean_flags(cat, rms, detect_k, prm)
    out = labels.copy()
    for r in cat[flag != 0]:
        y0, y1, x0, x1 = int(r["ymin"]), int(r["ymax"]) + 1, int(r["xmin"]), int(r["xmax"]) + 1
        box = out[y0:y1, x0:x1]
        box[box == int(r["label"])] = 0                                    # D12
    return out, cat[flag == 0], flag, fragile


def deblend_clean(sub, rms, labels, cat, detect_k, min_area, prm: DeblendParams, do_clean=True):
    """O10 then O6 on the new labels, then O11."""
    lab2, nobj, frag = deblend(sub, rms, labels, cat, detect_k, min_area, prm)
    cat2 = reduce_sources(lab2, sub, min_area)
    if not do_clean:
        return dict(labels=lab2, cat=cat2, n_objects=nobj, fragile_candidates=frag)
    lab3, cat3, flag, cfrag = clean(lab2, cat2, rms, detect_k, prm)
    return dict(labels=lab3, cat=cat3, labels_deblended=lab2, cat_deblended=cat2, n_objects=nobj,
                fragile_candidates=frag, clean_flags=flag, clean_fragile=cfrag)
