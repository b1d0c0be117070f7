"""Seeded synthetic frames shaped like the paper's workloads.

These stand in for the paper's SkyMaker simulations (2000^2..8000^2 px, 50-100 sources/deg^2,
PAPER.md:202, :224-232; background gradient as a % of the sky level) and its GWAC
frames (4196x4136 px, ~20 000 sources), none of which can be had here.  The five
configurations are BASELINE.json's ``configs`` (SURVEY.md section 8(d) fixes what that file leaves
open).  This module draws inputs only; it contains none of the method's arithmetic.

Recipe (every config): numpy ``Generator(PCG64(seed))``; float64 accumulation; draw order
  1. per-frame scalars where the config has them (sky level, read noise, n sources, FWHM),
  2. source x positions, 3. source y positions, 4. source fluxes,
  5. Poisson image ``P ~ Poisson(sky + sources)``, 6. read-noise image ``N(0, sigma_r)``,
  7. hot-pixel indices (config 3 only);
then clip / round where the config says so, and cast to float32.  Sources are sampled at pixel
centres (pixel (y, x) has its centre at coordinate (y, x)) and scaled so that the continuous
integral of the profile is the flux: Gaussian ``F/(2 pi s^2) exp(-r^2/(2 s^2))`` with
``s = FWHM/2.35482`` inside a square stamp of half-width ``ceil(8 s)``; Moffat
``F (beta-1)/(pi a^2) (1 + r^2/a^2)^(-beta)`` with ``a = FWHM / (2 sqrt(2^(1/beta) - 1))`` inside a
stamp of half-width 32.
"""
from __future__ import annotations

from dataclasses import dataclass, replace
import math

import numpy as np

FWHM_TO_SIGMA = 1.0 / 2.35482


@dataclass(frozen=True)
class FrameConfig:
    """Workload shape + the method parameters BASELINE.json attaches to it."""
    name: str
    B: int
    H: int
    W: int
    seed: int
    mesh: int
    filt: int
    clip_sigma: float = 3.0
    clip_iters: int = 5
    detect_k: float = 1.5
    min_area: int = 5
    kind: str = "cfg1"


CONFIGS = {
    # "512x512 ... seed 0: sky 1000 + 0.05 ADU/px, Poisson + N(0,5), 50 Gaussian FWHM 3"
    1: FrameConfig("cfg1_512", 1, 512, 512, 0, 64, 3, kind="cfg1"),
    # "4096x4096 (uint16) sky 800 + quadratic +-10%, N(0,8), 5000 Moffat beta 3 FWHM 2.5"
    2: FrameConfig("cfg2_4096_u16_moffat", 1, 4096, 4096, 1, 128, 3, kind="cfg2"),
    # "9216x9232 sky 300 + sinusoid, N(0,3), 40000 Gaussian FWHM 2-4, 0.1% hot pixels"
    3: FrameConfig("cfg3_9216x9232_cmos", 1, 9232, 9216, 2, 256, 5, kind="cfg3"),
    # "64 x 2048x2048 pipeline batch"
    4: FrameConfig("cfg4_batch64_2048", 64, 2048, 2048, 1000, 64, 3, kind="cfg4"),
    # "6144x6144 crowded, steep gradient, 250000 Gaussian FWHM 3 + 200 saturated"
    5: FrameConfig("cfg5_6144_crowded", 1, 6144, 6144, 4, 64, 3, detect_k=1.0, min_area=3, kind="cfg5"),
}


def _add_sources(img: np.ndarray, xs, ys, fluxes, fwhms, profile: str, beta: float = 3.0,
                 chunk: int = 4096) -> None:
    """Accumulate point sources into ``img`` (float64, in place)."""
    H, W = img.shape
    n = len(xs)
    if n == 0:
        return
    fwhms = np.broadcast_to(np.asarray(fwhms, dtype=np.float64), (n,))
    if profile == "gauss":
        sig = fwhms * FWHM_TO_SIGMA
        rad = np.ceil(8.0 * sig).astype(np.int64)
    else:
        alpha = fwhms / (2.0 * math.sqrt(2.0 ** (1.0 / beta) - 1.0))
        rad = np.full(n, 32, dtype=np.int64)
    flat = img.reshape(-1)
    order = np.argsort(rad, kind="stable")
    pos = 0
    while pos < n:
        r = int(rad[order[pos]])
        end = pos
        cap = max(1, min(chunk, 2_000_000 // ((2 * r + 1) ** 2)))
        while end < n and end - pos < cap and rad[order[end]] == r:
            end += 1
        idx = order[pos:end]
        pos = end
        off = np.arange(-r, r + 1, dtype=np.int64)
        cx = np.rint(xs[idx]).astype(np.int64)
        cy = np.rint(ys[idx]).astype(np.int64)
        px = cx[:, None] + off[None, :]                       # [m, S]
        py = cy[:, None] + off[None, :]
        dx2 = (px - xs[idx][:, None]) ** 2
        dy2 = (py - ys[idx][:, None]) ** 2
        r2 = dy2[:, :, None] + dx2[:, None, :]                # [m, S, S]
        if profile == "gauss":
            s2 = sig[idx] ** 2
            val = (fluxes[idx] / (2.0 * math.pi * s2))[:, None, None] * np.exp(-r2 / (2.0 * s2)[:, None, None])
        else:
            a2 = alpha[idx] ** 2
            val = (fluxes[idx] * (beta - 1.0) / (math.pi * a2))[:, None, None] * (1.0 + r2 / a2[:, None, None]) ** (-beta)
        ok = ((py >= 0) & (py < H))[:, :, None] & ((px >= 0) & (px < W))[:, None, :]
        lin = (py[:, :, None] * W + px[:, None, :])[ok]
        np.add.at(flat, lin, val[ok])


def _finish(rng, lam: np.ndarray, read_sigma: float) -> np.ndarray:
    out = rng.poisson(lam).astype(np.float64)
    out += rng.normal(0.0, read_sigma, size=lam.shape)
    return out


def _log_uniform(rng, n, lo_exp, hi_exp):
    return 10.0 ** rng.uniform(lo_exp, hi_exp, size=n)


def make_frame(cfg: FrameConfig, frame: int = 0, H: int | None = None, W: int | None = None,
               n_sources: int | None = None) -> np.ndarray:
    """One float32 frame ``[H, W]`` of config ``cfg`` (``frame`` selects the frame of a batch).

    ``H``/``W``/``n_sources`` override the size for scaled-down test cases; the source count is
    scaled with the area unless given.
    """
    fullH, fullW = cfg.H, cfg.W
    H = fullH if H is None else H
    W = fullW if W is None else W
    scale = (H * W) / float(fullH * fullW)
    yy = np.arange(H, dtype=np.float64)[:, None]
    xx = np.arange(W, dtype=np.float64)[None, :]
    kind = cfg.kind

    def nsrc(full):
        return int(round(full * scale)) if n_sources is None else n_sources

    if kind == "cfg1":
        rng = np.random.Generator(np.random.PCG64(cfg.seed))
        n = nsrc(50)
        xs = rng.uniform(0, W, n); ys = rng.uniform(0, H, n)
        fl = _log_uniform(rng, n, 3, 5)
        lam = 1000.0 + 0.05 * xx + np.zeros((H, 1))
        _add_sources(lam, xs, ys, fl, 3.0, "gauss")
        img = _finish(rng, lam, 5.0)
    elif kind == "cfg2":
        rng = np.random.Generator(np.random.PCG64(cfg.seed))
        n = nsrc(5000)
        xs = rng.uniform(0, W, n); ys = rng.uniform(0, H, n)
        # inverse CDF of N(>F) ~ F^-1.5 truncated to [500, 2e5]
        q = rng.uniform(0, 1, n)
        a, b = 500.0 ** -1.5, 2.0e5 ** -1.5
        fl = (a - q * (a - b)) ** (-1.0 / 1.5)
        u = 2.0 * xx / max(W - 1, 1) - 1.0
        v = 2.0 * yy / max(H - 1, 1) - 1.0
        lam = 800.0 * (1.0 + 0.1 * (u * u + v * v - 1.0))
        _add_sources(lam, xs, ys, fl, 2.5, "moffat", beta=3.0)
        img = _finish(rng, lam, 8.0)
        img = np.rint(np.clip(img, 0.0, 65535.0))          # uint16 detector, then float32
    elif kind == "cfg3":
        rng = np.random.Generator(np.random.PCG64(cfg.seed))
        n = nsrc(40000)
        xs = rng.uniform(0, W, n); ys = rng.uniform(0, H, n)
        fl = _log_uniform(rng, n, 3, 5)
        fwhm = 2.0 + 2.0 * xs / max(W - 1, 1)
        lam = 300.0 + 20.0 * np.sin(2 * math.pi * xx / 3000.0) * np.cos(2 * math.pi * yy / 3000.0)
        _add_sources(lam, xs, ys, fl, fwhm, "gauss")
        img = _finish(rng, lam, 3.0)
        nhot = int(round(0.001 * H * W))
        hot = rng.choice(H * W, size=nhot, replace=False)
        img.reshape(-1)[hot] = 60000.0
    elif kind == "cfg4":
        rng = np.random.Generator(np.random.PCG64(cfg.seed + frame))
        sky = rng.uniform(200.0, 2000.0)
        rs = rng.uniform(4.0, 10.0)
        n = int(rng.integers(500, 3001))
        fwhm = rng.uniform(2.0, 5.0)
        n = int(round(n * scale)) if n_sources is None else n_sources
        xs = rng.uniform(0, W, n); ys = rng.uniform(0, H, n)
        fl = _log_uniform(rng, n, 3, 5)
        lam = np.full((H, W), sky, dtype=np.float64)
        _add_sources(lam, xs, ys, fl, fwhm, "gauss")
        img = _finish(rng, lam, rs)
    elif kind == "cfg5":
        rng = np.random.Generator(np.random.PCG64(cfg.seed))
        n = nsrc(250000)
        nbright = min(n, int(round(200 * scale)) if n_sources is None else min(200, n))
        xs = rng.uniform(0, W, n); ys = rng.uniform(0, H, n)
        fl = _log_uniform(rng, n, 3, 5)
        fl[:nbright] = _log_uniform(rng, nbright, 6, 8)
        lam = 1500.0 + 0.3 * xx + np.zeros((H, 1))
        _add_sources(lam, xs, ys, fl, 3.0, "gauss")
        lam = np.minimum(lam, 1.0e7)
        img = _finish(rng, lam, 6.0)
        img = np.minimum(img, 65535.0)
    else:
        raise ValueError(kind)
    return img.astype(np.float32)


def make_frames(cfg: FrameConfig, H: int | None = None, W: int | None = None, B: int | None = None,
                n_sources: int | None = None) -> np.ndarray:
    """All frames of a config as one contiguous float32 array ``[B, H, W]``."""
    B = cfg.B if B is None else B
    out = np.empty((B, cfg.H if H is None else H, cfg.W if W is None else W), dtype=np.float32)
    for f in range(B):
        out[f] = make_frame(cfg, f, H, W, n_sources)
    return out


def small(cfg: FrameConfig, H: int, W: int, B: int | None = None) -> FrameConfig:
    """The same config with a reduced geometry (for parity cases the oracle finishes in seconds)."""
    return replace(cfg, H=H, W=W, B=cfg.B if B is None else B, name=f"{cfg.name}_{H}x{W}")


def noise_frame(seed: int, H: int, W: int, mean: float, sigma: float) -> np.ndarray:
    """Pure Gaussian noise N(mean, sigma^2) as float32 (used by statistical pins)."""
    rng = np.random.Generator(np.random.PCG64(seed))
    return rng.normal(mean, sigma, size=(H, W)).astype(np.float32)
