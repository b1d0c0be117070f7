#!/usr/bin/env python
"""bench.py -- background + detection throughput on B200.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config 3] [--unfused] [--impl reference]

One "step" = one pass of the whole hot path (steps a1..a5) over one synthetic frame batch of the chosen
BASELINE.json config (default: config 3, the 9216x9232 frame the metric's targets are quoted on), through the C ABI:
bkg_estimate -> bkg_subtract_detect (the fused a3+a4+a5 call; --unfused times bkg_subtract -> detect_sources).
`value` is Mpix/s with the frame resident in HBM; `e2e` is the same metric through bd_run_host with HOST buffers
(H2D of the frame and D2H of the catalogue inside the timed region).
`roofline` is for the dominant kernel, the fused tile kernel k4a_tile_label<fused> (pass a3 + pass a4 + the partial
sums of a5): algorithmic bytes 22 B/px (17 + 5) / its duration, taken with CUDA events that the
library records on the launching stream right before and after that kernel (outside the timed steps, same inputs),
against MEASURED_PEAKS.json's HBM copy bandwidth.  `roofline_k3_pass` is the stand-alone K3 pass (bkg_subtract),
the "fused interpolate/subtract/threshold pass" BASELINE.json's 70 % target names.
With N > 1 (torchrun) every rank processes its own frame (frames are independent units: no data-path
collective); value = all ranks' pixels / max-over-ranks time.
`--impl reference` times the CPU oracle, as it stands, on a bounded crop of the same workload.
The default run (config 3, N = 1) also reports, outside the timed region: `configs` -- the same step on configs 1, 2, 4, 5
(inputs of configs 1-2 rotated through > 256 MB of distinct copies so that L2 cannot serve them), each with its own clock
sample -- and `next_stages_ms` -- deblend_sources, clean_sources, photometry, image_subtract and image_reproject on config 3.
"""
from __future__ import annotations

import argparse
import hashlib
import json
import os
import subprocess
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

from synth import CONFIGS, make_frames  # noqa: E402

METRIC = "Mpix/s background+detection per frame"
K3_BYTES_PER_PX = 17.0          # img 4 read; sub 4 + bkg 4 + rms 4 + mask 1 written
TILE_BYTES_PER_PX = 22.0        # fused tile kernel = pass a3 (17) + pass a4 (mask 1 read, labels 4 written)
CHAIN_BYTES_PER_PX = 30.0       # K1 4 + K3 17 + K4 5 + K5 4
LAUNCHES_PER_STEP = 10          # K1, K2a, K2b, then bkg_subtract_detect: k_spline_tabs, k4a (fused), k4b, k5m, k5k, k5s, k5f
                                # (+2 memsets, not counted)
LAUNCHES_PER_STEP_UNFUSED = 10  # ... K3, then detect_sources: k4a, k4b, k5m, k5k, k5s, k5f
TRAFFIC_FILE = os.path.join("profiles", "traffic.json")   # ncu DRAM bytes per launch + the hash of the sources they were measured on
FALLBACK_HBM_GBS = 6650.0       # B200_PROFILING.md fallback if MEASURED_PEAKS.json is absent


def measured_peak():
    try:
        with open(os.path.join(ROOT, "MEASURED_PEAKS.json")) as f:
            return float(json.load(f)["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
    except Exception:
        return FALLBACK_HBM_GBS, "fallback (B200_PROFILING.md)"


class ClockSampler(threading.Thread):
    """SM clock and throttle reasons during the timed region: NVML (pynvml, ~1 ms per sample: the timed region of the
    default run is only ~20 ms long) when it is there, else nvidia-smi (~100 ms per sample)."""

    NAMES = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]

    def __init__(self, index: int):
        super().__init__(daemon=True)
        self.index, self.rows, self.stop_flag, self.source = index, [], False, "nvidia-smi"
        self.q = ("clocks.sm,clocks.max.sm,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
                  "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")
        self.nvml = None
        try:
            import pynvml
            pynvml.nvmlInit()
            # torch's device index follows CUDA_VISIBLE_DEVICES; NVML's does not
            vis = os.environ.get("CUDA_VISIBLE_DEVICES")
            phys = index
            if vis:
                ids = [v.strip() for v in vis.split(",") if v.strip()]
                if index < len(ids) and ids[index].isdigit():
                    phys = int(ids[index])
            self.handle = pynvml.nvmlDeviceGetHandleByIndex(phys)
            self.max_mhz = float(pynvml.nvmlDeviceGetMaxClockInfo(self.handle, pynvml.NVML_CLOCK_SM))
            self.nvml, self.source = pynvml, "nvml"
        except Exception:
            self.nvml = None

    def _sample_nvml(self):
        n = self.nvml
        mhz = n.nvmlDeviceGetClockInfo(self.handle, n.NVML_CLOCK_SM)
        r = n.nvmlDeviceGetCurrentClocksEventReasons(self.handle) if hasattr(n, "nvmlDeviceGetCurrentClocksEventReasons") \
            else n.nvmlDeviceGetCurrentClocksThrottleReasons(self.handle)
        bits = [getattr(n, "nvmlClocksThrottleReasonHwSlowdown", 0x8), getattr(n, "nvmlClocksThrottleReasonHwThermalSlowdown", 0x40),
                getattr(n, "nvmlClocksThrottleReasonSwThermalSlowdown", 0x20), getattr(n, "nvmlClocksThrottleReasonSwPowerCap", 0x4)]
        return [str(mhz), str(self.max_mhz)] + ["Active" if r & b else "Not Active" for b in bits]

    def run(self):
        while not self.stop_flag:
            try:
                if self.nvml:
                    self.rows.append(self._sample_nvml())
                    time.sleep(0.002)
                    continue
                out = subprocess.run(["nvidia-smi", f"--query-gpu={self.q}", "--format=csv,noheader,nounits", "-i", str(self.index)],
                                     capture_output=True, text=True, timeout=5).stdout.strip()
                if out:
                    self.rows.append([s.strip() for s in out.split(",")])
            except Exception:
                if self.nvml:
                    self.nvml = None     # fall back to nvidia-smi
            time.sleep(0.1)

    def summary(self):
        if not self.rows:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["unsampled"]}
        sm = sorted(float(r[0]) for r in self.rows if r[0].replace(".", "").isdigit())
        reasons = [n for i, n in enumerate(self.NAMES) if any(len(r) > 2 + i and r[2 + i].lower().startswith("active") for r in self.rows)]
        return {"sm_mhz": sm[len(sm) // 2] if sm else None, "sm_max_mhz": float(self.rows[0][1]), "reasons": reasons,
                "samples": len(self.rows), "source": self.source}


def source_hash(files):
    h = hashlib.sha256()
    for f in files:
        with open(os.path.join(ROOT, "paper_2502_10783_b200", "csrc", f), "rb") as fh:
            h.update(fh.read())
    return h.hexdigest()[:16]


def ncu_traffic(kernel):
    """DRAM bytes per launch from the committed ncu capture (profiles/traffic.json), or None when the kernel's sources have
    changed since that capture."""
    try:
        with open(os.path.join(ROOT, TRAFFIC_FILE)) as f:
            t = json.load(f)[kernel]
        return float(t["dram_bytes_per_launch"]) if source_hash(t["sources"]) == t["source_sha256_16"] else None
    except Exception:
        return None


def omp_threads(n):
    """Thread count of the oracle's OpenMP loops (a libgomp call; the oracle itself is not touched)."""
    import ctypes
    try:
        ctypes.CDLL("libgomp.so.1").omp_set_num_threads(int(n))
        return True
    except Exception:
        return False


def run_reference(args, cfg, threads=None):
    """CPU oracle, as it stands, on a bounded crop of the workload (host cores of this box)."""
    import oracle
    crop = min(cfg.H, args.ref_crop), min(cfg.W, args.ref_crop)
    img = make_frames(cfg, B=1)[0, :crop[0], :crop[1]].copy()
    p = oracle.BkgParams(mesh_h=cfg.mesh, mesh_w=cfg.mesh, filt_h=cfg.filt, filt_w=cfg.filt, clip_sigma=cfg.clip_sigma,
                         clip_iters=cfg.clip_iters)
    oracle.build()
    cores = int(os.environ.get("OMP_NUM_THREADS", os.cpu_count() or 1))
    if threads is not None and omp_threads(threads):
        cores = threads
    for _ in range(args.warmup_ref):
        oracle.chain(img, p, cfg.detect_k, cfg.min_area)
    t0 = time.perf_counter()
    nsrc = 0
    for _ in range(args.steps_ref):
        nsrc = len(oracle.chain(img, p, cfg.detect_k, cfg.min_area)["cat"])
    dt = (time.perf_counter() - t0) / args.steps_ref
    mpix = crop[0] * crop[1] / dt / 1e6
    # the oracle's steps one by one (same calls chain() makes), once
    st = {}
    t = time.perf_counter(); ms = oracle.mesh_stats(img, p); st["O1_mesh_stats"] = time.perf_counter() - t
    t = time.perf_counter()
    cb = oracle.spline_coeffs(oracle.grid_median(ms["bkg"], p.filt_h, p.filt_w)); cr = oracle.spline_coeffs(oracle.grid_median(ms["rms"], p.filt_h, p.filt_w))
    st["O2_grid_filter_prefilter"] = time.perf_counter() - t
    t = time.perf_counter()
    bkg = oracle.spline_eval(cb, crop[0], crop[1], p.mesh_h, p.mesh_w); rms = oracle.spline_eval(cr, crop[0], crop[1], p.mesh_h, p.mesh_w)
    st["O3_spline_eval"] = time.perf_counter() - t
    t = time.perf_counter(); _, sub32, mask, _ = oracle.subtract_threshold(img, bkg, rms, cfg.detect_k); st["O4_subtract_threshold"] = time.perf_counter() - t
    t = time.perf_counter(); lab = oracle.label(mask); st["O5_label"] = time.perf_counter() - t
    t = time.perf_counter(); oracle.reduce_sources(lab, sub32, cfg.min_area); st["O6_reduce"] = time.perf_counter() - t
    return dict(value=mpix, unit="Mpix/s", cores=cores, kind="oracle", ms_per_step=dt * 1e3,
                stages_ms={k: v * 1e3 for k, v in st.items()},
                sample=f"top-left {crop[0]}x{crop[1]} crop of {cfg.name}, whole chain O1-O6, float64, {nsrc} sources")


class Workload:
    """One config resident on the device: buffers, the step functions, the timing of K steps."""

    def __init__(self, bd, torch, ctx, cfg, img_h, cap, dev, rotate_bytes=0):
        self.bd, self.torch, self.ctx, self.cfg, self.cap = bd, torch, ctx, cfg, cap
        B, H, W = img_h.shape
        self.B, self.H, self.W, self.npx = B, H, W, B * H * W
        self.p = bd.BkgParams(mesh_h=cfg.mesh, mesh_w=cfg.mesh, filt_h=cfg.filt, filt_w=cfg.filt, clip_sigma=cfg.clip_sigma,
                              clip_iters=cfg.clip_iters)
        img = torch.from_numpy(img_h).to(dev)
        # L2 honesty: inputs smaller than L2 are rotated through enough distinct copies that L2 cannot serve them
        n_copies = 1 if self.npx * 4 >= rotate_bytes else int(-(-rotate_bytes // (self.npx * 4)))
        self.imgs = [img] + [img.clone() for _ in range(n_copies - 1)]
        self.k = 0
        self.ws_b = torch.empty(ctx.bkg_workspace_bytes(B, H, W, self.p), dtype=torch.uint8, device=dev)
        self.ws_d = torch.empty(ctx.detect_workspace_bytes(B, H, W, cap), dtype=torch.uint8, device=dev)
        f32 = lambda: torch.empty((B, H, W), dtype=torch.float32, device=dev)  # noqa: E731
        self.o3 = dict(sub=f32(), bkg=f32(), rms=f32(), mask=torch.empty((B, H, W), dtype=torch.uint8, device=dev))
        self.o5 = dict(labels=torch.empty((B, H, W), dtype=torch.int32, device=dev),
                       cat=torch.empty(cap * bd.SOURCE_DTYPE.itemsize, dtype=torch.uint8, device=dev),
                       n_sources=torch.empty(B, dtype=torch.int64, device=dev))

    def l2_note(self):
        mb = self.npx * 4 / 1e6
        if len(self.imgs) > 1:
            return (f"input {mb:.0f} MB per step: rotated through {len(self.imgs)} distinct copies ({mb * len(self.imgs):.0f} MB > 2 x 126 MB L2), "
                    "so no step finds its input in L2")
        return f"input {mb:.0f} MB per step > 126 MB L2 (no flush needed)"

    def next_img(self):
        self.k = (self.k + 1) % len(self.imgs)
        return self.imgs[self.k]

    def step_unfused(self, ev=None):
        bd, cfg, p, img = self.bd, self.cfg, self.p, self.next_img()
        if ev: ev[0].record()
        bm, rm, cb, cr = bd.bkg_estimate(self.ctx, img, p, ws=self.ws_b)
        if ev: ev[1].record()
        bd.bkg_subtract(self.ctx, img, p.mesh_h, p.mesh_w, cb, cr, cfg.detect_k, out=self.o3)
        if ev: ev[2].record()
        bd.detect_sources(self.ctx, self.o3["sub"], self.o3["rms"], self.o3["mask"], cfg.detect_k, cfg.min_area, self.cap, ws=self.ws_d,
                          out=self.o5)
        if ev: ev[3].record()

    def step_fused(self, ev=None):
        bd, cfg, p, img = self.bd, self.cfg, self.p, self.next_img()
        if ev: ev[0].record()
        bm, rm, cb, cr = bd.bkg_estimate(self.ctx, img, p, ws=self.ws_b)
        if ev: ev[1].record()
        o35 = dict(self.o3); o35.update(self.o5)
        bd.bkg_subtract_detect(self.ctx, img, p.mesh_h, p.mesh_w, cb, cr, cfg.detect_k, cfg.min_area, self.cap, ws=self.ws_d, out=o35)
        if ev: ev[2].record()
        if ev: ev[3].record()

    def timed(self, step, steps, warmup, barrier, local_rank):
        """warmup untimed steps, then exactly `steps` steps between two events; clocks sampled during the timed region."""
        torch = self.torch
        for _ in range(max(warmup, 3)):
            step()
        barrier()
        sampler = ClockSampler(local_rank); sampler.start()
        evs = [[torch.cuda.Event(enable_timing=True) for _ in range(4)] for _ in range(steps)]
        t_start, t_end = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        barrier()
        t_start.record()
        for k in range(steps):
            step(evs[k])
        t_end.record()
        barrier()
        sampler.stop_flag = True
        sampler.join(timeout=2.0)
        total_ms = t_start.elapsed_time(t_end)
        stage_ms = [float(np.mean([e[i].elapsed_time(e[i + 1]) for e in evs])) for i in range(3)]
        per_step = sorted(e[0].elapsed_time(e[3]) for e in evs)   # device time of each step alone (without the gap to the next)
        self.step_stats = {"median": float(per_step[len(per_step) // 2]), "best": float(per_step[0]), "worst": float(per_step[-1])}
        return total_ms, stage_ms, sampler.summary()

    def tile_kernel_ms(self, step, ev_tile, n=5):
        self.bd.tile_kernel_events(self.ctx, ev_tile[0], ev_tile[1])
        out = []
        for _ in range(n):
            step(); self.torch.cuda.synchronize()
            out.append(ev_tile[0].elapsed_time(ev_tile[1]))
        self.bd.tile_kernel_events(self.ctx, None, None)
        return float(np.mean(out))

    def free(self):
        for k in ("imgs", "ws_b", "ws_d", "o3", "o5"):
            setattr(self, k, None)
        self.torch.cuda.empty_cache()


def time_next_stages(bd, torch, ctx, wl, reps=5, sm_mhz=None, hbm_peak=None):
    """deblend_sources, clean_sources, photometry, image_subtract and image_reproject on the maps of the last step (outside the timed region)."""
    cfg, cap = wl.cfg, wl.cap
    sub, rms = wl.o3["sub"], wl.o3["rms"]
    ev = lambda: torch.cuda.Event(enable_timing=True)  # noqa: E731
    lab0 = wl.o5["labels"].clone()
    nb = bd.C.c_size_t()
    ctx.check(ctx.lib.bd_deblend_workspace_bytes(ctx.h, wl.B, wl.H, wl.W, bd.C.c_int64(cap), bd.C.c_int64(cap), bd.C.byref(nb)))
    ws = torch.empty(nb.value, dtype=torch.uint8, device=sub.device)
    ctx.check(ctx.lib.bd_clean_workspace_bytes(ctx.h, wl.B, wl.H, wl.W, bd.C.c_int64(cap), bd.C.byref(nb)))
    ws_c = torch.empty(nb.value, dtype=torch.uint8, device=sub.device)
    ctx.check(ctx.lib.bd_phot_workspace_bytes(ctx.h, bd.C.c_int64(cap), bd.C.byref(nb)))
    ws_p = torch.empty(nb.value, dtype=torch.uint8, device=sub.device)
    phot = torch.zeros(cap * bd.PHOT_DTYPE.itemsize, dtype=torch.uint8, device=sub.device)
    t = {"deblend_sources": [], "clean_sources": [], "photometry": [], "image_subtract": []}
    counts = {}
    cp = bd.ConvParams()
    gen = torch.Generator(device=sub.device); gen.manual_seed(7)
    kcoef = 1e-3 * torch.randn((wl.B, cp.n_basis, cp.n_sp), dtype=torch.float64, device=sub.device, generator=gen)
    kcoef[:, 0, 0] = 1.0
    bgcoef = torch.zeros((wl.B, cp.n_bg), dtype=torch.float64, device=sub.device)
    diff = torch.empty_like(sub)
    for _ in range(reps + 1):
        lab = lab0.clone()
        e = [ev() for _ in range(5)]
        e[0].record()
        d = bd.deblend_sources(ctx, sub, rms, lab, wl.o5["cat"], wl.o5["n_sources"], cap, cfg.detect_k, cfg.min_area, ws=ws)
        e[1].record()
        c = bd.clean_sources(ctx, rms, lab, d["cat"], d["n_sources"], cap, cfg.detect_k, ws=ws_c)
        e[2].record()
        bd.photometry(ctx, sub, rms, c["cat"], c["n_sources"], cap, out=phot, ws=ws_p)
        e[3].record()
        bd.image_subtract(ctx, wl.imgs[0], wl.imgs[0], cp, kcoef, bgcoef, out=dict(diff=diff))
        e[4].record()
        torch.cuda.synchronize()
        for i, k in enumerate(t):
            t[k].append(e[i].elapsed_time(e[i + 1]))
        counts = {"candidates": int(wl.o5["n_sources"].sum()), "deblended": int(d["n_sources"].sum()), "cleaned": int(c["n_sources"].sum())}
    out = {k: float(np.median(v[1:])) for k, v in t.items()}   # (workspaces are allocated once, outside the timed calls)
    out["objects"] = counts
    out["image_subtract_gflops"] = 2.0 * 441 * wl.npx / (out["image_subtract"] * 1e-3) / 1e9
    # K8 is bound by the float32 FMA pipe (K8): peak = SMs x 128 FMA/clk x 2 flop x the SM clock of the run
    prop = torch.cuda.get_device_properties(sub.device)
    clk_mhz = float(sm_mhz) if sm_mhz else 1965.0    # the SM clock sampled under load during the timed steps
    peak_tf = prop.multi_processor_count * 128 * 2 * clk_mhz * 1e6 / 1e12
    out["roofline_image_subtract"] = {"kernel": "k8_stamp_conv<10>", "bound": "alu", "achieved": out["image_subtract_gflops"] / 1e3, "peak": peak_tf,
                                      "unit": "TFLOP/s", "frac": out["image_subtract_gflops"] / 1e3 / peak_tf,
                                      "peak_source": f"SMs x 128 FP32 FMA/clk x 2 x {clk_mhz:.0f} MHz (B200_PROFILING.md unit counts; SM clock sampled under load)", "traffic": None}
    # K11: bilinear reprojection through a small rotation + shear + shift; 4 B/px read + 4 B/px written
    A = torch.tensor([[1.0007 * np.cos(0.004), -1.0007 * np.sin(0.004) + 0.0006, 3.37, 1.0007 * np.sin(0.004), 1.0007 * np.cos(0.004), -2.81]] * wl.B,
                     dtype=torch.float64, device=sub.device)
    tr = []
    for _ in range(reps + 1):
        e0, e1 = ev(), ev()
        e0.record()
        bd.image_reproject(ctx, wl.imgs[0], A, None, 0.0, out=diff)
        e1.record()
        torch.cuda.synchronize()
        tr.append(e0.elapsed_time(e1))
    out["image_reproject"] = float(np.median(tr[1:]))
    gbs = 8.0 * wl.npx / (out["image_reproject"] * 1e-3) / 1e9
    out["roofline_image_reproject"] = {"kernel": "k11_reproject", "bound": "hbm", "achieved": gbs, "peak": hbm_peak, "unit": "GB/s",
                                       "frac": gbs / hbm_peak if hbm_peak else None, "bytes_per_px": 8.0, "traffic": None}
    return out


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--config", type=int, default=3)
    ap.add_argument("--impl", default="b200", choices=["b200", "reference"])
    ap.add_argument("--ref-crop", type=int, default=3072)
    ap.add_argument("--steps-ref", type=int, default=1)
    ap.add_argument("--warmup-ref", type=int, default=0)
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-extras", action="store_true", help="skip the other configs and the NEXT stages (default run only)")
    ap.add_argument("--unfused", action="store_true", help="time bkg_subtract + detect_sources instead of bkg_subtract_detect")
    ap.add_argument("--cat-capacity", type=int, default=1 << 20)
    args = ap.parse_args()
    cfg = CONFIGS[args.config]
    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))

    if args.impl == "reference":
        if rank != 0:
            return
        if args.steps_ref == 1 and args.steps < 20:
            args.steps_ref = max(1, min(args.steps, 3))
        r = run_reference(args, cfg)
        line = {"impl": "reference", "metric": METRIC, "value": r["value"], "unit": "Mpix/s", "n_gpus": args.gpus,
                "steps": args.steps_ref, "warmup": args.warmup_ref, "ms_per_step": r["ms_per_step"], "higher_is_better": True,
                "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
                "config": {"workload": cfg.name, "sample": r["sample"]},
                "cpu_baseline": {k: r[k] for k in ("value", "unit", "cores", "kind", "sample", "stages_ms")},
                "e2e": {"value": r["value"], "unit": "Mpix/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}}
        print(json.dumps(line))
        return

    import torch
    import paper_2502_10783_b200 as bd
    from paper_2502_10783_b200 import shard

    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: there is no CPU fallback")
    torch.cuda.set_device(local_rank)
    dist = None
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=torch.device("cuda", local_rank))

    def barrier():
        if dist: dist.barrier()
        torch.cuda.synchronize()

    # ---- workload: each rank its own frame batch (seed offset by rank) -------------------------------
    from dataclasses import replace
    my_cfg = replace(cfg, seed=shard.rank_seed(cfg.seed, rank)) if rank else cfg
    img_h = make_frames(my_cfg)
    ctx = bd.Context(local_rank)
    dev = torch.device("cuda", local_rank)
    cap = args.cat_capacity
    ROTATE = 256 << 20
    wl = Workload(bd, torch, ctx, cfg, img_h, cap, dev, rotate_bytes=ROTATE)
    B, H, W, npx = wl.B, wl.H, wl.W, wl.npx
    ev_tile = [torch.cuda.Event(enable_timing=True) for _ in range(2)]
    for e in ev_tile:
        e.record()          # creates the handles
    step = wl.step_unfused if args.unfused else wl.step_fused

    total_ms, stage_ms, clocks = wl.timed(step, args.steps, args.warmup, barrier, local_rank)
    # outside the timed region: (i) the tile kernel alone (events recorded by the library around its launch),
    # (ii) the three calls one by one (bkg_subtract = the K3 pass alone, for the 17 B/px figure)
    tile_ms = wl.tile_kernel_ms(step, ev_tile)
    ev_u = [[torch.cuda.Event(enable_timing=True) for _ in range(4)] for _ in range(5)]
    wl.step_unfused(); torch.cuda.synchronize()
    for k in range(5):
        wl.step_unfused(ev_u[k])
    torch.cuda.synchronize()
    unfused_ms = [float(np.mean([e[i].elapsed_time(e[i + 1]) for e in ev_u])) for i in range(3)]
    step(); torch.cuda.synchronize()
    n_src = int(wl.o5["n_sources"].sum().item())
    total_ms = shard.max_over_ranks(total_ms, dist, dev)
    ms_per_step = total_ms / args.steps
    value = shard.whole_job_value(shard.sum_over_ranks(npx, dist, dev), ms_per_step * 1e-3) / 1e6

    # ---- end to end through bd_run_host: pinned host frame in, catalogue out, every step -------------
    e2e = None
    if not args.no_e2e:
        pinned = torch.from_numpy(img_h).pin_memory()
        cat_pin = torch.empty(cap * bd.SOURCE_DTYPE.itemsize, dtype=torch.uint8).pin_memory()   # (a pageable buffer is staged by the driver: ~1 ms more for 15 MB)
        cat_h = cat_pin.numpy().view(bd.SOURCE_DTYPE)
        host_img = pinned.numpy()
        for _ in range(2):
            bd.run_host(ctx, host_img, wl.p, cfg.detect_k, cfg.min_area, cap, cat=cat_h)
        barrier()
        n_e2e = max(3, min(args.steps, 10))
        t0 = time.perf_counter()
        for _ in range(n_e2e):
            recs, nn = bd.run_host(ctx, host_img, wl.p, cfg.detect_k, cfg.min_area, cap, cat=cat_h)
        torch.cuda.synchronize()
        dt = (time.perf_counter() - t0) / n_e2e
        dt = shard.max_over_ranks(dt, dist, dev)
        e2e = {"value": world * npx / dt / 1e6, "unit": "Mpix/s", "h2d_bytes_per_step": int(npx * 4),
               "d2h_bytes_per_step": int(len(recs) * bd.SOURCE_DTYPE.itemsize + B * 8), "ms_per_step": dt * 1e3,
               "api": "bd_run_host (pinned host frame -> catalogue in a pinned host buffer)"}
        del pinned, host_img, cat_h, cat_pin

    if rank != 0:
        if dist: dist.destroy_process_group()
        return
    peak, peak_src = measured_peak()

    def chain_roofline(n_px, ms):
        gbs = CHAIN_BYTES_PER_PX * n_px / (ms * 1e-3) / 1e9
        return {"bytes_per_px": CHAIN_BYTES_PER_PX, "achieved_gbs": gbs, "frac_of_measured": gbs / peak, "frac_of_8000": gbs / 8000.0}

    k3_gbs = K3_BYTES_PER_PX * npx / (unfused_ms[1] * 1e-3) / 1e9
    tile_bpp = 5.0 if args.unfused else TILE_BYTES_PER_PX
    tile_gbs = tile_bpp * npx / (tile_ms * 1e-3) / 1e9
    tile_traffic = ncu_traffic("k4a_tile_label<fused>") if not args.unfused and args.config == 3 else None
    line = {
        "metric": METRIC, "value": value, "unit": "Mpix/s", "n_gpus": world, "steps": args.steps, "warmup": max(args.warmup, 3),
        "ms_per_step": ms_per_step, "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f32/f64",
        "data": "synthetic",
        "config": {"workload": cfg.name, "B": B, "H": H, "W": W, "mesh": cfg.mesh, "filter": cfg.filt, "detect_k": cfg.detect_k,
                   "min_area": cfg.min_area, "sources_found": n_src, "parallelism": f"frames x{world} (no collective)",
                   "calls": "bkg_estimate + bkg_subtract + detect_sources" if args.unfused else "bkg_estimate + bkg_subtract_detect",
                   "l2": wl.l2_note()},
        "stages_ms": ({"bkg_estimate": stage_ms[0], "bkg_subtract": stage_ms[1], "detect_sources": stage_ms[2]} if args.unfused else
                      {"bkg_estimate": stage_ms[0], "bkg_subtract_detect": stage_ms[1]}),
        "stages_ms_separate_calls": {"bkg_estimate": unfused_ms[0], "bkg_subtract": unfused_ms[1], "detect_sources": unfused_ms[2]},
        "step_ms_device": wl.step_stats,
        "chain_roofline": chain_roofline(npx, ms_per_step),
        "roofline": {"kernel": "k4a_tile_label" + ("" if args.unfused else "<fused: a3 + a4 + partial sums of a5>"), "bound": "hbm",
                     "achieved": tile_gbs, "peak": peak, "unit": "GB/s", "frac": tile_gbs / peak, "frac_of_8000": tile_gbs / 8000.0,
                     "traffic": tile_traffic, "traffic_source": TRAFFIC_FILE if tile_traffic else None, "peak_source": peak_src,
                     "bytes_per_px": tile_bpp, "ms": tile_ms},
        "roofline_k3_pass": {"kernel": "k3_interp_subtract (bkg_subtract called alone)", "bound": "hbm", "achieved": k3_gbs, "peak": peak,
                             "unit": "GB/s", "frac": k3_gbs / peak, "frac_of_8000": k3_gbs / 8000.0,
                             "traffic": ncu_traffic("k3_interp_subtract") if args.config == 3 else None,
                             "bytes_per_px": K3_BYTES_PER_PX, "ms": unfused_ms[1]},
        "gpu_launches": (LAUNCHES_PER_STEP_UNFUSED if args.unfused else LAUNCHES_PER_STEP) * args.steps,
        "clocks": clocks,
        "host": {"nproc": os.cpu_count()},
    }
    if e2e:
        line["e2e"] = e2e
    extras = not args.no_extras and world == 1 and args.config == 3 and not args.unfused
    if extras:
        # SURVEY 8(f) stages on this config, then the other configs (parity-test cases; reported, not the headline)
        line["next_stages_ms"] = time_next_stages(bd, torch, ctx, wl, sm_mhz=(clocks or {}).get("sm_mhz"), hbm_peak=peak)
        wl.free()
        others = []
        for c in (1, 2, 4, 5):
            ocfg = CONFIGS[c]
            owl = Workload(bd, torch, ctx, ocfg, make_frames(ocfg), cap, dev, rotate_bytes=ROTATE)
            o_total, o_stage, o_clocks = owl.timed(owl.step_fused, 10, 3, barrier, local_rank)
            o_tile = owl.tile_kernel_ms(owl.step_fused, ev_tile, n=3)
            o_ms = o_total / 10
            others.append({"workload": ocfg.name, "B": owl.B, "H": owl.H, "W": owl.W, "ms_per_step": o_ms, "value": owl.npx / (o_ms * 1e-3) / 1e6,
                           "unit": "Mpix/s", "stages_ms": {"bkg_estimate": o_stage[0], "bkg_subtract_detect": o_stage[1]},
                           "tile_kernel_ms": o_tile, "chain_roofline": chain_roofline(owl.npx, o_ms), "l2": owl.l2_note(),
                           "sources_found": int(owl.o5["n_sources"].sum().item()), "clocks": o_clocks})
            owl.free()
        line["configs"] = others
    if not args.no_cpu_baseline and world == 1:
        r = run_reference(args, cfg)
        line["cpu_baseline"] = {k: r[k] for k in ("value", "unit", "cores", "kind", "sample", "stages_ms")}
        r1 = run_reference(args, cfg, threads=1)
        line["cpu_baseline"]["one_core"] = {"value": r1["value"], "unit": "Mpix/s", "cores": r1["cores"], "stages_ms": r1["stages_ms"]}
    print(json.dumps(line))
    if dist: dist.destroy_process_group()


if __name__ == "__main__":
    main()
