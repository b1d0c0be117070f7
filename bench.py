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
"""
from __future__ import annotations

import argparse
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
TILE_TRAFFIC_NCU = 1.8018e9     # dram__bytes_read.sum + dram__bytes_write.sum per launch of the fused tile kernel on config 3
                                # (351.2 MB + 1450.6 MB, profiles/r1_c_fused.md; algorithmic 22 B/px = 1.872 GB)
K3_TRAFFIC_NCU = 1.3888e9       # same for k3_interp_subtract (340.4 MB + 1048.4 MB; algorithmic 17 B/px = 1.446 GB)
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


def run_reference(args, cfg):
    """CPU oracle, as it stands, on a bounded crop of the workload (host cores of this box)."""
    import oracle
    crop = min(cfg.H, args.ref_crop), min(cfg.W, args.ref_crop)
    img = make_frames(cfg, B=1)[0, :crop[0], :crop[1]].copy()
    p = oracle.BkgParams(mesh_h=cfg.mesh, mesh_w=cfg.mesh, filt_h=cfg.filt, filt_w=cfg.filt, clip_sigma=cfg.clip_sigma,
                         clip_iters=cfg.clip_iters)
    oracle.build()
    for _ in range(args.warmup_ref):
        oracle.chain(img, p, cfg.detect_k, cfg.min_area)
    t0 = time.perf_counter()
    nsrc = 0
    for _ in range(args.steps_ref):
        nsrc = len(oracle.chain(img, p, cfg.detect_k, cfg.min_area)["cat"])
    dt = (time.perf_counter() - t0) / args.steps_ref
    cores = int(os.environ.get("OMP_NUM_THREADS", os.cpu_count() or 1))
    mpix = crop[0] * crop[1] / dt / 1e6
    return dict(value=mpix, unit="Mpix/s", cores=cores, kind="oracle", ms_per_step=dt * 1e3,
                sample=f"top-left {crop[0]}x{crop[1]} crop of {cfg.name}, whole chain O1-O6, float64, {nsrc} sources")


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
                "cpu_baseline": {k: r[k] for k in ("value", "unit", "cores", "kind", "sample")},
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

    # ---- workload: each rank its own frame batch (seed offset by rank) -------------------------------
    from dataclasses import replace
    my_cfg = replace(cfg, seed=shard.rank_seed(cfg.seed, rank)) if rank else cfg
    img_h = make_frames(my_cfg)
    B, H, W = img_h.shape
    npx = B * H * W
    p = bd.BkgParams(mesh_h=cfg.mesh, mesh_w=cfg.mesh, filt_h=cfg.filt, filt_w=cfg.filt, clip_sigma=cfg.clip_sigma,
                     clip_iters=cfg.clip_iters)
    ctx = bd.Context(local_rank)
    dev = torch.device("cuda", local_rank)
    img = torch.from_numpy(img_h).to(dev)
    cap = args.cat_capacity
    ws_b = torch.empty(ctx.bkg_workspace_bytes(B, H, W, p), dtype=torch.uint8, device=dev)
    ws_d = torch.empty(ctx.detect_workspace_bytes(B, H, W, cap), dtype=torch.uint8, device=dev)
    o3 = dict(sub=torch.empty((B, H, W), dtype=torch.float32, device=dev), bkg=torch.empty((B, H, W), dtype=torch.float32, device=dev),
              rms=torch.empty((B, H, W), dtype=torch.float32, device=dev), mask=torch.empty((B, H, W), dtype=torch.uint8, device=dev))
    o5 = dict(labels=torch.empty((B, H, W), dtype=torch.int32, device=dev),
              cat=torch.empty(cap * bd.SOURCE_DTYPE.itemsize, dtype=torch.uint8, device=dev),
              n_sources=torch.empty(B, dtype=torch.int64, device=dev))

    ev_tile = [torch.cuda.Event(enable_timing=True) for _ in range(2)]
    for e in ev_tile:
        e.record()          # creates the handles

    def step_unfused(ev=None):
        if ev: ev[0].record()
        bm, rm, cb, cr = bd.bkg_estimate(ctx, img, p, ws=ws_b)
        if ev: ev[1].record()
        bd.bkg_subtract(ctx, img, p.mesh_h, p.mesh_w, cb, cr, cfg.detect_k, out=o3)
        if ev: ev[2].record()
        bd.detect_sources(ctx, o3["sub"], o3["rms"], o3["mask"], cfg.detect_k, cfg.min_area, cap, ws=ws_d, out=o5)
        if ev: ev[3].record()

    def step_fused(ev=None):
        if ev: ev[0].record()
        bm, rm, cb, cr = bd.bkg_estimate(ctx, img, p, ws=ws_b)
        if ev: ev[1].record()
        o35 = dict(o3); o35.update(o5)
        bd.bkg_subtract_detect(ctx, img, p.mesh_h, p.mesh_w, cb, cr, cfg.detect_k, cfg.min_area, cap, ws=ws_d, out=o35)
        if ev: ev[2].record()
        if ev: ev[3].record()

    step = step_unfused if args.unfused else step_fused

    def barrier():
        if dist: dist.barrier()
        torch.cuda.synchronize()

    for _ in range(max(args.warmup, 3)):
        step()
    barrier()
    sampler = ClockSampler(local_rank); sampler.start()
    evs = [[torch.cuda.Event(enable_timing=True) for _ in range(4)] for _ in range(args.steps)]
    t_start, t_end = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    barrier()
    t_start.record()
    for k in range(args.steps):
        step(evs[k])
    t_end.record()
    barrier()
    sampler.stop_flag = True
    total_ms = t_start.elapsed_time(t_end)
    stage_ms = [float(np.mean([e[i].elapsed_time(e[i + 1]) for e in evs])) for i in range(3)]
    # outside the timed region: (i) the tile kernel alone (events recorded by the library around its launch),
    # (ii) the three calls one by one (bkg_subtract = the K3 pass alone, for the 17 B/px figure)
    tile_ms = []
    bd.tile_kernel_events(ctx, ev_tile[0], ev_tile[1])
    for _ in range(5):
        step(); torch.cuda.synchronize()
        tile_ms.append(ev_tile[0].elapsed_time(ev_tile[1]))
    bd.tile_kernel_events(ctx, None, None)
    tile_ms = float(np.mean(tile_ms))
    ev_u = [[torch.cuda.Event(enable_timing=True) for _ in range(4)] for _ in range(5)]
    step_unfused(); torch.cuda.synchronize()
    for k in range(5):
        step_unfused(ev_u[k])
    torch.cuda.synchronize()
    unfused_ms = [float(np.mean([e[i].elapsed_time(e[i + 1]) for e in ev_u])) for i in range(3)]
    n_src = int(o5["n_sources"].sum().item())
    total_ms = shard.max_over_ranks(total_ms, dist, dev)
    ms_per_step = total_ms / args.steps
    value = shard.whole_job_value(shard.sum_over_ranks(npx, dist, dev), ms_per_step * 1e-3) / 1e6

    # ---- end to end through bd_run_host: pinned host frame in, catalogue out, every step -------------
    e2e = None
    if not args.no_e2e:
        pinned = torch.from_numpy(img_h).pin_memory()
        cat_h = np.empty(cap, dtype=bd.SOURCE_DTYPE)
        host_img = pinned.numpy()
        for _ in range(2):
            bd.run_host(ctx, host_img, p, cfg.detect_k, cfg.min_area, cap, cat=cat_h)
        barrier()
        n_e2e = max(3, min(args.steps, 10))
        t0 = time.perf_counter()
        for _ in range(n_e2e):
            recs, nn = bd.run_host(ctx, host_img, p, cfg.detect_k, cfg.min_area, cap, cat=cat_h)
        torch.cuda.synchronize()
        dt = (time.perf_counter() - t0) / n_e2e
        dt = shard.max_over_ranks(dt, dist, dev)
        e2e = {"value": world * npx / dt / 1e6, "unit": "Mpix/s", "h2d_bytes_per_step": int(npx * 4),
               "d2h_bytes_per_step": int(len(recs) * bd.SOURCE_DTYPE.itemsize + B * 8), "ms_per_step": dt * 1e3,
               "api": "bd_run_host (pinned host frame -> catalogue on host)"}

    if rank != 0:
        if dist: dist.destroy_process_group()
        return
    peak, peak_src = measured_peak()
    k3_gbs = K3_BYTES_PER_PX * npx / (unfused_ms[1] * 1e-3) / 1e9
    tile_bpp = 5.0 if args.unfused else TILE_BYTES_PER_PX
    tile_gbs = tile_bpp * npx / (tile_ms * 1e-3) / 1e9
    line = {
        "metric": METRIC, "value": value, "unit": "Mpix/s", "n_gpus": world, "steps": args.steps, "warmup": max(args.warmup, 3),
        "ms_per_step": ms_per_step, "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f32/f64",
        "data": "synthetic",
        "config": {"workload": cfg.name, "B": B, "H": H, "W": W, "mesh": cfg.mesh, "filter": cfg.filt, "detect_k": cfg.detect_k,
                   "min_area": cfg.min_area, "sources_found": n_src, "parallelism": f"frames x{world} (no collective)",
                   "calls": "bkg_estimate + bkg_subtract + detect_sources" if args.unfused else "bkg_estimate + bkg_subtract_detect",
                   "l2": "input 340 MB per step > 126 MB L2 (no flush needed)" if npx * 4 > 200e6 else "inputs smaller than L2: L2-warm"},
        "stages_ms": ({"bkg_estimate": stage_ms[0], "bkg_subtract": stage_ms[1], "detect_sources": stage_ms[2]} if args.unfused else
                      {"bkg_estimate": stage_ms[0], "bkg_subtract_detect": stage_ms[1]}),
        "stages_ms_separate_calls": {"bkg_estimate": unfused_ms[0], "bkg_subtract": unfused_ms[1], "detect_sources": unfused_ms[2]},
        "chain_roofline": {"bytes_per_px": CHAIN_BYTES_PER_PX, "achieved_gbs": CHAIN_BYTES_PER_PX * npx / (ms_per_step * 1e-3) / 1e9,
                           "frac_of_measured": CHAIN_BYTES_PER_PX * npx / (ms_per_step * 1e-3) / 1e9 / peak,
                           "frac_of_8000": CHAIN_BYTES_PER_PX * npx / (ms_per_step * 1e-3) / 1e9 / 8000.0},
        "roofline": {"kernel": "k4a_tile_label" + ("" if args.unfused else "<fused: a3 + a4 + partial sums of a5>"), "bound": "hbm",
                     "achieved": tile_gbs, "peak": peak, "unit": "GB/s", "frac": tile_gbs / peak, "frac_of_8000": tile_gbs / 8000.0,
                     "traffic": TILE_TRAFFIC_NCU if not args.unfused and args.config == 3 else None, "peak_source": peak_src,
                     "bytes_per_px": tile_bpp, "ms": tile_ms},
        "roofline_k3_pass": {"kernel": "k3_interp_subtract (bkg_subtract called alone)", "bound": "hbm", "achieved": k3_gbs, "peak": peak,
                             "unit": "GB/s", "frac": k3_gbs / peak, "frac_of_8000": k3_gbs / 8000.0, "traffic": K3_TRAFFIC_NCU if args.config == 3 else None,
                             "bytes_per_px": K3_BYTES_PER_PX, "ms": unfused_ms[1]},
        "gpu_launches": (LAUNCHES_PER_STEP_UNFUSED if args.unfused else LAUNCHES_PER_STEP) * args.steps,
        "clocks": sampler.summary(),
        "host": {"nproc": os.cpu_count()},
    }
    if e2e:
        line["e2e"] = e2e
    if not args.no_cpu_baseline and world == 1:
        r = run_reference(args, cfg)
        line["cpu_baseline"] = {k: r[k] for k in ("value", "unit", "cores", "kind", "sample")}
    print(json.dumps(line))
    if dist: dist.destroy_process_group()


if __name__ == "__main__":
    main()
