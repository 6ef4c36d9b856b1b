#!/usr/bin/env python
"""bench.py -- headline benchmark of libblinkimg on B200.

One "step" = one pass of the whole hot path (steps a0..a5 of SURVEY.md section 8(a)) over one batch of
synthetic visibilities: blink_image() on BASELINE.json config 3 (50 timesteps x 768 channels -> 38400 dirty
images of 512 x 512, 8128 baselines) -- the configuration the metric is quoted on.

  python bench.py [--gpus N] [--steps K] [--warmup W] [--config 3] [--impl reference]

Prints ONE JSON line.  value = dirty images/s (whole job), device-resident inputs; e2e = the same through
blink_image_host() with pinned HOST buffers (H2D of visibilities and D2H of every image inside the timed
region); roofline = the bytes the fused implementation MUST move (M4 = 4 N^2 + 8 B per image + 12 T B: visibilities
in, images out) / kernel time / measured HBM peak, with the SURVEY 8(d) contract models M36 / M20 as
labelled companions; configs = short timed legs of BASELINE.json configs 1, 2, 4 (one timestep) and 5;
cpu_baseline = the CPU oracle, as it stands, on a bounded sample.
Multi-GPU (torchrun): every rank images its own independent batch ("replicas / independent shards",
PAPER.md L150, L322: each second of observation is independent) -- weak scaling, no collective on the data path.
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
import torch

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

from paper_2505_15204_b200 import shard, workloads  # noqa: E402

FALLBACK_HBM_GBS = 6650.0          # B200_PROFILING.md fallback when MEASURED_PEAKS.json is absent


def model_bytes(T, C, P, B, N):
    """Algorithmic bytes of one step: per image vis read (8B) + grid written (8N^2) + row pass
    read+write (16N^2) + column pass read (8N^2) + image written (4N^2); uvw read once per timestep."""
    n_img = T * C * P
    return {"M36": n_img * (36 * N * N + 8 * B) + 12 * T * B,
            "M20": n_img * (20 * N * N + 8 * B) + 12 * T * B,
            "M4": n_img * (4 * N * N + 8 * B) + 12 * T * B}


def hbm_peak():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        try:
            return float(json.load(open(p))["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
        except Exception:
            pass
    return FALLBACK_HBM_GBS, "fallback (B200_PROFILING.md)"


class ClockSampler:
    """nvidia-smi clocks / throttle reasons sampled every 100 ms from the warm-up to the end of the timed region
    (the timed region itself lasts only ~0.25 s: the warm-up keeps the same load running until the sampler is up)."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.index, self.proc, self.lines = index, None, []

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(self.index), f"--query-gpu={self.Q}",
                                          "--format=csv,noheader,nounits", "-lms", "100"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.th = threading.Thread(target=self._read, daemon=True)
            self.th.start()
        except Exception:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.lines.append(line.strip())

    def stop(self):
        if not self.proc:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        self.proc.terminate()
        try:
            self.proc.wait(timeout=5)
        except Exception:
            self.proc.kill()
        sm, mx, reasons = [], [], set()
        for ln in self.lines:
            f = [x.strip() for x in ln.split(",")]
            if len(f) < 7:
                continue
            try:
                sm.append(float(f[0])); mx.append(float(f[1]))
            except ValueError:
                continue
            for name, v in zip(("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"), f[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(name)
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "samples": len(sm), "reasons": sorted(reasons)}


def cpu_oracle_leg(w_small, target_s: float = 15.0):
    """Times the CPU oracle (oracle/, as it stands) on a bounded sample of the SAME workload shape."""
    import oracle
    cores = os.cpu_count() or 1
    vis, uvw = w_small.vis.cpu().numpy(), w_small.uvw_m.cpu().numpy()
    n_avail = w_small.T * w_small.C * w_small.P
    ids = np.arange(min(n_avail, 32 * cores))
    t0 = time.perf_counter()
    oracle.image_batch(vis, uvw, w_small.freqs_hz, w_small.n_pix, w_small.pixscale_rad, w_small.weighting, ids, nthreads=cores)
    dt = time.perf_counter() - t0
    # repeat the same sample until about target_s of wall time has been spent (the work per image is identical)
    reps = int(max(1, min(50, round(target_s / max(dt, 1e-3)))))
    t0 = time.perf_counter()
    for _ in range(reps):
        oracle.image_batch(vis, uvw, w_small.freqs_hz, w_small.n_pix, w_small.pixscale_rad, w_small.weighting, ids, nthreads=cores)
    dt = time.perf_counter() - t0
    n_done = reps * len(ids)
    return {"value": n_done / dt, "unit": "images/s", "cores": cores, "kind": "oracle",
            "sample": f"{len(ids)} images ({w_small.n_pix}x{w_small.n_pix}, {w_small.B} baselines) of the same workload, "
                      f"imaged {reps}x = {n_done} images in {dt:.1f} s wall, one image per task on {cores} threads"}


def sample_workload(cfg: int, n_images: int):
    """A slice of config `cfg` on the CPU with ~n_images images (first timesteps, channels spread over the band)."""
    shp = workloads.config_shape(cfg)
    C = max(1, min(shp["C"], n_images // max(1, shp["P"])))
    T = max(1, min(shp["T"], -(-n_images // (C * shp["P"]))))
    return workloads.make_config(cfg, device="cpu", T=T, C=C)


def run_reference(args, rank: int):
    """--impl reference: the oracle itself on the host cores (bounded sample per step)."""
    if rank != 0:
        return
    shp = workloads.config_shape(args.config)
    cores = os.cpu_count() or 1
    per_step = max(cores, 4 * cores)
    w = sample_workload(args.config, per_step)
    import oracle
    vis, uvw = w.vis.numpy(), w.uvw_m.numpy()
    ids = np.arange(min(per_step, w.T * w.C * w.P))
    run = lambda: oracle.image_batch(vis, uvw, w.freqs_hz, w.n_pix, w.pixscale_rad, w.weighting, ids, nthreads=cores)
    for _ in range(args.warmup):
        run()
    t0 = time.perf_counter()
    for _ in range(args.steps):
        run()
    dt = (time.perf_counter() - t0) / args.steps
    val = len(ids) / dt
    sample = f"{len(ids)} images per step of config {args.config} ({w.n_pix}x{w.n_pix}, {w.B} baselines), {cores} threads"
    print(json.dumps({
        "impl": "reference", "metric": "dirty_images_per_s", "value": val, "unit": "images/s", "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": dt * 1e3, "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": f"config{args.config}: bounded sample of {shp['T']}x{shp['C']}x{shp['P']} images "
                               f"{shp['n_pix']}x{shp['n_pix']}, B={shp['B']}", "sample": sample},
        "cpu_baseline": {"value": val, "unit": "images/s", "cores": cores, "kind": "oracle", "sample": sample},
        "e2e": {"value": val, "unit": "images/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0}))


def timed_ms(run, steps, warmup, dev, world, flush=None):
    """Mean device time of `run` (CUDA events on the current stream), max over ranks.  flush: a tensor larger than L2 that is
    rewritten before every timed call (small workloads whose inputs and outputs would otherwise stay in L2)."""
    for _ in range(warmup):
        run()
    torch.cuda.synchronize(dev)
    tot = 0.0
    if flush is None:
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        for _ in range(steps):
            run()
        e1.record()
        torch.cuda.synchronize(dev)
        tot = e0.elapsed_time(e1)
    else:
        for _ in range(steps):
            flush.add_(1)
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record()
            run()
            e1.record()
            torch.cuda.synchronize(dev)
            tot += e0.elapsed_time(e1)
    return shard.max_over_ranks(tot / steps, device=dev)


def bk_team_text(bk):
    v = __import__("ctypes").c_int(0)
    bk.lib().blink_get_option(bk.OPT_FUSED_TEAM, __import__("ctypes").byref(v))
    return "auto (cost model of blink_fused_kernel.cuh)" if v.value == 0 else f"forced {v.value} CTAs per image"


def config_leg(bk, cfg, T, dev, world, rank, steps, warmup, peak):
    """One short timed leg of BASELINE.json config `cfg` through blink_image (device-resident inputs)."""
    w = workloads.make_config(cfg, device=dev, T=T, seed=shard.rank_seed(cfg, rank))
    Tn, C, P, B, N = w.T, w.C, w.P, w.B, w.n_pix
    n_img = Tn * C * P
    image = torch.empty((n_img, N, N), dtype=torch.float32, device=dev)
    wsum = torch.empty(Tn * C, dtype=torch.float32, device=dev)
    rec, _ = bk.blink_workspace_bytes(bk.OP_IMAGE, Tn, C, P, B, N, w.weighting)
    ws = torch.empty(max(rec, 256), dtype=torch.uint8, device=dev)
    run = lambda: bk.blink_image(w.vis, w.uvw_m, w.freqs_hz, N, w.pixscale_rad, w.weighting, image=image, workspace=ws, wsum=wsum)
    small = n_img * N * N * 4 < (512 << 20)                     # outputs that would sit in the 126 MB L2: flush between calls
    flush = torch.zeros(256 << 20, dtype=torch.uint8, device=dev) if small else None
    l0 = bk.kernel_launches()
    ms = timed_ms(run, steps, warmup, dev, world, flush)
    launches = (bk.kernel_launches() - l0) // (steps + warmup)
    mb = model_bytes(Tn, C, P, B, N)
    shp = workloads.config_shape(cfg)
    out = {"workload": f"config{cfg}: {Tn} of {shp['T']} timesteps x {C} channels x {P} pol = {n_img} images of {N}x{N}, {B} baselines, "
                       f"{'natural' if w.weighting == 0 else 'uniform'} weighting",
           "ms_per_step": ms, "images_per_s": world * n_img / (ms * 1e-3), "gvis_per_s": world * n_img * B / (ms * 1e-3) / 1e9,
           "frac_M4": mb["M4"] / (ms * 1e-3) / 1e9 / peak, "model_speedup_M36": mb["M36"] / (ms * 1e-3) / 1e9 / peak,
           "team": bk_team_text(bk), "gpu_launches_per_step": int(launches), "l2": "flushed between timed calls (256 MB write)" if small else "outputs larger than L2; no flush"}
    if cfg == 1:
        out["us_per_image"] = ms * 1e3
        out["note"] = "one image: launch-latency bound, fractions not meaningful (SURVEY 8(d))"
    if Tn < shp["T"]:
        out["ms_full_config_extrapolated"] = ms * shp["T"] / Tn
    del image, ws, w
    torch.cuda.empty_cache()
    return out


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--config", type=int, default=3)
    ap.add_argument("--impl", default="blink")
    ap.add_argument("--path", type=int, default=0, help="BLINK_OPT_IMAGE_PATH: 0 auto, 1 unfused, 2 fused")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-cpu", action="store_true")
    ap.add_argument("--no-avg", action="store_true")
    ap.add_argument("--no-conv", action="store_true")
    ap.add_argument("--no-corr", action="store_true")
    ap.add_argument("--no-paper-size", action="store_true")
    ap.add_argument("--no-cufft", action="store_true")
    ap.add_argument("--no-configs", action="store_true", help="skip the timed legs of configs 1, 2, 4 (one timestep), 5")
    ap.add_argument("--conv-support", type=int, default=5, help="support of the gridding kernel timed in conv_mode (3, 5, 7)")
    ap.add_argument("--team", type=int, default=0, help="BLINK_OPT_FUSED_TEAM: CTAs per image in the fused kernel (0 = auto)")
    ap.add_argument("--T", type=int, default=None, help="reduce timesteps (debug only; invalidates the headline)")
    args = ap.parse_args()

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    if args.impl == "reference":
        run_reference(args, rank)
        return
    if args.warmup < 3:
        args.warmup = 3

    import torch.distributed as dist
    from paper_2505_15204_b200 import binding as bk
    torch.cuda.set_device(local_rank)
    dev = torch.device("cuda", local_rank)
    if world > 1:
        dist.init_process_group("nccl", device_id=dev)
    bk.lib()
    bk.set_option(bk.OPT_IMAGE_PATH, args.path)
    bk.set_option(bk.OPT_FUSED_TEAM, args.team)

    # independent batch per rank ("each second of observation can be processed independently")
    w = workloads.make_config(args.config, device=dev, T=args.T, seed=shard.rank_seed(args.config, rank))
    T, C, P, B, N = w.T, w.C, w.P, w.B, w.n_pix
    n_img = T * C * P
    image = torch.empty((n_img, N, N), dtype=torch.float32, device=dev)
    wsum = torch.empty(T * C, dtype=torch.float32, device=dev)
    rec, mn = bk.blink_workspace_bytes(bk.OP_IMAGE, T, C, P, B, N, w.weighting)
    ws = torch.empty(max(rec, 256), dtype=torch.uint8, device=dev)

    def step():
        bk.blink_image(w.vis, w.uvw_m, w.freqs_hz, N, w.pixscale_rad, w.weighting, image=image, workspace=ws, wsum=wsum)

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize(dev)

    sampler = ClockSampler(local_rank)
    if rank == 0:
        sampler.start()
    for _ in range(args.warmup):
        step()
    barrier()
    # same load, untimed, until nvidia-smi has delivered its first samples (bounded), so that the clocks line covers
    # the timed region that follows immediately
    t_wait = time.perf_counter()
    while rank == 0 and sampler.proc is not None and len(sampler.lines) < 2 and time.perf_counter() - t_wait < 4.0:
        step()
        torch.cuda.synchronize(dev)
    launches0 = bk.kernel_launches()
    ev = [torch.cuda.Event(enable_timing=True) for _ in range(args.steps + 1)]
    barrier()
    ev[0].record()
    for k in range(args.steps):
        step()
        ev[k + 1].record()
    barrier()
    launches = bk.kernel_launches() - launches0
    clocks = sampler.stop() if rank == 0 else None
    per_step = [ev[k].elapsed_time(ev[k + 1]) for k in range(args.steps)]
    total_ms = shard.max_over_ranks(ev[0].elapsed_time(ev[-1]), device=dev)      # slowest rank
    ms_per_step = total_ms / args.steps
    value = shard.aggregate_rate(n_img, world, ms_per_step)                      # whole job: every rank imaged n_img

    # ---- channel-averaged images (blink_image_avg), same inputs, device-resident -------
    avg = None
    if not args.no_avg:
        try:
            rec_a, _ = bk.blink_workspace_bytes(bk.OP_IMAGE_AVG, T, C, P, B, N, w.weighting)
            ws_a = torch.empty(max(rec_a, 16), dtype=torch.uint8, device=dev)
            img_a = torch.empty((T * P, N, N), dtype=torch.float32, device=dev)
            run_a = lambda: bk.blink_image_avg(w.vis, w.uvw_m, w.freqs_hz, N, w.pixscale_rad, w.weighting, avg_time=False,
                                               image_avg=img_a, workspace=ws_a, wsum=wsum)
            for _ in range(args.warmup):
                run_a()
            barrier()
            l0 = bk.kernel_launches()
            ea = [torch.cuda.Event(enable_timing=True) for _ in range(2)]
            ea[0].record()
            for _ in range(args.steps):
                run_a()
            ea[1].record()
            barrier()
            ms_a = torch.tensor([ea[0].elapsed_time(ea[1]) / args.steps], device=dev)
            if world > 1:
                dist.all_reduce(ms_a, op=dist.ReduceOp.MAX)
            ms_a = float(ms_a.item())
            bytes_a = n_img * 8 * B + 12 * T * B + T * P * 4 * N * N
            avg = {"api": "blink_image_avg (mean over the C channels of every timestep; PAPER.md L284)",
                   "ms_per_step": ms_a, "images_in_per_s": world * n_img / (ms_a * 1e-3),
                   "gvis_per_s": world * n_img * B / (ms_a * 1e-3) / 1e9, "images_out": T * P,
                   "gpu_launches_per_step": (bk.kernel_launches() - l0) // args.steps,
                   "algorithmic_bytes_per_step": bytes_a, "model": "n_img*8B + 12TB + T*P*4N^2 (vis + uvw read once, averaged images written)",
                   "hbm_gbs": bytes_a / (ms_a * 1e-3) / 1e9}
            del ws_a, img_a
            # the same call with UNIFORM weighting on one timestep of BASELINE config 4 (768 channels x 4 planes of 2048^2,
            # 10296 baselines): the column route of DESIGN.md 5.4 (per-sample weights by counting grid columns in shared memory)
            if args.T is None and rank == 0:
                w4 = workloads.make_config(4, device=dev, T=1)
                T4, C4, P4, B4 = w4.vis.shape
                rec4, _ = bk.blink_workspace_bytes(bk.OP_IMAGE_AVG, T4, C4, P4, B4, w4.n_pix, w4.weighting)
                ws4 = torch.empty(max(rec4, 16), dtype=torch.uint8, device=dev)
                img4 = torch.empty((T4 * P4, w4.n_pix, w4.n_pix), dtype=torch.float32, device=dev)
                wsum4 = torch.empty((T4 * C4,), dtype=torch.float32, device=dev)
                run4 = lambda: bk.blink_image_avg(w4.vis, w4.uvw_m, w4.freqs_hz, w4.n_pix, w4.pixscale_rad, w4.weighting,
                                                  avg_time=False, image_avg=img4, workspace=ws4, wsum=wsum4)
                for _ in range(args.warmup):
                    run4()
                e4 = [torch.cuda.Event(enable_timing=True) for _ in range(2)]
                e4[0].record()
                for _ in range(args.steps):
                    run4()
                e4[1].record()
                torch.cuda.synchronize()
                ms4 = e4[0].elapsed_time(e4[1]) / args.steps
                avg["uniform_config4_one_timestep"] = {"ms_per_step": ms4, "images_in": T4 * C4 * P4, "images_out": T4 * P4,
                                                        "gvis_per_s": T4 * C4 * P4 * B4 / (ms4 * 1e-3) / 1e9}
                del w4, ws4, img4, wsum4
        except Exception as ex:  # report, never hide
            avg = {"error": str(ex)[:200]}

    # ---- same-box context for the FFT step alone (the paper's FFT is the vendor library call, L194): cuFFT batched
    # C2C inverse through torch.fft.ifft2 on already materialised grids; bench-only comparator, not linked into libblinkimg,
    # not the oracle, no shift / normalisation / real part (those are extra passes for a library FFT)
    cufft = None
    if not args.no_cufft and rank == 0:
        try:
            nb = int(min(n_img, max(1, (4 << 30) // (N * N * 8))))
            g = torch.randn((nb, N, N, 2), device=dev, dtype=torch.float32)
            gc_ = torch.view_as_complex(g)
            for _ in range(2):
                torch.fft.ifft2(gc_)
            torch.cuda.synchronize()
            ef = [torch.cuda.Event(enable_timing=True) for _ in range(2)]
            ef[0].record()
            for _ in range(5):
                out_f = torch.fft.ifft2(gc_)
            ef[1].record()
            torch.cuda.synchronize()
            ms_f = ef[0].elapsed_time(ef[1]) / 5
            cufft = {"api": "torch.fft.ifft2 (cuFFT batched C2C, complex64, out of place)", "batch": nb,
                     "ms_per_batch": ms_f, "ms_per_step_extrapolated": ms_f * n_img / nb,
                     "images_per_s": nb / (ms_f * 1e-3), "note": "FFT only, on materialised grids; context, not a target"}
            del g, gc_, out_f
        except Exception as ex:
            cufft = {"error": str(ex)[:200]}

    # ---- convolutional gridding (blink_image_conv), same inputs and outputs -------------------
    conv = None
    if not args.no_conv and w.weighting == 0:
        try:
            S = args.conv_support
            rec_c, _ = bk.blink_workspace_bytes(bk.OP_IMAGE_CONV, T, C, P, B, N, 0)
            ws_c = torch.empty(max(rec_c, 16), dtype=torch.uint8, device=dev)
            run_c = lambda: bk.blink_image_conv(w.vis, w.uvw_m, w.freqs_hz, N, w.pixscale_rad, S, image=image,
                                                workspace=ws_c, wsum=wsum)
            for _ in range(args.warmup):
                run_c()
            barrier()
            ec = [torch.cuda.Event(enable_timing=True) for _ in range(2)]
            ec[0].record()
            for _ in range(args.steps):
                run_c()
            ec[1].record()
            barrier()
            ms_c = torch.tensor([ec[0].elapsed_time(ec[1]) / args.steps], device=dev)
            if world > 1:
                dist.all_reduce(ms_c, op=dist.ReduceOp.MAX)
            ms_c = float(ms_c.item())
            conv = {"api": f"blink_image_conv (Kaiser-Bessel, support {S}, beta {2.34 * S:.2f}; PAPER.md L192, L351; DESIGN.md R16)",
                    "support": S, "ms_per_step": ms_c, "images_per_s": world * n_img / (ms_c * 1e-3),
                    "gvis_per_s": world * n_img * B / (ms_c * 1e-3) / 1e9,
                    "g_tap_cells_per_s": world * n_img * B * S * S * 2 / (ms_c * 1e-3) / 1e9,
                    "frac_M4": (n_img * (4 * N * N + 8 * B) + 12 * T * B) / (ms_c * 1e-3) / 1e9 / hbm_peak()[0]}
            del ws_c
        except Exception as ex:  # report, never hide
            conv = {"error": str(ex)[:200]}

    # ---- the paper's own image side, 1200 x 1200 (Table 6) -----------
    # the same visibilities through blink_image's generic (mixed-radix, unfused) chain; 2 of the 50 timesteps per
    # timed run (1536 images, 8.8 GB of images > L2), scaled to the 38400 images of one second of data
    paper = None
    if not args.no_paper_size and args.config == 3 and args.T is None and w.weighting == 0:
        try:
            NP, TP = 1200, 2
            vis_p, uvw_p = w.vis[:TP].contiguous(), w.uvw_m[:TP].contiguous()
            img_p = image.view(-1)[:TP * C * P * NP * NP].view(TP * C * P, NP, NP)
            rec_p, _ = bk.blink_workspace_bytes(bk.OP_IMAGE, TP, C, P, B, NP, 0)
            ws_p = torch.empty(max(rec_p, 16), dtype=torch.uint8, device=dev)
            wsum_p = torch.empty(TP * C, dtype=torch.float32, device=dev)
            run_p = lambda: bk.blink_image(vis_p, uvw_p, w.freqs_hz, NP, 0.6 / NP, 0, image=img_p, workspace=ws_p, wsum=wsum_p)
            for _ in range(args.warmup):
                run_p()
            barrier()
            ep = [torch.cuda.Event(enable_timing=True) for _ in range(2)]
            ep[0].record()
            for _ in range(args.steps):
                run_p()
            ep[1].record()
            barrier()
            ms_p = torch.tensor([ep[0].elapsed_time(ep[1]) / args.steps], device=dev)
            if world > 1:
                dist.all_reduce(ms_p, op=dist.ReduceOp.MAX)
            ms_p = float(ms_p.item())
            n_p = TP * C * P
            m36 = n_p * (36 * NP * NP + 8 * B) + 12 * TP * B
            m4 = n_p * (4 * NP * NP + 8 * B) + 12 * TP * B
            paper = {"api": "blink_image at n_pix = 1200 (fused kernel of the paper's side, blink_fused_g.cu: 15 x 5 x 16 register-resident stages)",
                     "images_per_run": n_p, "ms_per_run": ms_p, "images_per_s": world * n_p / (ms_p * 1e-3),
                     "s_per_second_of_data": ms_p * 1e-3 * (T / TP),
                     "frac_M4": m4 / (ms_p * 1e-3) / 1e9 / hbm_peak()[0], "model_speedup_M36": m36 / (ms_p * 1e-3) / 1e9 / hbm_peak()[0],
                     "paper_context": "PAPER.md Table 6 (L339-340), gridding + 2D FFT of 38400 images of 1200^2: 1.77 s on an H100 (cuFFT), "
                                      "7.09 s on an MI250X GCD (rocFFT); other machines: context, not a target"}
            # the same images with a Kaiser-Bessel gridding kernel (blink_image_conv inside the fused 1200 kernel)
            S_p = args.conv_support
            rec_c, _ = bk.blink_workspace_bytes(bk.OP_IMAGE_CONV, TP, C, P, B, NP, 0)
            ws_c = torch.empty(max(rec_c, 16), dtype=torch.uint8, device=dev)
            run_pc = lambda: bk.blink_image_conv(vis_p, uvw_p, w.freqs_hz, NP, 0.6 / NP, S_p, image=img_p, workspace=ws_c, wsum=wsum_p)
            for _ in range(args.warmup):
                run_pc()
            barrier()
            ec = [torch.cuda.Event(enable_timing=True) for _ in range(2)]
            ec[0].record()
            for _ in range(args.steps):
                run_pc()
            ec[1].record()
            barrier()
            ms_pc = torch.tensor([ec[0].elapsed_time(ec[1]) / args.steps], device=dev)
            if world > 1:
                dist.all_reduce(ms_pc, op=dist.ReduceOp.MAX)
            paper["conv"] = {"api": f"blink_image_conv at n_pix = 1200, support {S_p}", "ms_per_run": float(ms_pc.item())}
            del ws_p, ws_c, vis_p, uvw_p, img_p
        except Exception as ex:  # report, never hide
            paper = {"error": str(ex)[:200]}

    # ---- SURVEY 8(f) rank 4 (last item): CMAC correlator on the int8 tensor cores (blink_correlate) --------------
    # one second of MWA Phase I voltages: 3072 fine channels of 10 kHz x 256 inputs x 10000
    # samples, correlated at 20 ms / 40 kHz -> 50 x 768 lower-triangular matrices (the visibilities config 3 images)
    corr = None
    if not args.no_corr and args.T is None:
        try:
            Fc, Ac, Nsc, n_t, n_avg = 3072, 256, 10000, 200, 4
            volt = torch.empty((Fc, Ac, Nsc, 2), dtype=torch.int8, device=dev)
            for f0 in range(0, Fc, 256):
                volt[f0:f0 + 256] = workloads.make_voltages(256, Ac, Nsc, seed=7000 + 100 * rank + f0, device=dev)
            visc = torch.empty((Nsc // n_t, Fc // n_avg, Ac * (Ac + 1) // 2), dtype=torch.complex64, device=dev)
            run_k = lambda: bk.blink_correlate(volt, n_t, n_avg, vis=visc)
            for _ in range(args.warmup):
                run_k()
            barrier()
            ek = [torch.cuda.Event(enable_timing=True) for _ in range(2)]
            ek[0].record()
            for _ in range(args.steps):
                run_k()
            ek[1].record()
            barrier()
            ms_k = torch.tensor([ek[0].elapsed_time(ek[1]) / args.steps], device=dev)
            if world > 1:
                dist.all_reduce(ms_k, op=dist.ReduceOp.MAX)
            ms_k = float(ms_k.item())
            n_mat = (Nsc // n_t) * (Fc // n_avg)
            cmacs = n_mat * (Ac * (Ac + 1) // 2) * n_t * n_avg
            # int8 multiply-adds the tensor cores are asked for: 3 tiles of 128 x 256 x (13 K-steps of 32 bytes per fine channel)
            issued_ops = 2 * n_mat * 3 * 128 * 256 * (13 * 32) * n_avg
            pk = json.load(open(os.path.join(ROOT, "MEASURED_PEAKS.json"))) if os.path.exists(os.path.join(ROOT, "MEASURED_PEAKS.json")) else {}
            i8_peak = 2.0 * float(pk.get("bf16_tflops", 2250.0 * 0.725))
            corr = {"api": "blink_correlate (tcgen05.mma kind::i8; PAPER.md eq. 3, L172-178; DESIGN.md R17)",
                    "workload": f"{Fc} fine channels x {Ac} inputs x {Nsc} samples (1 s of MWA Phase I VCS data), n_t {n_t}, n_avg {n_avg}",
                    "ms_per_step": ms_k, "seconds_of_data_per_s": world / (ms_k * 1e-3),
                    "tcmac_per_s": world * cmacs / (ms_k * 1e-3) / 1e12,
                    "roofline": {"bound": "tensor", "achieved": world * issued_ops / (ms_k * 1e-3) / 1e12, "unit": "TOP/s (int8)",
                                 "peak": i8_peak, "frac": issued_ops / (ms_k * 1e-3) / 1e12 / i8_peak,
                                 "peak_source": "2 x MEASURED_PEAKS.json bf16_tflops (nominal int8 : bf16 ratio)",
                                 "useful_frac": 8 * cmacs / (ms_k * 1e-3) / 1e12 / i8_peak},
                    "hbm_gbs": (volt.numel() + visc.numel() * 8) / (ms_k * 1e-3) / 1e9}
            if rank == 0 and not args.no_cpu:
                # the CPU oracle on a bounded sample of the same workload: 64 (t, c) matrices (32896 entries x 800 products each)
                import oracle
                sub = volt[:64 * n_avg, :, :n_t].contiguous().cpu().numpy()
                t0 = time.perf_counter()
                oracle.correlate(sub, n_t, n_avg)
                dt = time.perf_counter() - t0
                corr["cpu_baseline"] = {"value": 64 / dt / n_mat, "unit": "seconds of data/s", "cores": 1, "kind": "oracle",
                                        "sample": f"64 of the {n_mat} (interval, channel) matrices in {dt:.2f} s, one thread"}
            del volt, visc
        except Exception as ex:  # report, never hide
            corr = {"error": str(ex)[:200]}

    # ---- end to end through the host-buffer entry point (rank-local, then max over ranks) -----------------
    e2e = None
    if not args.no_e2e:
        try:
            vis_h = torch.empty(w.vis.shape, dtype=torch.complex64, pin_memory=True)
            vis_h.copy_(w.vis)
            uvw_h = torch.empty(w.uvw_m.shape, dtype=torch.float32, pin_memory=True)
            uvw_h.copy_(w.uvw_m)
            img_h = torch.empty((n_img, N, N), dtype=torch.float32, pin_memory=True)
            wsum_h = torch.empty(T * C, dtype=torch.float32, pin_memory=True)
            rec_h, _ = bk.blink_workspace_bytes(bk.OP_IMAGE_HOST, T, C, P, B, N, w.weighting)
            image = None                                          # config 3's 40 GB of device images: not needed any more
            torch.cuda.empty_cache()
            ws_h = torch.empty(rec_h, dtype=torch.uint8, device=dev)
            e_steps = max(1, min(args.steps, 3))
            bk.blink_image_host(vis_h, uvw_h, w.freqs_hz, N, w.pixscale_rad, w.weighting, img_h, wsum_h, ws_h)  # warm-up
            barrier()
            t0 = time.perf_counter()
            for _ in range(e_steps):
                bk.blink_image_host(vis_h, uvw_h, w.freqs_hz, N, w.pixscale_rad, w.weighting, img_h, wsum_h, ws_h)
            barrier()
            dt = torch.tensor([(time.perf_counter() - t0) / e_steps], device=dev)
            if world > 1:
                dist.all_reduce(dt, op=dist.ReduceOp.MAX)
            e2e = {"value": world * n_img / float(dt.item()), "unit": "images/s",
                   "h2d_bytes_per_step": int(vis_h.numel() * 8 + uvw_h.numel() * 4),
                   "d2h_bytes_per_step": int(img_h.numel() * 4 + wsum_h.numel() * 4),
                   "steps": e_steps, "ms_per_step": float(dt.item()) * 1e3,
                   "d2h_gbs": float((img_h.numel() * 4 + wsum_h.numel() * 4) / float(dt.item()) / 1e9),
                   "bound": "PCIe device->host: the images are 16x the visibilities; a pinned 2 GiB cudaMemcpy on the same kind of box "
                            "measures 54.1 GB/s device->host alone (DESIGN.md 5.3)",
                   "api": "blink_image_host (pinned host buffers, per-timestep H2D/compute/D2H pipeline)"}
            del img_h, vis_h, ws_h
        except Exception as ex:  # report, never hide
            e2e = {"value": None, "unit": "images/s", "error": str(ex)[:200]}

    # ---- the other configs, driver-timed (1, 2 and 5 whole; 4 = one of its 10 timesteps, 51.5 GB of images) ----
    configs = None
    if not args.no_configs and args.T is None and args.path == 0:
        image = None
        del ws
        torch.cuda.empty_cache()
        configs = {}
        for cfg, Tc in ((1, None), (2, None), (4, 1), (5, None)):
            if cfg == args.config:
                continue
            try:
                configs[f"config{cfg}"] = config_leg(bk, cfg, Tc, dev, world, rank, max(3, min(args.steps, 10)), args.warmup, hbm_peak()[0])
            except Exception as ex:  # report, never hide
                configs[f"config{cfg}"] = {"error": str(ex)[:200]}

    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return

    mb = model_bytes(T, C, P, B, N)
    peak, peak_src = hbm_peak()
    kern_ms = float(np.mean(per_step))
    fused = args.path != 1
    # The fused kernel never materialises the uv grid, so the bytes it MUST move are M4 (visibilities in, images out); the
    # unfused chain (--path 1) really moves M36.  M36 / M20 of SURVEY 8(d) stay as labelled model-speedup numbers.
    model = "M4" if fused else "M36"
    achieved = mb[model] / (kern_ms * 1e-3) / 1e9
    roofline = {"bound": "hbm", "achieved": achieved, "peak": peak, "unit": "GB/s", "frac": achieved / peak,
                "traffic": None, "peak_source": peak_src,
                "kernel": "fused_image_kernel (+ presort_kernel, < 0.1 % of the step): CUDA events on the launch stream over the timed region"
                          if fused else "grid_tiles_kernel + fft_rows_kernel + fft_cols_kernel (CUDA events on the launch stream)",
                "algorithmic_bytes_per_step": mb[model],
                "model": ("M4 = n_img*(4 N^2 + 8 B) + 12 T B: visibilities and uvw read once, images written (the grid never reaches HBM)"
                          if fused else "M36 = n_img*(36 N^2 + 8 B) + 12 T B (SURVEY 8(d): grid written, read and rewritten by two passes)"),
                "frac_M4": mb["M4"] / (kern_ms * 1e-3) / 1e9 / peak,
                "model_speedup_M36": mb["M36"] / (kern_ms * 1e-3) / 1e9 / peak,
                "model_speedup_M20": mb["M20"] / (kern_ms * 1e-3) / 1e9 / peak,
                "kernel_ms": kern_ms,
                "note": "frac is against the compulsory bytes of the implementation timed.  model_speedup_M36 / _M20 divide SURVEY 8(d)'s "
                        "contract models (three unfused kernels / gridder fused into the row pass) by the same time and peak: values above 1 "
                        "mean traffic the fusion removed, they are not roofline fractions."}
    prof = os.path.join(ROOT, "profiles", "traffic.csv")      # stored ncu figures of a committed capture (NOT measured by this run)
    if os.path.exists(prof):
        try:
            import csv
            key = f"config{args.config}_path{args.path}"
            for row in csv.DictReader(open(prof)):
                if row["key"] == key and args.T is None:
                    roofline["traffic"] = int(row["dram_bytes_per_step"])
                    roofline["traffic_is"] = "STORED ncu figure (dram__bytes_read.sum + dram__bytes_write.sum of one --set full capture), not measured by this run"
                    roofline["traffic_source"] = row["source"]
                    roofline["traffic_over_algorithmic"] = int(row["dram_bytes_per_step"]) / mb[model]
                    if row.get("limiter"):
                        roofline["limiter_stored_ncu"] = row["limiter"]
        except Exception:
            pass
    if avg and "hbm_gbs" in avg:
        avg["frac_of_hbm_peak"] = avg["hbm_gbs"] / peak
    cpu = None
    if not args.no_cpu:
        cores = os.cpu_count() or 1
        cpu = cpu_oracle_leg(sample_workload(args.config, 32 * cores))
    out = {
        "metric": "dirty_images_per_s", "value": value, "unit": "images/s", "n_gpus": world, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": ms_per_step, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f32", "data": "synthetic",
        "config": {"workload": f"config{args.config}: {T} timesteps x {C} channels x {P} pol = {n_img} images of {N}x{N}, "
                               f"{B} baselines, {'natural' if w.weighting == 0 else 'uniform'} weighting",
                   "per_gpu_images": n_img, "l2": "inputs (vis %.2f GB) and outputs (%.1f GB) larger than L2; no flush" %
                   (w.vis.numel() * 8 / 1e9, n_img * N * N * 4 / 1e9),
                   "image_path": args.path, "parallelism": f"independent batches x{world}"},
        "gvis_per_s": value * B / 1e9,
        "clocks": clocks, "e2e": e2e, "gpu_launches": int(launches), "roofline": roofline, "cpu_baseline": cpu, "avg_mode": avg, "conv_mode": conv, "paper_size_mode": paper, "corr_mode": corr, "cufft_context": cufft, "configs": configs,
        "ms_per_step_each": per_step,
    }
    print(json.dumps(out))
    if world > 1:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
