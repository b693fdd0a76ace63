#!/usr/bin/env python
"""bench.py -- rendered FPS over the config-3 trajectory (3 M Gaussians, 1080p): TemporalGS (AUTO schedule)
and full render every frame, on the CUDA path through the C-ABI (BASELINE.json: metric).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config 3] [--impl ours|reference]

A step = one frame of the trajectory = one pass of the whole hot path (A0-A10 of DESIGN.md §1).  With N > 1
(torchrun) every rank renders the same trajectory on its own GPU: the path does not shard ("replicas only",
DESIGN.md §8), so `value` is the sum of the ranks' frames over the slowest rank's time ("weak").
`--impl reference` times the CPU oracle as it stands on the host cores (rank 0 only).
Prints ONE JSON line (rank 0).
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
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "rendered FPS over trajectory (3M Gaussians, 1080p); speed-up vs full render"
# Lane-instructions one alive (pixel, Gaussian) interaction of the blend needs: 9.5 on the FMA pipe
# (exponent 2, weight, update of T', 3 colour FMAs, 2 moment FMAs; per run of 4 pixels d - d_ref, its square and the sum of
# the weights, 1/4 each; a packed FFMA2 half counts as 1) + 1 MUFU.EX2 + 3.5 on the ALU pipe (stop test, 2 selects; per run
# the any-pixel-composited test and the select of d_ref).
BLEND_LANE_INSTR = 14.0
# dram__bytes_read.sum + dram__bytes_write.sum of one one-piece k_blend<1,0,0,0> launch on config 3, from the ncu --set full capture
# summarised in profiles/r2z_top_kernels.md (the file names the command); per launch, like `achieved`.
BLEND_DRAM_TRAFFIC_BYTES = 35.8e6
BLEND_DRAM_TRAFFIC_SOURCE = "ncu --set full capture of one-piece k_blend<1,0,0,0> launches on config 3 (profiles/r2z_top_kernels.md: 35.0-35.8 MB), not re-measured by this run"
# Lane-instructions the pair binning needs: per (Gaussian, tile) test the tile coordinates and box (8), the
# selection bit (4), centre-in-box (5), four box edges of the conic form at the clamped optimum (4 x 12) and the margin
# compare (3) = 68; per emitted pair the rank, the staging and the two stores (12).
BIN_LANE_INSTR_PER_TEST = 68.0
BIN_LANE_INSTR_PER_PAIR = 12.0


def _peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        d = json.load(open(p))
        return float(d.get("hbm_gbs", 6650.0)), float(d.get("sm_max_mhz", 1965.0)), "measured"
    return 6650.0, 1965.0, "fallback"


class ClockSampler:
    """nvidia-smi clocks + throttle reasons during the timed region (B200_PROFILING.md recipe)."""

    Q = ("clocks.sm,clocks.max.sm,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        self.index = index
        self.proc = None
        self.lines = []

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(self.index), f"--query-gpu={self.Q}",
                                          "--format=csv,noheader,nounits", "-lms", "100"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            threading.Thread(target=self._pump, daemon=True).start()
        except Exception:
            self.proc = None

    def _pump(self):
        for line in self.proc.stdout:
            self.lines.append(line.strip())

    def stop(self):
        if self.proc:
            time.sleep(0.12)
            self.proc.terminate()
        sm, mx, reasons = [], 0.0, set()
        for ln in self.lines:
            f = [x.strip() for x in ln.split(",")]
            if len(f) < 6:
                continue
            try:
                sm.append(float(f[0])); mx = max(mx, float(f[1]))
            except ValueError:
                continue
            for name, v in zip(("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"), f[2:6]):
                if v.lower().startswith("active"):
                    reasons.add(name)
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": mx or None, "reasons": sorted(reasons),
                "samples": len(sm)}


def max_over_ranks(ms, world, device=None):
    """Replicas only: the job's time for K frames per rank is the slowest rank's device time."""
    if world <= 1:
        return float(ms)
    import torch
    import torch.distributed as dist
    t = torch.tensor([float(ms)], dtype=torch.float64, device=device or "cpu")
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def aggregate_fps(world, steps, ms):
    """Whole-job frames per second of `world` replicas that each rendered `steps` frames in `ms` (max over ranks)."""
    return world * steps / (ms * 1e-3)


def trajectory_pose(sc, f):
    """Frame f of an endless smooth trajectory: the config's poses played forward, then backward, ..."""
    F = len(sc.poses)
    k = f % (2 * F - 2) if F > 1 else 0
    return sc.poses[k if k < F else 2 * F - 2 - k]


def _ssim(a, b):
    """Mean SSIM of two [H][W][3] images in [0,1] (the paper's second quality metric, L138): Gaussian window sigma 1.5,
    C1 = 0.01^2, C2 = 0.03^2, per channel, on the host with scipy.  Reported only (quality is unpinned)."""
    from scipy.ndimage import gaussian_filter
    a, b = a.astype(np.float64), b.astype(np.float64)
    f = lambda x: gaussian_filter(x, sigma=(1.5, 1.5, 0), truncate=3.5)
    ma, mb = f(a), f(b)
    va, vb, cab = f(a * a) - ma * ma, f(b * b) - mb * mb, f(a * b) - ma * mb
    c1, c2 = 0.01 ** 2, 0.03 ** 2
    return float((((2 * ma * mb + c1) * (2 * cab + c2)) / ((ma * ma + mb * mb + c1) * (va + vb + c2))).mean())


STAGE_NAMES = ["init_warp_fill", "preprocess_select", "depth_sort", "bin_pairs", "sh_colour", "tile_sort_ranges", "blend_stitch", "post"]


def workload_string(sc, config):
    cam = sc.camera
    return (f"config {config} ({sc.name}): {sc.n} Gaussians, SH degree {sc.sh_degree}, {cam.W}x{cam.H}, {len(sc.poses)}-frame trajectory "
            f"played forward/backward, AUTO schedule (lambda_TDC=50, lambda_SR=5, eta=0.4)")


def stage_rooflines(stats, sc, hbm_gbs, alu_peak):
    """Achieved fraction of the roofline that bounds each stage (DESIGN.md §7.1 derives the units), for a list of frame
    statistics of ONE frame type.  Algorithmic bytes / needed lane-instructions come from the frames' own counters, the
    time from the stage events (single stream, kernel boundaries and launch gaps included)."""
    if not stats:
        return None
    cam = sc.camera
    mean = lambda key: float(np.mean([s[key] for s in stats]))
    t = np.mean([s["ms_stage"] for s in stats], axis=0) * 1e-3
    P, Nv, L, nt = mean("n_pairs"), mean("n_visible"), mean("n_interactions"), mean("n_tests_evaluated")   # tests really evaluated (slabs skip dead tiles)
    ftype = stats[0]["frame_type"]
    T_ = ((cam.W + 15) // 16) * ((cam.H + 15) // 16)
    tile_passes = (max(1, int(np.ceil(np.log2(T_)))) + 7) // 8
    K = (sc.sh_degree + 1) ** 2
    px = cam.W * cam.H
    # init + A1 warp + A2 fill: S frames 8 B/px init + 8 B/px read + 2 atomics (8 B) + 4 B read + 4 B written; R / P frames
    # only zero G_rendered' (N bytes) and a few words per tile
    init_bytes = (32.0 * px if ftype == 2 else float(sc.n)) + 25.0 * T_
    rows = {
        "init_warp_fill": ("hbm", init_bytes / 1e9, "GB"),
        "preprocess_select": ("hbm", (sc.n * (16 + 1) + Nv * (32 + 16 + 73)) / 1e9, "GB"),   # g2 + TGB lookups; written per visible Gaussian: A5a record 32, blend record 32, flag 1, staged key / index 8
        "depth_sort": ("hbm", Nv * 16 * 4 / 1e9, "GB"),
        "bin_pairs": ("alu", (nt * BIN_LANE_INSTR_PER_TEST + P * BIN_LANE_INSTR_PER_PAIR) / 1e12, "T lane-instr"),
        "sh_colour": ("hbm", Nv * (4 + 16 + 12 * K + 16) / 1e9, "GB"),
        "tile_sort_ranges": ("hbm", P * 16 * tile_passes / 1e9, "GB"),
        "blend_stitch": ("alu", L * BLEND_LANE_INSTR / 1e12, "T lane-instr"),
    }
    out = {}
    for i, name in enumerate(STAGE_NAMES[:7]):
        bound, work, unit = rows[name]
        peak = hbm_gbs if bound == "hbm" else alu_peak
        ach = work / t[i] if t[i] > 0 else 0.0
        out[name] = {"bound": bound, "ms": float(t[i] * 1e3), "achieved": ach, "peak": peak, "unit": unit + "/s", "frac": ach / peak}
    return out


def summarise(lst):
    if not lst:
        return None
    ms = np.mean([s["ms_stage"] for s in lst], axis=0)
    m = lambda key: float(np.mean([s[key] for s in lst]))
    return {"frames": len(lst), "ms_total": m("ms_total"), "ms_stage": {n: float(v) for n, v in zip(STAGE_NAMES, ms)},
            "n_pairs": m("n_pairs"), "n_tests": m("n_tests"), "n_tests_evaluated": m("n_tests_evaluated"), "n_visible": m("n_visible"),
            "n_sel_frac": float(np.mean([s["n_sel"] / s["n_tiles"] for s in lst])),
            "n_interactions": m("n_interactions"), "n_blended": m("n_blended"), "n_pixel_slots": m("n_pixel_slots"), "n_pairs_consumed": m("n_pairs_consumed")}


class Harness:
    """One scene on one GPU: timed frame loops (CUDA events on the context's stream), the per-stage pass, quality."""

    def __init__(self, tgs, torch, sc, local, world, warmup, depth_slabs=0):
        self.tgs, self.torch, self.sc, self.world, self.W = tgs, torch, sc, world, warmup
        self.stream = torch.cuda.Stream()
        self.ctx = tgs.Context(local, self.stream.cuda_stream)
        self.ctx.load_scene(sc)                         # scene resident in HBM before any timed region
        self.local = local
        self.depth_slabs = depth_slabs
        if depth_slabs:
            p = self.ctx.default_params(); p.depth_slabs = depth_slabs; self.ctx.set_params(p)

    def barrier(self):
        self.torch.cuda.synchronize()
        if self.world > 1:
            import torch.distributed as dist
            dist.barrier()
        self.torch.cuda.synchronize()

    def timed(self, mode, steps, readback=None):
        """Device time (ms, max over ranks) of `steps` frames of the trajectory, after W untimed warm-up frames."""
        torch, ctx, sc, cam = self.torch, self.ctx, self.sc, self.sc.camera
        ctx.reset_priors()
        for f in range(self.W):
            ctx.set_camera(trajectory_pose(sc, f), cam)
            ctx.render(mode)
        ctx.reset_priors()
        self.barrier()
        l0 = ctx.get_stats(check=False)["launches_total"]
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        with torch.cuda.stream(self.stream):
            e0.record(self.stream)
            for f in range(steps):
                ctx.set_camera(trajectory_pose(sc, f), cam)
                ctx.render(mode)
                if readback is not None:
                    ctx.read_image_async(readback[f & 1])   # device -> pinned host on the copy stream, overlaps the next frame
            if readback is not None:
                ctx.wait_reads()                    # every frame's image is on the host before the clock stops
            e1.record(self.stream)
        self.barrier()
        self.launches = ctx.get_stats(check=False)["launches_total"] - l0
        return max_over_ranks(e0.elapsed_time(e1), self.world, "cuda")

    def stage_pass(self, frames):
        """(a) stage events with the production instances of every kernel, everything on ONE stream so that the events
        bracket what they name (the production frame overlaps A2 / A4 / SH colours on side streams and is shorter than the
        sum); (b) the same frames with the counting instances of the blend (never timed): L, composited interactions and
        pixel slots are properties of the frames and are merged into the statistics of pass (a)."""
        tgs, ctx, sc, cam = self.tgs, self.ctx, self.sc, self.sc.camera
        ctx.debug_run_stage("timing_on")
        ctx.reset_priors()
        timed_stats = []
        for f in range(frames):
            ctx.set_camera(trajectory_pose(sc, f), cam)
            ctx.render(tgs.AUTO)
            timed_stats.append(ctx.get_stats())
        ctx.debug_run_stage("timing_off")
        ctx.debug_run_stage("count_interactions_on")
        ctx.reset_priors()
        per_type = {0: [], 1: [], 2: []}
        # pass (b) renders every frame in as many pieces as pass (a) did (the library's automatic choice depends on what it
        # has seen before, and the priors of one and two pieces differ in the last bits): the frames are then the same frames
        p = ctx.default_params()
        for f in range(frames):
            st = timed_stats[f]
            p.depth_slabs = int(st["n_slabs"])
            ctx.set_params(p)
            ctx.set_camera(trajectory_pose(sc, f), cam)
            ctx.render(tgs.AUTO)
            cs = ctx.get_stats()
            assert st["frame_type"] == cs["frame_type"] and st["n_visible"] == cs["n_visible"], (f, st["frame_type"], cs["frame_type"], st["n_visible"], cs["n_visible"])
            for key in ("n_interactions", "n_blended", "n_pixel_slots", "n_pairs_consumed"):
                st[key] = cs[key]
            per_type[st["frame_type"]].append(st)
        p.depth_slabs = self.depth_slabs
        ctx.set_params(p)
        ctx.debug_run_stage("count_interactions_off")
        return per_type

    def quality(self, frames):
        """PSNR / SSIM of the S frames against the full render of the same pose (reported; unpinned by the paper)."""
        tgs, ctx, sc, cam = self.tgs, self.ctx, self.sc, self.sc.camera
        psnr, ssim = [], []
        ctx.reset_priors()
        ref = tgs.Context(self.local, self.stream.cuda_stream)
        ref.load_scene(sc)
        for f in range(frames):
            ctx.set_camera(trajectory_pose(sc, f), cam)
            ctx.render(tgs.AUTO)
            if ctx.get_stats()["frame_type"] == tgs.FRAME_S:
                ref.set_camera(trajectory_pose(sc, f), cam)
                ref.render(tgs.FULL)
                a, b = ctx.read_image(), ref.read_image()
                mse = float(((a - b) ** 2).mean())
                psnr.append(10 * np.log10(1.0 / max(mse, 1e-12)))
                if len(ssim) < 3:
                    ssim.append(_ssim(a, b))
        ref.destroy()
        return (float(np.mean(psnr)) if psnr else None), (float(np.mean(ssim)) if ssim else None)

    def close(self):
        self.ctx.destroy()


def config_summary(h, hbm_gbs, alu_peak, stage_frames=60, quality_frames=12):
    """FPS of TemporalGS (AUTO) and of the full render over the WHOLE trajectory of the scene, their ratio, the share of
    selected tiles, quality of the S frames, and per-stage ms + roofline fractions by frame type."""
    tgs, sc = h.tgs, h.sc
    F = len(sc.poses)
    ms_tgs = h.timed(tgs.AUTO, F)
    ms_full = h.timed(tgs.FULL, F)
    per_type = h.stage_pass(min(F, stage_frames))
    psnr, ssim = h.quality(min(F, quality_frames))
    out = {"frames": F, "fps_tgs": aggregate_fps(h.world, F, ms_tgs), "fps_full": aggregate_fps(h.world, F, ms_full),
           "speedup": ms_full / ms_tgs, "psnr_S_vs_full_dB": psnr, "ssim_S_vs_full": ssim,
           "n_sel_frac_S": (summarise(per_type[2]) or {}).get("n_sel_frac"),
           "stages": {k: summarise(per_type[i]) for k, i in (("R", 0), ("P", 1), ("S", 2))},
           "stage_rooflines": {k: stage_rooflines(per_type[i], sc, hbm_gbs, alu_peak) for k, i in (("R", 0), ("P", 1), ("S", 2))}}
    return out, per_type


def run_ours(args):
    import torch
    import torch.distributed as dist
    from paper_2607_03390_b200 import build as tgs_build
    from synth import make_config

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    torch.cuda.set_device(local)
    tgs_build.build()
    from paper_2607_03390_b200 import tgs           # raises if libtgs.so is missing: no fallback

    sc = make_config(args.config, n=args.n, frames=None)
    cam = sc.camera
    K, W = args.steps, args.warmup
    h = Harness(tgs, torch, sc, local, world, W, args.depth_slabs)

    # ---- the headline: K frames of the trajectory, TemporalGS (AUTO); then the same frames end to end
    sampler = ClockSampler(local)
    if rank == 0:
        sampler.start()
    ms_tgs = h.timed(tgs.AUTO, K)
    launches = h.launches
    clocks = sampler.stop() if rank == 0 else None
    ms_full = h.timed(tgs.FULL, K)
    pinned = [torch.empty((cam.H, cam.W, 3), dtype=torch.float32).pin_memory() for _ in range(2)]
    ms_e2e = h.timed(tgs.AUTO, K, readback=[t.numpy() for t in pinned])

    hbm_gbs, sm_mhz_max, peak_kind = _peaks()
    sm_clk = (clocks or {}).get("sm_mhz") or sm_mhz_max
    alu_peak = 148 * 128 * sm_clk * 1e6 / 1e12          # T lane-instr/s at the clock seen under load
    # ---- the whole trajectory (BASELINE.json: "FPS over trajectory; speed-up vs full render"), whatever --steps says
    traj, per_type = config_summary(h, hbm_gbs, alu_peak)
    h.close()
    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return None

    # ---- the other synthetic trajectories (north_star: "on the synthetic trajectories below"): where selective rendering
    # and the stitch are actually timed (config 3 selects every tile)
    others = {}
    if world == 1 and args.n is None:
        for cfg in [int(x) for x in args.other_configs.split(",") if x.strip().isdigit()]:
            if cfg == args.config:
                continue
            sc2 = make_config(cfg, frames=None)
            h2 = Harness(tgs, torch, sc2, local, 1, W, args.depth_slabs)
            o2, _ = config_summary(h2, hbm_gbs, alu_peak, stage_frames=40, quality_frames=10)
            h2.close()
            o2["workload"] = workload_string(sc2, cfg)
            S = (o2["stage_rooflines"] or {}).get("S")
            o2["S_frame_roofline_fracs"] = {k: round(v["frac"], 4) for k, v in S.items()} if S else None
            others[f"config{cfg}"] = o2
            del sc2, h2

    # ---- roofline of the dominant kernel = the stage with the largest share of the profiled frames' time
    all_stats = [s for lst in per_type.values() for s in lst]
    tot = np.sum([np.asarray(s["ms_stage"]) for s in all_stats], axis=0)
    dom = int(np.argmax(tot[:7]))
    roofs_all = stage_rooflines(all_stats, sc, hbm_gbs, alu_peak)      # frame types pooled: the mix the timed region ran
    mean = lambda key: float(np.mean([s[key] for s in all_stats]))
    r = roofs_all[STAGE_NAMES[dom]]
    roof = {"kernel": "k_blend" if STAGE_NAMES[dom] == "blend_stitch" else STAGE_NAMES[dom], "bound": r["bound"], "achieved": r["achieved"],
            "peak": r["peak"], "unit": r["unit"], "frac": r["frac"], "ms_per_launch": r["ms"]}
    if STAGE_NAMES[dom] == "blend_stitch":
        roof.update({"traffic": BLEND_DRAM_TRAFFIC_BYTES, "traffic_source": BLEND_DRAM_TRAFFIC_SOURCE,
                     "interactions_per_launch": mean("n_interactions"), "blended_per_launch": mean("n_blended"),
                     "pixel_slots_per_launch": mean("n_pixel_slots"), "lane_instr_per_interaction": BLEND_LANE_INSTR,
                     "peak_note": f"148 SM x 4 schedulers x 32 lanes x {sm_clk:.0f} MHz (median SM clock during the run): one warp "
                                  f"instruction per scheduler and clock; the FMA pipe (128 lanes/clk/SM) and the ALU pipe (64) are not "
                                  f"tighter for this mix (DESIGN.md 7.2)"})
    else:
        roof.update({"traffic": None, "peak_note": f"{peak_kind} copy bandwidth" if r["bound"] == "hbm" else "issue peak"})
    roof["stages"] = {k: {n: {"ms": round(v["ms"], 5), "bound": v["bound"], "frac": round(v["frac"], 4)} for n, v in d.items()}
                      for k, d in traj["stage_rooflines"].items() if d}
    roof["stages_note"] = ("per-stage times are taken with every kernel on ONE stream (stage events must bracket what they name); the "
                           "production frame overlaps A2 / A4 / SH colours on side streams, so its ms_per_step is below the stage sum; where the library runs the depth sort as one launch (short visible lists) that launch also builds the flat test space (A5a), which the multi-launch pipeline does at the start of bin_pairs: depth_sort's fraction still counts the sort's bytes only")

    fps_tgs, fps_full, fps_e2e = aggregate_fps(world, K, ms_tgs), aggregate_fps(world, K, ms_full), aggregate_fps(world, K, ms_e2e)
    out = {
        "metric": METRIC, "value": fps_tgs, "unit": "frames/s", "n_gpus": world, "steps": K, "warmup": W,
        "ms_per_step": ms_tgs / K, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "f32", "data": "synthetic",
        "config": {"workload": workload_string(sc, args.config),
                   "l2": "scene arrays (>= 700 MB) exceed the 126 MB L2; no explicit flush", "parallelism": "replicas only",
                   "depth_slabs": "automatic (library default: one or two front-to-back pieces per frame, chosen from its own statistics)" if not args.depth_slabs else args.depth_slabs,
                   "fps_full_render": fps_full, "speedup_vs_full_render": fps_tgs / fps_full,
                   "trajectory": {k: traj[k] for k in ("frames", "fps_tgs", "fps_full", "speedup", "psnr_S_vs_full_dB", "ssim_S_vs_full", "n_sel_frac_S")},
                   "stages": traj["stages"],
                   "other_configs": {k: {kk: v[kk] for kk in ("workload", "frames", "fps_tgs", "fps_full", "speedup", "n_sel_frac_S", "psnr_S_vs_full_dB",
                                                             "ssim_S_vs_full", "S_frame_roofline_fracs", "stages", "stage_rooflines")} for k, v in others.items()}},
        "e2e": {"value": fps_e2e, "unit": "frames/s", "h2d_bytes_per_step": 16 * 4 + 8 * 4, "d2h_bytes_per_step": cam.W * cam.H * 3 * 4,
                "note": "camera by value through tgs_set_camera; every frame's image copied to pinned host memory (tgs_read_image_async: the copy of frame f overlaps the rendering of frame f+1), all copies complete inside the timed region"},
        "gpu_launches": int(launches),                 # counted by the library (tgs_stats.launches_total) over the timed region
        "roofline": roof, "clocks": clocks,
    }
    if world > 1:
        dist.destroy_process_group()
    return out


# ---------------------------------------------------------------------------------------------- ablation
def run_ablation(args):
    """Leave-one-out / one-at-a-time ablation of AFC, TOC and SR (the shape of the paper's Table IV) and the
    eta / lambda_SR sensitivity (Table VI) on the synthetic trajectory: FPS over `steps` frames of the AUTO
    schedule and PSNR of the S frames against the full render of the same pose.  Single GPU; prints one JSON line."""
    import torch
    from paper_2607_03390_b200 import build as tgs_build
    from synth import make_config
    tgs_build.build()
    from paper_2607_03390_b200 import tgs
    torch.cuda.set_device(0)
    sc = make_config(args.config, n=args.n, frames=None)
    stream = torch.cuda.Stream()
    ctx, ref = tgs.Context(0, stream.cuda_stream), tgs.Context(0, stream.cuda_stream)
    ctx.load_scene(sc); ref.load_scene(sc)
    cam, K, W = sc.camera, args.steps, max(args.warmup, 3)

    def variant(stride=1, **kw):
        """`stride`: every stride-th pose of the trajectory, i.e. the camera moves `stride` times faster per frame (the
        camera-speed axis of the paper's Table V)."""
        prm = ctx.default_params()
        for k, v in kw.items():
            setattr(prm, k, v)
        ctx.set_params(prm)
        ctx.reset_priors()
        for f in range(W):
            ctx.set_camera(trajectory_pose(sc, f * stride), cam); ctx.render(tgs.AUTO)
        ctx.reset_priors()
        torch.cuda.synchronize()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        with torch.cuda.stream(stream):
            e0.record(stream)
            for f in range(K):
                ctx.set_camera(trajectory_pose(sc, f * stride), cam); ctx.render(tgs.AUTO)
            e1.record(stream)
        torch.cuda.synchronize()
        fps = K / (e0.elapsed_time(e1) * 1e-3)
        ctx.reset_priors()
        psnr, types, sel = [], [], []
        for f in range(min(K, 40)):
            ctx.set_camera(trajectory_pose(sc, f * stride), cam); ctx.render(tgs.AUTO)
            st = ctx.get_stats()
            types.append("RPS"[st["frame_type"]])
            if st["frame_type"] == tgs.FRAME_S:
                sel.append(st["n_sel"] / st["n_tiles"])
                ref.set_camera(trajectory_pose(sc, f * stride), cam); ref.render(tgs.FULL)
                mse = float(((ctx.read_image() - ref.read_image()) ** 2).mean())
                psnr.append(10 * np.log10(1.0 / max(mse, 1e-12)))
        return {"fps": fps, "psnr_S_vs_full_dB": float(np.mean(psnr)) if psnr else None, "tgsf": types.count("S") / len(types),
                "mean_selected_fraction": float(np.mean(sel)) if sel else None}

    rows = {
        "full_render (lambda_sr=1)": variant(lambda_sr=1, lambda_tdc=1),
        "AFC only": variant(enable_afc=1, enable_toc=0, enable_sr=0),
        "TOC only": variant(enable_afc=0, enable_toc=1, enable_sr=0),
        "SR only": variant(enable_afc=0, enable_toc=0, enable_sr=1),
        "AFC+TOC (TDC)": variant(enable_sr=0),
        "TemporalGS (all)": variant(),
        "eta=0.2": variant(eta=0.2), "eta=0.6": variant(eta=0.6),
        "lambda_sr=2": variant(lambda_sr=2), "lambda_sr=10": variant(lambda_sr=10),
        "lambda_tdc=25": variant(lambda_tdc=25), "lambda_tdc=75": variant(lambda_tdc=75),
        # the paper's large-scene setting (L142) and the chained prior policy (R42, drift vs ANCHORED)
        "tgb_downscale=2": variant(tgb_downscale=2),
        "prior_policy=CHAINED": variant(prior_policy=1),
        "CHAINED, lambda_sr=10": variant(prior_policy=1, lambda_sr=10),
        "CHAINED + tgb_downscale=2": variant(prior_policy=1, tgb_downscale=2),
        # camera speed (Table V): every 2nd / 4th / 8th pose of the trajectory per frame
        "camera speed x2": variant(stride=2), "camera speed x4": variant(stride=4), "camera speed x8": variant(stride=8),
        "full render, camera speed x8": variant(stride=8, lambda_sr=1, lambda_tdc=1),
    }
    return {"metric": "ablation: FPS / PSNR(S vs full) / share of S frames per variant", "config": {"workload": f"config {args.config} ({sc.name})"},
            "steps": K, "warmup": W, "data": "synthetic", "ablation": rows}


# ---------------------------------------------------------------------------------------------- CPU oracle legs
def oracle_sample(config, n, frames_modes, budget_s=None):
    """Time the oracle, as it stands, on the given (frame index, mode) list of the config's trajectory."""
    from oracle import ora
    from oracle.ora import Oracle
    from synth import make_config
    sc = make_config(config, n=n, frames=None)
    o = Oracle()
    o.load_scene(sc)
    modes = {"full": ora.FULL, "auto": ora.AUTO, "temporal": ora.TEMPORAL}
    t_total, done, per = 0.0, 0, []
    for f, m in frames_modes:
        o.set_camera(trajectory_pose(sc, f), sc.camera)
        t0 = time.perf_counter()
        o.render(modes[m])
        dt = time.perf_counter() - t0
        st = o.stats()
        per.append({"frame": f, "type": "RPS"[st["frame_type"]], "s": dt, "ms_temporal": st["ms_temporal"], "ms_preprocess": st["ms_preprocess"],
                    "ms_sort": st["ms_sort"], "ms_blend": st["ms_blend"]})
        t_total += dt
        done += 1
        if budget_s is not None and t_total > budget_s:
            break
    return done, t_total, per, sc


def run_reference(args):
    """--impl reference: the CPU oracle on the same config / metric.  Each step is one trajectory frame in AUTO
    mode; the oracle needs seconds per 1080p frame, so the number of Gaussians is NOT reduced but the run is
    bounded by rendering the K (+W) frames with the SAME schedule and reporting frames / time."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return None
    K, W = args.steps, args.warmup
    # bounded sample: the oracle takes ~10-30 s per reference frame at config 3; keep the whole run within
    # a few minutes by bounding the number of timed frames (the JSON line says how many were timed)
    budget = float(os.environ.get("TGS_REF_BUDGET_S", "150"))
    frames = [(f, "auto") for f in range(W + K)]
    from oracle import ora
    from oracle.ora import Oracle
    from synth import make_config
    sc = make_config(args.config, n=args.n, frames=None)
    o = Oracle()
    o.load_scene(sc)
    t_used, timed_frames, t_timed, types = 0.0, 0, 0.0, []
    for i, (f, _) in enumerate(frames):
        o.set_camera(trajectory_pose(sc, f), sc.camera)
        t0 = time.perf_counter()
        ft = o.render(ora.AUTO)
        dt = time.perf_counter() - t0
        t_used += dt
        if i >= W:
            timed_frames += 1
            t_timed += dt
            types.append("RPS"[ft])
        if t_used > budget and timed_frames >= 1:
            break
    fps = timed_frames / t_timed
    cam = sc.camera
    sample = (f"{timed_frames} of the requested {K} frames (types {''.join(types)}) after {min(W, len(frames))} warm-up frames, "
              f"bounded to ~{budget:.0f} s of CPU time; full scene, full resolution")
    return {
        "impl": "reference", "metric": METRIC, "value": fps, "unit": "frames/s", "n_gpus": int(os.environ.get("WORLD_SIZE", "1")),
        "steps": K, "warmup": W, "ms_per_step": 1e3 * t_timed / timed_frames, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": workload_string(sc, args.config)},
        "cpu_baseline": {"value": fps, "unit": "frames/s", "cores": 1, "kind": "oracle", "sample": sample},
        "e2e": {"value": fps, "unit": "frames/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "steps_timed": timed_frames,
    }


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=300)
    ap.add_argument("--warmup", type=int, default=5)
    ap.add_argument("--config", type=int, default=3)
    ap.add_argument("--n", type=int, default=None, help="override the number of Gaussians (debug only)")
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--depth-slabs", type=int, default=0, help="tgs_params.depth_slabs: 0 = automatic (the default of the library), 1..4 = fixed (profiling runs)")
    ap.add_argument("--other-configs", default="2,5,4", help="configs also measured over their whole trajectories ('none' to skip)")
    ap.add_argument("--ablation", action="store_true", help="module ablation and sensitivity table instead of the bench line")
    args = ap.parse_args()
    args.warmup = max(args.warmup, 3) if args.impl == "ours" else args.warmup
    if args.impl == "reference":
        out = run_reference(args)
        if out is not None:
            print(json.dumps(out))
        return
    if args.ablation:
        print(json.dumps(run_ablation(args)))
        return
    out = run_ours(args)
    if out is None:
        return
    if out["n_gpus"] == 1 and not args.no_cpu_baseline:
        # the oracle as it stands on one host core: one lambda_SR cycle (6 frames) of the same trajectory in AUTO mode
        # (SURVEY 8(d)), with the oracle's own per-stage split
        done, t, per, _ = oracle_sample(args.config, args.n, [(f, "auto") for f in range(6)])
        split = {k: float(np.mean([p[k] for p in per])) for k in ("ms_temporal", "ms_preprocess", "ms_sort", "ms_blend")}
        out["cpu_baseline"] = {"value": done / t, "unit": "frames/s", "cores": 1, "kind": "oracle",
                               "sample": f"frames 0-{done - 1} of the same trajectory, AUTO schedule (one lambda_SR cycle), {t:.1f} s: " +
                                         ", ".join(f"{p['type']} {p['s']:.1f} s" for p in per),
                               "ms_per_frame_by_stage": split}
    print(json.dumps(out))


if __name__ == "__main__":
    main()
