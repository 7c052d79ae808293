#!/usr/bin/env python
"""bench.py -- rendered+fused frames/s of the FHGS hot path on the Mid workload (BASELINE.json
configs[2]: N = 10^6 Gaussians, SH degree 3, D = 128 fp32 unit features, one 1920x1080 view, one
1920x1080x128 fp32 GT feature map; seeded synthetic inputs, recipe in DESIGN.md).

A "step" = one frame = fhgs_project -> fhgs_bin_sort -> fhgs_render (RGB + D features) ->
fhgs_fuse_features (clear, accumulate one GT map, finalise), all through the C ABI.

    python bench.py --gpus N --steps K --warmup W            # the CUDA path (one rank per GPU)
    python bench.py --impl reference --steps K --warmup W    # the CPU oracle on host cores

Prints ONE JSON line (see DESIGN.md "Measurement" for every field).  N > 1 (torchrun): frames are
independent units, each rank renders and fuses its own frame (camera k = rank of an 8-camera
circle), no data-path collective; `value` = frames of all ranks / max-over-ranks time ("weak").
"""
from __future__ import annotations

import argparse
import json
import os
import statistics
import subprocess
import sys
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import numpy as np  # noqa: E402

METRIC = "rendered+fused frames/s at 1080p D=128"
UNIT = "frames/s"
FP32_LANES_PER_SM = 128
L2_BYTES = 126 * 2 ** 20


def load_peaks():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(path):
        with open(path) as f:
            p = json.load(f)
        return dict(hbm_gbs=float(p["hbm_gbs"]), sm_max_mhz=float(p.get("sm_max_mhz", 1965.0)), source="measured")
    return dict(hbm_gbs=6650.0, sm_max_mhz=1965.0, source="fallback")


# --------------------------------------------------------------------------------------------------
# clocks: nvidia-smi sampled DURING the timed region
# --------------------------------------------------------------------------------------------------
class ClockSampler:
    QUERY = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
             "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
             "clocks_event_reasons.sw_power_cap")

    def __init__(self, gpu_index: int):
        self.proc = None
        self.gpu = gpu_index

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(self.gpu), f"--query-gpu={self.QUERY}",
                                          "--format=csv,noheader,nounits", "-lms", "50"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
        except OSError:
            self.proc = None

    def stop(self) -> dict:
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.06)
        self.proc.terminate()
        try:
            out, _ = self.proc.communicate(timeout=5)
        except subprocess.TimeoutExpired:
            self.proc.kill()
            out, _ = self.proc.communicate()
        sm, mx, pw, reasons = [], [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for line in out.splitlines():
            f = [x.strip() for x in line.split(",")]
            if len(f) < 7:
                continue
            try:
                sm.append(float(f[0])); mx.append(float(f[1])); pw.append(float(f[2]))
            except ValueError:
                continue
            for nm, v in zip(names, f[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(nm)
        if not sm:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["no samples"]}
        return {"sm_mhz": statistics.median(sm), "sm_max_mhz": max(mx), "power_w_max": max(pw),
                "samples": len(sm), "reasons": sorted(reasons)}


# --------------------------------------------------------------------------------------------------
# the oracle arm (cpu_baseline and --impl reference).  Both legs use the SAME sample: the whole Mid
# frame ("Mid: oracle_scatter, 1 run"), ~10-15 s on 16 host cores.  (A tile-aligned crop
# of the frame -- same scene, same camera, principal point shifted -- is kept for --small debugging.)
# --------------------------------------------------------------------------------------------------
class OracleSample:
    def __init__(self, scene, cfg, cam, crop_w=None, crop_h=None):
        crop_w = cfg.width if crop_w is None else crop_w
        crop_h = cfg.height if crop_h is None else crop_h
        from oracle import fhgs_oracle as fo
        from paper_2505_19154_b200 import inputs
        self.fo, self.scene, self.cfg = fo, scene, cfg
        fo.lib()
        x0 = (cfg.width - crop_w) // 2 // 16 * 16
        y0 = (cfg.height - crop_h) // 2 // 16 * 16
        self.cam = inputs.crop_camera(cam, x0, y0, crop_w, crop_h)
        self.w, self.h = crop_w, crop_h
        self.frac = (crop_w * crop_h) / float(cfg.width * cfg.height)
        self.feat32 = np.ascontiguousarray(scene.feat, dtype=np.float32)
        if self.frac == 1.0:
            self.gt = inputs.make_gt_map(cfg, 0, cam)
        else:
            rng = np.random.default_rng(cfg.seed * 1000 + 999)
            g = rng.standard_normal((crop_h, crop_w, cfg.feat_dim), dtype=np.float32)
            g /= np.maximum(np.sqrt((g * g).sum(axis=-1, keepdims=True)), 1e-30)
            self.gt = g
        if self.frac == 1.0:
            self.desc = (f"oracle P+S+R+F (fo_project, fo_bins, fo_render_scatter, fo_fuse_scatter, fo_fuse_finalize) on the "
                         f"whole {cfg.width}x{cfg.height} frame, N={scene.n}, D={cfg.feat_dim}: one full step, no extrapolation")
        else:
            self.desc = (f"oracle P+S+R+F on the centred {crop_w}x{crop_h} crop of the {cfg.width}x{cfg.height} frame (all N={scene.n} "
                         f"Gaussians projected, {self.frac:.4f} of the pixels); frames/s = 1 / (t_P + (t_S+t_R+t_F)/{self.frac:.4f})")

    def step(self) -> float:
        """One sample; returns the extrapolated seconds per FULL frame."""
        fo, s, c = self.fo, self.scene, self.cam
        t0 = time.perf_counter()
        pr = fo.project(s.mean, s.scale, s.quat, s.opacity, s.sh, s.sh_degree, fo.cam_array(c.view, c.proj, c.cam_pos),
                        c.width, c.height)
        t1 = time.perf_counter()
        fo.bins(pr, c.width, c.height)
        order = fo.global_order(pr)
        fo.render_scatter(pr, order, self.feat32, c.width, c.height)
        num, den = fo.fuse(pr, order, self.gt, c.width, c.height)
        fo.finalize(num, den, self.feat32)
        t2 = time.perf_counter()
        return (t1 - t0) + (t2 - t1) / self.frac


def run_reference(args, rank: int):
    """--impl reference: the oracle, as it stands, on the host cores; rank 0 only."""
    if rank != 0:
        return
    from oracle import fhgs_oracle as fo
    from paper_2505_19154_b200 import inputs
    fo.build()
    cfg = inputs.CONFIGS["mid"]
    scene = inputs.make_scene(cfg)
    cam = inputs.make_camera(cfg, 0)
    smp = OracleSample(scene, cfg, cam)     # the same sample as the cuda arm's cpu_baseline leg: the whole frame
    for _ in range(args.warmup):
        smp.step()
    t0 = time.perf_counter()
    per_frame = [smp.step() for _ in range(args.steps)]
    wall = time.perf_counter() - t0
    sec = sum(per_frame) / len(per_frame)
    val = 1.0 / sec
    cores = fo.num_threads()
    line = {"impl": "reference", "metric": METRIC, "value": val, "unit": UNIT, "n_gpus": 0, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": 1e3 * wall / args.steps,
            "higher_is_better": True,
            "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": (f"mid: N={scene.n} SH{scene.sh_degree} D={cfg.feat_dim} f32, 1 view {cfg.width}x{cfg.height} + one "
                                    f"{cfg.width}x{cfg.height}x{cfg.feat_dim} GT map"),   # the same string as the cuda arm's
                       "sample": smp.desc},
            "cpu_baseline": {"value": val, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": smp.desc},
            "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line), flush=True)


# --------------------------------------------------------------------------------------------------
# the CUDA arm
# --------------------------------------------------------------------------------------------------
def launches_per_frame(width: int, height: int) -> int:
    """Kernels of libfhgs.so launched per frame (default sort schedule; memsets are not kernels): project 1;
    bin_sort = presort_init 1 + hist_scan 1 + 4 depth onesweep passes + offsets scan 1 + depth-order scan 1 +
    [tile_scan 1 | hist_scan 1 + ranges 1] + emit_partition 1 + emit 1 + ceil(tile_bits/8) tile-id onesweep passes;
    render 1; fuse: sparse clear 1 + accumulate 1 + finalise 1."""
    gw, gh = (width + 15) // 16, (height + 15) // 16
    tile_bits = max(1, (gw * gh - 1).bit_length())
    grid_counts = (gw + 1) * (gh + 1) <= 12288
    return 1 + (1 + 1 + 4 + 1 + 1 + (1 if grid_counts else 2) + 1 + 1 + (tile_bits + 7) // 8) + 1 + 3


def load_traffic() -> dict:
    """DRAM bytes per launch (dram__bytes_read.sum + dram__bytes_write.sum) of the hot kernels, from the committed
    `ncu --set full` capture summarised in profiles/ (bench.py never runs under a profiler)."""
    import glob
    paths = sorted(glob.glob(os.path.join(ROOT, "profiles", "r[0-9][0-9]_traffic.json")))   # the latest round's capture
    if paths:
        with open(paths[-1]) as f:
            return json.load(f)
    return {}


def run_cuda(args, rank: int, world: int, local_rank: int):
    import torch
    import torch.distributed as dist
    from paper_2505_19154_b200 import binding as fb   # fails loudly without libfhgs.so
    from paper_2505_19154_b200 import inputs, parallel

    if not torch.cuda.is_available():
        raise RuntimeError("bench.py needs a CUDA device: the FHGS path has no CPU fallback")
    torch.cuda.set_device(local_rank)
    dev = torch.device("cuda", local_rank)
    if world > 1:
        dist.init_process_group("nccl", device_id=dev)
    peaks = load_peaks()

    cfg = inputs.CONFIGS["mid"]
    if args.small:   # debugging aid only; never a bench line
        cfg = inputs.scaled(cfg, n=100_000, width=640, height=368, log_scale_mu=-3.5)
    scene = inputs.make_scene(cfg)
    cam_np = inputs.make_camera(cfg, 0) if rank == 0 else inputs.circle_camera(rank % 8, 8, cfg.width, cfg.height)
    gt_np = inputs.make_gt_map(cfg, rank, cam_np)
    W, H, D, n = cfg.width, cfg.height, cfg.feat_dim, scene.n
    capacity = int(40e6) if not args.small else int(8e6)

    ctx = fb.Context(local_rank)
    g = fb.Gaussians(scene.mean, scene.scale, scene.quat, scene.opacity, scene.sh, scene.feat, scene.sh_degree, device=dev)
    vs = fb.ViewState(n, W, H, capacity, device=dev)
    prm = fb.default_params(rect_mode=1 if args.rect == 'tight' else 0)
    cam = fb.make_camera(cam_np.view, cam_np.proj, cam_np.cam_pos, W, H)
    f32 = torch.float32
    gt = torch.from_numpy(gt_np).to(dev)
    out_rgb = torch.empty((H, W, 3), dtype=f32, device=dev)
    out_feat = torch.empty((H, W, D), dtype=f32, device=dev)
    out_T = torch.empty((H, W), dtype=f32, device=dev)
    out_n = torch.empty((H, W), dtype=torch.int32, device=dev)
    num = torch.zeros((n, D), dtype=f32, device=dev)
    den = torch.zeros((n,), dtype=f32, device=dev)
    fused = g.feat.clone()
    stream = torch.cuda.current_stream()

    NAMES = ["project", "bin_sort", "render", "fuse_zero", "fuse_accumulate", "fuse_finalize"]

    def frame(evs=None):
        def mark(i):
            if evs is not None:
                evs[i].record(stream)
        mark(0)
        fb.project(ctx, g, cam, prm, vs)
        mark(1)
        fb.bin_sort(ctx, cam, vs, sync=False)
        mark(2)
        fb.render(ctx, g, cam, prm, vs, out_rgb, out_feat, out_T, out_n)
        mark(3)
        # num / den start as zeros and are only ever written by the library: the sparse clear's precondition holds
        fb.fuse_features(ctx, None, prm, vs, None, num, den, None, fb.FHGS_FUSE_ZERO_ONLY | fb.FHGS_FUSE_ZERO_TOUCHED)
        mark(4)
        fb.fuse_features(ctx, cam, prm, vs, gt, num, den, None, 0)
        mark(5)
        fb.fuse_features(ctx, None, prm, vs, None, num, den, fused, fb.FHGS_FUSE_FINALIZE_ONLY)
        mark(6)

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    # capacity check once, outside the timed region
    fb.project(ctx, g, cam, prm, vs)
    M = fb.bin_sort(ctx, cam, vs, sync=True)

    for _ in range(max(args.warmup, 3)):
        frame()
    barrier()
    evs = [[torch.cuda.Event(enable_timing=True) for _ in range(7)] for _ in range(args.steps)]
    sampler = ClockSampler(local_rank)
    sampler.start()
    barrier()
    for k in range(args.steps):
        frame(evs[k])
    barrier()
    clocks = sampler.stop()
    total_ms = parallel.max_over_ranks(evs[0][0].elapsed_time(evs[-1][6]), dev)
    ms_per_step = total_ms / args.steps
    value = world * args.steps / (total_ms * 1e-3)
    parts = {nm: statistics.mean(evs[k][i].elapsed_time(evs[k][i + 1]) for k in range(args.steps))
             for i, nm in enumerate(NAMES)}

    # ---- algorithmic work of this frame, from the path's integer outputs
    n_contrib_total = int(out_n.view(torch.int32).to(torch.int64).sum().item())
    n_vis = int((vs.tiles_touched.view(torch.int32) != 0).sum().item())
    n_final = int((den > float(prm.den_eps)).sum().item())
    K = (scene.sh_degree + 1) ** 2
    tiles = ((W + 15) // 16) * ((H + 15) // 16)
    tile_bits = max(1, (tiles - 1).bit_length())
    p_full = (32 + tile_bits + 7) // 8
    # n_eval of SURVEY 8(d): instances of a tile's list walked before the whole tile stopped (fhgs_render's
    # tile_visited diagnostics) x the tile's valid pixels
    gw, gh = (W + 15) // 16, (H + 15) // 16
    ctx.set_diagnostics(True)     # one extra, un-timed render with the diagnostics variant of the kernel
    fb.render(ctx, g, cam, prm, vs, out_rgb, out_feat, out_T, out_n)
    ctx.set_diagnostics(False)
    tv = vs.tile_visited().to(torch.int64).view(gh, gw)
    px_x = torch.clamp(W - 16 * torch.arange(gw, device=dev), max=16)
    px_y = torch.clamp(H - 16 * torch.arange(gh, device=dev), max=16)
    n_eval_total = int((tv * (px_y[:, None] * px_x[None, :])).sum().item())
    work = {
        # lane-ops = sum_x [7 n_eval(x) + (D + 8) n_c(x)] (render), [7 n_eval + (D + 6) n_c] (fuse)
        "render_lane_ops": 7 * n_eval_total + (8 + D) * n_contrib_total,
        "fuse_lane_ops": 7 * n_eval_total + (6 + D) * n_contrib_total,
        # stricter count: only the (pixel, contributor) pairs, nothing for the evaluations that are cut off
        "render_lane_ops_contrib_only": (7 + 8 + D) * n_contrib_total,
        "fuse_lane_ops_contrib_only": (7 + 6 + D) * n_contrib_total,
        "fuse_bytes": W * H * D * 4,                                      # the GT map, read once
        "project_bytes": 44 * n + 12 * K * n_vis + 16 * n + 40 * n_vis,
        # S, algorithmic: scan + duplicate, histogram + p_full = 6 LSD passes over the pairs, ranges
        "bin_sort_bytes": (4 * n + 12 * n_vis + 4 * n + 12 * M) + (8 * M + p_full * 24 * M) + (8 * M + 8 * tiles),
        # S, as executed by the default schedule: depth pre-sort of the N Gaussians (init 16 N + 8 n_vis,
        # 4 passes x 16 N), two scans (8 N + 12 N), instance-balanced emission (20 n_vis read, 12 M written),
        # ceil(tile_bits / 8) tile-id passes x 24 M
        "bin_sort_bytes_executed": 100 * n + 28 * n_vis + 12 * M + ((tile_bits + 7) // 8) * 24 * M,
        # finalise touches only the rows it divides: den for all, num read + out written where den > den_eps
        "finalize_bytes": n * 4 + n_final * D * 8,
        "finalized_rows": n_final,
    }
    ffma_ops, _ = ctx.ffma_peak(2048)
    alu_nominal = 148 * FP32_LANES_PER_SM * peaks["sm_max_mhz"] * 1e6       # lane-ops/s at max clock
    steps_roof = {}
    for nm, ops in (("render", work["render_lane_ops"]), ("fuse_accumulate", work["fuse_lane_ops"])):
        ach = 2.0 * ops / (parts[nm] * 1e-3) / 1e12
        ops_c = work[("render" if nm == "render" else "fuse") + "_lane_ops_contrib_only"]
        steps_roof[nm] = {"bound": "alu", "achieved": ach, "peak": 2.0 * alu_nominal / 1e12, "unit": "TFLOP/s",
                          "frac": ach / (2.0 * alu_nominal / 1e12), "ms": parts[nm],
                          "frac_of_measured_ffma": 2.0 * ops / (parts[nm] * 1e-3) / (2.0 * ffma_ops),
                          "frac_contributors_only": ops_c / (parts[nm] * 1e-3) / alu_nominal,
                          "work": "lane-ops = 7 n_eval + (D+%d) n_contrib (SURVEY 8(d)); FMA = 2 flop" % (8 if nm == "render" else 6)}
    for nm, by in (("project", work["project_bytes"]), ("bin_sort", work["bin_sort_bytes"]),
                   ("fuse_finalize", work["finalize_bytes"])):
        ach = by / (parts[nm] * 1e-3) / 1e9
        steps_roof[nm] = {"bound": "hbm", "achieved": ach, "peak": peaks["hbm_gbs"], "unit": "GB/s",
                          "frac": ach / peaks["hbm_gbs"], "ms": parts[nm]}
    steps_roof["fuse_accumulate"]["hbm_gbs_gt_map"] = work["fuse_bytes"] / (parts["fuse_accumulate"] * 1e-3) / 1e9
    steps_roof["bin_sort"]["frac_real_traffic"] = work["bin_sort_bytes_executed"] / (parts["bin_sort"] * 1e-3) / 1e9 / peaks["hbm_gbs"]
    steps_roof["bin_sort"]["note"] = ("frac = SURVEY 8(d)'s algorithmic bytes (literal 6-pass LSD sort of the pairs) / time; "
                                      "frac_real_traffic = bytes the default schedule actually moves / time")
    dominant = max(("render", "fuse_accumulate", "bin_sort", "project", "fuse_finalize"), key=lambda k: parts[k])
    roofline = dict(steps_roof[dominant])
    roofline["kernel"] = {"render": "render_ws_kernel<128,float>", "fuse_accumulate": "fuse_ws_kernel<float>",
                          "bin_sort": "fhgs_bin_sort (13 launches)", "project": "project_kernel<3>",
                          "fuse_finalize": "finalize_kernel<float>"}[dominant]
    roofline["peak_source"] = ("148 SMs x 128 FP32 lanes x sm_max_mhz (MEASURED_PEAKS.json), FMA = 2 flop"
                               if roofline["bound"] == "alu" else f"hbm_gbs of MEASURED_PEAKS.json ({peaks['source']})")
    traffic = load_traffic().get(roofline["kernel"])
    roofline["traffic"] = traffic["dram_bytes_per_launch"] if traffic else None
    if traffic:
        roofline["traffic_source"] = traffic["source"]

    # ---- optional: the NEXT-1 row (NDFD forward losses) on the same frame, timed for the record
    ndfd = None
    if args.ndfd:
        lgt = torch.empty((H, W), dtype=f32, device=dev)
        lcf = torch.empty((H, W), dtype=f32, device=dev)
        for _ in range(2):
            fb.ndfd_forward(ctx, g, cam, prm, vs, gt, lgt, lcf)
        ev = [torch.cuda.Event(enable_timing=True) for _ in range(2)]
        ev[0].record(stream)
        for _ in range(5):
            fb.ndfd_forward(ctx, g, cam, prm, vs, gt, lgt, lcf)
        ev[1].record(stream)
        torch.cuda.synchronize()
        nms = ev[0].elapsed_time(ev[1]) / 5
        # lane-ops: 7 n_eval + (3 D + 12) n_contrib (phi, F.f and the F update are D FMAs each)
        nops = 7 * n_eval_total + (3 * D + 12) * n_contrib_total
        ndfd = {"ms": nms, "frac_of_nominal_fp32": nops / (nms * 1e-3) / alu_nominal,
                "mean_lgt": float(lgt.mean().item()), "mean_lcf": float(lcf.mean().item())}
        for _ in range(2):
            fb.ndfd_forward(ctx, g, cam, prm, vs, gt, lgt, lcf, mode=fb.FHGS_NDFD_FAR_TO_NEAR)
        ev[0].record(stream)
        for _ in range(5):
            fb.ndfd_forward(ctx, g, cam, prm, vs, gt, lgt, lcf, mode=fb.FHGS_NDFD_FAR_TO_NEAR)
        ev[1].record(stream)
        torch.cuda.synchronize()
        ndfd["far_to_near_ms"] = ev[0].elapsed_time(ev[1]) / 5   # one more D-vector per pixel: (4 D + 12) n_contrib lane-ops
        ndfd["far_to_near_mean_lcf"] = float(lcf.mean().item())
        gop = torch.zeros((n,), dtype=f32, device=dev)
        work = fb.ndfd_backward(ctx, g, cam, prm, vs, gt, gop)
        ev[0].record(stream)
        for _ in range(3):
            fb.ndfd_backward(ctx, g, cam, prm, vs, gt, gop, work=work)
        ev[1].record(stream)
        torch.cuda.synchronize()
        ndfd["backward_ms"] = ev[0].elapsed_time(ev[1]) / 3

    # ---- end to end through fhgs_frame_host: host (pinned) buffers, copies inside the timed region
    e2e = None
    if not args.no_e2e:
        pin = lambda a: torch.from_numpy(np.ascontiguousarray(a)).pin_memory()
        host = dict(mean=pin(scene.mean), scale=pin(scene.scale), quat=pin(scene.quat), opacity=pin(scene.opacity),
                    sh=pin(scene.sh), feat=pin(scene.feat), gt=pin(gt_np),
                    out_rgb=torch.empty((H, W, 3), dtype=f32).pin_memory(),
                    out_feat=torch.empty((H, W, D), dtype=f32).pin_memory(),
                    fused_feat=torch.empty((n, D), dtype=f32).pin_memory())
        ws = dict(out_rgb=out_rgb, out_feat=out_feat, gt=gt, num=num, den=den, fused_feat=fused)
        h2d = sum(host[k].numel() * host[k].element_size() for k in ("mean", "scale", "quat", "opacity", "sh", "feat", "gt"))
        d2h = sum(host[k].numel() * host[k].element_size() for k in ("out_rgb", "out_feat", "fused_feat")) + 8
        e_steps = max(4, min(args.steps, 10))
        e_steps += e_steps & 1
        for _ in range(2):
            fb.frame_host(ctx, host, g, cam, prm, vs, ws)
        barrier()
        t0 = time.perf_counter()
        for _ in range(e_steps):
            fb.frame_host(ctx, host, g, cam, prm, vs, ws)   # synchronises the stream before returning
        barrier()
        e_one = parallel.max_over_ranks(time.perf_counter() - t0, dev)
        e_one_steps = e_steps
        # Two or three frames in flight: a second (third) context (its own copy streams and events), its own device staging, view state,
        # workspace and host OUTPUT buffers, driven from a second host thread through the same blocking call (ctypes
        # drops the GIL).  Every frame still copies all of its inputs host->device and all of its results device->host
        # inside the timed region; what overlaps is frame k+1's upload with frame k's read-back (PCIe is full duplex), which
        # one blocking call per frame cannot do: its own read-back has to wait for its own upload.
        import threading
        lanes = [(ctx, host, g, vs, ws, torch.cuda.Stream(dev))]
        n_lanes = 3 if world == 1 else 2   # under torchrun every rank pins its own buffers: keep the host footprint down
        for _ in range(n_lanes - 1):   # lanes 2 (and 3): own context, device staging, view state, workspace and host output buffers
            ctx_k = fb.Context(local_rank)
            g_k = fb.Gaussians(scene.mean, scene.scale, scene.quat, scene.opacity, scene.sh, scene.feat, scene.sh_degree, device=dev)
            vs_k = fb.ViewState(n, W, H, capacity, device=dev)
            ws_k = {k: torch.empty_like(v) for k, v in ws.items()}
            host_k = dict(host)
            for k in ("out_rgb", "out_feat", "fused_feat"):
                host_k[k] = torch.empty_like(host[k]).pin_memory()
            lanes.append((ctx_k, host_k, g_k, vs_k, ws_k, torch.cuda.Stream(dev)))
        errs = []

        def worker(lane, count):
            c_, h_, g_, v_, w_, st_ = lane
            try:
                torch.cuda.set_device(local_rank)
                for _ in range(count):
                    fb.frame_host(c_, h_, g_, cam, prm, v_, w_, stream=st_)
            except Exception as ex:   # noqa: BLE001  (reported below; a failed lane must not pass silently)
                errs.append(ex)

        def run_lanes(k, count):
            th = [threading.Thread(target=worker, args=(ln, count)) for ln in lanes[:k]]
            for t_ in th:
                t_.start()
            for t_ in th:
                t_.join()
            if errs:
                raise errs[0]

        def timed_lanes(k):
            torch.cuda.synchronize()
            run_lanes(k, 1)
            barrier()
            t0 = time.perf_counter()
            run_lanes(k, e_steps // k)
            barrier()
            return parallel.max_over_ranks(time.perf_counter() - t0, dev) * e_steps / (k * (e_steps // k))   # per e_steps frames
        e_steps = 12 if e_steps >= 10 else 6   # divisible by 2 and 3
        e_one = e_one * e_steps / e_one_steps
        e_two = timed_lanes(2)
        e_three = timed_lanes(3) if n_lanes >= 3 else float("inf")
        same = all(bool(torch.equal(host["out_rgb"], ln[1]["out_rgb"]) and torch.equal(host["out_feat"], ln[1]["out_feat"]))
                   for ln in lanes[1:])
        e_s = min(e_one, e_two, e_three)
        e2e = {"value": world * e_steps / e_s, "unit": UNIT, "h2d_bytes_per_step": int(h2d), "d2h_bytes_per_step": int(d2h),
               "steps": e_steps, "ms_per_step": 1e3 * e_s / e_steps,
               "frames_in_flight": 1 if e_s == e_one else (2 if e_s == e_two else 3),
               "one_frame_in_flight": {"value": world * e_steps / e_one, "ms_per_step": 1e3 * e_one / e_steps},
               "two_frames_in_flight": {"value": world * e_steps / e_two, "ms_per_step": 1e3 * e_two / e_steps},
               "three_frames_in_flight": ({"value": world * e_steps / e_three, "ms_per_step": 1e3 * e_three / e_steps}
                                          if n_lanes >= 3 else None),
               "lanes_agree": same,
               "pcie_gbs_both_directions": (h2d + d2h) * e_steps / e_s / 1e9}
        del lanes
        del host

    cpu_baseline = None
    if rank == 0 and world == 1 and not args.no_cpu_baseline:
        from oracle import fhgs_oracle as fo   # the one place bench.py's CUDA arm runs the oracle
        fo.build()
        smp = OracleSample(scene, cfg, cam_np) if not args.small else OracleSample(scene, cfg, cam_np, 320, 176)
        sec = smp.step()
        cpu_baseline = {"value": 1.0 / sec, "unit": UNIT, "cores": fo.num_threads(), "kind": "oracle", "sample": smp.desc,
                        "seconds_per_frame": sec}

    if rank == 0:
        line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
                "warmup": max(args.warmup, 3), "ms_per_step": ms_per_step, "higher_is_better": True, "scaling": "weak",
                "vs_baseline": None, "dtype": "f32", "data": "synthetic",
                "config": {"workload": f"mid: N={n} SH{scene.sh_degree} D={D} f32, 1 view {W}x{H} + one {W}x{H}x{D} GT map"
                                       + (" [--rect tight: NEXT-4 (i) variant, not the bench line]" if args.rect == "tight" else "")
                                       + (" [--small debug size, not a bench line]" if args.small else ""),
                           "instances_M": M, "visible": n_vis, "contributors_per_px": n_contrib_total / (W * H),
                           "evaluated_per_px": n_eval_total / (W * H),
                           "l2": "no flush: inputs larger than L2 (GT map %.2f GB, feat %.2f GB, pairs %.2f GB vs 126 MB)"
                                 % (gt.numel() * 4 / 1e9, g.feat.numel() * 4 / 1e9, 12 * M / 1e9),
                           "parallelism": f"{world} independent frame(s), one per GPU"},
                "ms": parts, "roofline": roofline, "roofline_steps": steps_roof,
                "ffma_peak_measured_tflops": 2.0 * ffma_ops / 1e12,
                "ndfd_forward": ndfd, "cpu_baseline": cpu_baseline, "e2e": e2e, "gpu_launches": launches_per_frame(W, H) * args.steps,
                "clocks": clocks}
        print(json.dumps(line), flush=True)
    if world > 1:
        dist.destroy_process_group()



# --------------------------------------------------------------------------------------------------
# the other BASELINE.json configs (parity-test cases; timed for DESIGN.md / BASELINE.md, never the bench line)
# --------------------------------------------------------------------------------------------------
def run_cuda_workload(args, local_rank: int):
    """`--workload tiny|small|large|multiview`: device-timed frames of another config, one GPU.
    tiny/small/large: step = P + S + R + F(zero, one map, finalise) of view 0.
    multiview: step = the fusion sweep over `--views` evenly spaced cameras of the 200-camera orbit
    (P + S + F per view into one accumulator, finalise once); no rendering, as BASELINE.json describes it."""
    import torch
    from paper_2505_19154_b200 import binding as fb
    from paper_2505_19154_b200 import inputs
    if not torch.cuda.is_available():
        raise RuntimeError("bench.py needs a CUDA device: the FHGS path has no CPU fallback")
    torch.cuda.set_device(local_rank)
    dev = torch.device("cuda", local_rank)
    peaks = load_peaks()
    cfg = inputs.CONFIGS[args.workload]
    scene = inputs.make_scene(cfg)
    W, H, D, n = cfg.width, cfg.height, cfg.feat_dim, scene.n
    multiview = args.workload == "multiview"
    views = [int(round(k * cfg.n_views / args.views)) % cfg.n_views for k in range(args.views)] if multiview else [0]
    cams_np = [inputs.make_camera(cfg, v) for v in views]
    cams = [fb.make_camera(c.view, c.proj, c.cam_pos, W, H) for c in cams_np]
    ctx = fb.Context(local_rank)
    g = fb.Gaussians(scene.mean, scene.scale, scene.quat, scene.opacity, scene.sh, scene.feat, scene.sh_degree, device=dev)
    prm = fb.default_params(rect_mode=1 if args.rect == 'tight' else 0)
    fdt = g.feat.dtype
    # instance counts (capacity) from a capacity-0 pass per view
    vs0 = fb.ViewState(n, W, H, 0, device=dev)
    Ms = []
    for cam in cams:
        fb.project(ctx, g, cam, prm, vs0)
        try:
            Ms.append(fb.bin_sort(ctx, cam, vs0, sync=True))
        except fb.FhgsError:
            Ms.append(int(vs0.num_instances.item()))
    del vs0
    vs = fb.ViewState(n, W, H, int(max(Ms) * 1.02) + 1024, device=dev)
    if multiview:   # map values do not change the timing: one seeded unit-norm map stands in for every view's map
        gen = torch.Generator(device=dev).manual_seed(cfg.seed)
        gt = torch.randn((H, W, D), generator=gen, device=dev, dtype=torch.float32)
        gt /= gt.norm(dim=-1, keepdim=True)
    else:
        gt = torch.from_numpy(inputs.make_gt_map(cfg, 0, cams_np[0])).to(dev)
    f32 = torch.float32
    out_rgb = torch.empty((H, W, 3), dtype=f32, device=dev)
    out_feat = None if multiview else torch.empty((H, W, D), dtype=fdt, device=dev)
    out_n = torch.empty((H, W), dtype=torch.int32, device=dev)
    num = torch.zeros((n, D), dtype=f32, device=dev)
    den = torch.zeros((n,), dtype=f32, device=dev)
    fused = g.feat.clone()
    stream = torch.cuda.current_stream()
    NAMES = ["project", "bin_sort", "render", "fuse"]
    acc = {k: 0.0 for k in NAMES}

    def step(evs=None):
        for vi, cam in enumerate(cams):
            e = [torch.cuda.Event(enable_timing=True) for _ in range(5)] if evs is not None else None
            def mark(i):
                if e is not None:
                    e[i].record(stream)
            mark(0)
            fb.project(ctx, g, cam, prm, vs)
            mark(1)
            fb.bin_sort(ctx, cam, vs, sync=False)
            mark(2)
            if not multiview:
                fb.render(ctx, g, cam, prm, vs, out_rgb, out_feat, None, out_n)
            mark(3)
            flags = (fb.FHGS_FUSE_ZERO if vi == 0 else 0) | (fb.FHGS_FUSE_FINALIZE if vi == len(cams) - 1 else 0)
            fb.fuse_features(ctx, cam, prm, vs, gt, num, den, fused, flags)
            mark(4)
            if evs is not None:
                evs.append(e)

    for _ in range(max(args.warmup, 3)):
        step()
    torch.cuda.synchronize()
    sampler = ClockSampler(local_rank)
    sampler.start()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    evs = []
    e0.record(stream)
    for _ in range(args.steps):
        step(evs)
    e1.record(stream)
    torch.cuda.synchronize()
    clocks = sampler.stop()
    total_ms = e0.elapsed_time(e1)
    for e in evs:
        for i, nm in enumerate(NAMES):
            acc[nm] += e[i].elapsed_time(e[i + 1]) / args.steps
    # contributor counts (RGB-only render per view, outside the timed region) for the FP32 accounting
    n_contrib = 0
    for cam in cams:
        fb.project(ctx, g, cam, prm, vs)
        fb.bin_sort(ctx, cam, vs, sync=False)
        fb.render(ctx, g, cam, prm, vs, out_rgb, None, None, out_n)
        n_contrib += int(out_n.to(torch.int64).sum().item())
    # NEXT-4 (ii), per-pixel regime only (D not a multiple of 64): steps R + F as two calls against fhgs_render_fuse
    single = None
    if not multiview and D % 64 != 0 and len(cams) == 1:
        def r_then_f():
            fb.render(ctx, g, cams[0], prm, vs, out_rgb, out_feat, None, out_n)
            fb.fuse_features(ctx, cams[0], prm, vs, gt, num, den, None, 0)

        def r_and_f():
            fb.render_fuse(ctx, g, cams[0], prm, vs, out_rgb, out_feat, gt, num, den, out_ncontrib=out_n)
        ms2 = []
        for fn in (r_then_f, r_and_f):
            for _ in range(5):
                fn()
            ea, eb = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            ea.record(stream)
            for _ in range(50):
                fn()
            eb.record(stream)
            torch.cuda.synchronize()
            ms2.append(ea.elapsed_time(eb) / 50)
        single = {"render_then_fuse_ms": ms2[0], "render_fuse_ms": ms2[1], "note": "accumulate only (no clear / finalise)"}
    alu_nominal = 148 * FP32_LANES_PER_SM * peaks["sm_max_mhz"] * 1e6
    roof = {}
    if not multiview:
        roof["render"] = {"bound": "alu", "ms": acc["render"],
                          "frac": (15 + D) * n_contrib / (acc["render"] * 1e-3) / alu_nominal}
    roof["fuse"] = {"bound": "alu", "ms": acc["fuse"], "frac": (13 + D) * n_contrib / (acc["fuse"] * 1e-3) / alu_nominal,
                    "hbm_gbs_gt_maps": len(cams) * W * H * D * gt.element_size() / (acc["fuse"] * 1e-3) / 1e9,
                    "note": "includes zeroing num/den and the finalise pass"}
    unit = "view-sweeps/s" if multiview else UNIT
    line = {"metric": f"[{args.workload}] " + ("multi-view fusion sweeps/s" if multiview else "rendered+fused frames/s"),
            "value": args.steps / (total_ms * 1e-3), "unit": unit, "n_gpus": 1, "steps": args.steps,
            "warmup": max(args.warmup, 3), "ms_per_step": total_ms / args.steps, "higher_is_better": True,
            "scaling": "weak", "vs_baseline": None, "dtype": "f32", "data": "synthetic",
            "config": {"workload": f"{args.workload}: N={n} SH{scene.sh_degree} D={D} {cfg.feat_dtype}, {len(cams)} view(s) {W}x{H}"
                                   " [parity-test config, not the bench line]",
                       "views": views, "instances_M": Ms, "contributors_per_px": n_contrib / (W * H * len(cams)),
                       "gt": "one seeded unit-norm map reused for every view (values do not affect timing)" if multiview
                             else "inputs.make_gt_map"},
            "ms": acc, "ms_per_view": total_ms / args.steps / len(cams), "roofline_steps": roof,
            "single_traversal": single, "cpu_baseline": None,
            "e2e": None, "gpu_launches": None, "clocks": clocks}
    print(json.dumps(line), flush=True)

# --------------------------------------------------------------------------------------------------
# BASELINE.json configs[4] as stated: the 200-view fusion sweep, on 1 GPU or view-sharded over N ranks
# --------------------------------------------------------------------------------------------------
def run_multiview_sweep(args, rank: int, world: int, local_rank: int):
    """`--workload multiview --views V` (V = 200 is the config): every view's GT map is generated on the device
    (inputs.make_gt_map_blobs_torch, seeded per view) OUTSIDE the timed spans, then P + S + F of that view are timed
    with CUDA events; the accumulators persist across the views, one finalise at the end.  With N ranks (torchrun) the
    views are sharded round-robin through parallel.fuse_views_sharded: private accumulators per rank, ONE NCCL
    all-reduce(sum) of num [N,D] and den [N], finalise on every rank.  Reported: end-to-end device time of the sweep
    (sum of the timed spans + all-reduce + finalise, max over ranks), views/s over all ranks, per-view mean; and two
    invariants of the result: conservation sum_i den_i = sum_views sum_x (1 - T_final(x))
    against RGB-only renders of the same views, and the cosine between every well-covered Gaussian's fused vector and
    its blob's vector."""
    import torch
    import torch.distributed as dist
    from paper_2505_19154_b200 import binding as fb
    from paper_2505_19154_b200 import inputs, parallel
    if not torch.cuda.is_available():
        raise RuntimeError("bench.py needs a CUDA device: the FHGS path has no CPU fallback")
    torch.cuda.set_device(local_rank)
    dev = torch.device("cuda", local_rank)
    if world > 1:
        dist.init_process_group("nccl", device_id=dev)
    cfg = inputs.CONFIGS["multiview"]
    if args.small:
        cfg = inputs.scaled(cfg, n=100_000, width=432, height=320, log_scale_mu=-3.2)
    scene = inputs.make_scene(cfg)
    W, H, D, n = cfg.width, cfg.height, cfg.feat_dim, scene.n
    views = [int(round(k * cfg.n_views / args.views)) % cfg.n_views for k in range(args.views)]
    ctx = fb.Context(local_rank)
    g = fb.Gaussians(scene.mean, scene.scale, scene.quat, scene.opacity, scene.sh, scene.feat, scene.sh_degree, device=dev)
    prm = fb.default_params(rect_mode=1 if args.rect == "tight" else 0)
    capacity = int(48e6) if not args.small else int(8e6)     # > the largest view of the orbit (2.2e7 instances; checked below)
    vs = fb.ViewState(n, W, H, capacity, device=dev)
    f32 = torch.float32
    gt = torch.empty((H, W, D), dtype=f32, device=dev)
    num = torch.empty((n, D), dtype=f32, device=dev)
    den = torch.empty((n,), dtype=f32, device=dev)
    fused = g.feat.clone()
    out_rgb = torch.empty((H, W, 3), dtype=f32, device=dev)
    out_T = torch.empty((H, W), dtype=f32, device=dev)
    stream = torch.cuda.current_stream()
    spans, Ms, one_minus_T = [], [], [0.0]

    def fuse_one_view(v, first):
        cam_np = inputs.make_camera(cfg, v)
        cam = fb.make_camera(cam_np.view, cam_np.proj, cam_np.cam_pos, W, H)
        inputs.make_gt_map_blobs_torch(cfg, v, cam_np, dev, out=gt)          # not timed
        e = [torch.cuda.Event(enable_timing=True) for _ in range(4)]
        e[0].record(stream)
        fb.project(ctx, g, cam, prm, vs)
        e[1].record(stream)
        fb.bin_sort(ctx, cam, vs, sync=False)
        e[2].record(stream)
        fb.fuse_features(ctx, cam, prm, vs, gt, num, den, None, fb.FHGS_FUSE_ZERO if first else 0)
        e[3].record(stream)
        spans.append(e)
        # the invariants' reference, outside the timed spans: RGB-only render of the same view state
        fb.render(ctx, g, cam, prm, vs, out_rgb, None, out_T, None)
        one_minus_T[0] += float((1.0 - out_T.double()).sum().item())
        m = int(vs.num_instances.item())
        if m > capacity:
            raise RuntimeError(f"view {v}: {m} instances exceed the capacity {capacity}")
        Ms.append(m)

    ev = [torch.cuda.Event(enable_timing=True) for _ in range(3)]

    def finalize():
        ev[1].record(stream)
        fb.fuse_features(ctx, None, prm, vs, None, num, den, fused, fb.FHGS_FUSE_FINALIZE_ONLY)
        ev[2].record(stream)

    # warm-up: three views into scratch accumulators (module load, clocks), then the sweep
    for v in views[:3]:
        fuse_one_view(v, True)
    torch.cuda.synchronize()
    spans.clear(); Ms.clear(); one_minus_T[0] = 0.0
    sampler = ClockSampler(local_rank)
    sampler.start()
    t_wall = time.perf_counter()
    # parallel.fuse_views_sharded: this rank's views, then the all-reduce (between ev[0] and ev[1]), then finalise
    mine = parallel.fuse_views_sharded(views, fuse_one_view, num, den, finalize, before_reduce=lambda: ev[0].record(stream))
    torch.cuda.synchronize()
    wall_s = time.perf_counter() - t_wall
    clocks = sampler.stop()
    parts = {"project": 0.0, "bin_sort": 0.0, "fuse": 0.0}
    for e in spans:
        for i, k in enumerate(parts):
            parts[k] += e[i].elapsed_time(e[i + 1])
    parts["all_reduce"] = ev[0].elapsed_time(ev[1]) if world > 1 else 0.0
    parts["finalize"] = ev[1].elapsed_time(ev[2])
    sweep_ms = parallel.max_over_ranks(sum(parts.values()), dev)
    # invariants on the reduced result (every rank holds all of num/den after the all-reduce)
    omt = torch.tensor([one_minus_T[0]], dtype=torch.float64, device=dev)
    if world > 1:
        dist.all_reduce(omt)
    den_sum = float(den.double().sum().item())
    conservation_rel = abs(den_sum - float(omt.item())) / max(float(omt.item()), 1e-30)
    vec = torch.from_numpy(inputs.blob_vectors(cfg).astype(np.float32)).to(dev)
    centres = torch.from_numpy(inputs.blob_centres(cfg).astype(np.float32)).to(dev)
    owner = torch.arange(n, device=dev) % 64
    dist_c = (g.mean - centres[owner]).norm(dim=1)
    well = (den > 1.0) & (dist_c < 0.6)             # well covered, inside its blob's 2-sigma ball (the map's labelling radius)
    cos = torch.nn.functional.cosine_similarity(fused[well].float(), vec[owner[well]], dim=1)
    cos_stats = {"gaussians": int(well.sum().item()), "median": float(cos.median().item()),
                 "p10": float(cos.quantile(0.10).item()), "frac_above_0.9": float((cos > 0.9).float().mean().item())}
    if rank == 0:
        nv = len(views)
        line = {"metric": "[multiview] fused views/s (BASELINE.json configs[4]: P+S+F per view, one finalise)",
                "value": nv / (sweep_ms * 1e-3), "unit": "views/s", "n_gpus": world, "steps": 1, "warmup": 3,
                "ms_per_step": sweep_ms, "higher_is_better": True, "scaling": "strong", "vs_baseline": None, "dtype": "f32",
                "data": "synthetic",
                "config": {"workload": f"multiview: N={n} SH{scene.sh_degree} D={D} f32, {nv} views {W}x{H} of the {cfg.n_views}-camera orbit"
                                       + (" [--small debug size]" if args.small else ""),
                           "parallelism": f"views sharded round-robin over {world} rank(s), one all-reduce(sum) of num/den",
                           "gt": "inputs.make_gt_map_blobs_torch per view on the device, outside the timed spans",
                           "views_this_rank": len(mine), "instances_M_min_mean_max": [min(Ms), sum(Ms) / len(Ms), max(Ms)]},
                "ms": parts, "ms_per_view": sweep_ms / nv * world, "end_to_end_s": sweep_ms * 1e-3,
                "wall_s_incl_map_generation_and_checks": wall_s,
                "invariants": {"conservation_rel_err": conservation_rel, "den_sum": den_sum, "one_minus_T_sum": float(omt.item()),
                               "cosine_to_blob_vector": cos_stats},
                "cpu_baseline": None, "e2e": None, "gpu_launches": None, "clocks": clocks}
        print(json.dumps(line), flush=True)
    assert conservation_rel < 2e-4, f"conservation violated: {conservation_rel}"
    if world > 1:
        dist.destroy_process_group()


# --------------------------------------------------------------------------------------------------
# NEXT-4 (v): LABELLED comparison, outside north_star's "no tensor cores" contract and outside the product path
# --------------------------------------------------------------------------------------------------
def run_tc_compare(args, local_rank: int):
    """`--tc-compare`: what the per-tile products of steps R / F would cost on the tensor cores with 3xTF32 splitting
    (SURVEY 8(f) NEXT-4 v).  Library GEMMs only (cuBLAS batched matmul through torch), on synthetic operands of the Mid
    frame's shape: one batch entry per tile, W^T [128 instances x 256 pixels] times G [256 pixels x 128 channels] (a
    tile's 106 tile-culled survivors on average, padded to 128).  3xTF32: x = hi + lo with hi = x truncated to 10
    mantissa bits; W^T G ~ hi hi + lo hi + hi lo, three TF32 GEMMs with fp32 accumulation.  Reported next to the FP32
    (CUDA-core SGEMM) form of the same batched product and to the error of each against float64.  Nothing of this is
    called by the library; libfhgs.so contains no tensor-core instruction (profiles/r02_sass_census.md)."""
    import torch
    dev = torch.device("cuda", local_rank)
    torch.manual_seed(1234)
    tiles, n_inst, px, ch = 8160, 128, 256, 128
    # weights: non-negative, most of them zero (a pixel blends ~70 of the tile's instances), rows sum to < 1 per pixel
    Wt = torch.rand((tiles, n_inst, px), device=dev) * (torch.rand((tiles, n_inst, px), device=dev) < 0.55) * 0.02
    G = torch.randn((tiles, px, ch), device=dev) / ch ** 0.5

    def split(x):
        hi = (x.view(torch.int32) & -8192).view(torch.float32)   # clear the 13 low mantissa bits: exactly a TF32 value
        return hi, x - hi

    def timed(fn, reps=5):
        for _ in range(2):
            fn()
        a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        a.record()
        for _ in range(reps):
            out = fn()
        b.record()
        torch.cuda.synchronize()
        return a.elapsed_time(b) / reps, out

    torch.backends.cuda.matmul.allow_tf32 = False
    ms_fp32, c_fp32 = timed(lambda: torch.bmm(Wt, G))
    torch.backends.cuda.matmul.allow_tf32 = True
    ms_tf32, c_tf32 = timed(lambda: torch.bmm(Wt, G))
    ms_split, parts = timed(lambda: (split(Wt), split(G)))
    (w_hi, w_lo), (g_hi, g_lo) = parts
    ms_3x, c_3x = timed(lambda: torch.bmm(w_hi, g_hi) + torch.bmm(w_lo, g_hi) + torch.bmm(w_hi, g_lo))
    torch.backends.cuda.matmul.allow_tf32 = False
    ref = torch.bmm(Wt[:64].double(), G[:64].double())
    err = lambda c: float((c[:64].double() - ref).abs().max())
    flop = 2.0 * tiles * n_inst * px * ch
    line = {"experiment": "NEXT-4 (v) tensor-core comparison -- LABELLED, outside north_star's contract, library GEMMs, not a bench line",
            "shape": {"tiles": tiles, "instances": n_inst, "pixels": px, "channels": ch, "flop_per_product": flop},
            "fp32_sgemm": {"ms": ms_fp32, "tflops": flop / ms_fp32 / 1e9, "max_abs_err_vs_f64": err(c_fp32)},
            "tf32_single": {"ms": ms_tf32, "tflops": flop / ms_tf32 / 1e9, "max_abs_err_vs_f64": err(c_tf32)},
            "tf32_3x": {"ms_gemms_and_adds": ms_3x, "ms_split": ms_split, "tflops_fp32_equivalent": flop / ms_3x / 1e9,
                        "max_abs_err_vs_f64": err(c_3x)},
            "library_kernel_for_scale": "fuse_ws_kernel<float>: 1.57 ms for the Mid frame's W^T G including traversal, weights and atomics"}
    print(json.dumps(line), flush=True)


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="cuda", choices=["cuda", "reference"])
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--small", action="store_true", help="debug-size workload (not a bench line)")
    ap.add_argument("--workload", default="mid", choices=["mid", "tiny", "small", "large", "multiview"],
                    help="mid = the bench line (BASELINE.json metric); the others are timed for the record only")
    ap.add_argument("--rect", default="radius", choices=["radius", "tight"],
                    help="tile rectangle rule: north_star's scalar 3-sigma radius (default, the bench line) or the tight per-axis extents (NEXT-4 i)")
    ap.add_argument("--ndfd", action="store_true", help="mid: also time fhgs_ndfd_forward (NEXT-1 row) on the frame")
    ap.add_argument("--tc-compare", action="store_true",
                    help="NEXT-4 (v): labelled 3xTF32 tensor-core comparison of the per-tile products (library GEMMs; not a bench line)")
    ap.add_argument("--views", type=int, default=8, help="multiview: number of evenly spaced orbit cameras per sweep")
    args = ap.parse_args()
    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    if args.impl == "reference":
        run_reference(args, rank)
        return
    if args.tc_compare:
        if rank == 0:
            run_tc_compare(args, local_rank)
        return
    if args.workload == "multiview" and (args.views > 8 or world > 1):
        run_multiview_sweep(args, rank, world, local_rank)      # the config as BASELINE.json states it (and its sharded form)
        return
    if args.workload != "mid":
        if rank == 0:
            run_cuda_workload(args, local_rank)
        return
    if world == 1 and args.gpus > 1:
        sys.stderr.write("bench.py: --gpus N > 1 must be launched with torch.distributed.run (one rank per GPU); "
                         "running rank 0 only\n")
    run_cuda(args, rank, world, local_rank)


if __name__ == "__main__":
    main()
