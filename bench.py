#!/usr/bin/env python
"""bench.py -- frames/sec of the forward 3DGS render (BASELINE.json `metric`) on synthetic scenes, 1 line of JSON.

  python bench.py [--gpus N] [--steps K] [--warmup W] [--config C] [--impl reference]

A STEP is one pass of the whole hot path (preprocess -> duplication + sort -> render) over every
camera pose of a configuration: `poses` frames.  BASELINE.json's metric is "frames/sec per config", so WITHOUT --config
all five configurations are measured, each with its own W warm-up and K timed steps; the top-level `value`, `config`,
`roofline`, `e2e` and `cpu_baseline` are those of configs[4] (10 M Gaussians, 3840x2160: the largest single-GPU
workload, whose sort and render times BASELINE.json wants reported separately) and `per_config` holds the same fields
for every configuration.  All five fit one GPU (config 4 needs ~21.5 GB of workspace).  With --config C only that one is
measured and it is the headline.  Every configuration also gets a companion entry `with_tile_cull` (configs 3-5 also `with_exact_tile_cull`, gs_set_tile_cull(2)): the same measurement
(no e2e, no CPU baseline) with gs_set_tile_cull(1) -- tighter tile rects, same image; the top-level
numbers are always the standard 3-sigma rect of BASELINE.json's north_star.
`value` = frames/s with the scene resident in HBM, device-timed (CUDA events on the launching stream around every step,
L2 flushed before every step, max over ranks).  `latency` = one frame at a time, L2 flushed before every frame.
`e2e` = the same metric through the public API with HOST buffers: every step copies the scene host->device from pinned
memory, renders every pose and copies every image back.  N > 1 runs N independent replicas (DESIGN.md "Multi-GPU":
replicas only; no data-path collective); `--gpus N` without a torchrun environment re-launches itself under
torch.distributed.run with N ranks.

`--impl reference` times the CPU oracle (oracle/, test infrastructure) on the same workload: one bounded sample per step.
"""
from __future__ import annotations

import argparse
import json
import os
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "frames/sec (fwd render)"
UNIT = "frames/s"
FP32_LANES_PER_SM = 128          # FP32 FMA lanes per SM per clock (mb probe: FFMA 3.8-4.0 warp-instr/clk/SM)
INSTR_PER_PAIR = 14              # FP32-pipe thread-instructions per evaluated (pixel, Gaussian) pair
L2_FLUSH_BYTES = 256 << 20       # > 126 MB L2
HEADLINE_CONFIG = 5               # BASELINE.json configs[4]: the largest single-GPU workload


def _peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        d = json.load(open(p))
        return dict(hbm_gbs=float(d["hbm_gbs"]), sm_max_mhz=float(d.get("sm_max_mhz", 1965.0)), source="measured")
    return dict(hbm_gbs=6650.0, sm_max_mhz=1965.0, source="fallback")


class ClockSampler(threading.Thread):
    """Samples SM clock and clock-event reasons through NVML while the timed region runs."""

    def __init__(self, torch_index: int, period_s: float = 0.005):
        super().__init__(daemon=True)
        self.period, self.samples, self.reasons, self.stop_flag = period_s, [], set(), False
        self.h, self.sm_max, self.nv = None, None, None
        try:
            import pynvml as nv
            import torch
            nv.nvmlInit()
            self.nv = nv
            try:
                uuid = str(torch.cuda.get_device_properties(torch_index).uuid)
                self.h = nv.nvmlDeviceGetHandleByUUID(("GPU-" + uuid) if not uuid.startswith("GPU-") else uuid)
            except Exception:
                vis = os.environ.get("CUDA_VISIBLE_DEVICES")
                idx = int(vis.split(",")[torch_index]) if vis and vis.split(",")[torch_index].isdigit() else torch_index
                self.h = nv.nvmlDeviceGetHandleByIndex(idx)
            self.sm_max = int(nv.nvmlDeviceGetMaxClockInfo(self.h, nv.NVML_CLOCK_SM))
        except Exception as e:  # NVML unavailable: report it, never fake numbers
            self.err = repr(e)

    NAMES = (("hw_slowdown", 0x8), ("hw_thermal_slowdown", 0x40), ("sw_thermal_slowdown", 0x20), ("sw_power_cap", 0x4),
             ("hw_power_brake_slowdown", 0x80), ("sync_boost", 0x10), ("applications_clocks_setting", 0x2))

    def run(self):
        if self.h is None:
            return
        nv = self.nv
        while not self.stop_flag:
            try:
                self.samples.append(int(nv.nvmlDeviceGetClockInfo(self.h, nv.NVML_CLOCK_SM)))
                r = int(nv.nvmlDeviceGetCurrentClocksEventReasons(self.h))
                for name, bit in self.NAMES:
                    if r & bit:
                        self.reasons.add(name)
            except Exception:
                pass
            time.sleep(self.period)

    def result(self):
        self.stop_flag = True
        if self.h is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": [], "error": getattr(self, "err", "nvml unavailable")}
        self.join(timeout=1.0)
        s = sorted(self.samples)
        return {"sm_mhz": (s[len(s) // 2] if s else None), "sm_max_mhz": self.sm_max, "reasons": sorted(self.reasons),
                "samples": len(s)}


def _dist():
    ws = int(os.environ.get("WORLD_SIZE", "1"))
    return ws, int(os.environ.get("RANK", "0")), int(os.environ.get("LOCAL_RANK", "0"))


# Replicas only: the ranks never exchange data-path bytes; torch.distributed carries the barrier
# around the timed region and the max-over-ranks of the device time.  Backend-agnostic so that the world-size-2 gloo
# test (tests/test_replicas_gloo.py) exercises exactly these functions on CPU.
def replica_barrier(ws):
    if ws > 1:
        import torch.distributed as dist
        dist.barrier()


def replica_max(x, ws, device):
    if ws == 1:
        return float(x)
    import torch
    import torch.distributed as dist
    t = torch.tensor([float(x)], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def aggregate_fps(ws, frames_per_rank, slowest_rank_ms):
    """Whole-job frames/s: every rank rendered `frames_per_rank` frames; time = the slowest rank's device time."""
    return ws * frames_per_rank / (slowest_rank_ms * 1e-3)


# ----------------------------------------------------------------------------------------------------------------
# the CPU oracle, as it stands, on the host cores: `cpu_baseline` of our arm and the whole reference arm
# ----------------------------------------------------------------------------------------------------------------
ORACLE_SAMPLE_TILES = {1: None, 2: None, 3: None, 4: 8, 5: 96}   # None: whole frames; else tiles per sampled frame


class OracleSampler:
    """Times the oracle on a BOUNDED sample of a configuration.  Configs 1-3: whole frames (one pose per call, cycling).
    Configs 4-5 (minutes per frame): per call the per-Gaussian preprocess and the duplication pass of the WHOLE frame plus
    the sorted lists and the pixels of a fixed random subset of tiles; a frame is then estimated as t_fixed + (t_sample -
    t_fixed) * n_tiles / n_sample, with t_fixed (the same call on ONE tile: preprocess + duplication pass) measured once.
    The estimate is a reported baseline, not a target."""

    def __init__(self, sc, config, cores):
        import numpy as np
        from oracle import oracle
        self.oracle, self.sc, self.config, self.cores = oracle, sc, config, cores
        self.n_pose = len(sc.cameras)
        self.k = 0
        self.n_sample = ORACLE_SAMPLE_TILES.get(config)
        cam = sc.cameras[0]
        self.n_tiles = ((cam.W + 15) // 16) * ((cam.H + 15) // 16)
        self.t_pre = None
        if self.n_sample is not None:
            self.tiles = np.sort(np.random.default_rng(config).choice(self.n_tiles, size=self.n_sample, replace=False)).astype(np.int32)
            t0 = time.perf_counter()
            oracle.render(sc, 0, tile_subset=self.tiles[:1], n_threads=cores)
            self.t_pre = time.perf_counter() - t0

    def step(self):
        """One sample; returns the estimated seconds per FRAME."""
        pose = self.k % self.n_pose
        self.k += 1
        t0 = time.perf_counter()
        if self.n_sample is None:
            self.oracle.render(self.sc, pose, n_threads=self.cores)
            return time.perf_counter() - t0
        self.oracle.render(self.sc, pose, tile_subset=self.tiles, n_threads=self.cores)
        t = time.perf_counter() - t0
        return self.t_pre + max(t - self.t_pre, 0.0) * self.n_tiles / self.n_sample

    def describe(self, n, dt):
        if self.n_sample is None:
            return "%d whole frames (poses cycling over %d) of the same workload, oracle tile-parallel on %d threads, %.1f s" % (
                n, self.n_pose, self.cores, dt)
        return ("%d samples, each the whole-frame preprocess + duplication pass and the sorted lists and pixels of %d of the %d tiles "
                "(fixed random subset); a frame is estimated as t_fixed + (t_sample - t_fixed) x %d / %d with t_fixed = %.2f s (the "
                "same call on one tile, single thread); lists and pixels on %d threads; %.1f s in all") % (n, self.n_sample, self.n_tiles, self.n_tiles, self.n_sample, self.t_pre, self.cores, dt)


def run_reference(args):
    ws, rank, _ = _dist()
    if rank != 0:
        return 0
    from paper_2606_16566_b200 import scenes
    config = args.config if args.config else HEADLINE_CONFIG
    cfg = scenes.config_defaults(config)
    sc = scenes.make_scene(config)
    cores = os.cpu_count() or 1
    smp = OracleSampler(sc, config, cores)
    for _ in range(args.warmup):
        smp.step()
    t0 = time.perf_counter()
    est = [smp.step() for _ in range(args.steps)]
    dt = time.perf_counter() - t0
    frame_s = sum(est) / len(est)
    fps = 1.0 / frame_s
    line = {"impl": "reference", "metric": METRIC, "value": fps, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": 1e3 * dt / args.steps, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "f64 blend / f32 preprocess (CPU oracle)", "data": "synthetic",
            "config": _config_dict(config, cfg, sc),
            "cpu_baseline": {"value": fps, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": smp.describe(args.steps, dt)},
            "e2e": {"value": fps, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "step": "one bounded sample of the workload per step (see cpu_baseline.sample); value = 1 / estimated seconds per frame",
            "gpu_launches": 0}
    print(json.dumps(line))
    return 0


def _config_dict(config, cfg, sc):
    return {"workload": "BASELINE.json configs[%d]: %s, %d Gaussians, %dx%d, f=%g, SH degree %d, %d poses, 16x16 tiles, seed %d" % (
        config - 1, cfg["name"], sc.P, cfg["W"], cfg["H"], cfg["f"], sc.sh_degree, len(sc.cameras), config - 1),
        "gaussians": sc.P, "width": cfg["W"], "height": cfg["H"], "sh_degree": sc.sh_degree, "poses": len(sc.cameras)}


# ----------------------------------------------------------------------------------------------------------------
# our arm: the CUDA path through the C ABI
# ----------------------------------------------------------------------------------------------------------------
def _stage_bytes(P, K_sh, n_vis, n_dup, n_coarse, n_sort_passes, max_dup):
    """Algorithmic HBM bytes per frame of the memory-bound stages.  n_coarse > 0:
    two-level binning -- the entries that are duplicated and sorted are the n_coarse (super-tile, Gaussian) pairs, and
    the expansion reads every sorted id (4) + its rect (8) and writes the n_dup ids of the tile lists once."""
    compact = P >= (1 << 20)                  # common.cuh COMPACT_MIN_P: small scenes sort all P keys
    n_sort = n_vis if compact else P
    fused = max_dup <= (4 << 20)              # common.cuh FUSED_DUP_MAX (= one-level binning)
    n_ent = n_coarse if n_coarse > 0 else n_dup
    packed = n_sort_passes == 2 and P <= (1 << 24)
    rank_bytes = n_vis * 20                   # depth-ordered id (8) + offset (4) + rect (8), read by the duplication
    if n_sort_passes == 1:
        first, rest = (4, 0) if fused else (8 + 8 + 4, 0)
    elif packed:
        first, rest = (4, 8) if fused else (8 + 8 + 4, 8)      # packed 4-byte entries between the two passes
    else:
        first, rest = (8, 16 * (n_sort_passes - 2) + 12) if fused else (8 + 16, 16 * (n_sort_passes - 2) + 12)
    dup_only = rank_bytes + n_ent * (first if fused else 8)
    sort_rest = n_ent * ((first - 8 if not fused else 0) + rest)
    if n_coarse > 0:
        sort_rest += n_coarse * 12 + n_dup * 4
    return {
        "preprocess": P * 40 + n_vis * (4 + 12 * K_sh) + P * 16 + n_vis * 64 + n_sort * 8,
        "depth_sort": 4 * 16 * n_sort,
        "offset_scan": n_vis * (8 + 16 + 4 + 8),
        "duplicate": dup_only,
        "tile_sort": sort_rest,
    }


# ncu `--set full` captures of render_b200_kernel committed under profiles/ (file named beside each number): DRAM bytes
# of one launch, and the hardware pipe utilisation / executed-work figures (A) and (B) of SURVEY.md 8(d).
PROFILED = {
    # (A) and (B) of SURVEY.md 8(d) and the DRAM traffic of one launch, from profiles/r02_render_ncu.md (ncu --set full, pose 0)
    2: {"file": "profiles/r02_render_ncu.md", "dram_bytes": 10131968, "us_under_ncu": 44.4, "fma_pipe_pct": 44.1, "xu_pipe_pct": 45.3,
        "issue_slots_pct": 68.7, "branch_uniformity_pct": 96.4, "threads_per_inst": 31.7,
        "executed_fp32_thread_ops": 539267784, "executed_mufu_thread_ops": 57513600, "executed_work_roofline_frac": 0.338},
    5: {"file": "profiles/r02_render_ncu.md", "dram_bytes": 314942976, "us_under_ncu": 582.8, "fma_pipe_pct": 42.3, "xu_pipe_pct": 47.5,
        "issue_slots_pct": 71.1, "branch_uniformity_pct": 95.0, "threads_per_inst": 31.4,
        "executed_fp32_thread_ops": 7513506416, "executed_mufu_thread_ops": 797693696, "executed_work_roofline_frac": 0.364},
}


def measure_config(config, args, ctx, tile_cull=None, light=False):
    """All measurements of one configuration on this rank; returns the result dict (rank 0 uses it).  tile_cull: override of
    the process-wide switch for this measurement; light: no e2e and no CPU baseline (the tile-cull companion entries)."""
    import torch
    from paper_2606_16566_b200 import binding, scenes
    from paper_2606_16566_b200.renderer import Renderer
    ws, rank, dev, peaks, n_sm = ctx["ws"], ctx["rank"], ctx["dev"], ctx["peaks"], ctx["n_sm"]

    cfg = scenes.config_defaults(config)
    if args.res_scale != 1:   # PAPER.md Table VI's 1x / 2x resolution axis: same scene, image and focal length scaled
        cfg = dict(cfg, W=cfg["W"] * args.res_scale, H=cfg["H"] * args.res_scale, f=cfg["f"] * args.res_scale)
    if config not in ctx["scenes"]:      # generated once per run (the 10 M-Gaussian scene takes ~25 s of numpy)
        sc0 = scenes.make_scene(config, W=cfg["W"], H=cfg["H"], f=cfg["f"]) if args.res_scale != 1 else scenes.make_scene(config)
        ctx["scenes"][config] = (sc0, Renderer.pin_scene(sc0))   # the host copy lives in pinned memory (what e2e uploads from)
    sc, pinned = ctx["scenes"][config]
    cams = sc.cameras
    n_pose = len(cams)
    W, H = cfg["W"], cfg["H"]
    if tile_cull is not None:
        binding.gs_set_tile_cull(tile_cull)

    def barrier():
        replica_barrier(ws)

    def rank_max(x):
        return replica_max(x, ws, dev)

    # ---- size the workspace: largest N_dup over the poses (+5 %) -----------------------------------------------------
    # gs_set_tile_cull(2) culls where the super-tile lists are expanded: it needs the two-level binning (capacity > 4 Mi entries)
    min_dup = (5 << 20) if binding.gs_get_tile_cull() == 2 else 0
    max_dup, need = max(1 << 21, min_dup), 0
    graph = None if args.graph < 0 else bool(args.graph)
    r = Renderer(sc.P, W, H, max_dup, device=dev, count_contrib=True, graph=graph)
    r.upload(pinned)
    overflowed = False
    for cam in cams:
        r.render(cam, count_contrib=False)
        try:
            need = max(need, r.intermediates(copy=()).n_dup)
        except binding.GsError as e:
            if e.code != binding.GS_ERR_OVERFLOW:
                raise
            need, overflowed = max(need, e.n_dup), True
    if need > max_dup or overflowed:
        del r
        torch.cuda.empty_cache()
        max_dup = max(int(need * 1.05) + 4096, min_dup)
        r = Renderer(sc.P, W, H, max_dup, device=dev, count_contrib=True, graph=graph)
        r.upload(pinned)
    # ---- statistics pass (untimed): units of the rooflines -------------------------------------------------------------
    binding.gs_set_stats(True)
    stats, per_pose = [], []
    for cam in cams:
        r.render(cam, count_contrib=True)
        stats.append(binding.gs_get_stats(r.workspace))
        it = r.intermediates(copy=())
        per_pose.append((it.n_visible, it.n_dup, it.n_coarse, int(r.out_tile_counts.sum().item())))
        max_dup = int(it.max_dup)   # the capacity the library recovered from the workspace size
    binding.gs_set_stats(False)
    launches_per_frame = binding.gs_last_launch_count()
    mean = lambda xs: float(sum(xs)) / max(len(xs), 1)
    pairs_eval = mean([s["pairs_evaluated"] for s in stats])
    pairs_blend = mean([s["pairs_blended"] for s in stats])
    staged = mean([s["entries_staged"] for s in stats])
    n_vis_m, n_dup_m, n_coarse_m = mean([p[0] for p in per_pose]), mean([p[1] for p in per_pose]), mean([p[2] for p in per_pose])
    n_list_m = mean([p[3] for p in per_pose])   # entries of the tile lists (= N_dup except with gs_set_tile_cull(2))

    flush = ctx["flush"]

    def frame(cam, e0=None, e1=None):
        flush.zero_()                       # L2 flush before every frame (outside the event pair)
        if e0 is not None:
            e0.record()
        r.render(cam, count_contrib=False)
        if e1 is not None:
            e1.record()

    # A step = every pose of the configuration once, through the public batch call: `lanes` frames in flight on their own
    # streams and workspaces (Renderer.render_batch).  The L2 is flushed before every step, outside the event pair.
    lanes = args.lanes if args.lanes > 0 else 1     # 0: chosen below, by timing warm-up steps

    def step(e0=None, e1=None):
        flush.zero_()
        if e0 is not None:
            e0.record()
        r.render_batch(cams, lanes=lanes)
        if e1 is not None:
            e1.record()

    # ---- pre-warm (clock ramp), choice of the frames in flight, W warm-up steps -----------------------------------------
    t0 = time.perf_counter()
    while time.perf_counter() - t0 < 0.3:
        step()
        torch.cuda.synchronize()
    if args.lanes <= 0:   # untimed tuning: the fastest of 1, 2, 3, 4, 6 frames in flight over a few warm-up steps (rank 0 decides)
        cands = [1, 2, 3, 4, 6] if r.workspace.numel() < (4 << 30) else [1, 2]
        best = (None, 1)
        for cand in cands:
            lanes = cand
            step(); step()
            torch.cuda.synchronize()
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            tt = 0.0
            for _ in range(3):
                step(e0, e1)
                torch.cuda.synchronize()
                tt += e0.elapsed_time(e1)
            if best[0] is None or tt < best[0]:
                best = (tt, cand)
        lanes = int(rank_max(best[1])) if ws > 1 else best[1]
    for _ in range(args.warmup):
        step()
    # ---- timed region: exactly K steps ---------------------------------------------------------------------------------------
    K = args.steps
    evs = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(K)]
    sampler = ClockSampler(ctx["lrank"])
    barrier()
    torch.cuda.synchronize()
    sampler.start()
    wall0 = time.perf_counter()
    launches = 0
    for s in range(K):
        e0, e1 = evs[s]
        step(e0, e1)
        launches += launches_per_frame * n_pose
    torch.cuda.synchronize()
    wall = time.perf_counter() - wall0
    clocks = sampler.result()
    barrier()
    dev_ms = rank_max(sum(e0.elapsed_time(e1) for e0, e1 in evs))
    ms_per_step = dev_ms / K
    fps = aggregate_fps(ws, n_pose * K, dev_ms)

    # ---- latency: one frame at a time on one stream, L2 flushed before every frame ------------------------------------------
    for cam in cams:
        frame(cam)
    n_lat = max(1, min(K, 20))
    fevs = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(n_lat * n_pose)]
    torch.cuda.synchronize()
    for s in range(n_lat):
        for i, cam in enumerate(cams):
            e0, e1 = fevs[s * n_pose + i]
            frame(cam, e0, e1)
    torch.cuda.synchronize()
    serial_ms_per_frame = rank_max(sum(e0.elapsed_time(e1) for e0, e1 in fevs) / len(fevs))

    # ---- per-stage device times: a second pass with the library's own CUDA events between its kernels -----------
    binding.gs_set_timing(True)
    acc = {n: 0.0 for n in binding.TIMING_NAMES}
    n_t = 0
    for s in range(n_lat):
        for cam in cams:
            flush.zero_()
            r.render(cam, count_contrib=False)
            t = binding.gs_get_timings(r.workspace)
            for n in acc:
                acc[n] += t[n]
            n_t += 1
    binding.gs_set_timing(False)
    stage_ms = {n: acc[n] / n_t for n in acc}

    # ---- e2e: host (pinned) buffers in, host images out, every step ---------------------------------------------------------
    e2e_fps, h2d_bytes, d2h_bytes = None, 0, 0

    def e2e_step():
        h2d = r.upload(pinned)
        r.render_batch(cams, lanes=lanes, to_host=True)   # device -> pinned host copies overlap the later frames
        r.synchronize_readback()
        return h2d
    for _ in range(0 if light else 2):
        h2d_bytes = e2e_step()
    barrier()
    torch.cuda.synchronize()
    # K steps, each with its own host -> device copy of the scene and its own device -> host copies of the images; the
    # upload of step k+1 goes to a second set of device buffers on an upload stream while step k is rendered and read back
    if not light:
        t0 = time.perf_counter()
        r.upload_async(pinned)
        for k in range(K):
            r.activate_uploaded()
            if k + 1 < K:
                r.upload_async(pinned)
            r.render_batch(cams, lanes=lanes, to_host=True)
        r.synchronize_readback()
        torch.cuda.synchronize()
        e2e_s = rank_max(time.perf_counter() - t0)
        h2d_bytes += n_pose * (16 + 16 + 3) * 4
        d2h_bytes = n_pose * 3 * H * W * 4
        e2e_fps = ws * n_pose * K / e2e_s

    # ---- rooflines ---------------------------------------------------------------------------------------------------------------------
    issue = ctx["issue"]                                    # measured on this device, this run (gs_selftest_issue_peak)
    alu_peak = max(issue["ffma"], issue["ffma2"]) / 1e12    # T FP32 thread-operations / s
    render_s = stage_ms["render"] * 1e-3
    achieved = pairs_eval * INSTR_PER_PAIR / render_s / 1e12
    prof = PROFILED.get(config) if (args.res_scale == 1 and binding.gs_get_tile_cull() == 0 and args.render_variant in (None, 4)) else None
    roofline = {"kernel": "render_b200_kernel", "bound": "alu", "achieved": achieved, "peak": alu_peak,
                "unit": "T FP32-pipe thread-instr/s", "frac": achieved / alu_peak,
                "traffic": (prof["dram_bytes"] if prof else None),
                "peak_source": "measured in this run: gs_selftest_issue_peak, max of scalar FFMA (%.2f T/s) and packed FFMA2 (%.2f T/s); "
                               "derived figure for comparison: %d SMs x %d lanes x %.0f MHz = %.2f T/s" % (
                                   issue["ffma"] / 1e12, issue["ffma2"] / 1e12, n_sm, FP32_LANES_PER_SM, peaks["sm_max_mhz"],
                                   n_sm * FP32_LANES_PER_SM * peaks["sm_max_mhz"] * 1e6 / 1e12),
                "what": "(C) of SURVEY.md 8(d): ALGORITHMIC work = (pixel, Gaussian) pairs whose alpha the blend loop evaluated x 14 "
                        "FP32-pipe thread-instructions, over the render kernel's own time",
                "sfu": {"achieved": pairs_eval / render_s / 1e12, "peak": issue["ex2"] / 1e12, "unit": "T ex2/s",
                        "frac": pairs_eval / render_s / issue["ex2"]},
                "units_per_launch": {"pairs_evaluated": pairs_eval, "instr_per_pair": INSTR_PER_PAIR,
                                     "pairs_blended": pairs_blend, "entries_staged": staged},
                "ms_per_launch": stage_ms["render"]}
    if prof:   # (A) hardware pipe utilisation and (B) executed-work roofline of the committed ncu capture of this config
        roofline["from_profile"] = dict(prof)
    gx, gy = (W + 15) // 16, (H + 15) // 16
    n_sorted_cells = ((gx + 7) // 8) * ((gy + 7) // 8) if n_coarse_m > 0 else gx * gy   # super-tiles or tiles
    n_sort_passes = (max(1, (n_sorted_cells - 1).bit_length()) + 7) // 8
    sb = _stage_bytes(sc.P, (sc.sh_degree + 1) ** 2, n_vis_m, n_dup_m, n_coarse_m, n_sort_passes, max_dup)
    kernels = []
    for n in ("preprocess", "depth_sort", "tile_grid", "offset_scan", "duplicate", "tile_sort", "render"):
        k = {"stage": n, "ms": stage_ms[n], "share": stage_ms[n] / max(stage_ms["frame"], 1e-9)}
        if n in sb:
            gbs = sb[n] / (stage_ms[n] * 1e-3) / 1e9 if stage_ms[n] > 0 else 0.0
            k.update(bound="hbm", achieved=gbs, peak=peaks["hbm_gbs"], unit="GB/s", frac=gbs / peaks["hbm_gbs"],
                     algorithmic_bytes=sb[n])
        elif n == "render":
            k.update(bound="alu", frac=roofline["frac"])
        kernels.append(k)
    sort_ms = stage_ms["depth_sort"] + stage_ms["tile_grid"] + stage_ms["offset_scan"] + stage_ms["duplicate"] + stage_ms["tile_sort"]

    cpu_baseline = None
    if rank == 0 and ws == 1 and not args.no_cpu_baseline and not light:
        cores = os.cpu_count() or 1
        smp = OracleSampler(sc, config, cores)
        budget = args.cpu_seconds
        t0 = time.perf_counter()
        est = []
        while not est or (time.perf_counter() - t0 < budget and len(est) < 4 * n_pose):
            est.append(smp.step())
        dt = time.perf_counter() - t0
        cpu_baseline = {"value": len(est) / sum(est), "unit": UNIT, "cores": cores, "kind": "oracle", "sample": smp.describe(len(est), dt)}

    res = {"metric": METRIC, "value": fps, "unit": UNIT, "n_gpus": ws, "steps": K, "warmup": args.warmup,
           "ms_per_step": ms_per_step, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
           "dtype": "f32", "data": "synthetic",
           "config": _config_dict(config, cfg, sc),
           "run": {"frames_per_step": n_pose, "l2": "flushed (256 MiB write) before every step", "frames_in_flight": lanes,
                   "parallelism": "replicas x%d" % ws, "n_dup_mean": n_dup_m, "n_list_entries_mean": n_list_m, "n_visible_mean": n_vis_m, "n_coarse_mean": n_coarse_m,
                   "binning": "two-level (8x8-tile super-tiles)" if n_coarse_m > 0 else "one-level", "res_scale": args.res_scale,
                   "render_variant": binding.gs_get_render_variant(), "tile_cull": binding.gs_get_tile_cull(), "cuda_graph": bool(r.graph), "workspace_bytes": int(r.workspace.numel())},
           "ms_per_frame": ms_per_step / n_pose, "wall_ms_per_step_incl_flush": 1e3 * wall / K,
           "latency": {"ms_per_frame": serial_ms_per_frame, "frames_per_s": ws * 1e3 / serial_ms_per_frame,
                       "how": "one frame in flight, one stream, L2 flushed before every frame"},
           "sort_ms_per_frame": sort_ms, "render_ms_per_frame": stage_ms["render"],
           "clocks": clocks,
           "e2e": {"value": e2e_fps, "unit": UNIT, "h2d_bytes_per_step": h2d_bytes, "d2h_bytes_per_step": d2h_bytes,
                   "input": "scene arrays in pinned host memory (Renderer.pin_scene), copied host -> device every step; images "
                            "copied device -> pinned host every frame; steps pipelined through a second device buffer set"},
           "gpu_launches": launches, "launches_per_frame": launches_per_frame,
           "roofline": roofline, "kernels": kernels, "stage_ms_per_frame": stage_ms,
           "cpu_baseline": cpu_baseline}
    r.close()
    del r
    torch.cuda.empty_cache()
    if tile_cull is not None:
        binding.gs_set_tile_cull(args.tile_cull)
    return res


def run_ours(args):
    import torch
    import torch.distributed as dist
    from paper_2606_16566_b200 import binding

    ws, rank, lrank = _dist()
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device -- the product path has no CPU fallback")
    torch.cuda.set_device(lrank)
    dev = torch.device("cuda", lrank)
    if ws > 1:
        dist.init_process_group("nccl", device_id=dev)
    binding.lib()  # raises if libgs.so is missing and cannot be built
    if args.render_variant is not None:
        binding.gs_set_render_variant(args.render_variant)
    binding.gs_set_tile_cull(args.tile_cull)
    ctx = {"ws": ws, "rank": rank, "lrank": lrank, "dev": dev, "peaks": _peaks(),
           "n_sm": torch.cuda.get_device_properties(dev).multi_processor_count,
           "flush": torch.empty(L2_FLUSH_BYTES, dtype=torch.uint8, device=dev), "scenes": {},
           "issue": binding.gs_selftest_issue_peak(2000)}
    configs = [args.config] if args.config else [1, 2, 3, 4, 5]
    headline = args.config if args.config else HEADLINE_CONFIG
    results = {}
    # everything runs on an ordinary (capturable) stream: the legacy default stream cannot replay CUDA graphs (gs_set_graph)
    main_stream = torch.cuda.Stream(device=dev)
    culled, exact = {}, {}
    for c in configs:
        with torch.cuda.stream(main_stream):
            results[c] = measure_config(c, args, ctx)
            if args.tile_cull == 0 and not args.no_tile_cull_entries:
                # companion entry: the same configuration with gs_set_tile_cull(1) (tighter rects, same image)
                culled[c] = measure_config(c, args, ctx, tile_cull=1, light=True)
                if c >= 3:   # ... and with gs_set_tile_cull(2), the exact ellipse-tile test (the frames that bin in two levels)
                    exact[c] = measure_config(c, args, ctx, tile_cull=2, light=True)
        if c != configs[-1]:
            ctx["scenes"].pop(c, None)   # one multi-GB scene at a time
    if rank == 0:
        line = dict(results[headline])
        line["peaks"] = dict(ctx["peaks"], issue_peak_measured=ctx["issue"])
        line["gpu_launches"] = sum(r["gpu_launches"] for r in results.values()) + sum(r["gpu_launches"] for r in culled.values()) + sum(r["gpu_launches"] for r in exact.values())
        cull_keep = ("value", "unit", "ms_per_frame", "latency", "sort_ms_per_frame", "render_ms_per_frame", "roofline", "stage_ms_per_frame", "run", "clocks")
        for c, rc in culled.items():
            results[c]["with_tile_cull"] = {k: rc[k] for k in cull_keep}
        for c, rc in exact.items():
            results[c]["with_exact_tile_cull"] = {k: rc[k] for k in cull_keep}
        if headline in culled:
            line["with_tile_cull"] = results[headline]["with_tile_cull"]
        if headline in exact:
            line["with_exact_tile_cull"] = results[headline]["with_exact_tile_cull"]
        if len(configs) > 1:
            keep = ("config", "value", "unit", "ms_per_step", "ms_per_frame", "latency", "sort_ms_per_frame", "render_ms_per_frame",
                    "e2e", "roofline", "cpu_baseline", "clocks", "gpu_launches", "launches_per_frame", "stage_ms_per_frame", "kernels", "run",
                    "with_tile_cull", "with_exact_tile_cull")
            line["per_config"] = [{k: results[c][k] for k in keep if k in results[c]} for c in configs]
            line["headline"] = "configs[%d] (top-level fields); every configuration has its own %d warm-up and %d timed steps" % (
                headline - 1, args.warmup, args.steps)
        print(json.dumps(line))
    if ws > 1:
        dist.destroy_process_group()
    return 0


def _respawn_under_torchrun(args):
    """`--gpus N` without a torchrun environment: run the same command under torch.distributed.run with N ranks."""
    import socket
    import subprocess
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        port = s.getsockname()[1]
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", str(args.gpus),
           "--master-addr", "127.0.0.1", "--master-port", str(port), os.path.abspath(__file__)] + sys.argv[1:]
    return subprocess.call(cmd)


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--config", type=int, default=0, choices=(0, 1, 2, 3, 4, 5),
                    help="0 (default): all five configurations, configs[4] as the headline; 1..5: that configuration only")
    ap.add_argument("--impl", default="ours", choices=("ours", "reference"))
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--cpu-seconds", type=float, default=8.0, help="budget of the cpu_baseline leg per configuration")
    ap.add_argument("--lanes", type=int, default=0, help="frames in flight in a step (0 = the fastest of 1-6 over a few warm-up steps)")
    ap.add_argument("--res-scale", type=int, default=1, choices=(1, 2), help="render at 1x or 2x the configuration's resolution (our arm only)")
    ap.add_argument("--tile-cull", type=int, default=0, choices=(0, 1, 2), help="gs_set_tile_cull: 1 = rects intersected with the alpha >= 1/255 bounding box, 2 = and the exact ellipse-tile test per list entry (our arm only; the default is the standard 3-sigma rect)")
    ap.add_argument("--graph", type=int, default=-1, choices=(-1, 0, 1), help="CUDA graph replay of the frame (gs_set_graph): -1 = the Renderer's default (on up to 2^21 Gaussians), 0 off, 1 on")
    ap.add_argument("--no-tile-cull-entries", action="store_true", help="skip the companion measurement of every configuration with gs_set_tile_cull(1)")
    ap.add_argument("--render-variant", type=int, default=None, help="ablation: gs_set_render_variant (default: the library default)")
    args = ap.parse_args()
    if args.gpus < 1:
        ap.error("--gpus must be >= 1")
    ws = int(os.environ.get("WORLD_SIZE", "1"))
    if args.gpus > 1 and "WORLD_SIZE" not in os.environ:
        return _respawn_under_torchrun(args)
    if ws != args.gpus:
        print("bench.py: --gpus %d but WORLD_SIZE=%d" % (args.gpus, ws), file=sys.stderr)
        return 2
    args.warmup = max(args.warmup, 3) if args.impl == "ours" else args.warmup
    if args.impl == "reference":
        return run_reference(args)
    return run_ours(args)


if __name__ == "__main__":
    sys.exit(main())
