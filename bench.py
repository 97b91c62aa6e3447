#!/usr/bin/env python
"""bench.py — throughput of the render hot path on the paper-scale workload (BASELINE.json configs[2]).

One step = one pass of the whole path over one frame of synthetic input: pose update (a0) ->
camera setup + frustum cull + compaction (a1, a2) -> render (a3-a9) of 1024 worlds x 64 agents at
128x128, all four planes.  Poses of consecutive frames (speed / yaw-rate dynamics at dt = 0.1 s) are
resident in HBM before the timed region.  Prints ONE JSON line (see the driver's contract).

  python bench.py [--gpus N] [--steps K] [--warmup W] [--impl reference] [--workload paper|small|...]
"""
from __future__ import annotations

import argparse
import json
import os
import statistics
import subprocess
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import gp_scenes as gs  # noqa: E402

METRIC = "agent-views rendered/sec at 128x128 (1024 worlds x 64 agents, class+instance+depth+RGB)"
UNIT = "agent-views/s"
FP32_OPS_PER_TEST = 29          # contract C5 per executed slab test


def parse():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=200)
    ap.add_argument("--warmup", type=int, default=5)
    ap.add_argument("--impl", default="b200", choices=["b200", "reference"])
    ap.add_argument("--workload", default="paper", choices=list(gs.CONFIGS))
    ap.add_argument("--worlds", type=int, default=0, help="override the number of worlds (debug)")
    ap.add_argument("--res", type=int, default=0, help="override H = W (resolution sweep)")
    ap.add_argument("--hw", type=int, nargs=2, default=None, metavar=("H", "W"), help="override the image size")
    ap.add_argument("--strip-px", type=int, default=0, help="GP_OPT_STRIP_PX override (0 = library default)")
    ap.add_argument("--gather", type=int, default=-1, help="GP_OPT_GATHER override (-1 = library default)")
    ap.add_argument("--stage-cap", type=int, default=0, help="GP_OPT_STAGE_CAP override (0 = library default)")
    ap.add_argument("--variant", type=int, default=-1, help="GP_OPT_VARIANT: 0 ray strips, 1 raster tiles, -1 library default")
    ap.add_argument("--tile-px", type=int, default=0, help="GP_OPT_TILE_PX override (0 = library default)")
    ap.add_argument("--pipeline", type=int, default=0, help="GP_OPT_PIPELINE override (0 = library default = 1 = serial)")
    ap.add_argument("--t-max", type=float, default=0.0,
                    help="override the far plane (m); 0.01 empties every list: the floor of the render pass (diagnostic, not a bench config)")
    ap.add_argument("--chunk-worlds", type=int, default=0,
                    help="worlds per gp_render_batch call (0 = as many as keep the planes under 40 GB)")
    ap.add_argument("--graph", action="store_true",
                    help="capture each step (pose update + cull + render) in a CUDA graph and time the replays")
    ap.add_argument("--e2e-steps", type=int, default=2)
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-sim", action="store_true", help="skip the dynamics + O_vec + render leg (agent steps / s)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-configs", action="store_true",
                    help="skip the `configs` block (the other BASELINE.json configurations, timed after the headline region)")
    ap.add_argument("--launch-check", action="store_true",
                    help="CPU dry run of the multi-rank launch: rendezvous over gloo, one max-over-ranks reduction, one JSON line")
    return ap.parse_args()


def peaks():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(path):
        with open(path) as f:
            return float(json.load(f)["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs, copy read+write)"
    return 6650.0, "fallback (B200_PROFILING.md 6.65 TB/s)"


class ClockSampler:
    """nvidia-smi clocks and throttle reasons DURING the timed region."""
    Q = ("clocks.sm,clocks.max.sm,clocks.mem,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        self.index, self.rows, self.proc = index, [], None

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(self.index), "--query-gpu=" + self.Q,
                                          "--format=csv,noheader,nounits", "-lms", "100"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.t = threading.Thread(target=self._read, daemon=True)
            self.t.start()
        except OSError:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append([x.strip() for x in line.split(",")])

    def stop(self):
        if not self.proc:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.15)
        self.proc.terminate()
        try:
            self.proc.wait(timeout=5)
        except subprocess.TimeoutExpired:
            self.proc.kill()
        sm, mx, mem, reasons = [], [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for r in self.rows:
            if len(r) < 7:
                continue
            try:
                sm.append(float(r[0])); mx.append(float(r[1])); mem.append(float(r[2]))
            except ValueError:
                continue
            for n, v in zip(names, r[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(n)
        return {"sm_mhz": statistics.median(sm) if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "mem_mhz": statistics.median(mem) if mem else None, "samples": len(sm), "reasons": sorted(reasons)}


def workload_cfg(args):
    cfg = gs.config(args.workload)
    if args.worlds:
        cfg = cfg.replace(n_worlds=args.worlds)
    if args.res:
        cfg = cfg.replace(H=args.res, W=args.res)
    if args.hw:
        cfg = cfg.replace(H=args.hw[0], W=args.hw[1])
    if getattr(args, "t_max", 0.0) > 0.0:
        cfg = cfg.replace(t_max=args.t_max)
    return cfg


def config_dict(cfg, extra=None):
    d = {"workload": "%s: %d worlds x %d agents x %d camera(s) + %d quads, %dx%d px (HxW), %.0f m extent, 4 planes" % (
        cfg.name, cfg.n_worlds, cfg.agents, cfg.cams, cfg.quads, cfg.H, cfg.W, cfg.extent),
        "baseline_config": "BASELINE.json configs[2] (paper-scale)" if cfg.name == "paper" else cfg.name,
        "views_per_step": cfg.views, "pixels_per_step": cfg.views * cfg.H * cfg.W,
        "worlds_per_render_call": (extra or {}).get("worlds_per_render_call", cfg.n_worlds),
        "l2": "outputs per step (%.2f GB) far exceed the 126 MB L2; no explicit flush" % (cfg.views * cfg.H * cfg.W * 12 / 1e9)}
    if cfg.t_max != gs.config(cfg.name).t_max:
        d["diagnostic"] = "far plane overridden to %g m (--t-max): NOT a BASELINE.json configuration" % cfg.t_max
    if extra:
        d.update(extra)
    return d


# ------------------------------------------------------------------------------------------------
def oracle_sample(cfg, n_views, threads):
    """The oracle as it stands over the first n_views views of the workload (frame 0); returns seconds."""
    import oracle
    vpw = cfg.agents * cfg.cams
    n_w = (n_views + vpw - 1) // vpw
    sub = cfg.replace(n_worlds=n_w)
    agents, quads = gs.gen_world_prims(sub)
    prims = np.concatenate([agents, quads], axis=1)
    pitch = gs.gen_pitch(sub) if cfg.pitch_deg_max > 0 else None
    par = oracle.make_params(cam_height=cfg.cam_height, t_max=cfg.t_max, fov_rad=float(np.float32(cfg.fov_rad)))
    rig = gs.rig_array(cfg.rig)
    views = [(v // vpw, (v % vpw) // cfg.cams, v % cfg.cams) for v in range(n_views)]
    oracle.render_views(prims, views[:threads], cfg.H, cfg.W, par, pitch_cs=pitch, threads=threads, rig=rig)   # page in
    t0 = time.perf_counter()
    oracle.render_views(prims, views, cfg.H, cfg.W, par, pitch_cs=pitch, threads=threads, rig=rig)
    return time.perf_counter() - t0


def run_reference(args):
    """--impl reference: the CPU oracle timed on the host cores (rank 0 only)."""
    if int(os.environ.get("RANK", "0")) != 0:
        return
    cfg = workload_cfg(args)
    threads = max(1, min(64, os.cpu_count() or 1))
    per_core_s = 0.09 * (cfg.H * cfg.W * cfg.prims) / (128 * 128 * 264)
    # bounded sample: the whole --steps/--warmup run should end within ~2.5 minutes
    step_s = min(20.0, max(0.2, 150.0 / max(1, args.steps + args.warmup)))
    n_views = max(threads, int(min(cfg.views, max(1, round(step_s * threads / per_core_s)))))
    for _ in range(args.warmup):
        oracle_sample(cfg, n_views, threads)
    t = [oracle_sample(cfg, n_views, threads) for _ in range(args.steps)]
    total = sum(t)
    value = n_views * args.steps / total
    sample = "%d views of the workload (frame 0) per step, all-primitive fp32 oracle, %d threads" % (n_views, threads)
    print(json.dumps({
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * total / args.steps,
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f32", "data": "synthetic",
        "config": config_dict(cfg, {"sample": sample}),
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": threads, "kind": "oracle", "sample": sample},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0}))


# ------------------------------------------------------------------------------------------------
# The other BASELINE.json configurations (configs[1], [3], [4]: "reporting views/sec and roofline fraction at each
# resolution") and the paper's 4-camera rig, each timed the same way after the headline region: W warm-up steps, K steps back
# to back between two CUDA events, then a short pass with per-kernel events for k_render's own time.
OTHER_CONFIGS = (
    ("small", "small", {}, "BASELINE.json configs[1]"),
    ("sweep32", "sweep", {"H": 32, "W": 32}, "BASELINE.json configs[3] at 32 px"),
    ("sweep64", "sweep", {"H": 64, "W": 64}, "BASELINE.json configs[3] at 64 px"),
    ("sweep128", "sweep", {"H": 128, "W": 128}, "BASELINE.json configs[3] at 128 px"),
    ("sweep192", "sweep", {"H": 192, "W": 192}, "BASELINE.json configs[3] at 192 px"),
    ("sweep256", "sweep", {"H": 256, "W": 256}, "BASELINE.json configs[3] at 256 px"),
    ("dense_chunk", "dense", {"n_worlds": 256}, "BASELINE.json configs[4], one 256-world chunk of its 2048 (all planes of all "
                                                "worlds are 206 GB: the full run renders such chunks into a reused buffer)"),
    ("rig4", "rig4", {}, "SURVEY 8(f) NEXT-2: 4 cameras per agent at 210 x 126 (PAPER.md:434)"),
)


def configs_block(local_rank, peak, steps=20, warmup=5):
    import torch
    from paper_2606_19641_b200 import Renderer, gp
    dev = torch.device("cuda", local_rank)
    out = {}
    for key, name, over, what in OTHER_CONFIGS:
        try:
            cfg = gs.config(name, **over)
            agents, quads = gs.gen_world_prims(cfg)
            speed, yaw_rate = gs.gen_dynamics(cfg)
            n_frames = steps + warmup
            poses = gs.poses_at_frames(cfg, agents, speed, yaw_rate, range(n_frames))
            d_pose = torch.from_numpy(np.stack([poses[f] for f in range(n_frames)])).to(dev)
            fov = float(np.float32(cfg.fov_rad))
            r = Renderer(local_rank)
            r.scene_upload(agents, quads, cam_height=cfg.cam_height, t_max=cfg.t_max)
            if cfg.pitch_deg_max > 0:
                r.cameras_set(torch.from_numpy(gs.gen_pitch(cfg)).to(dev))
            if cfg.rig != gs.RIG_FRONT:
                r.camera_rig_set(gs.rig_array(cfg.rig))
            outs = r.alloc_outputs(cfg.views, cfg.H, cfg.W, rgb=True)

            def step(f):
                r.agents_update(d_pose[f])
                r.render_batch(0, cfg.n_worlds, cfg.H, cfg.W, fov, *outs)

            for f in range(warmup):
                step(f)
            ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            torch.cuda.synchronize()
            l0 = r.launch_count()
            ev0.record()
            for f in range(warmup, n_frames):
                step(f)
            ev1.record()
            torch.cuda.synchronize()
            step_ms = ev0.elapsed_time(ev1) / steps
            launches = r.launch_count() - l0
            r.set_option(gp.GP_OPT_TIMING, 1)
            for k in (gp.GP_KERNEL_UPDATE, gp.GP_KERNEL_CULL, gp.GP_KERNEL_RENDER):
                r.kernel_time(k)
            n_k = min(8, steps)
            for f in range(warmup, warmup + n_k):
                step(f)
            kt = {nm: r.kernel_time(k)[0] / n_k for nm, k in (("update", gp.GP_KERNEL_UPDATE), ("cull", gp.GP_KERNEL_CULL),
                                                               ("render", gp.GP_KERNEL_RENDER))}
            r.set_option(gp.GP_OPT_TIMING, 0)
            npx = cfg.views * cfg.H * cfg.W
            alg_bytes = npx * 12 + cfg.n_worlds * cfg.prims * 48 + cfg.views * 64
            out[key] = {"workload": config_dict(cfg)["workload"], "baseline_config": what, "steps": steps, "warmup": warmup,
                        "ms_per_step": step_ms, "views_per_s": cfg.views / (step_ms * 1e-3),
                        "mpixels_per_s": npx / (step_ms * 1e-3) / 1e6, "kernels_ms_per_step": kt,
                        "gpu_launches": int(launches), "algorithmic_bytes_per_step": alg_bytes,
                        "k_render_frac": alg_bytes / (kt["render"] * 1e-3) / 1e9 / peak,
                        "step_frac": alg_bytes / (peak * 1e9) * 1e3 / step_ms}
            r.close()
            del outs, d_pose, r
            torch.cuda.empty_cache()
        except Exception as ex:  # noqa: BLE001 - report, do not hide
            out[key] = {"error": repr(ex)[:300]}
    out["how"] = ("each configuration: %d warm-up steps, then %d steps (pose update + cull + render of all its worlds) back to back "
                  "between two CUDA events; kernels_ms_per_step from a separate pass of up to 8 steps with an event pair around every "
                  "launch; k_render_frac = algorithmic bytes / k_render time / peak, step_frac = algorithmic bytes / peak / step "
                  "time, peak = %.1f GB/s (the headline roofline's); outputs of every configuration (>= 0.4 GB per step) exceed "
                  "the 126 MB L2; the peak is the read + write copy figure and this path only writes, so a fraction can pass 1 "
                  "(the write-only probe of the headline line is the harder ceiling)" % (warmup, steps, peak))
    return out


# ------------------------------------------------------------------------------------------------
def run_b200(args):
    import torch
    import torch.distributed as dist
    from paper_2606_19641_b200 import Renderer, gp, shard

    rank = int(os.environ.get("RANK", "0"))
    world_size = int(os.environ.get("WORLD_SIZE", "1"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    distributed = world_size > 1
    torch.cuda.set_device(local_rank)
    if distributed:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local_rank))
    dev = torch.device("cuda", local_rank)

    cfg = workload_cfg(args)
    # weak scaling: every rank renders its own cfg.n_worlds worlds (rank-disjoint world ids), no collective
    # on the data path (the path has no exchange step: PAPER.md:319).
    w0, _ = shard.weak_world_range(rank, cfg.n_worlds)
    agents, quads = gs.gen_world_prims(cfg.replace(n_worlds=w0 + cfg.n_worlds), w0, cfg.n_worlds)
    big = cfg.replace(n_worlds=w0 + cfg.n_worlds)
    speed, yaw_rate = gs.gen_dynamics(big, w0, cfg.n_worlds)
    n_frames = args.steps + args.warmup
    poses = gs.poses_at_frames(cfg, agents, speed, yaw_rate, range(n_frames))
    d_pose = torch.from_numpy(np.stack([poses[f] for f in range(n_frames)])).to(dev)   # resident in HBM
    fov = float(np.float32(cfg.fov_rad))

    r = Renderer(local_rank)
    if args.strip_px:
        r.set_option(gp.GP_OPT_STRIP_PX, args.strip_px)
    if args.stage_cap:
        r.set_option(gp.GP_OPT_STAGE_CAP, args.stage_cap)
    if args.gather >= 0:
        r.set_option(gp.GP_OPT_GATHER, args.gather)
    if args.variant >= 0:
        r.set_option(gp.GP_OPT_VARIANT, args.variant)
    if args.tile_px:
        r.set_option(gp.GP_OPT_TILE_PX, args.tile_px)
    if args.pipeline:
        r.set_option(gp.GP_OPT_PIPELINE, args.pipeline)
    r.scene_upload(agents, quads, cam_height=cfg.cam_height, t_max=cfg.t_max)
    if cfg.pitch_deg_max > 0:
        r.cameras_set(torch.from_numpy(gs.gen_pitch(big, w0, cfg.n_worlds)).to(dev))
    if cfg.rig != gs.RIG_FRONT:
        r.camera_rig_set(gs.rig_array(cfg.rig))
    # worlds per render call: the whole batch when its planes fit (paper scale: 12.9 GB), else world chunks into a
    # reused buffer (dense: 206 GB of planes in all)
    vpw = cfg.agents * cfg.cams
    chunk = args.chunk_worlds or max(1, int(40e9 // (vpw * cfg.H * cfg.W * 12)))
    chunk = min(chunk, cfg.n_worlds)
    chunks = [(w, min(chunk, cfg.n_worlds - w)) for w in range(0, cfg.n_worlds, chunk)]
    outs = r.alloc_outputs(chunk * vpw, cfg.H, cfg.W, rgb=True)
    subs = {nw: [o[:nw * vpw] for o in outs] for _, nw in chunks}

    def step(f, stats_acc=None):
        r.agents_update(d_pose[f])
        for w_begin, nw in chunks:
            r.render_batch(w_begin, nw, cfg.H, cfg.W, fov, *subs[nw])
            if stats_acc is not None:
                for k, v in r.stats().items():
                    stats_acc[k] = stats_acc.get(k, 0) + v

    def barrier():
        if distributed:
            dist.barrier()
        torch.cuda.synchronize()

    launches_per_step = 0
    for f in range(args.warmup):
        l0 = r.launch_count()
        step(f)
        launches_per_step = r.launch_count() - l0
    barrier()
    graphs = None
    if args.graph:                      # one graph per frame (each reads its own resident pose slice)
        side = torch.cuda.Stream()
        graphs = []
        with torch.cuda.stream(side):
            for f in range(args.warmup, n_frames):
                g = torch.cuda.CUDAGraph()
                with torch.cuda.graph(g, stream=side):
                    step(f)
                graphs.append(g)
        barrier()
    # per-kernel CUDA events on every 4th step of the timed region (events between all launches would space them out:
    # +0.8 % on the paper-scale step, +12 % on the small one)
    timing_every = 4 if args.steps >= 16 else 1
    r.set_option(gp.GP_OPT_TIMING, 0 if args.graph else timing_every)
    for k in (gp.GP_KERNEL_UPDATE, gp.GP_KERNEL_CULL, gp.GP_KERNEL_RENDER):
        r.kernel_time(k)
    sampler = ClockSampler(local_rank)
    if rank == 0:
        sampler.start()
    launches0 = r.launch_count()
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    barrier()
    ev0.record()
    if graphs:
        for g in graphs:
            g.replay()
    else:
        for f in range(args.warmup, n_frames):
            step(f)
    ev1.record()
    barrier()
    ms = ev0.elapsed_time(ev1)
    clocks = sampler.stop() if rank == 0 else None
    launches = r.launch_count() - launches0
    if graphs:
        # replays launch the captured kernels (1 update + cull + render per world chunk and step); per-kernel times
        # come from a short un-graphed pass after the timed region
        launches = args.steps * launches_per_step
        r.set_option(gp.GP_OPT_TIMING, 1)
        for k in (gp.GP_KERNEL_UPDATE, gp.GP_KERNEL_CULL, gp.GP_KERNEL_RENDER):
            r.kernel_time(k)
        for f in range(args.warmup, args.warmup + min(10, args.steps)):
            step(f)
    ktimes = {name: r.kernel_time(k) for name, k in (("update", gp.GP_KERNEL_UPDATE), ("cull", gp.GP_KERNEL_CULL),
                                                       ("render", gp.GP_KERNEL_RENDER))}
    r.set_option(gp.GP_OPT_TIMING, 0)
    ms = shard.max_over_ranks(ms, dev)

    # per-step distribution ("the per-frame distribution"): a separate pass after the timed region, every step
    # bracketed by its own pair of events (which spaces the launches a little: the headline stays the back-to-back figure)
    n_dist = min(args.steps, 256)
    evs = [torch.cuda.Event(enable_timing=True) for _ in range(n_dist + 1)]
    torch.cuda.synchronize()
    evs[0].record()
    for q in range(n_dist):
        step(args.warmup + q)
        evs[q + 1].record()
    torch.cuda.synchronize()
    per_step = sorted(evs[q].elapsed_time(evs[q + 1]) for q in range(n_dist))
    step_dist = {"n": n_dist, "min": per_step[0], "median": per_step[n_dist // 2], "p95": per_step[min(n_dist - 1, (n_dist * 95) // 100)],
                 "max": per_step[-1], "unit": "ms", "how": "one CUDA-event pair per step, separate pass after the timed region"}

    # one instrumented frame (not timed): executed tests and listed pairs for the FP32 roof
    r.set_option(gp.GP_OPT_STATS, 1)
    stats = {}
    step(n_frames - 1, stats)
    r.set_option(gp.GP_OPT_STATS, 0)

    # calibration probes: write-only bandwidth with the render pass's store pattern over the same output
    # planes, and the FP32 FMA rate at the clock this GPU runs it at; after the timed region, never inside it
    probes = None
    try:
        n_probe = (min(cfg.views, chunk * vpw) * cfg.H * cfg.W) // 128 * 128
        st_best, st_med = r.probe(gp.GP_PROBE_STORE, n_probe, 10, outs)
        fma_best, fma_med = r.probe(gp.GP_PROBE_FMA, 0, 10)
        sv_best = sv_med = None
        if (cfg.H * cfg.W) % 128 == 0:          # the same stream, one CTA per view as k_render maps it
            n_view = min(cfg.views, chunk * vpw) * cfg.H * cfg.W
            sv_best, sv_med = r.probe(gp.GP_PROBE_STORE_VIEW, n_view, 10, outs)
        probes = {"store_gbs_best": st_best, "store_gbs_median": st_med, "store_bytes": n_probe * 12,
                  "fma_tflops_best": fma_best, "fma_tflops_median": fma_med,
                  "store_view_gbs_best": sv_best, "store_view_gbs_median": sv_med,
                  "how": "gp_probe: 10 launches after 1 warm-up each, CUDA events; store = 12 B/px plane pattern of k_render over "
                         "the bench's own output planes; fma = 8 FFMA chains/thread, (SM count)x8 CTAs x 256 threads"}
    except Exception as ex:  # noqa: BLE001
        probes = {"error": repr(ex)[:200]}

    # the whole simulator step on the device: jerk-bicycle dynamics fused
    # with the pose update -> O_vec (nearest 16 agents, nearest 32 road segments within 100 m) -> cull -> render, no
    # host transfer; actions are resident in HBM.  Not the headline metric: reported beside it as agent steps / s.
    agent_step = None
    if not args.no_sim:
        try:
            K_OBS, M_OBS, RADIUS = 16, 32, 100.0
            sim_steps = min(args.steps, 50)
            gen = torch.Generator(device=dev); gen.manual_seed(1234 + rank)
            actions = torch.randint(0, 12, (sim_steps + 3, cfg.n_worlds, cfg.agents), dtype=torch.int32, device=dev, generator=gen)
            psi = np.arctan2(agents["sin_yaw"].astype(np.float64), agents["cos_yaw"].astype(np.float64))
            st0 = np.zeros((cfg.n_worlds, cfg.agents, 8), np.float32)
            st0[..., 0] = speed                                  # the generator's per-agent speed
            st0[..., 4] = psi
            d_state = torch.from_numpy(st0).to(dev)
            d_sp = torch.from_numpy(poses[0].copy()).to(dev)
            obs = (torch.empty((cfg.n_worlds, cfg.agents, K_OBS), dtype=torch.int32, device=dev),
                   torch.empty((cfg.n_worlds, cfg.agents, K_OBS, 8), dtype=torch.float32, device=dev),
                   torch.empty((cfg.n_worlds, cfg.agents, M_OBS), dtype=torch.int32, device=dev),
                   torch.empty((cfg.n_worlds, cfg.agents, M_OBS, 8), dtype=torch.float32, device=dev))
            dyn = gp.DynParams(0.1, 6.0, 4.0, 20.0, 0.6, 0.8, 0.5, float(cfg.extent))

            def sim_step(i):
                r.dynamics_step(dyn, actions[i], d_state, d_sp)
                r.observe_vec(d_state, K_OBS, M_OBS, RADIUS, *obs)
                for w_begin, nw in chunks:
                    r.render_batch(w_begin, nw, cfg.H, cfg.W, fov, *subs[nw])

            for i in range(3):
                sim_step(i)
            r.set_option(gp.GP_OPT_TIMING, 4 if sim_steps >= 16 else 1)
            kids = (("dynamics", gp.GP_KERNEL_DYNAMICS), ("observe", gp.GP_KERNEL_OBSERVE), ("cull", gp.GP_KERNEL_CULL),
                    ("render", gp.GP_KERNEL_RENDER))
            for _, k in kids:
                r.kernel_time(k)
            l0 = r.launch_count()
            barrier()
            ev0.record()
            for i in range(3, 3 + sim_steps):
                sim_step(i)
            ev1.record()
            barrier()
            sim_ms = shard.max_over_ranks(ev0.elapsed_time(ev1), dev)
            kt = {name: r.kernel_time(k) for name, k in kids}
            r.set_option(gp.GP_OPT_TIMING, 0)
            n_s = max(1, kt["dynamics"][1])
            agent_step = {"value": world_size * cfg.n_worlds * cfg.agents * sim_steps / (sim_ms * 1e-3), "unit": "agent steps/s",
                          "ms_per_step": sim_ms / sim_steps, "steps": sim_steps,
                          "views_per_s": world_size * cfg.views * sim_steps / (sim_ms * 1e-3),
                          "kernels_ms_per_step": {k: v[0] / n_s for k, v in kt.items()},
                          "gpu_launches": int(r.launch_count() - l0),
                          "roofline_observe": (lambda b, t: {
                              "bound": "hbm", "kernel": "k_observe_vec", "algorithmic_bytes": b, "avg_launch_ms": t,
                              "achieved": b / (t * 1e-3) / 1e9, "peak": peaks()[0], "unit": "GB/s", "frac": b / (t * 1e-3) / 1e9 / peaks()[0],
                              "note": "bytes = Wn P 48 (records) + Wn A 32 (state) read + Wn A (K + M) 36 written; the kernel is bound by "
                                      "instruction issue, not by HBM (profiles/r03_observe.md): 1528 warp instructions per agent, 75 % of "
                                      "the issue slots"})(
                              cfg.n_worlds * cfg.prims * 48 + cfg.n_worlds * cfg.agents * (32 + (K_OBS + M_OBS) * 36),
                              kt["observe"][0] / n_s),
                          "what": "gp_dynamics_step (12 random actions, dt 0.1 s, torus %g m) + gp_observe_vec (K=%d agents, M=%d road "
                                  "segments, %g m) + gp_render_batch, all on the device" % (cfg.extent, K_OBS, M_OBS, RADIUS),
                          "context": "PAPER.md:8 quotes ~50k agent steps/s on 1 GPU for its simulator with rendering (other hardware, "
                                     "nuPlan scenes, resolution unstated): context, not a like-for-like baseline"}
        except Exception as ex:  # noqa: BLE001 - report, do not hide
            agent_step = {"value": None, "unit": "agent steps/s", "error": repr(ex)[:300]}

    # end to end through the host-buffer entry point (pinned host memory, copies inside the timed region)
    e2e = None
    if not args.no_e2e:
        try:
            e2e_worlds = chunk                      # host planes of one render call (all worlds when they fit)
            V, H, W = e2e_worlds * vpw, cfg.H, cfg.W
            h = [torch.empty((V, H, W), dtype=torch.uint8), torch.empty((V, H, W), dtype=torch.int32),
                 torch.empty((V, H, W), dtype=torch.float32), torch.empty((V, 3, H, W), dtype=torch.uint8)]
            pinned = True
            try:
                h = [x.pin_memory() for x in h]
            except RuntimeError:
                pinned = False
            h_pose = [torch.from_numpy(poses[f]).pin_memory() if pinned else torch.from_numpy(poses[f])
                      for f in range(min(n_frames, args.e2e_steps + 1))]
            r.render_batch_host(h_pose[0], 0, e2e_worlds, H, W, fov, *h)            # warm-up, allocates staging
            barrier()
            t0 = time.perf_counter()
            for i in range(args.e2e_steps):
                r.render_batch_host(h_pose[(i + 1) % len(h_pose)], 0, e2e_worlds, H, W, fov, *h)   # synchronises
            barrier()
            e_s = time.perf_counter() - t0
            e_s = shard.max_over_ranks(e_s, dev)
            e2e = {"value": world_size * V * args.e2e_steps / e_s, "unit": UNIT, "worlds_per_call": e2e_worlds,
                   "h2d_bytes_per_step": int(h_pose[0].numel() * 4),
                   "d2h_bytes_per_step": int(sum(x.numel() * x.element_size() for x in h)),
                   "steps": args.e2e_steps, "pinned_host": pinned,
                   "api": "gp_render_batch_host (H2D poses, render in chunks, D2H of all four planes)"}
            del h
        except Exception as ex:  # noqa: BLE001 - report, do not hide
            e2e = {"value": None, "unit": UNIT, "error": repr(ex)[:200]}

    if rank != 0:
        if distributed:
            dist.destroy_process_group()
        return

    views_total = world_size * cfg.views * args.steps
    value = views_total / (ms * 1e-3)
    npx = cfg.views * cfg.H * cfg.W
    peak, peak_src = peaks()
    alg_bytes = npx * 12 + cfg.n_worlds * cfg.prims * 48 + cfg.views * 64
    r_ms, r_n = ktimes["render"]
    r_avg_ms = r_ms / max(1, r_n)
    steps_sampled = max(1, ktimes["update"][1])                # one pose update per step
    render_launches_per_step = max(1.0, r_n / steps_sampled)   # render calls x pipeline chunks per call (GP_OPT_PIPELINE)
    alg_bytes_launch = alg_bytes / render_launches_per_step    # one render launch = one world chunk of the pipeline
    achieved = alg_bytes_launch / (r_avg_ms * 1e-3) / 1e9
    # dram bytes of one k_render launch from a COMMITTED ncu --set full capture of this command (not measured live:
    # a run under the profiler is never a bench run); the file names its source captures
    traffic, traffic_source = None, None
    for tname in ("r03_traffic.txt", "r02_traffic.txt"):
        tpath = os.path.join(ROOT, "profiles", tname)
        if traffic is None and os.path.exists(tpath) and not args.worlds and not args.hw:
            for line in open(tpath):
                part = line.split()
                if len(part) >= 2 and part[0] == (cfg.name if not args.res else "%s%d" % (cfg.name, args.res)):
                    traffic = int(part[1])
                    traffic_source = "profiles/%s (dram__bytes_read.sum + dram__bytes_write.sum of one k_render launch, earlier " \
                                     "ncu --set full capture; see profiles/r02_render_cull_full.md)" % tname
    sm_mhz = (clocks or {}).get("sm_mhz") or 1965.0
    fp32_nominal = 148 * 128 * 2 * sm_mhz * 1e6
    fp32_peak = (probes or {}).get("fma_tflops_best", 0) * 1e12 or fp32_nominal
    wr_peak = (probes or {}).get("store_gbs_best")
    wv_peak = (probes or {}).get("store_view_gbs_best")
    t_fp32_ms = stats["executed_tests"] * FP32_OPS_PER_TEST / fp32_peak * 1e3
    t_hbm_ms = alg_bytes / (peak * 1e9) * 1e3
    step_ms = ms / args.steps
    out = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world_size, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": step_ms, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f32", "data": "synthetic",
        "config": config_dict(cfg, {"worlds_per_render_call": chunk}),
        "mpixels_per_s": value * cfg.H * cfg.W / 1e6,
        "clocks": clocks,
        "gpu_launches": int(launches),
        "kernels_ms_per_step": {k: v[0] / steps_sampled for k, v in ktimes.items()},
        "kernel_samples": {k: int(v[1]) for k, v in ktimes.items()},
        "kernels_note": "per-kernel times come from the steps sampled with GP_OPT_TIMING (every %d-th): those launches carry a CUDA "
                        "event between the cull and the render, so the programmatic-dependent-launch overlap of the back-to-back "
                        "steps (ms_per_step) is not in them" % timing_every,
        "cuda_graph": bool(graphs),
        "step_ms_distribution": step_dist,
        "roofline": {"bound": "hbm", "kernel": "k_render", "achieved": achieved, "peak": peak, "unit": "GB/s",
                     "frac": achieved / peak, "traffic": traffic, "traffic_source": traffic_source, "peak_source": peak_src,
                     "peak_write_only": wr_peak, "frac_write_only": (achieved / wr_peak) if wr_peak else None,
                     "peak_write_only_source": "gp_probe(GP_PROBE_STORE) in this run: write-only kernel with k_render's store pattern",
                     "peak_view_pattern": wv_peak, "frac_view_pattern": (achieved / wv_peak) if wv_peak else None,
                     "peak_view_pattern_source": "gp_probe(GP_PROBE_STORE_VIEW) in this run: the same write-only stream with "
                                                 "k_render's CTA -> address mapping (one CTA per view)",
                     "algorithmic_bytes_per_launch": alg_bytes_launch, "avg_launch_ms": r_avg_ms,
                     "launches_per_step": render_launches_per_step, "share_of_step": r_ms / steps_sampled / step_ms,
                     "note": ("GP_OPT_PIPELINE = %d: the culls of later world chunks run concurrently with these launches on a second "
                              "stream" % args.pipeline) if args.pipeline > 1 else
                             "one k_render launch per render call, launched with programmatic stream serialisation behind the cull"},
        "roofline_step": {"t_hbm_ms": t_hbm_ms, "t_fp32_ms": t_fp32_ms, "frac_of_slower_roof": max(t_hbm_ms, t_fp32_ms) / step_ms,
                          "executed_tests": stats["executed_tests"], "listed_pairs": stats["listed_pairs"],
                          "frac_of_write_only_roof": (alg_bytes / (wr_peak * 1e9) * 1e3 / step_ms) if wr_peak else None,
                          "tests_per_pixel": stats["executed_tests"] / npx, "fp32_peak_tflops": fp32_peak / 1e12,
                          "fp32_peak_source": "gp_probe(GP_PROBE_FMA) in this run" if (probes or {}).get("fma_tflops_best") else
                                              "nominal 148 SM x 128 lanes x 2 x sampled SM clock",
                          "fp32_nominal_tflops": fp32_nominal / 1e12,
                          "fp32_ops_per_test": FP32_OPS_PER_TEST},
        "e2e": e2e,
        "agent_step": agent_step,
        "probes": probes,
    }
    if not args.no_cpu_baseline and world_size == 1:
        threads = max(1, min(64, os.cpu_count() or 1))
        per_core_s = 0.09 * (cfg.H * cfg.W * cfg.prims) / (128 * 128 * 264)
        n_views = int(min(cfg.views, max(threads, round(40.0 * threads / per_core_s))))
        sec = oracle_sample(cfg, n_views, threads)
        n1 = max(1, min(cfg.views, int(round(1.5 / per_core_s))))
        sec1 = oracle_sample(cfg, n1, 1)
        out["cpu_baseline"] = {"value": n_views / sec, "unit": UNIT, "cores": threads, "kind": "oracle",
                               "note": "the oracle is the plain definition: every primitive of the world per pixel, scalar C, no culling; "
                                       "a reported baseline, not a tuned CPU renderer",
                               "one_core": {"value": n1 / sec1, "unit": UNIT, "sample": "%d views, 1 thread, %.1f s" % (n1, sec1)},
                               "sample": "%d views of the workload (frame 0), all-primitive fp32 oracle (oracle/gp_oracle.c), %d threads, %.1f s"
                                         % (n_views, threads, sec)}
    if cfg.name == "paper" and not (args.no_configs or args.worlds or args.res or args.hw or distributed):
        r.close()
        del outs, subs, d_pose
        torch.cuda.empty_cache()
        out["configs"] = configs_block(local_rank, peak)
    print(json.dumps(out))
    if distributed:
        dist.destroy_process_group()


def launch_check(args):
    """CPU dry run of the N-rank launch (no GPU): every rank joins a gloo group, the ranks take one max-over-ranks reduction
    as the timed region does, rank 0 prints one JSON line."""
    import torch.distributed as dist
    from paper_2606_19641_b200 import shard
    rank, world_size = int(os.environ.get("RANK", "0")), int(os.environ.get("WORLD_SIZE", "1"))
    if world_size > 1:
        dist.init_process_group("gloo")
    w0, nw = shard.weak_world_range(rank, 4)
    slowest = shard.max_over_ranks(1.0 + rank)
    if world_size > 1:
        dist.barrier()
        dist.destroy_process_group()
    if rank == 0:
        print(json.dumps({"launch_check": True, "n_gpus": world_size, "asked_gpus": args.gpus, "slowest_rank_ms": slowest,
                          "rank0_worlds": [w0, nw]}))


def spawn_ranks(args):
    """`python bench.py --gpus N` started without a launcher: start the N ranks here, one per GPU, the way the driver's
    torchrun line does, and pass their exit code on."""
    import socket
    s = socket.socket(); s.bind(("127.0.0.1", 0)); port = s.getsockname()[1]; s.close()
    env = dict(os.environ)
    if "NCCL_DEBUG" not in env:         # keep NCCL's communicator log, but out of stdout (ONE JSON line is printed there)
        env["NCCL_DEBUG"] = "INFO"
        env.setdefault("NCCL_DEBUG_FILE", "/tmp/gp_bench_nccl.%h.%p.log")
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", str(args.gpus),
           "--master-addr", "127.0.0.1", "--master-port", str(port), os.path.abspath(__file__), *sys.argv[1:]]
    return subprocess.call(cmd, env=env)


def main():
    args = parse()
    if args.impl == "reference":
        run_reference(args)
        return
    if args.gpus > 1 and "WORLD_SIZE" not in os.environ:
        sys.exit(spawn_ranks(args))
    if args.launch_check:
        launch_check(args)
    else:
        run_b200(args)


if __name__ == "__main__":
    main()
