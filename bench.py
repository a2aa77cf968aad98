#!/usr/bin/env python
"""bench.py -- the headline benchmark: reprojected frames/s at 1920x1080 (BASELINE.json metric).

Workload (N=1): BASELINE.json configs[3] -- 256^3 volume, 1920x1080 source frames, 60 display
frames with the camera dollying towards the centre, a splat + BVH rebuild every 4th frame.
One *step* = one pass of the whole hot path over one source frame: 1 splats_update (bounds,
unproject+Morton+compaction, onesweep sort, gather+box pyramid, hierarchy, node boxes; 6 launches)
followed by the 4 splats_render calls of the display frames that use that BVH.  Step k uses source frame k mod 15,
so 15 steps are exactly the scripted 60-frame sequence.  value = display frames / second, timed
with CUDA events around exactly K steps of the library as a user runs it (programmatic dependent
launches; the four renders of a step write four images and may overlap, SPLATS_OPT_OVERLAP).  The
per-kernel table and the roofline come from a second pass over the same K steps with per-stage
events on the library's stream (which serialises the stages; its rate is value_with_stage_events).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference]

N > 1 (torchrun, one rank per GPU): the path does not shard usefully below one frame
(replicas only), so every rank runs the same sequence on its own GPU
with no data-path collective ("scaling": "weak"); value = N * frames / max-over-ranks time.

--impl reference: the CPU oracle (oracle/, single thread) on the same metric and config, each
step a bounded sample of the same work.  This is the only other place oracle/ is executed.
"""
from __future__ import annotations

import argparse
import json
import os
import statistics
import sys
import threading
import time
from pathlib import Path

import numpy as np

ROOT = Path(__file__).resolve().parent
sys.path.insert(0, str(ROOT))

METRIC = "reprojected frames/s at 1920x1080 (1 BVH rebuild per 4 frames)"
UNIT = "frames/s"
FALLBACK_HBM_GBS = 6650.0   # /opt/skills/guides/B200_PROFILING.md fallback

# DRAM bytes per launch from the `ncu --set full` captures summarised under profiles/
# (dram__bytes_read.sum + dram__bytes_write.sum); None until a capture exists for that kernel.
NCU_TRAFFIC_BYTES = {
    # profiles/r01c_ncu_full_summary.txt and r01e_ncu_render_summary.txt, source frame 10 (N = 297 k), cold L2
    "bounds": 8.32e6,
    "unproject_morton_compact": 4.23e6,
    "sort": 2.73e6,        # the keys and values stay in L2 between the passes
    "tree_1": 5.39e6,
    "tree_2": 12.2e6,
    "render": 21.7e6,      # BVH + splats read once; the image stays in L2 under ncu's cache control
}


def log(*a):
    print(*a, file=sys.stderr, flush=True)


def hbm_peak():
    p = ROOT / "MEASURED_PEAKS.json"
    if p.exists():
        try:
            return float(json.loads(p.read_text())["hbm_gbs"]), "measured (MEASURED_PEAKS.json)"
        except Exception:
            pass
    return FALLBACK_HBM_GBS, "fallback (B200_PROFILING.md)"


# --------------------------------------------------------------------------- workload
def make_workload(config_index: int, n_groups: int | None):
    import synth
    cfg = synth.make_config(config_index)
    n_builds = len(cfg.src_cams) if n_groups is None else min(n_groups, len(cfg.src_cams))
    frames = []
    t0 = time.time()
    for b in range(n_builds):
        color, depth = synth.source_frame(cfg, b)
        dst = [cfg.dst_cams[i] for i, s in enumerate(cfg.dst_src) if s == b]
        frames.append(dict(color=color, depth=depth, src_cam=cfg.src_cams[b], dst_cams=dst,
                           N=int((np.isfinite(depth) & (depth > 0)).sum())))
    log(f"[bench] generated {n_builds} source frames of {cfg.name} in {time.time() - t0:.1f}s; "
        f"N per frame: {[f['N'] for f in frames]}")
    return cfg, frames


def synth_volume(cfg):
    import synth
    return synth.volume(cfg)


def algorithmic_bytes(P: int, N: int, P2: int) -> dict:
    """Compulsory DRAM traffic per launch for the layout in DESIGN.md sec. 5 (bytes)."""
    return {
        "bounds": 4 * P + 4 * (P // 2048 + 1),
        "unproject_morton_compact": 4 * P + 12 * N,
        # hybrid onesweep (default): 4 passes over the top 31 code bits x (read 12 N + write 12 N)
        # + the neighbour check reading the keys once (8 N); the all-8-pass fallback is not counted
        "sort": 4 * 24 * N + 8 * N,
        # pyramid mode: gather (perm 4, depth 4, colour 16) -> sphere 16 + rgba 16 + pyramid 32 (N entries)
        "tree_1": (4 + 4 + 16) * N + (16 + 16 + 32) * N,
        # hierarchy_kernel: keys 8 read, ranges 16 written; boxes_kernel: ranges 16 + sphere 16 + pyramid 32
        # read once, 64-byte node records written once
        "tree_2": (8 + 16) * N + (16 + 16 + 32) * N + 64 * N,
        "render": 16 * P2 + (64 + 16 + 16 + 4) * N,  # image written once + BVH/splats read once
    }


# --------------------------------------------------------------------------- clocks
class ClockSampler:
    """Samples SM clock and throttle reasons through NVML while the GPU is under load."""

    REASONS = {0x1: "gpu_idle", 0x2: "applications_clocks_setting", 0x4: "sw_power_cap", 0x8: "hw_slowdown",
               0x10: "sync_boost", 0x20: "sw_thermal_slowdown", 0x40: "hw_thermal_slowdown",
               0x80: "hw_power_brake_slowdown", 0x100: "display_clock_setting"}

    def __init__(self, index: int, period: float = 0.02):
        self.samples, self.reasons, self.max_mhz = [], set(), None
        self._stop = threading.Event()
        self._thread = None
        self.period = period
        try:
            import pynvml
            pynvml.nvmlInit()
            self.nv = pynvml
            vis = os.environ.get("CUDA_VISIBLE_DEVICES")
            if vis:
                tok = vis.split(",")[index].strip()
                index = int(tok) if tok.isdigit() else index
            self.h = pynvml.nvmlDeviceGetHandleByIndex(index)
            self.max_mhz = int(pynvml.nvmlDeviceGetMaxClockInfo(self.h, pynvml.NVML_CLOCK_SM))
        except Exception as e:  # pragma: no cover
            log(f"[bench] NVML unavailable: {e}")
            self.nv = None

    def _run(self):
        nv = self.nv
        while not self._stop.is_set():
            try:
                self.samples.append(int(nv.nvmlDeviceGetClockInfo(self.h, nv.NVML_CLOCK_SM)))
                r = int(nv.nvmlDeviceGetCurrentClocksEventReasons(self.h))
                for bit, name in self.REASONS.items():
                    if r & bit and name != "gpu_idle":
                        self.reasons.add(name)
            except Exception:
                pass
            time.sleep(self.period)

    def start(self):
        if self.nv is not None:
            self._thread = threading.Thread(target=self._run, daemon=True)
            self._thread.start()

    def stop(self) -> dict:
        self._stop.set()
        if self._thread is not None:
            self._thread.join()
        return {"sm_mhz": statistics.median(self.samples) if self.samples else None,
                "sm_max_mhz": self.max_mhz, "reasons": sorted(self.reasons), "samples": len(self.samples)}


# --------------------------------------------------------------------------- our arm
def run_ours(args):
    import torch
    from paper_2006_14726_b200 import binding as sp
    from paper_2006_14726_b200 import replicas

    world, rank, local_rank = replicas.world_info()
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device (there is no CPU fallback; use --impl reference for the oracle)")
    torch.cuda.set_device(local_rank)
    replicas.init("nccl")
    assert world == args.gpus or world == 1, f"--gpus {args.gpus} but WORLD_SIZE={world}"

    cfg, frames = make_workload(args.config, args.groups)
    W, H = cfg.W, cfg.H
    P = W * H
    G = len(frames)
    renders_per_step = len(frames[0]["dst_cams"])
    d_color = [torch.from_numpy(f["color"]).cuda() for f in frames]
    d_depth = [torch.from_numpy(f["depth"]).cuda() for f in frames]
    d_out = [torch.empty((H, W, 4), dtype=torch.float32, device="cuda") for _ in range(renders_per_step)]
    sp.splats_create(W, H)

    def step(k: int):
        f = frames[k % G]
        sp.splats_update(d_color[k % G], d_depth[k % G], f["src_cam"], W, H, cfg.r_scale)
        for j, cam in enumerate(f["dst_cams"]):
            sp.splats_render(cam, W, H, d_out[j])

    barrier = replicas.barrier

    def timed(fn, K: int, fin=None) -> float:
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        barrier()
        e0.record()
        for k in range(K):
            fn(k)
        if fin is not None:
            fin()   # e.g. wait for the library's copy streams: e1 must come after the last read-back
        e1.record()
        barrier()
        return replicas.max_over_ranks(e0.elapsed_time(e1))

    K, Wm = args.steps, args.warmup
    # the four renders of a step go to four different images: let them overlap (include/splats.h)
    sp.splats_set_option(sp.OPT_OVERLAP, 1)
    for k in range(Wm):
        step(k)
    barrier()

    sampler = ClockSampler(local_rank)
    sampler.start()
    # ---- timed region: exactly K steps, the library as a user runs it (no per-stage events)
    launches0 = sp.splats_launch_count()
    ms_total = timed(step, K)
    launches = sp.splats_launch_count() - launches0
    n_in_region = len(sampler.samples)
    # ---- the same K steps again with per-stage CUDA events on the library's stream (the events
    # serialise the stages, so this pass is a little slower; kernels / roofline come from it)
    sp.splats_set_profiling(True)
    ms_staged = timed(step, K)
    stage = sp.splats_stage_ms()
    sp.splats_set_profiling(False)

    # ---- the paper's first-hit query on the same sequence: renders only,
    # reported beside the headline, not part of it
    def step_first(k: int):
        f = frames[k % G]
        if k < G:   # one pass over the source frames is enough
            sp.splats_update(d_color[k % G], d_depth[k % G], f["src_cam"], W, H, cfg.r_scale)
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record()
            for j, cam in enumerate(f["dst_cams"]):
                sp.splats_render_first_hit(cam, W, H, d_out[j])
            e1.record()
            first_events.append((e0, e1, len(f["dst_cams"])))
            p0, p1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            p0.record()
            for j, cam in enumerate(f["dst_cams"]):
                sp.splats_render_points(cam, W, H, 2, d_out[j])
            p1.record()
            point_events.append((p0, p1, len(f["dst_cams"])))

    first_events, point_events = [], []
    for k in range(min(K, G)):
        step_first(k)
    torch.cuda.synchronize()
    first_ms = sum(a.elapsed_time(b) for a, b, _ in first_events) / max(1, sum(n for _, _, n in first_events))
    points_ms = sum(a.elapsed_time(b) for a, b, _ in point_events) / max(1, sum(n for _, _, n in point_events))

    # ---- the paper's wire format: server-side pack + compaction and the
    # client-side build from packed samples, once per source frame; reported beside the headline
    import math
    half_diag = math.sqrt(3.0) / cfg.vol_n / 2          # half a voxel's diagonal
    quant = [0.0, 0.0, 0.0, 1.0, 1.0, 1.0, 4 * half_diag]
    w_samples = torch.empty(P, dtype=torch.int64, device="cuda")
    w_colors = torch.empty(P, dtype=torch.int32, device="cuda")
    w_count = torch.zeros(1, dtype=torch.int32, device="cuda")
    d_vol = torch.from_numpy(synth_volume(cfg)).cuda()
    m_color = torch.empty((H, W, 4), dtype=torch.float32, device="cuda")
    m_depth = torch.empty((H, W), dtype=torch.float32, device="cuda")
    tf = sp.make_transfer([(0.35, 0.8, (0.95, 0.55, 0.15)), (0.70, 0.95, (0.25, 0.60, 0.95))])
    march_ms = []
    for rep in range(2):
        for g in range(0, G, max(1, G // 4)):
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record()
            sp.splats_march(d_vol, cfg.vol_n, tf, frames[g]["src_cam"], W, H, m_color, m_depth)
            e1.record()
            torch.cuda.synchronize()
            if rep:
                march_ms.append(e0.elapsed_time(e1))
    del d_vol
    sp.splats_set_radius(sp.RADIUS_CONSTANT, half_diag)
    pack_ms, upd_ms, wire_n = [], [], []
    for rep in range(2):                                # first pass warms up
        for g in range(G):
            f = frames[g]
            ev = [torch.cuda.Event(enable_timing=True) for _ in range(4)]
            ev[0].record()
            sp.splats_pack(d_color[g], d_depth[g], f["src_cam"], W, H, cfg.r_scale, quant, w_samples, w_colors, w_count)
            ev[1].record()
            n_s = int(w_count.item())                   # the count travels with the frame
            ev[3].record()
            sp.splats_update_packed(w_samples, w_colors, n_s, quant)
            ev[2].record()
            sp.splats_render_first_hit(f["dst_cams"][-1], W, H, d_out[0])
            torch.cuda.synchronize()
            if rep:
                pack_ms.append(ev[0].elapsed_time(ev[1]))
                upd_ms.append(ev[3].elapsed_time(ev[2]))
                wire_n.append(n_s)
    sp.splats_set_radius(sp.RADIUS_FOOTPRINT, 0.0)
    pack_avg, upd_avg, n_avg = sum(pack_ms) / len(pack_ms), sum(upd_ms) / len(upd_ms), sum(wire_n) / len(wire_n)
    pack_bytes = 8 * P + 28 * n_avg                     # depth read twice, colour read + 12 B written per sample

    # ---- end-to-end through the host-buffer entry points (H2D of the frame, D2H of every image)
    h_color = [torch.from_numpy(f["color"]).pin_memory() for f in frames]
    h_depth = [torch.from_numpy(f["depth"]).pin_memory() for f in frames]
    h_out = [torch.empty((H, W, 4), dtype=torch.float32).pin_memory() for _ in range(renders_per_step)]

    def step_e2e(k: int):
        f = frames[k % G]
        sp.splats_update_host(h_color[k % G], h_depth[k % G], f["src_cam"], W, H, cfg.r_scale)
        for j, cam in enumerate(f["dst_cams"]):
            sp.splats_render_host(cam, W, H, h_out[j])

    for k in range(min(Wm, 3)):
        step_e2e(k)
    sp.splats_synchronize()
    barrier()
    t0 = time.perf_counter()
    ms_e2e_dev = timed(step_e2e, K, fin=sp.splats_synchronize)
    wall_e2e = (time.perf_counter() - t0) * 1e3
    ms_e2e = max(ms_e2e_dev, 0.0)
    # ---- the same end-to-end steps with the 8-bit display image read back (extra key, not the e2e)
    h_out8 = [torch.empty((H, W), dtype=torch.int32).pin_memory() for _ in range(renders_per_step)]

    def step_e2e8(k: int):
        f = frames[k % G]
        sp.splats_update_host(h_color[k % G], h_depth[k % G], f["src_cam"], W, H, cfg.r_scale)
        for j, cam in enumerate(f["dst_cams"]):
            sp.splats_render_host_rgba8(cam, W, H, h_out8[j])

    for k in range(min(Wm, 3)):
        step_e2e8(k)
    sp.splats_synchronize()
    ms_e2e8 = timed(step_e2e8, K, fin=sp.splats_synchronize)
    # ---- the paper's own client, end to end: packed samples arrive in host memory (12 B per sample,
    # PAPER.md:103), BVH build, 8-bit display images read back (extra key, not the e2e)
    sp.splats_set_radius(sp.RADIUS_CONSTANT, half_diag)
    h_samples, h_colors, n_packed = [], [], []
    for g in range(G):
        sp.splats_pack(d_color[g], d_depth[g], frames[g]["src_cam"], W, H, cfg.r_scale, quant, w_samples, w_colors, w_count)
        n_s = int(w_count.item())
        h_samples.append(w_samples[:n_s].cpu().pin_memory())
        h_colors.append(w_colors[:n_s].cpu().pin_memory())
        n_packed.append(n_s)
    sp.splats_set_radius(sp.RADIUS_FOOTPRINT, 0.0)

    def step_client(k: int):
        g = k % G
        sp.splats_update_packed_host(h_samples[g], h_colors[g], n_packed[g], quant)
        for j, cam in enumerate(frames[g]["dst_cams"]):
            sp.splats_render_host_rgba8(cam, W, H, h_out8[j])

    for k in range(min(Wm, 3)):
        step_client(k)
    sp.splats_synchronize()
    ms_client = timed(step_client, K, fin=sp.splats_synchronize)
    clocks = sampler.stop()
    clocks["samples_in_timed_region"] = n_in_region

    frames_done = K * renders_per_step * world
    value = frames_done / (ms_total * 1e-3)
    peak, peak_src = hbm_peak()

    # ---- per-kernel roofline from the events recorded inside the timed region
    steps_N = [frames[k % G]["N"] for k in range(K)]
    kernels = []
    bytes_sum = {}
    for k in range(K):
        ab = algorithmic_bytes(P, steps_N[k], P)
        for name, b in ab.items():
            mult = renders_per_step if name == "render" else 1
            bytes_sum[name] = bytes_sum.get(name, 0) + b * mult
    for name, (ms_sum, calls) in stage.items():
        if calls == 0:
            continue
        gbs = bytes_sum[name] / (ms_sum * 1e-3) / 1e9 if ms_sum > 0 else 0.0
        kernels.append({"stage": name, "launches_per_call": 1, "calls": calls,
                        "ms_avg": ms_sum / calls, "share": ms_sum / ms_staged, "algorithmic_bytes_avg": bytes_sum[name] / calls,
                        "achieved_gbs": gbs, "frac_of_hbm_peak": gbs / peak,
                        "traffic_ncu": NCU_TRAFFIC_BYTES.get(name)})
    dominant = max(kernels, key=lambda r: r["share"])
    build = [r for r in kernels if r["stage"] != "render"]
    build_ms = sum(r["ms_avg"] for r in build)
    build_bytes = sum(r["algorithmic_bytes_avg"] for r in build)
    render_ms = next(r["ms_avg"] for r in kernels if r["stage"] == "render")

    out = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": K, "warmup": Wm,
        "ms_per_step": ms_total / K, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "f32", "data": "synthetic",
        "config": {"workload": f"BASELINE.json configs[{args.config}]: {cfg.vol_n}^3 volume, {W}x{H} source frames, "
                               f"{G} source frames cycled, 1 rebuild + {renders_per_step} renders per step, "
                               f"r_scale {cfg.r_scale}, dolly x0.5 over the sequence",
                   "splats_per_frame_min_max": [min(steps_N), max(steps_N)],
                   "l2_policy": f"inputs larger than L2: {G} source frames x {P * 20 / 1e6:.1f} MB cycled",
                   "launch_mode": "programmatic dependent launches, consecutive renders of a step overlap "
                                  "(SPLATS_OPT_PDL, SPLATS_OPT_OVERLAP); kernels / roofline from a second pass of the same "
                                  "steps with per-stage events, stages serialised",
                   "parallelism": "replicas" if world > 1 else "single GPU"},
        "clocks": clocks,
        "e2e": {"value": frames_done / (ms_e2e * 1e-3), "unit": UNIT,
                "h2d_bytes_per_step": P * 20, "d2h_bytes_per_step": P * 16 * renders_per_step,
                "wall_ms_per_step": wall_e2e / K},
        "e2e_rgba8": {"value": frames_done / (ms_e2e8 * 1e-3), "unit": UNIT, "h2d_bytes_per_step": P * 20,
                      "d2h_bytes_per_step": P * 4 * renders_per_step,
                      "note": "same steps with splats_render_host_rgba8 (8-bit display image read back instead of float32)"},
        "e2e_paper_client": {"value": frames_done / (ms_client * 1e-3), "unit": UNIT,
                             "h2d_bytes_per_step": 12 * sum(n_packed) / G, "d2h_bytes_per_step": P * 4 * renders_per_step,
                             "note": "splats_update_packed_host (64-bit samples + RGBA8 colours from pinned host memory, "
                                     "constant half-voxel-diagonal radius) + 4 x splats_render_host_rgba8 per step"},
        "gpu_launches": int(launches),
        "value_with_stage_events": frames_done / (ms_staged * 1e-3), "ms_per_step_with_stage_events": ms_staged / K,
        "build_ms": build_ms, "render_ms": render_ms, "mrays_per_s": P / (render_ms * 1e-3) / 1e6,
        "roofline": {"kernel": dominant["stage"], "bound": "hbm", "achieved": dominant["achieved_gbs"], "peak": peak,
                     "unit": "GB/s", "frac": dominant["achieved_gbs"] / peak,
                     "traffic": NCU_TRAFFIC_BYTES.get(dominant["stage"]), "peak_source": peak_src,
                     "note": "dominant kernel by time; traversal is L2/latency bound, its algorithmic DRAM floor is "
                             "the image written once plus BVH and splats read once (DESIGN.md sec. 6)"},
        "roofline_build": {"bound": "hbm", "achieved": build_bytes / (build_ms * 1e-3) / 1e9, "peak": peak, "unit": "GB/s",
                           "frac": build_bytes / (build_ms * 1e-3) / 1e9 / peak, "algorithmic_bytes": build_bytes,
                           "note": "all build kernels of one splats_update (6 launches), per-stage events of the staged pass"},
        "kernels": kernels,
        "wire_format": {"march_ms": sum(march_ms) / len(march_ms), "pack_ms": pack_avg, "pack_gbs": pack_bytes / (pack_avg * 1e-3) / 1e9,
                        "pack_frac_of_hbm_peak": pack_bytes / (pack_avg * 1e-3) / 1e9 / peak,
                        "update_packed_ms": upd_avg, "samples_avg": n_avg, "payload_bytes_avg": 12 * n_avg,
                        "note": "splats_march (the server's ray marcher on this config's volume, a few source cameras), "
                                "splats_pack (Eq. 1, constant half-voxel-diagonal radius, 64-bit samples + RGBA8, GPU "
                                "compaction; the paper's serial CPU compaction takes 23 ms at 1024x1024, PAPER.md:79) and "
                                "splats_update_packed on the same source frames"},
        "point_baseline": {"render_ms": points_ms,
                           "note": "splats_render_points, 2x2-pixel points: CUDA restatement of the OpenGL point rendering of "
                                   "[ZAL12] that the paper compares against (PAPER.md:37,89); GL itself is unavailable on this box"},
        "first_hit": {"render_ms": first_ms, "mrays_per_s": P / (first_ms * 1e-3) / 1e6,
                      "note": "splats_render_first_hit (the paper's own query, PAPER.md:53,59) on the same frames and cameras"},
    }
    if rank == 0 and world == 1 and not args.no_cpu_baseline:
        out["cpu_baseline"] = cpu_baseline(cfg, frames)
    sp.splats_destroy()
    replicas.shutdown()
    if rank == 0:
        print(json.dumps(out), flush=True)


# --------------------------------------------------------------------------- oracle arms
def oracle_step(cfg, frame, sample_every: int, seed: int):
    """One step of the oracle on a bounded sample: the full build (O1-O7) and, for each of the
    step's display frames, the BVH-walk render (O8-O9) of every `sample_every`-th pixel (random
    subset); returns (build seconds, render seconds extrapolated to full frames)."""
    import oracle
    W, H = cfg.W, cfg.H
    t0 = time.perf_counter()
    sc = oracle.build_scene(frame["color"], frame["depth"], frame["src_cam"], W, H, cfg.r_scale)
    t_build = time.perf_counter() - t0
    rng = np.random.default_rng(seed)
    n_px = max(1, (W * H) // sample_every)
    t_render = 0.0
    for cam in frame["dst_cams"]:
        px = np.sort(rng.choice(W * H, size=n_px, replace=False)).astype(np.int64)
        t0 = time.perf_counter()
        oracle.render(sc, cam, W, H, "bvh", pixels=px)
        t_render += (time.perf_counter() - t0) * (W * H / n_px)
    return t_build, t_render


def cpu_baseline(cfg, frames):
    g = len(frames) // 2
    tb, tr = oracle_step(cfg, frames[g], sample_every=2, seed=1)
    n = len(frames[g]["dst_cams"])
    return {"value": n / (tb + tr), "unit": UNIT, "cores": 1, "kind": "oracle",
            "sample": f"source frame {g} of {len(frames)} (N={frames[g]['N']}): full oracle build ({tb * 1e3:.0f} ms) + "
                      f"BVH-walk render of a random half of the pixels of its {n} display frames, render time x2",
            "build_ms": tb * 1e3, "render_ms_per_frame": tr / n * 1e3, "host_cores_available": os.cpu_count()}


def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    cfg, frames = make_workload(args.config, args.groups)
    G = len(frames)
    n = len(frames[0]["dst_cams"])
    sample_every = 16
    for k in range(args.warmup):
        oracle_step(cfg, frames[k % G], sample_every, k)
    total = 0.0
    for k in range(args.steps):
        tb, tr = oracle_step(cfg, frames[k % G], sample_every, 100 + k)
        total += tb + tr
    value = args.steps * n / total
    sample = (f"per step: full oracle build + BVH-walk render of a random 1/{sample_every} of the pixels of each of the "
              f"{n} display frames, render time x{sample_every}")
    out = {"impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
           "warmup": args.warmup, "ms_per_step": total / args.steps * 1e3, "higher_is_better": True, "scaling": "weak",
           "vs_baseline": None, "dtype": "f32", "data": "synthetic",
           "config": {"workload": f"BASELINE.json configs[{args.config}] ({cfg.W}x{cfg.H}), oracle on a bounded sample: {sample}"},
           "cpu_baseline": {"value": value, "unit": UNIT, "cores": 1, "kind": "oracle", "sample": sample},
           "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
           "gpu_launches": 0}
    print(json.dumps(out), flush=True)


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=300, help="15 steps = one scripted 60-frame sequence")
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", choices=["ours", "reference"], default="ours")
    ap.add_argument("--config", type=int, default=3, help="BASELINE.json config index (headline: 3)")
    ap.add_argument("--groups", type=int, default=None, help="use only the first G source frames (debug)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    args = ap.parse_args()
    if args.warmup < 3:
        log("[bench] warmup raised to 3 (timing rules)")
        args.warmup = 3
    if args.impl == "reference":
        run_reference(args)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()
