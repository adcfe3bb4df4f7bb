#!/usr/bin/env python
"""bench.py -- frames/s of the HiGS forward render path on B200 (BASELINE.json metric).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl higs|reference] [--n N_GAUSSIANS]

A *step* is one frame: one pass of the whole hot path (a1 project+SH .. a8 merge, SURVEY.md section
8a) over the seeded synthetic 5.8 M-gaussian scene (BASELINE.json configs[3], SH degree 3) at
1920x1080; step i renders orbit view i % 32 (view 0 is configs[3]'s pose).  The scene arrays
(1.37 GB) are resident in HBM before the timed region and are far larger than the 126 MB L2, so no
L2 flush is needed between frames.  The 4K number (configs[4]: same scene, 3840x2160, 32 orbit
views) is reported next to it under "fps_4k".

Printed (rank 0, ONE JSON line): the base contract keys plus
  roofline      dominant kernel, algorithmic work / CUDA-event time against the measured peak
  stages        per-stage ms (CUDA events on the render stream) with each stage's own roofline
  cpu_baseline  the oracle as it stands, timed on this host's cores (rank 0, N = 1 only)
  e2e           same metric through higs_render_host: pinned HOST buffers in, HOST image out
  fps_4k        configs[4] sweep: median / min / max FPS, stage means, unit-load statistics

N > 1 (torchrun, one rank per GPU): frames are independent, so ranks render disjoint views of the
replicated scene with no data-path collective ("replicas only"); value = frames
of all ranks / max-over-ranks time.

--impl reference times the CPU oracle (oracle/, plain C, untuned) on this host: the base
contract's reference arm for this tier.
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import threading
import time
from pathlib import Path

import numpy as np

ROOT = Path(__file__).resolve().parent
if str(ROOT) not in sys.path:
    sys.path.insert(0, str(ROOT))

METRIC = "frames_per_sec_1080p_5.8M_gaussians"
UNIT = "frames/s"
N_PAPER = 5_800_000
FP32_LANES_PER_SM = 128          # ALU peak = SMs x 128 lanes x SM clock
RASTER_FP32_INST_PER_EVAL = 13.0  # FP32-pipe instructions per pixel-gaussian evaluation (SASS count)


def source_sha() -> str:
    """sha256 over the library's sources: ties the committed ncu traffic figures to the code they were captured on."""
    import hashlib
    h = hashlib.sha256()
    for p in sorted((ROOT / "paper_2606_00352_b200" / "csrc").glob("*.cu*")) + [ROOT / "include" / "higs.h"]:
        h.update(p.name.encode()); h.update(p.read_bytes())
    return h.hexdigest()[:16]


def committed_traffic() -> dict:
    """DRAM bytes per launch (dram__bytes_read.sum + dram__bytes_write.sum) of the stage kernels from the committed
    `ncu --set full` capture (profiles/r02_traffic.json, written from profiles/r02_final.md's capture).  ncu cannot run
    inside a timed bench, so the figures are tied to the source hash they were captured on and dropped (null) when the
    library's sources have changed since."""
    p = ROOT / "profiles" / "r02_traffic.json"
    if not p.exists():
        return {"note": "no committed capture"}
    d = json.loads(p.read_text())
    if d.get("src_sha") != source_sha():
        return {"note": f"stale: captured on sources {d.get('src_sha')}, now {source_sha()}"}
    return dict(d["traffic"], note=f"ncu --set full capture on sources {d['src_sha']}")


def measured_peaks() -> dict:
    p = ROOT / "MEASURED_PEAKS.json"
    if p.exists():
        d = json.loads(p.read_text())
        return {"hbm_gbs": float(d["hbm_gbs"]), "sm_max_mhz": float(d.get("sm_max_mhz", 1965.0)), "which": "measured"}
    return {"hbm_gbs": 6650.0, "sm_max_mhz": 1965.0, "which": "fallback"}


# ---- rank plumbing (pure functions: covered by the gloo world_size-2 test) -------------------------
def views_for_rank(step: int, rank: int, world: int, n_views: int) -> int:
    """Orbit view rendered by `rank` at `step`: ranks walk disjoint, interleaved views."""
    return (step * world + rank) % n_views


def aggregate_fps(frames_per_rank: int, world: int, max_seconds: float) -> float:
    return frames_per_rank * world / max_seconds if max_seconds > 0 else 0.0


def dist_setup():
    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    return rank, local, world


class ClockSampler:
    """nvidia-smi clocks + throttle reasons sampled DURING a timed region (B200_PROFILING.md)."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.index, self.rows, self.proc = index, [], None

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(self.index), f"--query-gpu={self.Q}",
                                          "--format=csv,noheader,nounits", "-lms", "20"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.thr = threading.Thread(target=self._pump, daemon=True)
            self.thr.start()
            t_end = time.time() + 10.0                  # nvidia-smi needs a second or two before its first row
            while not self.rows and time.time() < t_end and self.proc.poll() is None:
                time.sleep(0.05)
        except OSError:
            self.proc = None

    def _pump(self):
        for line in self.proc.stdout:
            self.rows.append((time.time(), line.strip()))

    def mark(self):
        return time.time()

    def stop(self):
        if self.proc:
            self.proc.terminate()
            try:
                self.proc.wait(timeout=2)
            except Exception:
                self.proc.kill()

    def summary(self, t0: float, t1: float) -> dict:
        sm, mx, reasons = [], [], set()
        rows = [r for t, r in self.rows if t0 <= t <= t1 + 0.06]
        if not rows and self.rows:                      # timed region shorter than a sampling period: nearest samples
            mid = 0.5 * (t0 + t1)
            rows = [r for _, r in sorted(self.rows, key=lambda tr: abs(tr[0] - mid))[:3]]
        for r in rows:
            f = [x.strip() for x in r.split(",")]
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
                "reasons": sorted(reasons), "samples": len(sm)}


def build_scene(n: int):
    import higs_scenes as hs
    return hs.scene_large(N=n, W=1920, H=1080)


def subsample(scene, stride: int):
    import higs_scenes as hs
    if stride <= 1:
        return scene
    c = lambda a: np.ascontiguousarray(a[::stride])
    return hs.Scene(scene.name + f"_every{stride}", c(scene.means), c(scene.scales), c(scene.quats), c(scene.opacities),
                    c(scene.sh), scene.degree, scene.cameras)


# ---- the CPU oracle, timed (cpu_baseline leg and --impl reference) ---------------------------------
def oracle_frame_seconds(scene, cam) -> float:
    import oracle
    t0 = time.perf_counter()
    oracle.render_scene(scene, cam)          # project -> global (key,id) sort -> O-IMG compositing
    return time.perf_counter() - t0


def run_reference(args) -> int:
    rank, _, world = dist_setup()
    if rank != 0:
        return 0
    import oracle
    oracle.build()
    scene = build_scene(args.n)
    stride = args.ref_stride
    sub = subsample(scene, stride)
    cores = oracle.n_threads()
    n_views = len(scene.cameras)
    for i in range(args.warmup):
        oracle_frame_seconds(sub, scene.cameras[i % n_views])
    t = [oracle_frame_seconds(sub, scene.cameras[i % n_views]) for i in range(args.steps)]
    total = float(np.sum(t))
    fps = args.steps / (total * stride)
    sample = (f"whole frames (all {scene.N:,} gaussians, 1920x1080), orbit views i%{n_views}" if stride == 1 else
              f"every {stride}th gaussian of the scene ({sub.N:,} of {scene.N:,}), full 1920x1080 frame, orbit views "
              f"i%{n_views}; time scaled x{stride} (an over-estimate: occlusion makes the work sub-linear in N)")
    line = {"impl": "reference", "metric": METRIC, "value": fps, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": 1000.0 * total * stride / args.steps, "higher_is_better": True,
            "scaling": "weak", "vs_baseline": None, "dtype": "f64 (decisions f32)", "data": "synthetic",
            "config": workload_config(scene, args, world),
            "cpu_baseline": {"value": fps, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample},
            "e2e": {"value": fps, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line), flush=True)
    return 0


def workload_config(scene, args, world) -> dict:
    return {"workload": "configs[3]: large scene, paper scale (heavy-tailed planes/shells + 20% background + 10% hot region)",
            "n_gaussians": scene.N, "sh_degree": scene.degree, "image": "1920x1080", "fov_x_deg": 60,
            "views": f"orbit of {len(scene.cameras)} poses, step i -> view (i*{world}+rank) % {len(scene.cameras)}; view 0 = configs[3]'s pose",
            "tiles": f"8x8 px render tiles, 8x4 macro-tiles (64x32 px), B_r={args.batch_cap}, partition batches = 2 persistent CTAs per SM over 128-id chunks",
            "l2": "inputs (1.37 GB) and per-frame records (0.46 GB) exceed the 126 MB L2; no flush between frames",
            "parallelism": f"replicas x{world} (views sharded, no collective)"}


# ---- the CUDA path ------------------------------------------------------------------------------------
def run_higs(args) -> int:
    import torch
    import torch.distributed as dist
    import higs_scenes as hs
    import paper_2606_00352_b200 as hg

    rank, local, world = dist_setup()
    if not torch.cuda.is_available():
        raise RuntimeError("bench.py needs a CUDA device: the HiGS path has no CPU fallback")
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    peaks = measured_peaks()
    scene = build_scene(args.n)
    n_views = len(scene.cameras)
    cams_1080 = scene.cameras
    cams_4k = hs.retarget(scene, 3840, 2160).cameras
    dev = hg.scene_to_device(scene, f"cuda:{local}")
    max_w, max_h = (3840, 2160) if not args.no_4k else (1920, 1080)
    ctx = hg.higs_create(local, scene.N, max_w, max_h, 0)
    if args.batch_cap != 1024:
        hg.higs_set_batch_cap(ctx, args.batch_cap)
    ccams_1080 = [hg.make_camera(c) for c in cams_1080]
    ccams_4k = [hg.make_camera(c) for c in cams_4k]
    img = torch.empty((1080, 1920, 3), dtype=torch.float32, device=f"cuda:{local}")
    stream = torch.cuda.current_stream()

    def frame(i, cams=ccams_1080, W=1920, H=1080, out=img):
        hg.higs_render(ctx, *dev, scene.degree, cams[views_for_rank(i, rank, world, n_views)], W, H, out, stream.cuda_stream)

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    # -- timed region: K frames, CUDA events on the render stream, clocks sampled meanwhile --
    sampler = ClockSampler(local)
    if rank == 0:
        sampler.start()
    hg.higs_set_flags(ctx, args.flags)
    for i in range(args.warmup):
        frame(i)
    barrier()
    evs = [torch.cuda.Event(enable_timing=True) for _ in range(args.steps + 1)]
    t_mark0 = sampler.mark()
    evs[0].record(stream)
    for i in range(args.steps):
        frame(args.warmup + i)
        evs[i + 1].record(stream)              # between frames only: the kernel chains inside a frame are untouched
    barrier()
    t_mark1 = sampler.mark()
    secs = evs[0].elapsed_time(evs[-1]) / 1000.0
    frame_ms = np.array([evs[i].elapsed_time(evs[i + 1]) for i in range(args.steps)])
    st_last = hg.higs_get_stats(ctx)
    launches_per_frame = int(st_last["n_launches"])
    if world > 1:
        t = torch.tensor([secs], dtype=torch.float64, device=f"cuda:{local}")
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        secs = float(t.item())
    fps = aggregate_fps(args.steps, world, secs)
    clocks = sampler.summary(t_mark0, t_mark1) if rank == 0 else None

    # -- per-stage pass: the same K views with stage events on, one sync per frame --
    hg.higs_set_flags(ctx, args.flags | hg.HIGS_FLAG_STAGE_TIMERS)
    stage_names = ["project", "count", "scan", "fill", "sort", "raster", "merge", "total"]
    rows, frames_stats = [], []
    for i in range(args.steps):
        frame(args.warmup + i)
        s = hg.higs_get_stats(ctx)
        rows.append([s["ms_" + k] for k in stage_names])
        frames_stats.append(s)
    stage_ms = dict(zip(stage_names, np.mean(np.array(rows), axis=0).tolist()))
    stage_med = dict(zip(stage_names, np.median(np.array(rows), axis=0).tolist()))
    mean_of = lambda k: float(np.mean([s[k] for s in frames_stats]))

    # -- instrumented pass: evaluations actually executed by the rasterizer (same views) --
    hg.higs_set_flags(ctx, args.flags | hg.HIGS_FLAG_COUNT_EVALS)
    evals, tile_pairs = [], []
    for i in range(min(args.steps, 8)):
        frame(args.warmup + i)
        s = hg.higs_get_stats(ctx)
        evals.append(s["n_evals"]); tile_pairs.append(s["n_tile_pairs"])
    hg.higs_set_flags(ctx, args.flags)
    n_evals, n_tile_pairs = float(np.mean(evals)), float(np.mean(tile_pairs))

    # -- rooflines (algorithmic work per launch / mean CUDA-event duration of that stage) --
    K = (scene.degree + 1) ** 2
    n_sm_early = torch.cuda.get_device_properties(local).multi_processor_count
    N, n_vis, n_pairs, n_units = scene.N, mean_of("n_visible"), mean_of("n_pairs"), mean_of("n_units")
    n_b, n_m = 2 * n_sm_early, 30 * 34                                   # partition CTAs = histogram rows (2 per SM), macro-tiles at 1080p
    hbm = peaks["hbm_gbs"]
    alg_bytes = {
        "project": 44.0 * N + (12.0 * K + 80.0) * n_vis + 4.0 * n_b * n_m,           # inputs, SH rows, 64-B + 16-B records, histogram rows (count is folded in)
        "fill": 16.0 * n_vis + 12.0 * n_b * n_m + 8.0 * n_pairs,                    # 16-B bin record per survivor, bases, pairs written
        "sort": 16.0 * n_pairs,
    }
    NCU_TRAFFIC = committed_traffic()
    def hbm_roof(stage, nbytes):
        ms = stage_ms[stage]
        ach = nbytes / (ms * 1e-3) / 1e9 if ms > 0 else 0.0
        return {"bound": "hbm", "achieved": ach, "peak": hbm, "unit": "GB/s", "frac": ach / hbm, "traffic": NCU_TRAFFIC.get(stage),
                "traffic_source": NCU_TRAFFIC.get("note"), "peak_source": peaks["which"], "algorithmic_bytes": nbytes, "ms": ms}
    sm_hz = peaks["sm_max_mhz"] * 1e6
    n_sm = torch.cuda.get_device_properties(local).multi_processor_count
    alu_peak = n_sm * FP32_LANES_PER_SM * sm_hz / 1e9                      # G FP32-pipe thread-instructions / s
    ras_ms = stage_ms["raster"]
    ras_ach = n_evals * RASTER_FP32_INST_PER_EVAL / (ras_ms * 1e-3) / 1e9 if ras_ms > 0 else 0.0
    roof = {k: hbm_roof(k, v) for k, v in alg_bytes.items()}
    survey_bytes = 44.0 * N + (12.0 * K + 56.0) * n_vis                      # SURVEY.md 8(d)'s own per-unit figure (56 B written per survivor)
    roof["project"]["frac_survey_formula"] = survey_bytes / (stage_ms["project"] * 1e-3) / 1e9 / hbm if stage_ms["project"] > 0 else 0.0
    roof["raster"] = {"bound": "alu", "achieved": ras_ach, "peak": alu_peak, "unit": "G FP32 thread-inst/s",
                      "frac": ras_ach / alu_peak, "traffic": NCU_TRAFFIC.get("raster"), "peak_source": f"{n_sm} SMs x {FP32_LANES_PER_SM} lanes x {peaks['sm_max_mhz']:.0f} MHz",
                      "evals_per_frame": n_evals, "tile_pairs_per_frame": n_tile_pairs,
                      "gevals_per_s": n_evals / (ras_ms * 1e-3) / 1e9 if ras_ms > 0 else 0.0,
                      "fp32_inst_per_eval": RASTER_FP32_INST_PER_EVAL, "ms": ras_ms}
    dominant = max(("project", "fill", "sort", "raster"), key=lambda k: stage_ms[k])

    e2e = None
    if not args.no_e2e:
        # -- e2e: the same frames through higs_render_host (pinned host arrays in, host image out) --
        pin = lambda a: torch.from_numpy(np.ascontiguousarray(a, dtype=np.float32)).pin_memory()
        host = [pin(scene.means), pin(scene.scales), pin(scene.quats), pin(scene.opacities), pin(scene.sh)]
        host_img = torch.empty((1080, 1920, 3), dtype=torch.float32).pin_memory()
        # bytes that cross PCIe per frame: the four small arrays are copied; of the page-locked SH array the projection
        # kernel reads the rows of the survivors in place (include/higs.h, higs_render_host): n_visible rows of that frame
        row_bytes = int(host[4].numel()) // scene.N * 4
        h2d = sum(int(t.numel()) * 4 for t in host[:4]) + int(round(n_vis)) * row_bytes + 80
        h2d_arrays = sum(int(t.numel()) * 4 for t in host) + 80
        d2h = int(host_img.numel()) * 4
        def e2e_frame(i):
            hg.higs_render_host(ctx, *host, scene.degree, ccams_1080[views_for_rank(i, rank, world, n_views)], 1920, 1080, host_img)
        e2e_steps = max(1, min(args.steps, args.e2e_steps))
        for i in range(min(args.warmup, 3)):
            e2e_frame(i)
        barrier()
        t0 = time.perf_counter()
        for i in range(e2e_steps):
            e2e_frame(args.warmup + i)
        barrier()
        e2e_secs = time.perf_counter() - t0
        # resident-scene variant: per frame only the camera goes in and the image comes out
        hg.higs_scene_upload(ctx, *host, scene.degree)
        for i in range(3):
            hg.higs_render_view_host(ctx, ccams_1080[i % n_views], 1920, 1080, host_img)
        barrier()
        t0 = time.perf_counter()
        for i in range(args.steps):
            hg.higs_render_view_host(ctx, ccams_1080[views_for_rank(args.warmup + i, rank, world, n_views)], 1920, 1080, host_img)
        barrier()
        res_secs = time.perf_counter() - t0
        if world > 1:
            t = torch.tensor([e2e_secs, res_secs], dtype=torch.float64, device=f"cuda:{local}")
            dist.all_reduce(t, op=dist.ReduceOp.MAX)
            e2e_secs, res_secs = (float(x) for x in t.tolist())
        e2e = {"value": aggregate_fps(e2e_steps, world, e2e_secs), "unit": UNIT, "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": d2h,
               "steps": e2e_steps, "host_array_bytes": h2d_arrays,
               "api": "higs_render_host, pinned host arrays: means/scales/quats/opacities copied every frame, SH rows of the survivors "
                      "read in place by the projection kernel (h2d_bytes_per_step = copies + n_visible x row bytes)",
               "resident_scene": {"value": aggregate_fps(args.steps, world, res_secs), "unit": UNIT, "h2d_bytes_per_step": 80,
                                  "d2h_bytes_per_step": d2h, "api": "higs_scene_upload once, then higs_render_view_host per frame"}}

    # -- load map (Fig. 1): per render tile, gaussians that pass the per-tile test / units of its macro-tile --
    def load_map(cams, W, H, out, view):
        hg.higs_set_flags(ctx, args.flags | hg.HIGS_FLAG_COUNT_EVALS | hg.HIGS_FLAG_NO_XBATCH_CUT)
        hg.higs_render(ctx, *dev, scene.degree, cams[view], W, H, out, stream.cuda_stream)
        ls = hg.higs_get_lists(ctx)
        hg.higs_set_flags(ctx, args.flags)
        nb = np.diff(ls["batch_offset"]).astype(np.float64)
        tl = ls["tile_load"].astype(np.float64)
        has = nb > 0
        per_unit = tl[has] / nb[has, None]                    # what one (macro-tile, batch) unit brings to the tile on average
        touched = tl[has] > 0
        seg = ls["mt_count"].astype(np.int64)
        unit_len = np.concatenate([np.minimum(args.batch_cap, np.maximum(0, n - args.batch_cap * np.arange((n + args.batch_cap - 1) // args.batch_cap)))
                                   for n in seg[seg > 0]]) if (seg > 0).any() else np.zeros(1)
        return {"view": view, "per_tile_gaussians_max": float(tl.max()), "per_tile_gaussians_mean": float(tl[has][touched].mean()) if touched.any() else 0.0,
                "per_tile_load_per_unit_max": float(per_unit.max()) if has.any() else 0.0,
                "per_tile_load_per_unit_mean": float(per_unit[touched].mean()) if touched.any() else 0.0,
                "unit_len_max": int(unit_len.max()), "unit_len_mean": float(unit_len.mean()), "n_units": int(ls["n_units"]),
                "what": "per render tile: gaussians overlapping the tile (inline visibility test, no cross-batch cut) summed over the macro-tile's "
                        "units = the per-tile list length of a per-tile renderer; divided by the units of the macro-tile = the per-unit load"}
    load_1080 = load_map(ccams_1080, 1920, 1080, img, 0)

    # -- 4K sweep (configs[4]): every orbit view, timed like the 1080p number (no stage events inside the timed frames) --
    fps_4k = None
    if not args.no_4k:
        img4 = torch.empty((2160, 3840, 3), dtype=torch.float32, device=f"cuda:{local}")
        per_view, st4 = [], []
        my_views = [v for v in range(n_views) if v % world == rank]
        reps = max(3, args.reps_4k)
        for v in my_views:
            hg.higs_set_flags(ctx, args.flags)
            for _ in range(2):
                hg.higs_render(ctx, *dev, scene.degree, ccams_4k[v], 3840, 2160, img4, stream.cuda_stream)
            ev4 = [torch.cuda.Event(enable_timing=True) for _ in range(reps + 1)]
            ev4[0].record(stream)
            for r_ in range(reps):
                hg.higs_render(ctx, *dev, scene.degree, ccams_4k[v], 3840, 2160, img4, stream.cuda_stream)
                ev4[r_ + 1].record(stream)
            torch.cuda.synchronize()
            per_view.append(1000.0 / float(np.median([ev4[r_].elapsed_time(ev4[r_ + 1]) for r_ in range(reps)])))
            hg.higs_set_flags(ctx, args.flags | hg.HIGS_FLAG_STAGE_TIMERS)     # one more frame for the stage breakdown
            hg.higs_render(ctx, *dev, scene.degree, ccams_4k[v], 3840, 2160, img4, stream.cuda_stream)
            st4.append(hg.higs_get_stats(ctx))
        hg.higs_set_flags(ctx, args.flags)
        pv = np.array(per_view)
        fps_4k = {"workload": "configs[4]: same scene at 3840x2160, 32 orbit views", "views": len(my_views), "frames_per_view": reps,
                  "timing": "median over the frames of a view, CUDA events between frames, no stage events",
                  "median": float(np.median(pv)), "min": float(pv.min()), "max": float(pv.max()),
                  "per_view": [round(float(x), 1) for x in pv],
                  "stages_ms_mean": {k: float(np.mean([s_["ms_" + k] for s_ in st4])) for k in stage_names},
                  "n_pairs_mean": float(np.mean([s_["n_pairs"] for s_ in st4])), "n_units_mean": float(np.mean([s_["n_units"] for s_ in st4])),
                  "unit_load_mean": float(np.mean([s_["n_pairs"] / max(1, s_["n_units"]) for s_ in st4])),
                  "max_segment": int(max(s_["max_segment"] for s_ in st4)),
                  "load_map": [load_map(ccams_4k, 3840, 2160, img4, v) for v in (0, 8, 16, 24) if v in my_views]}
        del img4

    # -- variants: fp16 data path, 16x16 render tiles, 32-byte SH codes; same views, same timing --
    variants = None
    if not args.no_variants:
        def timed(render, n):
            for i in range(3):
                render(i)
            evv = [torch.cuda.Event(enable_timing=True) for _ in range(n + 1)]
            evv[0].record(stream)
            for i in range(n):
                render(args.warmup + i)
                evv[i + 1].record(stream)
            torch.cuda.synchronize()
            return evv[0].elapsed_time(evv[-1]) / n

        def stage_means(render, n):
            rows_ = []
            for i in range(n):
                render(args.warmup + i)
                s_ = hg.higs_get_stats(ctx)
                rows_.append([s_["ms_" + k] for k in stage_names])
            return dict(zip(stage_names, np.mean(np.array(rows_), axis=0).tolist()))

        nv = min(args.steps, 32)
        variants = {}
        def run_variant(name, flags, render, note):
            hg.higs_set_flags(ctx, args.flags | flags)
            ms = timed(render, nv)
            hg.higs_set_flags(ctx, args.flags | flags | hg.HIGS_FLAG_STAGE_TIMERS)
            variants[name] = {"fps": 1000.0 / ms, "ms_per_frame": ms, "stages_ms_mean": stage_means(render, min(nv, 8)), "note": note}
            hg.higs_set_flags(ctx, args.flags)
        run_variant("fp32_8x8", 0, frame, "the headline configuration, re-timed here over the same frames as the variants")
        run_variant("fp16_8x8", hg.HIGS_FLAG_FP16, frame,
                    "PAPER.md:180-226, 280: Cholesky conics, tile-unit coordinates, half2 blending, 16 KB fp16 partials per unit (fp32: 32 KB)")
        hg.higs_set_tile(ctx, 16)
        run_variant("fp32_16x16", 0, frame, "PAPER.md:286-299 (Table 2): 16x16 render tiles, macro-tiles of 128x64 px")
        run_variant("fp16_16x16", hg.HIGS_FLAG_FP16, frame, "both")
        hg.higs_set_tile(ctx, 8)
        for tx, ty in ((4, 8), (16, 2)):                                # macro-tile shape sweep: 32 render tiles grouped otherwise
            hg.higs_set_macro_tile(ctx, tx, ty)
            run_variant(f"fp32_8x8_mt{tx}x{ty}", 0, frame, f"macro-tiles of {tx} x {ty} render tiles = {8 * tx} x {8 * ty} px instead of 8 x 4 (PAPER.md:73)")
        hg.higs_set_macro_tile(ctx, 8, 4)
        hg.higs_scene_upload(ctx, *[np.ascontiguousarray(a, dtype=np.float32) for a in (scene.means, scene.scales, scene.quats, scene.opacities, scene.sh)], scene.degree)
        hg.higs_scene_compress_sh(ctx)
        view = lambda i: hg.higs_render_view(ctx, ccams_1080[views_for_rank(i, rank, world, n_views)], 1920, 1080, img, stream.cuda_stream)
        run_variant("resident_fp32sh", 0, view, "resident scene (higs_scene_upload + higs_render_view), 192-byte fp32 SH rows")
        run_variant("resident_sh32", hg.HIGS_FLAG_SH32, view, "PAPER.md:245: 32-byte SH codes decoded inline in the projection kernel")
        run_variant("resident_sh32_fp16", hg.HIGS_FLAG_SH32 | hg.HIGS_FLAG_FP16, view, "the paper's default configuration: fp16 data path + 32-byte SH")
        hg.higs_scene_sort_spatial(ctx, scene.N)
        hg.higs_scene_compress_sh(ctx)
        run_variant("sorted_fp32sh", 0, view, "resident scene stored along a Morton curve (higs_scene_sort_spatial): survivors of the cull are contiguous")
        run_variant("sorted_sh32", hg.HIGS_FLAG_SH32, view, "Morton order + 32-byte SH codes")
        run_variant("sorted_sh32_fp16", hg.HIGS_FLAG_SH32 | hg.HIGS_FLAG_FP16, view, "Morton order + 32-byte SH codes + fp16 data path")

    hg.higs_destroy(ctx)
    if rank == 0:
        sampler.stop()
    cpu_baseline = None
    if rank == 0 and world == 1 and not args.no_cpu_baseline:
        import oracle
        oracle.build()
        stride = args.cpu_stride
        sub = subsample(scene, stride)
        secs_cpu = oracle_frame_seconds(sub, scene.cameras[0]) * stride
        cpu_baseline = {"value": 1.0 / secs_cpu, "unit": UNIT, "cores": oracle.n_threads(), "kind": "oracle",
                        "ms_per_frame": 1000.0 * secs_cpu,
                        "sample": ("one whole frame, view 0, all gaussians" if stride == 1 else
                                   f"every {stride}th gaussian ({sub.N:,} of {scene.N:,}), whole frame, view 0, time scaled x{stride}")}
    if world > 1:
        dist.barrier()
        dist.destroy_process_group()
    if rank != 0:
        return 0
    line = {"metric": METRIC, "value": fps, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
            "ms_per_step": 1000.0 * secs / args.steps, "ms_per_step_median": float(np.median(frame_ms)),
            "fps_from_median_frame": 1000.0 / float(np.median(frame_ms)), "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": "f32", "data": "synthetic", "config": workload_config(scene, args, world),
            "clocks": clocks, "gpu_launches": launches_per_frame * args.steps, "gpu_launches_per_frame": launches_per_frame,
            "roofline": dict(roof[dominant], kernel=dominant), "stages": {"ms_mean": stage_ms, "ms_median": stage_med, "roofline": roof},
            "frame": {"n_visible": n_vis, "n_pairs": n_pairs, "n_units": n_units, "max_segment": mean_of("max_segment"),
                      "n_oversize": mean_of("n_oversize"), "unit_load_mean": n_pairs / max(1.0, n_units), "load_map": load_1080},
            "e2e": e2e, "fps_4k": fps_4k, "variants": variants, "cpu_baseline": cpu_baseline,
            "paper_context": "1,124 FPS at 1080p on a 5.8 M-gaussian scene, RTX PRO 6000 Blackwell, fp16 + 32-byte SH (PAPER.md:9): other hardware, other scene, not a target"}
    print(json.dumps(line), flush=True)
    return 0


def main() -> int:
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=None, help="timed frames (default 100 for higs: the paper's protocol, PAPER.md:309; 10 for reference)")
    ap.add_argument("--warmup", type=int, default=5)
    ap.add_argument("--impl", default="higs", choices=["higs", "reference"])
    ap.add_argument("--n", type=int, default=N_PAPER, help="gaussians in the scene (default: the paper-scale 5.8 M)")
    ap.add_argument("--batch-cap", type=int, default=1024, help="B_r, gaussians per rasterizer work unit (PAPER.md:81 fixes 1,024; smaller values for the sweep)")
    ap.add_argument("--flags", type=int, default=0, help="extra HIGS_FLAG_* bits for every frame (4 = no cross-batch cut, 8 = merge-sort tiers)")
    ap.add_argument("--no-4k", action="store_true")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true", help="skip the host-buffer end-to-end legs (gaussian-count sweeps beyond host memory for pinned copies)")
    ap.add_argument("--no-variants", action="store_true", help="skip the fp16 / 16x16 / SH32 variant timings")
    ap.add_argument("--reps-4k", type=int, default=5, help="timed frames per 4K view (median)")
    ap.add_argument("--e2e-steps", type=int, default=16)
    ap.add_argument("--cpu-stride", type=int, default=1, help="cpu_baseline renders every k-th gaussian (1 = the whole frame)")
    ap.add_argument("--ref-stride", type=int, default=1, help="--impl reference renders every k-th gaussian per step")
    args = ap.parse_args()
    if args.steps is None:
        args.steps = 100 if args.impl == "higs" else 10
    if args.steps < 1 or args.warmup < 0:
        ap.error("steps >= 1, warmup >= 0")
    if args.impl == "higs" and args.warmup < 3:
        args.warmup = 3                                  # timing rule: at least 3 warm-up frames
    return run_reference(args) if args.impl == "reference" else run_higs(args)


if __name__ == "__main__":
    sys.exit(main())
