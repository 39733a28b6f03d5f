#!/usr/bin/env python
"""bench.py -- throughput of the SSS-GS forward relighting render path on B200.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config C] [--impl reference]

A step = one pass of the whole hot path (MLP + projection + sort + tile binning + G-buffer
compositing + deferred shading) over one batch of synthetic input = one sssgs_render call
producing every frame of one view of the workload (BASELINE.json configs[C-1]; default C=2, the
configuration the metric is quoted on).  Prints ONE JSON line.

  value     Mpix/s, inputs resident in HBM, CUDA events around each step, L2 flushed between
            steps, step replayed from a CUDA graph (the launch configuration the tests check)
  e2e       same metric through sssgs_render_host with pinned HOST buffers (H2D + D2H inside)
  roofline  the step's dominant kernel against its bound, timed with events inside the library
  cpu_baseline  the CPU oracle, as it stands, on this box's host cores (rank 0, N = 1)

--impl reference times the CPU oracle alone (the reference arm of this tier).
N > 1 (torchrun): frames are independent, every rank renders the same number of frames with no
data-path collective ("weak" scaling); value = all ranks' pixels / max-over-ranks time.
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

from paper_2408_12282_b200 import multi, scenes  # noqa: E402

METRIC = "Mpix/s (MLP + G-buffer splat + deferred shading)"
# dram__bytes_read.sum + dram__bytes_write.sum of one launch of a stage's kernel, from the
# `ncu --set full` captures summarised under profiles/ (r01_ncu_full.md): (config, stage) -> bytes
NCU_DRAM_BYTES_PER_LAUNCH = {(2, "raster"): 11665664, (3, "mlp"): 31867392, (3, "raster"): 267091712,
                             (4, "raster"): 274415360, (5, "mlp"): 221394688, (5, "raster"): 1027052288}
FP32_LANES_PER_SM = 128


def load_peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        d = json.load(open(p))
        return dict(hbm=float(d["hbm_gbs"]), bf16_burst=float(d["bf16_tflops"]),
                    bf16_sustained=float(d.get("bf16_tflops_sustained", d["bf16_tflops"])),
                    sm_max_mhz=float(d.get("sm_max_mhz", 1965.0)), source="measured")
    return dict(hbm=6650.0, bf16_burst=1590.0, bf16_sustained=1400.0, sm_max_mhz=1965.0, source="fallback")


class ClockSampler:
    """Samples nvidia-smi clocks / throttle reasons while the timed region runs."""

    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        self.index, self.rows, self.proc = index, [], None

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
            self.rows.append([c.strip() for c in line.split(",")])

    def stop(self):
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        self.proc.terminate()
        try:
            self.proc.wait(timeout=2)
        except Exception:
            self.proc.kill()
        sm, mx, reasons = [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for r in self.rows:
            try:
                sm.append(float(r[0]))
                mx.append(float(r[1]))
                for k, nm in enumerate(names):
                    if r[3 + k].lower().startswith("active"):
                        reasons.add(nm)
            except Exception:
                pass
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "samples": len(sm), "reasons": sorted(reasons)}


def workload(cfg):
    """(scene, cams of one step, lights of one step, frames per step)."""
    s = scenes.make_scene(cfg)
    return s, s.cameras[:1], s.lights[0], len(s.lights[0])


def oracle_sample(scene, min_seconds=0.0, max_frames=1):
    """Times the CPU oracle, as it stands, on a bounded sample: whole-path renders of the first
    (view, light) frame, repeated until `min_seconds` of CPU work (at least `max_frames` = 1 frame)."""
    import oracle
    t0 = time.perf_counter()
    frames, res = 0, None
    while frames < max_frames or time.perf_counter() - t0 < min_seconds:
        res = oracle.render_frame(scene, 0, 0, mlp_mode=1)   # projection, lists, MLP, compositing, shading
        frames += 1
    dt = time.perf_counter() - t0
    cam = scene.cameras[0]
    return dict(seconds=dt, frames=frames, mpix_s=frames * cam.width * cam.height / dt / 1e6,
                cores=oracle.num_threads(), res=res)


def mlp_flops_per_row(mlp):
    d, fl = mlp.in_dim, 0
    for w in mlp.trunk_width:
        fl += 2 * d * w
        d = w
    fl += 2 * d * 3
    di = d
    for w in mlp.inc_hidden_width:
        fl += 2 * di * w
        di = w
    return fl + 2 * di


def stage_models(scene, nl, n_vis, inst, counters, peaks, num_sms, mlp_rows):
    """Algorithmic work of each stage for ONE step."""
    n = scene.n
    cam = scene.cameras[0]
    npix = cam.width * cam.height
    feat = scene.feat.shape[1]
    alu_peak = num_sms * FP32_LANES_PER_SM * 2 * peaks["sm_max_mhz"] * 1e6 / 1e12  # TFLOP/s
    m = {
        "project": ("hbm", 44.0 * n + 48.0 * n_vis),
        "depth_sort": ("hbm", (3 * 16.0 + 12.0) * n),
        "emit": ("hbm", 16.0 * n + 8.0 * inst),
        "tile_sort": ("hbm", 16.0 * inst * (2 if (cam.width + 15) // 16 * ((cam.height + 15) // 16) > 256 else 1)),
        # rows the MLP actually evaluated (in a sweep: the Gaussians blended at some pixel of the view)
        "mlp": ("tensor", float(mlp_flops_per_row(scene.mlp)) * mlp_rows * nl),
    }
    if counters is not None:
        p_eval, p_blend = counters
        m["raster"] = ("alu", 10.0 * p_eval + (17.0 + 8.0 * (nl - 1)) * p_blend)
    else:
        m["raster"] = ("alu", None)
    pk = {"hbm": (peaks["hbm"], "GB/s"), "tensor": (peaks["bf16_burst"], "TFLOP/s"), "alu": (alu_peak, "TFLOP/s")}
    return m, pk


def run_reference(args, rank):
    """Reference arm of this tier: the CPU oracle, as it stands, on the host cores."""
    if rank != 0:
        return
    scene, cams, lights, fps = workload(args.config)
    cam = cams[0]
    for _ in range(args.warmup if args.config <= 2 else 0):
        oracle_sample(scene)
    t, frames, cores = 0.0, 0, 1
    for _ in range(args.steps):
        r = oracle_sample(scene)
        t += r["seconds"]
        frames += r["frames"]
        cores = r["cores"]
    val = frames * cam.width * cam.height / t / 1e6
    sample = f"first (view, light) frame of configs[{args.config - 1}] per step, whole path, bf16-emulating MLP"
    print(json.dumps({
        "impl": "reference", "metric": METRIC, "value": val, "unit": "Mpix/s", "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": t / args.steps * 1e3,
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": f"configs[{args.config - 1}] {scene.name}", "frames_per_step": 1},
        "cpu_baseline": {"value": val, "unit": "Mpix/s", "cores": cores, "kind": "oracle", "sample": sample},
        "e2e": {"value": val, "unit": "Mpix/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0}))


def run_gpu(args, rank, world, local_rank):
    import torch
    from paper_2408_12282_b200 import binding

    torch.cuda.set_device(local_rank)
    dev = torch.device("cuda", local_rank)
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=dev)
    peaks = load_peaks()
    scene, cams, lights, fps = workload(args.config)
    cam = cams[0]
    npix = cam.width * cam.height
    nl = len(lights)
    R = binding.Renderer(scene, max_instances=int(20 * scene.n), device=local_rank)
    outs = R.alloc_outputs(1, nl, cam.width, cam.height, ("rgb", "counters"))
    num_sms = torch.cuda.get_device_properties(dev).multi_processor_count

    # nvidia-smi samples clocks / throttle reasons from here to the end of the e2e loop: the timed
    # region itself lasts only tens of milliseconds, so every sample is taken under this load
    sampler = ClockSampler(local_rank)
    if rank == 0:
        sampler.start()
    # ---- warm-up (un-captured), then capture one step into a CUDA graph -------------------------
    for _ in range(2):
        R.render(cams=cams, lights=lights, outputs=outs, sum_lights=args.sum_lights, forward=args.forward)
    torch.cuda.synchronize()
    cnt = outs["counters"][0].tolist()
    if cnt[binding.CNT_OVERFLOW] or cnt[binding.CNT_SORT_ERROR]:
        raise RuntimeError(f"render failed: counters {cnt}")
    launches_per_step = R.launch_count()
    graph = torch.cuda.CUDAGraph()
    with torch.cuda.graph(graph):
        R.render(cams=cams, lights=lights, outputs=outs, sum_lights=args.sum_lights, forward=args.forward)
    flush = torch.empty(256 << 20, dtype=torch.uint8, device=dev)  # > 126 MB L2

    def barrier():
        torch.cuda.synchronize()
        multi.barrier()
        torch.cuda.synchronize()

    stream = torch.cuda.current_stream(dev)
    for _ in range(max(args.warmup, 3)):
        flush.zero_()
        graph.replay()
    barrier()
    ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(args.steps)]
    t_wall = time.perf_counter()
    for a, b in ev:
        flush.zero_()            # L2 flush between timed iterations (outside the event pair)
        a.record(stream)
        graph.replay()
        b.record(stream)
    barrier()
    t_wall = time.perf_counter() - t_wall
    step_ms = [a.elapsed_time(b) for a, b in ev]
    total_ms = float(sum(step_ms))
    total_ms = multi.max_over_ranks(total_ms, dev)
    value = multi.whole_job_mpix_per_s(world, args.steps, fps, npix, total_ms)

    # ---- per-stage device times (events inside the library, same step, L2 flushed) --------------
    binding.sssgs_profile_enable(R.ctx, True)
    acc, nlaunch = None, None
    for _ in range(args.steps):
        flush.zero_()
        R.render(cams=cams, lights=lights, outputs=outs, sum_lights=args.sum_lights, forward=args.forward)
        ms, nlaunch = binding.sssgs_profile_read(R.ctx)
        acc = ms if acc is None else {k: acc[k] + ms[k] for k in ms}
    binding.sssgs_profile_enable(R.ctx, False)
    stage_ms = {k: v / args.steps for k, v in acc.items()}

    # ---- end to end through the C ABI with pinned host buffers -------------------------------------
    H = binding.HostRenderer(scene, max_instances=int(20 * scene.n), device=local_rank)
    for _ in range(2):
        H.render(cams, lights)
    barrier()
    t0 = time.perf_counter()
    e2e_steps = max(3, min(args.steps, 20))
    for _ in range(e2e_steps):
        H.render(cams, lights)
    t_e2e = time.perf_counter() - t0
    t_e2e = multi.max_over_ranks(t_e2e, dev)
    e2e_val = multi.whole_job_mpix_per_s(world, e2e_steps, fps, npix, t_e2e * 1e3)
    h2d, d2h = H.h2d_bytes, H.d2h_bytes
    H.close()
    if rank == 0 and len(sampler.rows) < 3:   # keep the GPU busy until a few samples exist
        t_end = time.perf_counter() + 1.5
        while time.perf_counter() < t_end and len(sampler.rows) < 3:
            flush.zero_()
            graph.replay()
            torch.cuda.synchronize()
    clocks = sampler.stop() if rank == 0 else None

    if rank == 0:
        cpu = None
        counters = None
        if world == 1 and not args.no_cpu_baseline:
            r = oracle_sample(scene, min_seconds=12.0)
            cpu = {"value": r["mpix_s"], "unit": "Mpix/s", "cores": r["cores"], "kind": "oracle",
                   "sample": f"{r['frames']} whole-path renders of the first (view, light) frame of "
                             f"configs[{args.config - 1}] (bf16-emulating MLP), {r['seconds']:.1f} s of CPU work"}
            counters = (r["res"].comp.p_eval, r["res"].comp.p_blend)
        mlp_rows = cnt[binding.CNT_MLP_ROWS] or scene.n
        models, pk = stage_models(scene, nl, cnt[binding.CNT_NVIS], min(cnt[binding.CNT_INSTANCES], 20 * scene.n),
                                  counters, peaks, num_sms, mlp_rows)
        stages = {}
        for k, ms in stage_ms.items():
            e = {"ms": round(ms, 5), "launches": nlaunch[k]}
            if k in models and models[k][1] is not None and ms > 0:
                bound, work = models[k]
                ach = work / (ms * 1e-3) / (1e9 if bound == "hbm" else 1e12)
                e.update(bound=bound, achieved=round(ach, 3), unit=pk[bound][1], frac=round(ach / pk[bound][0], 4))
            stages[k] = e
        dom = max(stage_ms, key=stage_ms.get)
        roof = {"kernel": dom, "bound": stages[dom].get("bound"), "achieved": stages[dom].get("achieved"),
                "peak": round(pk[stages[dom]["bound"]][0], 2) if "bound" in stages[dom] else None,
                "unit": stages[dom].get("unit"), "frac": stages[dom].get("frac"),
                "traffic": NCU_DRAM_BYTES_PER_LAUNCH.get((args.config, dom)),
                "peak_source": peaks["source"] if stages[dom].get("bound") != "alu" else
                "derived: SMs x 128 fp32 lanes x 2 x clocks.max.sm (DESIGN.md)",
                "share_of_step": round(stage_ms[dom] / sum(stage_ms.values()), 3)}
        print(json.dumps({
            "metric": METRIC, "value": value, "unit": "Mpix/s", "n_gpus": world, "steps": args.steps,
            "warmup": max(args.warmup, 3), "ms_per_step": total_ms / args.steps, "higher_is_better": True,
            "scaling": "weak", "vs_baseline": None, "dtype": "f32 (raster/shade) + bf16 x bf16 -> f32 (MLP)",
            "data": "synthetic",
            "config": {"workload": f"configs[{args.config - 1}] {scene.name}", "gaussians": scene.n,
                       "width": cam.width, "height": cam.height, "frames_per_step": fps,
                       "l2": "flushed between timed steps (256 MiB memset)", "launch": "CUDA graph replay",
                       "instances": cnt[binding.CNT_INSTANCES], "mlp_rows_per_light": mlp_rows,
                       "sum_lights": bool(args.sum_lights), "forward_shading": bool(args.forward)},
            "ms_per_frame": total_ms / args.steps / fps,
            "gaussians_per_s": world * args.steps * fps * scene.n / (total_ms * 1e-3),
            "clocks": clocks,
            "e2e": {"value": e2e_val, "unit": "Mpix/s", "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": d2h,
                    "steps": e2e_steps},
            "gpu_launches": launches_per_step * args.steps,
            "roofline": roof, "stages": stages, "cpu_baseline": cpu,
            "wall_s_timed_region": round(t_wall, 4)}))
    R.close()
    if world > 1:
        dist.destroy_process_group()


def fibonacci_dirs(K):
    k = np.arange(K) + 0.5
    z = 1 - 2 * k / K
    phi = k * np.pi * (3 - np.sqrt(5))
    r = np.sqrt(1 - z * z)
    return np.stack([r * np.cos(phi), r * np.sin(phi), z], 1).astype(np.float32), np.full(K, 4 * np.pi / K, np.float32)


def run_bake(args, local_rank):
    """--bake K: times sssgs_bake_visibility on the config's Gaussians, K Fibonacci directions.
    A side measurement: its JSON line has its own metric (rays/s) and is not the headline."""
    import torch
    from paper_2408_12282_b200 import binding
    torch.cuda.set_device(local_rank)
    dev = torch.device("cuda", local_rank)
    scene, cams, lights, fps = workload(args.config)
    K, t_min = args.bake, 0.05
    dirs, wts = fibonacci_dirs(K)
    R = binding.Renderer(scene, max_instances=int(20 * scene.n), device=local_rank)
    d_dirs, d_wts = torch.from_numpy(dirs).to(dev), torch.from_numpy(wts).to(dev)
    for _ in range(max(args.warmup, 3)):
        sh, _ = R.bake_visibility(d_dirs, d_wts, t_min)
    torch.cuda.synchronize()
    launches = R.launch_count()
    stream = torch.cuda.current_stream(dev)
    flush = torch.empty(256 << 20, dtype=torch.uint8, device=dev)
    ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(args.steps)]
    for a, b in ev:
        flush.zero_()
        a.record(stream)
        sh, _ = R.bake_visibility(d_dirs, d_wts, t_min)
        b.record(stream)
    torch.cuda.synchronize()
    ms = float(np.mean([a.elapsed_time(b) for a, b in ev]))
    cpu = None
    if not args.no_cpu_baseline:
        import oracle   # cpu_baseline leg only
        rows = np.random.default_rng(0).choice(scene.n, size=min(scene.n, max(8, int(2e9 / (scene.n * K)))), replace=False)
        t0 = time.perf_counter()
        oracle.bake_visibility(scene, dirs, wts, t_min, rows=rows)
        dt = time.perf_counter() - t0
        cpu = {"value": len(rows) * K / dt / 1e6, "unit": "Mrays/s", "cores": oracle.num_threads(), "kind": "oracle",
               "sample": f"{len(rows)} of {scene.n} Gaussians x {K} directions, brute force over all pairs, {dt:.1f} s"}
    R.close()
    print(json.dumps({"metric": "Mrays/s (BVH build + traversal + SH fit)", "value": scene.n * K / ms / 1e3, "unit": "Mrays/s",
                      "n_gpus": 1, "steps": args.steps, "warmup": max(args.warmup, 3), "ms_per_step": ms,
                      "higher_is_better": True, "vs_baseline": None, "dtype": "f32", "data": "synthetic",
                      "config": {"workload": f"configs[{args.config - 1}] {scene.name}", "gaussians": scene.n, "dirs": K,
                                 "t_min": t_min, "l2": "flushed between timed steps (256 MiB memset)"},
                      "gpu_launches": launches * args.steps, "cpu_baseline": cpu}))


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=50)
    ap.add_argument("--warmup", type=int, default=5)
    ap.add_argument("--config", type=int, default=2, choices=[1, 2, 3, 4, 5, 6])
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--forward", action="store_true",
                    help="the paper's 'w/o deferred' variant (SSSGS_FORWARD_SHADING): Eq. 7 per Gaussian, RGB composited")
    ap.add_argument("--sum-lights", action="store_true",
                    help="image-based-lighting mode (SSSGS_SUM_LIGHTS): the lights of a step are summed into one frame")
    ap.add_argument("--bake", type=int, default=0, metavar="K",
                    help="time sssgs_bake_visibility with K directions instead of the render step (side measurement)")
    args = ap.parse_args()
    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    if args.impl == "reference":
        if args.steps > 60:
            args.steps = 60  # bounded: each step is seconds of CPU work
        run_reference(args, rank)
        return
    if args.bake:
        if rank == 0:
            run_bake(args, local_rank)
        return
    run_gpu(args, rank, world, local_rank)


if __name__ == "__main__":
    main()
