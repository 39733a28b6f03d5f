#!/usr/bin/env python
"""bench.py -- throughput of the SSS-GS forward relighting render path on B200.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config C] [--impl reference]

A step = one pass of the whole hot path (MLP + projection + sort + tile binning + G-buffer
compositing + deferred shading) over one batch of synthetic input = ONE sssgs_render call producing
every frame of one view of the workload.  BASELINE.json's `metric` names no configuration, so the
default workload is the largest single-GPU one, configs[4] (C = 5): 3 M Gaussians, 1024 x 1024, one
view x its 16 lights per step.  Prints ONE JSON line:

  value     Mpix/s, inputs resident in HBM, CUDA events around each step, L2 flushed between
            steps, step replayed from a CUDA graph (the launch configuration the tests check);
            ms_per_step is the mean over the K timed steps, ms_per_step_median / _min beside it
  e2e       same metric through sssgs_render_host with pinned HOST buffers (H2D + D2H inside)
  roofline  the step's dominant kernel against its bound, timed with events inside the library
  stages    every stage of the step: ms, launches, achieved vs measured (and nominal) peak
  configs   the same protocol on all five BASELINE configs (ms/step median and min, Mpix/s,
            Gaussians/s, dominant stage and its roofline fraction)
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
# dram__bytes_read.sum + dram__bytes_write.sum of ONE launch of a stage's heaviest kernel, from the `ncu --set full`
# captures summarised in profiles/r03_ncu_full.md (configs[4]) and profiles/r02_ncu_full.md (configs[1], [2]); tight
# lists, one view x all lights: (config, stage) -> bytes.  Constants: a kernel change needs a new capture.
NCU_DRAM_BYTES_PER_LAUNCH = {
    ("5", "prepass"): 375.5e6 + 617.1e6,   # raster_shade_kernel<1,1,4,4,1,0>: lists + rows in, weight cache + T out
    ("5", "raster"): 795.4e6 + 98.1e6,     # raster_cached_kernel<8,0>: weight cache + rows in, 8 frames out
    ("5", "mlp"): 190.6e6 + 30.0e6,        # mlp_kernel<8,1,1>: kept rows' inputs in, 8 x 16 B per kept row out
    ("3", "raster"): 148.3e6 + 61.6e6,     # raster_cached_kernel<8,1> (cfg 3, one of the 7 later batches)
    ("2", "raster"): 13.5e6 + 17.9e6,      # raster_shade_kernel<1,4,8,2,0,0> (cfg 2)
}
# the same two ncu metrics summed over EVERY kernel launch of one default step (tight lists, one view x all lights)
NCU_DRAM_BYTES_PER_STEP = {
    "5": 4.603e9,   # profiles/r03_ncu_full.md: the 19 launches of the step
}
FP32_LANES_PER_SM = 128
HBM_NOMINAL_GBS = 8000.0   # BASELINE.json north_star: "~8 TB/s"
MAX_INSTANCES_PER_GAUSSIAN = 20


def load_peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        d = json.load(open(p))
        return dict(hbm=float(d["hbm_gbs"]), bf16_burst=float(d["bf16_tflops"]),
                    bf16_sustained=float(d.get("bf16_tflops_sustained", d["bf16_tflops"])),
                    sm_max_mhz=float(d.get("sm_max_mhz", 1965.0)), source="measured")
    return dict(hbm=6650.0, bf16_burst=1590.0, bf16_sustained=1400.0, sm_max_mhz=1965.0, source="fallback")


def load_oracle_counters():
    """Work counters of every config's first frame, written by oracle/make_workload_counters.py
    (oracle only).  They are the denominators of the raster / pre-pass roofline figures."""
    p = os.path.join(ROOT, "oracle", "workload_counters.json")
    return json.load(open(p)) if os.path.exists(p) else {}


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
        sm, mx, pw, reasons = [], [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for r in self.rows:
            try:
                sm.append(float(r[0]))
                mx.append(float(r[1]))
                pw.append(float(r[2]))
                for k, nm in enumerate(names):
                    if r[3 + k].lower().startswith("active"):
                        reasons.add(nm)
            except Exception:
                pass
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "power_w_max": max(pw) if pw else None, "samples": len(sm), "reasons": sorted(reasons)}


BACKWARD_CONFIGS = (2, 4)   # configs whose backward pass (one view, one light) is timed beside the forward table


def workload(cfg, rank=0, world=1):
    """(scene, cams of one step, lights of one step, frames per step).  Under torchrun each rank renders its own
    view of the config's orbit (multi.frames_of_rank: round-robin by view; view 0 at N = 1)."""
    s = scenes.make_scene(cfg)
    mine = multi.frames_of_rank(len(s.cameras), rank, world)
    v = mine[0] if mine else rank % len(s.cameras)
    return s, s.cameras[v:v + 1], s.lights[v], len(s.lights[v])


def config_dict(cfg, scene, fps):
    """The `config` object: identical in the GPU arm and in the reference arm (same workload)."""
    cam = scene.cameras[0]
    m = scene.mlp
    return {"workload": f"configs[{cfg - 1}] {scene.name}: {scene.n} Gaussians, {cam.width}x{cam.height}, "
                        f"one view x {fps} light(s) per step (view 0 of {len(scene.cameras)}; rank r of N renders view r)",
            "gaussians": int(scene.n), "width": int(cam.width), "height": int(cam.height),
            "frames_per_step": int(fps), "views_in_config": len(scene.cameras),
            "mlp": f"{m.in_dim} -> {'x'.join(str(w) for w in m.trunk_width)} -> 3+1",
            "mlp_compute": "fp16 x fp16 -> fp32 (weights bf16-exact)", "tile_lists": "tight (SURVEY S5)",
            "l2": "flushed between timed steps (256 MiB memset)", "launch": "CUDA graph replay"}


# ---------------------------------------------------------------------------------------------------
# CPU oracle legs (cpu_baseline, --impl reference): the only places bench.py executes oracle/
# ---------------------------------------------------------------------------------------------------
def oracle_sample(scene, count_on=None):
    """count_on = (vals, ranges) of another tile list of the same view (the device's tight list): the oracle's
    compositor also counts the evaluated pairs of THAT list (outside the timed seconds) -> "p_eval_counted".

    One whole-path render of the first (view, light) frame by the CPU oracle, as it stands: projection, lists,
    the fp16-emulating MLP on ALL rows, compositing and shading of the whole frame.  Every second reported was
    spent; nothing is extrapolated.  Bounded by construction: ONE frame (the GPU step renders `frames_per_step`)."""
    import oracle
    cam, lt = scene.cameras[0], scene.lights[0][0]
    t0 = time.perf_counter()
    proj = oracle.project(scene, cam)
    keys, vals, ranges = oracle.build_lists(proj)
    t_geo = time.perf_counter() - t0
    t0 = time.perf_counter()
    x = oracle.mlp_inputs(scene, cam, lt.position)
    mlp_out = oracle.mlp_forward(x, scene.mlp, 2)
    t_mlp = time.perf_counter() - t0
    t0 = time.perf_counter()
    comp = oracle.composite(scene, cam, proj, oracle.channels(scene, proj, mlp_out), vals, ranges)
    oracle.shade(cam, lt, comp.gbuf)
    t_img = time.perf_counter() - t0
    total = t_geo + t_mlp + t_img
    counted = None
    if count_on is not None:
        c2 = oracle.composite(scene, cam, proj, oracle.channels(scene, proj, mlp_out), count_on[0], count_on[1])
        assert c2.p_blend == comp.p_blend, "the device's tight list does not blend the pairs the canonical list blends"
        counted = c2.p_eval
    return dict(seconds=total, frames=1, p_eval_counted=counted, mpix_s=cam.width * cam.height / total / 1e6, cores=oracle.num_threads(),
                p_eval=comp.p_eval, p_blend=comp.p_blend,
                sample=(f"one whole-path render of the first (view, light) frame of {scene.name}, all measured: "
                        f"projection + lists {t_geo:.1f} s, fp16-emulating MLP on all {int(scene.n)} rows {t_mlp:.1f} s, "
                        f"compositing + shading of the whole frame {t_img:.1f} s"))


def run_reference(args, rank):
    """Reference arm of this tier: the CPU oracle, as it stands, on the host cores (rank 0 only)."""
    if rank != 0:
        return
    scene, cams, lights, fps = workload(args.config)
    cam = cams[0]
    # bounded: a step (one frame) is up to ~20 s of CPU work on the largest config; the whole run ends within
    # a few minutes and `steps` / `ms_per_step` are what was really run and timed
    steps = max(1, min(args.steps, 3 if scene.n > 200_000 else 30))
    warm = min(args.warmup, 1 if scene.n > 200_000 else 3)
    for _ in range(warm):
        oracle_sample(scene)
    t, cores, sample = 0.0, 1, ""
    for _ in range(steps):
        r = oracle_sample(scene)
        t += r["seconds"]
        cores, sample = r["cores"], r["sample"]
    val = steps * cam.width * cam.height / t / 1e6
    cfg_d = config_dict(args.config, scene, 1)     # this arm renders ONE (view, light) frame per step
    cfg_d["gpu_arm_frames_per_step"] = int(fps)
    cfg_d["l2"] = cfg_d["launch"] = "n/a (CPU)"
    print(json.dumps({
        "impl": "reference", "metric": METRIC, "value": val, "unit": "Mpix/s", "n_gpus": args.gpus,
        "steps": steps, "warmup": warm, "ms_per_step": t / steps * 1e3,
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": cfg_d,
        "cpu_baseline": {"value": val, "unit": "Mpix/s", "cores": cores, "kind": "oracle",
                         "sample": sample + "; one frame per step (the oracle has no light batching)"},
        "e2e": {"value": val, "unit": "Mpix/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0}))


# ---------------------------------------------------------------------------------------------------
# Work models: algorithmic bytes / flops of each stage for ONE step
# ---------------------------------------------------------------------------------------------------
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


def stage_models(scene, nl, n_vis, inst, ocnt, peaks, num_sms, mlp_rows, swept, tight):
    """-> (work model per stage for the list mode being timed, the same with the canonical-list counters where that
    differs, peaks).  With tight lists the evaluated-pair count is the oracle's count on the MINIMAL S5 list
    (oracle/workload_counters.json p_eval_min): the device's tight list is a superset of it, so the figure is a lower
    bound of the pairs the walk evaluated and the fraction is conservative."""
    n = scene.n
    alu_peak = num_sms * FP32_LANES_PER_SM * 2 * peaks["sm_max_mhz"] * 1e6 / 1e12  # TFLOP/s
    m = {
        "project": ("hbm", 44.0 * n + 48.0 * n_vis),
        "depth_sort": ("hbm", (3 * 16.0 + 12.0) * n),
        "emit": ("hbm", 16.0 * n + 8.0 * inst),
        "tile_sort": ("hbm", 16.0 * inst),     # ONE stable pass over (tile, index) pairs is the algorithmic minimum
        "ranges": ("hbm", 4.0 * inst),
        # rows the MLP actually evaluated (in a sweep: the Gaussians blended at some pixel of the view)
        "mlp": ("tensor", float(mlp_flops_per_row(scene.mlp)) * mlp_rows * nl),
    }
    alt = {}
    if ocnt:
        def walks(pe, pb, out):
            if swept:   # pre-pass: alpha + transmittance chain once per view; walks: blends only
                out["prepass"] = ("alu", 10.0 * pe + 3.0 * pb)
                out["raster"] = ("alu", 2.0 * (11.0 + 4.0 * nl) * pb)
            else:
                out["raster"] = ("alu", 10.0 * pe + (17.0 + 8.0 * (nl - 1)) * pb)
        pb = float(ocnt["p_blend"])
        if tight and "p_eval_min" in ocnt:
            walks(float(ocnt["p_eval_min"]), pb, m)
            walks(float(ocnt["p_eval"]), pb, alt)
        else:
            walks(float(ocnt["p_eval"]), pb, m)
    pk = {"hbm": (peaks["hbm"], "GB/s"), "tensor": (peaks["bf16_burst"], "TFLOP/s"), "alu": (alu_peak, "TFLOP/s")}
    return m, alt, pk


class ConfigRun:
    """One config on one GPU: device-resident scene, a CUDA graph of one step, timed replays, per-stage
    device times.  The timing protocol of the headline number and of every row of `configs`."""

    def __init__(self, cfg, local_rank, args, scene=None):
        import torch
        from paper_2408_12282_b200 import binding
        self.torch, self.binding, self.cfg = torch, binding, cfg
        self.dev = torch.device("cuda", local_rank)
        if scene is None:
            self.scene, self.cams, self.lights, self.fps = workload(cfg, *multi.env_ranks()[:2])
        else:
            self.scene, self.cams, self.lights, self.fps = scene, scene.cameras[:1], scene.lights[0], len(scene.lights[0])
        self.cam = self.cams[0]
        self.npix = self.cam.width * self.cam.height
        self.kw = dict(sum_lights=args.sum_lights, forward=args.forward, tight=not args.canonical_lists)
        self.R = binding.Renderer(self.scene, max_instances=int(MAX_INSTANCES_PER_GAUSSIAN * self.scene.n),
                                  device=local_rank,
                                  compute=binding.SSSGS_COMPUTE_BF16 if args.bf16 else binding.SSSGS_COMPUTE_FP16)
        self.outs = self.R.alloc_outputs(1, len(self.lights), self.cam.width, self.cam.height, ("rgb", "counters"))
        for _ in range(2):
            self.render()
        torch.cuda.synchronize()
        self.cnt = self.outs["counters"][0].tolist()
        if self.cnt[binding.CNT_OVERFLOW] or self.cnt[binding.CNT_SORT_ERROR]:
            raise RuntimeError(f"render failed: counters {self.cnt}")
        self.launches = self.R.launch_count()
        self.graph = torch.cuda.CUDAGraph()
        with torch.cuda.graph(self.graph):
            self.render()

    def render(self):
        self.R.render(cams=self.cams, lights=self.lights, outputs=self.outs, **self.kw)

    def timed(self, steps, warmup, flush, barrier=lambda: None):
        torch = self.torch
        stream = torch.cuda.current_stream(self.dev)
        for _ in range(max(warmup, 3)):
            flush.zero_()
            self.graph.replay()
        barrier()
        ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(steps)]
        t_wall = time.perf_counter()
        for a, b in ev:
            flush.zero_()            # L2 flush between timed iterations (outside the event pair)
            a.record(stream)
            self.graph.replay()
            b.record(stream)
        barrier()
        torch.cuda.synchronize()
        t_wall = time.perf_counter() - t_wall
        return [a.elapsed_time(b) for a, b in ev], t_wall

    def stage_times(self, reps, flush):
        """Per-stage device times: events inside the library, stages serialised, L2 flushed."""
        b = self.binding
        b.sssgs_profile_enable(self.R.ctx, True)
        acc, nlaunch = None, None
        for _ in range(reps):
            flush.zero_()
            self.render()
            ms, nlaunch = b.sssgs_profile_read(self.R.ctx)
            acc = ms if acc is None else {k: acc[k] + ms[k] for k in ms}
        b.sssgs_profile_enable(self.R.ctx, False)
        return {k: v / reps for k, v in acc.items()}, nlaunch

    def stages(self, stage_ms, nlaunch, ocnt, peaks, num_sms):
        b = self.binding
        nl = len(self.lights)
        mlp_rows = self.cnt[b.CNT_MLP_ROWS] or self.scene.n
        swept = nlaunch.get("prepass", 0) > 0
        inst = min(self.cnt[b.CNT_INSTANCES], MAX_INSTANCES_PER_GAUSSIAN * self.scene.n)
        models, alt, pk = stage_models(self.scene, nl, self.cnt[b.CNT_NVIS], inst, ocnt, peaks, num_sms, mlp_rows, swept,
                                       self.kw["tight"])
        out = {}
        for k, ms in stage_ms.items():
            if nlaunch[k] == 0:
                continue
            e = {"ms": round(ms, 5), "launches": nlaunch[k]}
            if k in models and ms > 0:
                bound, work = models[k]
                ach = work / (ms * 1e-3) / (1e9 if bound == "hbm" else 1e12)
                e.update(bound=bound, achieved=round(ach, 3), unit=pk[bound][1], frac=round(ach / pk[bound][0], 4))
                if bound == "hbm":
                    e["frac_of_nominal_8TBs"] = round(ach / HBM_NOMINAL_GBS, 4)
                if k in alt and alt[k][1] != work:
                    e["counters"] = "minimal S5 list (p_eval_min): lower bound of the pairs a tight-list walk evaluates"
                    e["frac_with_canonical_list_counters"] = round(alt[k][1] / (ms * 1e-3) / 1e12 / pk[bound][0], 4)
            out[k] = e
        return out, pk

    def backward_ms(self, reps=3):
        """sssgs_render_backward of the step's view and lights: median device time over `reps`
        calls, G-buffer of a forward call and a seeded dL/drgb resident in HBM."""
        torch = self.torch
        fwd = self.R.render(cams=self.cams, lights=self.lights, want=("rgb", "gbuffer"), tight=self.kw["tight"])
        gen = torch.Generator(device=self.dev).manual_seed(7)
        G = torch.randn(fwd["rgb"].shape, generator=gen, device=self.dev)
        def timed(**kw):
            ms = []
            for _ in range(reps + 1):
                a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                a.record()
                self.R.render_backward(self.cam, self.lights, G, fwd["gbuffer"], tight=self.kw["tight"], **kw)
                b.record()
                torch.cuda.synchronize()
                ms.append(a.elapsed_time(b))
            return round(float(np.median(ms[1:])), 4)
        ms_all = timed(through_inputs=True)     # + step a1: feature, visibility SH, input-side shares
        ms = timed()
        return {"ms": ms, "ms_with_input_gradients": ms_all, "launches": self.R.launch_count(),
                "lights": len(self.lights), "mlp_backward": "tcgen05, binary16 operands (fp32 CUDA-core path: SSSGS_BACKWARD_FP32)"}

    def close(self):
        self.graph = None
        self.R.close()


def summarize(step_ms):
    a = np.asarray(step_ms, np.float64)
    return float(a.mean()), float(np.median(a)), float(a.min())


def run_gpu(args, rank, world, local_rank):
    import torch
    from paper_2408_12282_b200 import binding

    torch.cuda.set_device(local_rank)
    dev = torch.device("cuda", local_rank)
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=dev)
    peaks = load_peaks()
    ocnt_all = load_oracle_counters()
    num_sms = torch.cuda.get_device_properties(dev).multi_processor_count
    flush = torch.empty(256 << 20, dtype=torch.uint8, device=dev)  # > 126 MB L2

    # nvidia-smi samples clocks / throttle reasons from here to the end of the e2e loop
    sampler = ClockSampler(local_rank)
    if rank == 0:
        sampler.start()

    def barrier():
        torch.cuda.synchronize()
        multi.barrier()
        torch.cuda.synchronize()

    run = ConfigRun(args.config, local_rank, args)
    scene, cam, fps, npix = run.scene, run.cam, run.fps, run.npix
    step_ms, t_wall = run.timed(args.steps, args.warmup, flush, barrier)
    total_ms = multi.max_over_ranks(float(sum(step_ms)), dev)
    value = multi.whole_job_mpix_per_s(world, args.steps, fps, npix, total_ms)
    mean_ms, med_ms, min_ms = summarize(step_ms)
    stage_ms, nlaunch = run.stage_times(min(args.steps, 10), flush)

    # ---- end to end through the C ABI with pinned host buffers -------------------------------------
    H = binding.HostRenderer(scene, max_instances=int(MAX_INSTANCES_PER_GAUSSIAN * scene.n), device=local_rank)
    for _ in range(2):
        H.render(run.cams, run.lights, tight=not args.canonical_lists)
    barrier()
    t0 = time.perf_counter()
    e2e_steps = max(3, min(args.steps, 10))
    for _ in range(e2e_steps):
        H.render(run.cams, run.lights, tight=not args.canonical_lists)
    t_e2e = multi.max_over_ranks(time.perf_counter() - t0, dev)
    e2e_val = multi.whole_job_mpix_per_s(world, e2e_steps, fps, npix, t_e2e * 1e3)
    h2d, d2h = H.h2d_bytes, H.d2h_bytes
    H.close()
    del H
    if rank == 0 and len(sampler.rows) < 3:   # keep the GPU busy until a few samples exist
        t_end = time.perf_counter() + 1.5
        while time.perf_counter() < t_end and len(sampler.rows) < 3:
            flush.zero_()
            run.graph.replay()
            torch.cuda.synchronize()
    clocks = sampler.stop() if rank == 0 else None

    if rank == 0:
        key = f"configs[{args.config - 1}]"
        ocnt = ocnt_all.get(key)
        stages, pk = run.stages(stage_ms, nlaunch, ocnt, peaks, num_sms)
        if ocnt and not args.sum_lights and not args.forward:   # the device's own counters against the oracle's
            assert ocnt["n_vis"] == run.cnt[binding.CNT_NVIS], (ocnt, run.cnt)
            if args.canonical_lists:
                assert ocnt["instances"] == run.cnt[binding.CNT_INSTANCES], (ocnt, run.cnt)
            else:   # tight lists: a sub-sequence of the canonical list
                assert run.cnt[binding.CNT_INSTANCES] <= ocnt["instances"], (ocnt, run.cnt)
        dom = max(stage_ms, key=stage_ms.get)
        sd = stages[dom]
        roof = {"kernel": dom, "bound": sd.get("bound"), "achieved": sd.get("achieved"),
                "peak": round(pk[sd["bound"]][0], 2) if "bound" in sd else None,
                "unit": sd.get("unit"), "frac": sd.get("frac"),
                "traffic": NCU_DRAM_BYTES_PER_LAUNCH.get((str(args.config), dom)),
                "launches_per_step": sd.get("launches"),
                "peak_source": peaks["source"] if sd.get("bound") != "alu" else
                "derived: SMs x 128 fp32 lanes x 2 x clocks.max.sm (DESIGN.md)",
                "share_of_step": round(stage_ms[dom] / sum(stage_ms.values()), 3)}
        if sd.get("bound") == "hbm":
            roof["frac_of_nominal_8TBs"] = sd.get("frac_of_nominal_8TBs")
        for extra in ("counters", "frac_with_canonical_list_counters"):
            if extra in sd:
                roof[extra] = sd[extra]
        roof["traffic_source"] = ("constant from one `ncu --set full` capture of this kernel (profiles/r03_ncu_full.md), "
                                  "not measured by this run" if roof["traffic"] else None)
        # BASELINE.json's metric asks for the pipeline's share of the HBM roofline: DRAM bytes of ALL kernels of one
        # step (same capture) over the measured step time.  The path is instruction-issue-bound, not HBM-bound.
        step_bytes = NCU_DRAM_BYTES_PER_STEP.get(str(args.config)) if not args.canonical_lists else None
        if step_bytes:
            roof["hbm_frac_of_step"] = round(step_bytes / (med_ms * 1e-3) / 1e9 / peaks["hbm"], 4)
            roof["hbm_bytes_per_step"] = step_bytes
            roof["hbm_frac_of_step_source"] = ("sum of dram__bytes_read + dram__bytes_write over every kernel of one step "
                                               "(profiles/r03_ncu_full.md) / median step time / measured HBM peak")
        roof["pipeline_bound"] = "instruction issue (fp32 / integer ALU work of the list walks) + tensor pipe (MLP); not HBM"

        row = dict(ms_per_step_median=round(med_ms, 5), ms_per_step_min=round(min_ms, 5), frames_per_step=fps,
                   mpix_s=round(fps * npix / med_ms / 1e3, 1), gaussians_per_s=round(fps * scene.n / (med_ms * 1e-3), 0),
                   dominant_stage=dom, dominant_frac=sd.get("frac"), dominant_bound=sd.get("bound"),
                   mlp_tensor_frac=stages.get("mlp", {}).get("frac"),
                   stage_ms={k: v["ms"] for k, v in stages.items()})
        table = {key: row}
        backward = {}
        if args.config in BACKWARD_CONFIGS and world == 1 and not args.no_table:
            backward[key] = run.backward_ms()
        launches_per_step = run.launches
        cnt_head, mlp_rows_head = run.cnt, (run.cnt[binding.CNT_MLP_ROWS] or scene.n)
        dev_list = None
        if world == 1 and not args.no_cpu_baseline and not args.canonical_lists and not args.forward and not args.sum_lights:
            # the tight list the timed step walked (geometry-only call), for the oracle to count its evaluated pairs
            o = run.R.render(cams=run.cams, lights=run.lights[:1], want=("sorted_vals", "tile_ranges", "counters"),
                             tight=True, precomputed=torch.zeros((1, max(scene.n, 1), 4), device=dev))
            torch.cuda.synchronize()
            n_inst = int(o["counters"][0][binding.CNT_INSTANCES])
            dev_list = (o["sorted_vals"][0][:n_inst].cpu().numpy().view(np.uint32), o["tile_ranges"][0].cpu().numpy().view(np.uint32))
            del o
        run.close()
        del run
        torch.cuda.empty_cache()
        # ---- the same protocol on the other BASELINE configs ---------------------------------------
        if world == 1 and not args.no_table and not args.sum_lights and not args.forward:
            for c in (1, 2, 3, 4, 5):
                k = f"configs[{c - 1}]"
                if k in table:
                    continue
                r = ConfigRun(c, local_rank, args)
                sm, _ = r.timed(min(args.steps, 10), 3, flush)
                st_ms, nl_ = r.stage_times(3, flush)
                st, _pk = r.stages(st_ms, nl_, ocnt_all.get(k), peaks, num_sms)
                _, med, mn = summarize(sm)
                d = max(st_ms, key=st_ms.get)
                table[k] = dict(ms_per_step_median=round(med, 5), ms_per_step_min=round(mn, 5), frames_per_step=r.fps,
                                mpix_s=round(r.fps * r.npix / med / 1e3, 1),
                                gaussians_per_s=round(r.fps * r.scene.n / (med * 1e-3), 0),
                                dominant_stage=d, dominant_frac=st[d].get("frac"), dominant_bound=st[d].get("bound"),
                                mlp_tensor_frac=st.get("mlp", {}).get("frac"),
                                stage_ms={kk: v["ms"] for kk, v in st.items()})
                if c in BACKWARD_CONFIGS:
                    backward[k] = r.backward_ms()
                r.close()
                del r
                torch.cuda.empty_cache()
        cpu = None
        if world == 1 and not args.no_cpu_baseline:
            r = oracle_sample(scene, count_on=dev_list)
            cpu = {"value": r["mpix_s"], "unit": "Mpix/s", "cores": r["cores"], "kind": "oracle",
                   "sample": r["sample"] + f"; {r['seconds']:.1f} s of CPU work"}
            if r["p_eval_counted"] is not None and roof.get("bound") == "alu" and dom in ("prepass", "raster"):
                # the dominant walk's fraction on the pairs of the list it really walked (counted by the oracle's
                # compositor on the device's exported tight list; not part of the timed seconds)
                pe, pb = float(r["p_eval_counted"]), float(r["p_blend"])
                nl_ = len(scene.lights[0])
                work = (10.0 * pe + 3.0 * pb) if dom == "prepass" else \
                    (10.0 * pe + (17.0 + 8.0 * (nl_ - 1)) * pb if "prepass" not in stages else None)
                if work:
                    roof["p_eval_device_tight_list"] = int(pe)
                    roof["frac_on_device_tight_list"] = round(work / (stage_ms[dom] * 1e-3) / 1e12 / roof["peak"], 4)
        cfg_d = config_dict(args.config, scene, fps)
        print(json.dumps({
            "metric": METRIC, "value": value, "unit": "Mpix/s", "n_gpus": world, "steps": args.steps,
            "warmup": max(args.warmup, 3), "ms_per_step": total_ms / args.steps,
            "ms_per_step_median": med_ms, "ms_per_step_min": min_ms, "higher_is_better": True,
            "scaling": "weak", "vs_baseline": None,
            "dtype": "f32 (raster/shade) + " + ("bf16 x bf16" if args.bf16 else "fp16 x fp16") + " -> f32 (MLP)",
            "data": "synthetic", "config": cfg_d,
            "variant": {"sum_lights": bool(args.sum_lights), "forward_shading": bool(args.forward),
                        "tile_lists": "canonical" if args.canonical_lists else
                        "tight (SSSGS_TIGHT_LISTS, SURVEY S5: sub-sequence of the canonical list, bit-identical frames)"},
            "counters": {"n_vis": cnt_head[binding.CNT_NVIS], "instances": cnt_head[binding.CNT_INSTANCES],
                         "mlp_rows_per_light": mlp_rows_head, "oracle": ocnt},
            "ms_per_frame": med_ms / fps,
            "gaussians_per_s": world * args.steps * fps * scene.n / (total_ms * 1e-3),
            "clocks": clocks,
            "e2e": {"value": e2e_val, "unit": "Mpix/s", "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": d2h,
                    "steps": e2e_steps,
                    "note": "sssgs_render_host uploads the WHOLE scene and downloads every frame in each call "
                            "(one crossing per call by design): PCIe-bound"},
            "gpu_launches": launches_per_step * args.steps,
            "roofline": roof, "stages": stages, "configs": table, "backward": backward, "cpu_baseline": cpu,
            "peaks": {"hbm_gbs_measured": peaks["hbm"], "hbm_gbs_nominal": HBM_NOMINAL_GBS,
                      "bf16_tflops_burst": peaks["bf16_burst"], "bf16_tflops_sustained": peaks["bf16_sustained"],
                      "source": peaks["source"]},
            "wall_s_timed_region": round(t_wall, 4)}))
    else:
        run.close()
    if world > 1:
        dist.destroy_process_group()


def fibonacci_dirs(K):
    k = np.arange(K) + 0.5
    z = 1 - 2 * k / K
    phi = k * np.pi * (3 - np.sqrt(5))
    r = np.sqrt(1 - z * z)
    return np.stack([r * np.cos(phi), r * np.sin(phi), z], 1).astype(np.float32), np.full(K, 4 * np.pi / K, np.float32)


def run_relight(args, local_rank):
    """--relight: times sssgs_relight on an OLAT stack of the config's frame shape
    (frames_per_step lights), resident in HBM.  A side measurement with its own metric; HBM roofline: 12 (L + 1) P
    bytes per call over the measured copy bandwidth."""
    import torch
    from paper_2408_12282_b200 import binding
    torch.cuda.set_device(local_rank)
    dev = torch.device("cuda", local_rank)
    scene, cams, lights, fps = workload(args.config)
    cam, L = cams[0], max(len(lights), 1)
    P = cam.width * cam.height
    gen = torch.Generator(device=dev).manual_seed(1)
    frames = torch.rand((L, cam.height, cam.width, 3), generator=gen, device=dev)
    w = torch.rand((L, 3), generator=gen, device=dev)
    out = torch.empty((cam.height, cam.width, 3), device=dev)
    flush = torch.empty(256 << 20, dtype=torch.uint8, device=dev)
    stream = torch.cuda.current_stream(dev)
    call = lambda: binding.sssgs_relight(local_rank, frames.data_ptr(), L, P, w.data_ptr(), out.data_ptr(), stream.cuda_stream)  # noqa: E731
    for _ in range(max(args.warmup, 3)):
        call()
    ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(args.steps)]
    for a, b in ev:
        flush.zero_()
        a.record(stream)
        call()
        b.record(stream)
    torch.cuda.synchronize()
    ms = float(np.median([a.elapsed_time(b) for a, b in ev]))
    peaks = load_peaks()
    nbytes = 12.0 * (L + 1) * P
    gbs = nbytes / (ms * 1e-3) / 1e9
    print(json.dumps({
        "metric": "relit Mpix/s (sssgs_relight: sum over a precomputed reflectance field, PAPER.md L301)",
        "value": P / (ms * 1e-3) / 1e6, "unit": "Mpix/s", "n_gpus": 1, "steps": args.steps, "warmup": max(args.warmup, 3),
        "ms_per_step": ms, "higher_is_better": True, "dtype": "f32", "data": "synthetic",
        "config": {"workload": f"OLAT stack of {L} frames {cam.width}x{cam.height} (frame shape of configs[{args.config - 1}])",
                   "l2": "flushed between timed calls (256 MiB memset)"},
        "gpu_launches": args.steps,
        "roofline": {"kernel": "relight_vec_kernel", "bound": "hbm", "achieved": round(gbs, 1), "peak": peaks["hbm"],
                     "unit": "GB/s", "frac": round(gbs / peaks["hbm"], 4), "traffic": None,
                     "algorithmic_bytes": nbytes, "peak_source": peaks["source"]}}))


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
    R = binding.Renderer(scene, max_instances=int(MAX_INSTANCES_PER_GAUSSIAN * scene.n), device=local_rank)
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
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=5)
    ap.add_argument("--config", type=int, default=5, choices=[1, 2, 3, 4, 5, 6],
                    help="BASELINE.json configs[C-1]; default 5 = the largest single-GPU configuration")
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--relight", action="store_true", help="time sssgs_relight on an OLAT stack of the config's frame shape")
    ap.add_argument("--no-table", action="store_true", help="skip the per-config table (`configs`)")
    ap.add_argument("--canonical-lists", action="store_true",
                    help="render from the canonical tile lists instead of the tight ones (SSSGS_TIGHT_LISTS)")
    ap.add_argument("--bf16", action="store_true", help="MLP with bf16 layer inputs (SSSGS_COMPUTE_BF16) instead of fp16")
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
        run_reference(args, rank)
        return
    if args.bake:
        if rank == 0:
            run_bake(args, local_rank)
        return
    if args.relight:
        if rank == 0:
            run_relight(args, local_rank)
        return
    run_gpu(args, rank, world, local_rank)


if __name__ == "__main__":
    main()
