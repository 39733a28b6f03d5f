"""Writes oracle/workload_counters.json: the oracle's work counters of the first (view, light) frame of
every BASELINE config at full size.  They are the denominators of bench.py's roofline figures
("Counters come from the oracle and define the roofline denominators"):

  n_vis      Gaussians that survive projection / culling (step 3)
  instances  I = sum of tiles touched (canonical tile lists, step 4)
  p_eval     list entries a per-pixel walker visits, up to and including the entry it stops at (step 5)
  p_blend    blended (pixel, entry) pairs
  g_contrib  Gaussians blended at >= 1 pixel (the rows an MLP-skipping sweep must still evaluate)
  unstable_pixels  pixels with a decision inside the margin of a threshold (S7)
(The size of the minimal S5 list is not stored: oracle.tile_hits is brute force over every pixel of every listed
tile, which the full-size tests run on 256 sampled tiles per view instead.)

Calls only oracle/ and the seeded input generators; no value comes from the CUDA path.

    python oracle/make_workload_counters.py
"""
import json
import os
import sys
import time

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)

import oracle  # noqa: E402
from paper_2408_12282_b200 import scenes  # noqa: E402


def main():
    out = {}
    for cfg in (1, 2, 3, 4, 5):
        t0 = time.perf_counter()
        s = scenes.make_scene(cfg, views=1, lights=1)
        cam = s.cameras[0]
        proj = oracle.project(s, cam)
        keys, vals, ranges = oracle.build_lists(proj)
        ch = oracle.channels(s, proj, np.zeros((s.n, 4)))
        comp = oracle.composite(s, cam, proj, ch, vals, ranges)
        out[f"configs[{cfg - 1}]"] = dict(
            name=s.name, gaussians=int(s.n), width=int(cam.width), height=int(cam.height), view=0,
            n_vis=int(proj.visible.sum()), instances=int(len(keys)), p_eval=comp.p_eval, p_blend=comp.p_blend,
            g_contrib=int(comp.contrib.sum()), unstable_pixels=comp.n_unstable)
        print(cfg, out[f"configs[{cfg - 1}]"], f"{time.perf_counter() - t0:.1f} s", flush=True)
    with open(os.path.join(ROOT, "oracle", "workload_counters.json"), "w") as f:
        json.dump(out, f, indent=1)
        f.write("\n")


if __name__ == "__main__":
    main()
