"""Writes oracle/workload_counters.json: the oracle's work counters of the first (view, light) frame of
every BASELINE config at full size.  They are the denominators of bench.py's roofline figures
("Counters come from the oracle and define the roofline denominators"):

  n_vis      Gaussians that survive projection / culling (step 3)
  instances  I = sum of tiles touched (canonical tile lists, step 4)
  p_eval     list entries a per-pixel walker visits, up to and including the entry it stops at (step 5)
  p_blend    blended (pixel, entry) pairs
  g_contrib  Gaussians blended at >= 1 pixel (the rows an MLP-skipping sweep must still evaluate)
  unstable_pixels  pixels with a decision inside the margin of a threshold (S7)
  instances_min, p_eval_min   the same two counters on the MINIMAL tile list of reading S5 (oracle.tile_hits, brute
             force over every pixel of every listed tile: a pair is kept iff the Gaussian reaches alpha >= 1/255 at
             some pixel of the tile).  Every valid tight list (SSSGS_TIGHT_LISTS) lies between the minimal and the
             canonical one, so these are the lower bounds of the work a tight-list render evaluates; p_blend and
             g_contrib are the same on all three lists (asserted here).

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
        hit = oracle.tile_hits(s, cam, proj, vals, ranges)
        tile_of = (keys >> np.uint64(32)).astype(np.int64)
        kept = np.bincount(tile_of[hit], minlength=len(ranges))
        ends = np.cumsum(kept)
        ranges_min = np.stack([ends - kept, ends], axis=1).astype(np.uint32)
        comp_min = oracle.composite(s, cam, proj, ch, vals[hit], ranges_min)
        assert comp_min.p_blend == comp.p_blend and int(comp_min.contrib.sum()) == int(comp.contrib.sum())
        assert np.array_equal(comp_min.gbuf, comp.gbuf)     # dropped pairs blend nowhere: same frame, bit for bit
        out[f"configs[{cfg - 1}]"] = dict(
            name=s.name, gaussians=int(s.n), width=int(cam.width), height=int(cam.height), view=0,
            n_vis=int(proj.visible.sum()), instances=int(len(keys)), p_eval=comp.p_eval, p_blend=comp.p_blend,
            g_contrib=int(comp.contrib.sum()), unstable_pixels=comp.n_unstable,
            instances_min=int(hit.sum()), p_eval_min=comp_min.p_eval)
        print(cfg, out[f"configs[{cfg - 1}]"], f"{time.perf_counter() - t0:.1f} s", flush=True)
    with open(os.path.join(ROOT, "oracle", "workload_counters.json"), "w") as f:
        json.dump(out, f, indent=1)
        f.write("\n")


if __name__ == "__main__":
    main()
