"""Writes tests/golden/tiny_scene_expected.json: expected values of a small seeded scene,
computed by the CPU oracle ONLY (never by the CUDA path).

    python tests/golden/make_golden.py

The paper prints no worked numeric example of the render path (no per-pixel values,
no intermediate tensors), so there is no paper fixture to store; this file pins the oracle to its
own committed output instead, so that an accidental change of the oracle's arithmetic is noticed
(tests/test_golden.py), and gives the CUDA path a stored target that does not come from itself.
The inputs are regenerated from the seed by paper_2408_12282_b200.scenes (input generator only).
"""
import json
import os
import sys

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
sys.path.insert(0, ROOT)

import oracle  # noqa: E402
from paper_2408_12282_b200 import scenes  # noqa: E402

SCENE = dict(cfg=1, n=600, width=48, height=40)
PIXELS = [(20, 24), (13, 30), (27, 17), (5, 5), (33, 41), (20, 8)]  # (row, col)


def compute():
    scene = scenes.make_scene(SCENE["cfg"], n=SCENE["n"], width=SCENE["width"], height=SCENE["height"])
    r = oracle.render_frame(scene, mlp_mode=2)  # fp16-emulating MLP: what the tensor-core path computes by default
    out = {
        "scene": SCENE,
        "n_vis": r.n_vis,
        "n_instances": r.n_instances,
        "keys_head": [int(k) for k in r.keys[:8]],
        "vals_head": [int(v) for v in r.vals[:8]],
        "ranges_sum": int(r.ranges.astype(np.int64).sum()),
        "p_eval": r.comp.p_eval,
        "p_blend": r.comp.p_blend,
        "pixels": [
            {"row": y, "col": x, "unstable": bool(r.comp.unstable[y, x]),
             "gbuffer": [float(v) for v in r.gbuf[y, x]], "rgb": [float(v) for v in r.rgb[y, x]]}
            for (y, x) in PIXELS],
        "mlp_out_head": [[float(v) for v in row] for row in r.mlp_out[:4]],
    }
    return out


if __name__ == "__main__":
    path = os.path.join(os.path.dirname(os.path.abspath(__file__)), "tiny_scene_expected.json")
    with open(path, "w") as f:
        json.dump(compute(), f, indent=1)
    print("wrote", path)
