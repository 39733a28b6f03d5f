"""Test helpers: hand-built scenes (inputs only; no method arithmetic)."""
import dataclasses

import numpy as np

from paper_2408_12282_b200 import scenes


def custom_scene(means, scales, rotations=None, opacities=None, normals=None, base_color=None,
                 roughness=None, metallic=None, subsurface=None, width=64, height=64,
                 eye=(0.0, -4.0, 0.0), fov=40.0, lights=((0.0, -3.0, 1.0),), feat_dim=0,
                 trunk=(16,), inc_hidden=(), act=scenes.ACT_RELU, seed=0, bg=(0.0, 0.0, 0.0)):
    rng = np.random.default_rng(seed)
    means = np.asarray(means, np.float32).reshape(-1, 3)
    n = means.shape[0]

    def arr(v, shape, default):
        if v is None:
            v = default
        return np.ascontiguousarray(np.broadcast_to(np.asarray(v, np.float32), shape)).copy()

    scales = arr(scales, (n, 3), 0.05)
    rotations = arr(rotations, (n, 4), (1.0, 0.0, 0.0, 0.0))
    opacities = arr(opacities, (n,), 0.5)
    normals = arr(normals, (n, 3), (0.0, -1.0, 0.0))
    base_color = arr(base_color, (n, 3), 0.5)
    roughness = arr(roughness, (n,), 0.5)
    metallic = arr(metallic, (n,), 0.0)
    subsurface = arr(subsurface, (n,), 0.5)
    vis = np.zeros((n, 4), np.float32)
    vis[:, 0] = 0.5 / scenes.Y00
    vis[:, 1] = 0.5 * normals[:, 1] / scenes.Y1
    vis[:, 2] = 0.5 * normals[:, 2] / scenes.Y1
    vis[:, 3] = 0.5 * normals[:, 0] / scenes.Y1
    feat = rng.standard_normal((n, feat_dim)).astype(np.float32)
    mlp = scenes._make_mlp(rng, 40 + feat_dim, list(trunk), list(inc_hidden), act)
    cam = scenes.look_at_camera(eye, width, height, fov, bg=bg)
    lts = [scenes.Light(np.asarray(p, np.float32), np.ones(3, np.float32)) for p in lights]
    return scenes.Scene(name="custom", n=n, means=means, scales=scales, rotations=rotations,
                        opacities=opacities, normals=normals, base_color=base_color,
                        roughness=roughness, metallic=metallic, subsurface=subsurface, vis_sh=vis,
                        vis_sh_degree=1, feat=feat, mlp=mlp, cameras=[cam], lights=[lts])


def with_mlp_params(scene, params):
    mlp = dataclasses.replace(scene.mlp, params=np.ascontiguousarray(params, np.float32))
    return dataclasses.replace(scene, mlp=mlp)
