"""Seeded synthetic scene generators (numpy only).

This module serves BOTH the CPU oracle tests and the CUDA path.  It holds none of
the method's arithmetic: it only draws inputs (Gaussians, MLP parameters, cameras,
lights) with the shapes and distributions of BASELINE.json's five configs, which
stand in for the paper's OLAT light-stage workloads (object
centric, inward facing cameras, point lights on a sphere, 800^2-class images).
The exact recipe is restated in DESIGN.md ("Input recipe").

Conventions (shared with include/sssgs.h):
  * scales / opacities are ACTIVATED (exp / sigmoid already applied),
  * rotations are unit quaternions (w, x, y, z),
  * camera: world->camera R (row-major) and t; camera looks down +z, x right, y down,
    pixel k is centred at integer coordinate k,
  * MLP parameters: packed float32, per layer W[out][in] row-major then b[out];
    order = trunk layers, SSS head (3 outputs), incident-head hidden layers,
    incident-head output (1).  Weights are rounded to bf16 once here so that both
    sides see identical weights (BASELINE.json cfg 4: "bf16 MLP weights").
"""
from __future__ import annotations

import dataclasses
import math
from typing import List, Optional

import numpy as np

ACT_RELU = 0
ACT_LEAKY_RELU = 1

Y00 = 0.2820948
Y1 = 0.4886025


def round_to_bf16(x: np.ndarray) -> np.ndarray:
    """Round float32 values to the nearest bf16 (ties to even); result kept as float32."""
    x = np.ascontiguousarray(x, dtype=np.float32)
    u = x.view(np.uint32).astype(np.uint64)
    lsb = (u >> 16) & 1
    u = (u + 0x7FFF + lsb) & 0xFFFF0000
    return u.astype(np.uint32).view(np.float32).reshape(x.shape)


@dataclasses.dataclass
class MlpSpec:
    in_dim: int
    trunk_width: List[int]
    inc_hidden_width: List[int]
    activation: int
    leaky_slope: float
    params: np.ndarray  # packed float32

    def layer_shapes(self):
        """[(out, in, kind)] in packing order; kind in trunk|sss|inc_hidden|inc_out."""
        shapes = []
        d = self.in_dim
        for w in self.trunk_width:
            shapes.append((w, d, "trunk"))
            d = w
        shapes.append((3, d, "sss"))
        di = d
        for w in self.inc_hidden_width:
            shapes.append((w, di, "inc_hidden"))
            di = w
        shapes.append((1, di, "inc_out"))
        return shapes

    def unpack(self):
        """-> list of (W[out,in], b[out], kind) views into params."""
        out = []
        off = 0
        for (o, i, kind) in self.layer_shapes():
            W = self.params[off:off + o * i].reshape(o, i)
            off += o * i
            b = self.params[off:off + o]
            off += o
            out.append((W, b, kind))
        assert off == self.params.size
        return out


@dataclasses.dataclass
class Camera:
    R: np.ndarray  # [3,3] float32 world->camera
    t: np.ndarray  # [3] float32
    fx: float
    fy: float
    cx: float
    cy: float
    tan_half_fovx: float
    tan_half_fovy: float
    width: int
    height: int
    znear: float
    bg: np.ndarray  # [3] float32
    position: np.ndarray  # [3] float32 world position (= -R^T t), for convenience


@dataclasses.dataclass
class Light:
    position: np.ndarray  # [3] float32
    intensity: np.ndarray  # [3] float32


@dataclasses.dataclass
class Scene:
    name: str
    n: int
    means: np.ndarray
    scales: np.ndarray
    rotations: np.ndarray
    opacities: np.ndarray
    normals: np.ndarray
    base_color: np.ndarray
    roughness: np.ndarray
    metallic: np.ndarray
    subsurface: np.ndarray
    vis_sh: np.ndarray
    vis_sh_degree: int
    feat: np.ndarray
    mlp: MlpSpec
    cameras: List[Camera]
    lights: List[List[Light]]  # lights[view] -> list of lights rendered for that view
    tile: int = 16


def look_at_camera(eye, width, height, fov_deg, fov_axis="y", target=(0.0, 0.0, 0.0),
                   up=(0.0, 0.0, 1.0), znear=0.2, bg=(0.0, 0.0, 0.0)) -> Camera:
    eye = np.asarray(eye, dtype=np.float64)
    f = np.asarray(target, dtype=np.float64) - eye
    f /= np.linalg.norm(f)
    r = np.cross(f, np.asarray(up, dtype=np.float64))
    r /= np.linalg.norm(r)
    d = np.cross(f, r)
    R = np.stack([r, d, f]).astype(np.float32)
    t = (-(R.astype(np.float64) @ eye)).astype(np.float32)
    half = math.tan(math.radians(fov_deg) / 2.0)
    extent = height if fov_axis == "y" else width
    fl = np.float32((extent / 2.0) / half)
    cam = Camera(R=R, t=t, fx=float(fl), fy=float(fl),
                 cx=float(np.float32((width - 1) / 2.0)), cy=float(np.float32((height - 1) / 2.0)),
                 tan_half_fovx=float(np.float32((width / 2.0) / fl)),
                 tan_half_fovy=float(np.float32((height / 2.0) / fl)),
                 width=int(width), height=int(height), znear=float(np.float32(znear)),
                 bg=np.asarray(bg, dtype=np.float32),
                 position=eye.astype(np.float32))
    return cam


def sph_dir(az_deg, el_deg):
    az, el = math.radians(az_deg), math.radians(el_deg)
    return np.array([math.cos(el) * math.cos(az), math.cos(el) * math.sin(az), math.sin(el)])


def fibonacci_sphere(n, radius):
    i = np.arange(n) + 0.5
    z = 1.0 - 2.0 * i / n
    phi = i * math.pi * (3.0 - math.sqrt(5.0))
    rr = np.sqrt(np.maximum(0.0, 1.0 - z * z))
    return radius * np.stack([rr * np.cos(phi), rr * np.sin(phi), z], axis=1)


def _unit_dirs(rng, n):
    v = rng.standard_normal((n, 3))
    v /= np.linalg.norm(v, axis=1, keepdims=True)
    return v


def _make_mlp(rng, in_dim, trunk, inc_hidden, activation, leaky_slope=0.01) -> MlpSpec:
    spec = MlpSpec(in_dim=in_dim, trunk_width=list(trunk), inc_hidden_width=list(inc_hidden),
                   activation=activation, leaky_slope=leaky_slope, params=np.zeros(0, np.float32))
    chunks = []
    for (o, i, _kind) in spec.layer_shapes():
        W = rng.standard_normal((o, i)) * math.sqrt(2.0 / i)  # He init
        b = rng.uniform(-0.1, 0.1, size=o)
        chunks.append(round_to_bf16(W.astype(np.float32)).ravel())
        chunks.append(b.astype(np.float32))
    spec.params = np.ascontiguousarray(np.concatenate(chunks), dtype=np.float32)
    return spec


def _attributes(rng, n, normals, log_scale, opacity_logit, feat_dim):
    ls = rng.normal(log_scale[0], log_scale[1], size=(n, 3))
    scales = np.exp(ls).astype(np.float32)
    q = rng.standard_normal((n, 4))
    q /= np.linalg.norm(q, axis=1, keepdims=True)
    q = q.astype(np.float32)
    q /= np.linalg.norm(q.astype(np.float64), axis=1, keepdims=True).astype(np.float32)
    ol = rng.normal(opacity_logit[0], opacity_logit[1], size=n)
    opac = (1.0 / (1.0 + np.exp(-ol))).astype(np.float32)
    base = rng.uniform(0.0, 1.0, size=(n, 3)).astype(np.float32)
    rough = rng.uniform(0.05, 1.0, size=n).astype(np.float32)
    metal = (rng.uniform(size=n) < 0.2).astype(np.float32)
    sss = rng.uniform(0.0, 1.0, size=n).astype(np.float32)
    nrm = normals / np.linalg.norm(normals, axis=1, keepdims=True)
    # degree-1 visibility SH: closed form 0.5 + 0.5 n.w (SURVEY 8(c) pins) + N(0,0.05)
    sh = np.empty((n, 4))
    sh[:, 0] = 0.5 / Y00
    sh[:, 1] = 0.5 * nrm[:, 1] / Y1  # Y_1,-1 ~ y
    sh[:, 2] = 0.5 * nrm[:, 2] / Y1  # Y_1,0  ~ z
    sh[:, 3] = 0.5 * nrm[:, 0] / Y1  # Y_1,1  ~ x
    sh += rng.normal(0.0, 0.05, size=(n, 4))
    feat = rng.standard_normal((n, feat_dim)).astype(np.float32)
    return dict(scales=scales, rotations=q, opacities=opac, base_color=base, roughness=rough,
                metallic=metal, subsurface=sss, normals=nrm.astype(np.float32),
                vis_sh=sh.astype(np.float32), feat=feat)


def _blob_points(rng, n):
    a = rng.uniform(0.02, 0.08, size=8)
    w = 1.5 * rng.standard_normal((8, 3))
    phi = rng.uniform(0.0, 2.0 * math.pi, size=8)
    d = _unit_dirs(rng, n)
    r = 1.0 + (a[None, :] * np.sin(2.0 * math.pi * (d @ w.T) + phi[None, :])).sum(axis=1)
    return d * r[:, None], d


CONFIGS = {
    1: dict(name="cfg1_tiny_sphere", n=2000, width=128, height=128, shape="sphere",
            log_scale=(-4.5, 0.5), opacity=(1.0, 1.5), feat=16, trunk=[64, 64], inc_hidden=[],
            act=ACT_RELU, views=1, lights=1),
    2: dict(name="cfg2_torus_100k", n=100_000, width=512, height=512, shape="torus",
            log_scale=(-4.5, 0.5), opacity=(1.0, 1.5), feat=16, trunk=[64, 64, 64], inc_hidden=[],
            act=ACT_RELU, views=1, lights=1),
    3: dict(name="cfg3_blob_300k_olat64", n=300_000, width=800, height=800, shape="blob",
            log_scale=(-4.5, 0.5), opacity=(1.0, 1.5), feat=16, trunk=[128, 128, 128],
            inc_hidden=[], act=ACT_RELU, views=1, lights=64),
    4: dict(name="cfg4_blob_1m_1080p", n=1_000_000, width=1920, height=1080, shape="blob",
            log_scale=(-5.5, 0.6), opacity=(1.0, 1.5), feat=16, trunk=[128, 128, 128],
            inc_hidden=[], act=ACT_RELU, views=8, lights=1),
    5: dict(name="cfg5_blob_3m_16x16", n=3_000_000, width=1024, height=1024, shape="blob",
            log_scale=(-4.8, 0.7), opacity=(2.0, 1.0), feat=32, trunk=[128, 128, 128, 128],
            inc_hidden=[], act=ACT_RELU, views=16, lights=16),
    # parity-only "paper-arch": 40 -> [64,32,32], incident head 32 -> 32 -> 1,
    # SSS head 32 -> 3, Leaky-ReLU; no extra feature (F = 0).
    6: dict(name="cfg6_paper_arch", n=20_000, width=256, height=256, shape="sphere",
            log_scale=(-4.0, 0.5), opacity=(1.0, 1.5), feat=0, trunk=[64, 32, 32], inc_hidden=[32],
            act=ACT_LEAKY_RELU, views=1, lights=2),
}


def make_scene(cfg: int, n: Optional[int] = None, width: Optional[int] = None,
               height: Optional[int] = None, views: Optional[int] = None,
               lights: Optional[int] = None, seed: Optional[int] = None) -> Scene:
    """Build config `cfg` (1..6).  Overrides shrink a config for parity tests; the
    distributions are unchanged.  seed defaults to the config index."""
    c = dict(CONFIGS[cfg])
    n = int(n if n is not None else c["n"])
    W = int(width if width is not None else c["width"])
    H = int(height if height is not None else c["height"])
    nv = int(views if views is not None else c["views"])
    nl = int(lights if lights is not None else c["lights"])
    rng = np.random.default_rng(cfg if seed is None else seed)

    if c["shape"] == "sphere":
        d = _unit_dirs(rng, n)
        means = d + rng.normal(0.0, 0.02, size=(n, 3))
        normals = d
    elif c["shape"] == "torus":
        u = rng.uniform(0.0, 2.0 * math.pi, size=n)
        v = rng.uniform(0.0, 2.0 * math.pi, size=n)
        R0, r0 = 1.0, 0.35
        means = np.stack([(R0 + r0 * np.cos(v)) * np.cos(u), (R0 + r0 * np.cos(v)) * np.sin(u),
                          r0 * np.sin(v)], axis=1) + rng.normal(0.0, 0.01, size=(n, 3))
        normals = np.stack([np.cos(v) * np.cos(u), np.cos(v) * np.sin(u), np.sin(v)], axis=1)
    else:
        means, normals = _blob_points(rng, n)
    attrs = _attributes(rng, n, normals, c["log_scale"], c["opacity"], c["feat"])
    mlp = _make_mlp(rng, 40 + c["feat"], c["trunk"], c["inc_hidden"], c["act"])

    cams, lights_per_view = [], []
    if cfg in (1, 2, 3, 6):
        for k in range(nv):
            cams.append(look_at_camera(4.0 * sph_dir(30.0 + 45.0 * k, 20.0), W, H, 40.0))
        if cfg == 3:
            lp = fibonacci_sphere(max(nl, 1), 3.0)[:nl]
        else:
            lp = np.stack([3.0 * sph_dir(75.0 + 50.0 * j, 40.0) for j in range(nl)]) if nl else np.zeros((0, 3))
        for k in range(nv):
            lights_per_view.append([Light(p.astype(np.float32), np.ones(3, np.float32)) for p in lp])
    elif cfg == 4:
        for k in range(nv):
            az = 45.0 * k
            cams.append(look_at_camera(4.0 * sph_dir(az, 20.0), W, H, 40.0, fov_axis="y"))
            lights_per_view.append([
                Light((3.0 * sph_dir(az + 45.0 + 30.0 * j, 40.0)).astype(np.float32),
                      np.ones(3, np.float32)) for j in range(nl)])
    else:  # cfg 5: azimuth orbit x 4x4 azimuth-elevation light grid, upper hemisphere
        grid = []
        for j in range(4):
            for i in range(4):
                grid.append(3.0 * sph_dir(90.0 * (i + 0.5), 22.5 * (j + 0.5)))
        grid = grid[:nl] if nl <= 16 else grid
        for k in range(nv):
            cams.append(look_at_camera(4.0 * sph_dir(360.0 / max(nv, 1) * k, 20.0), W, H, 40.0))
            lights_per_view.append([Light(p.astype(np.float32), np.ones(3, np.float32)) for p in grid])

    return Scene(name=c["name"], n=n, means=means.astype(np.float32), mlp=mlp, cameras=cams,
                 lights=lights_per_view, vis_sh_degree=1, **attrs)


def subset(scene: Scene, idx) -> Scene:
    """Scene restricted / permuted to Gaussian indices `idx` (for permutation tests)."""
    idx = np.asarray(idx)
    kw = {}
    for f in ("means", "scales", "rotations", "opacities", "normals", "base_color", "roughness",
              "metallic", "subsurface", "vis_sh", "feat"):
        kw[f] = np.ascontiguousarray(getattr(scene, f)[idx])
    return dataclasses.replace(scene, n=len(idx), **kw)
