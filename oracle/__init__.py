"""CPU oracle of the SSS-GS forward relighting render path -- TEST INFRASTRUCTURE ONLY.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs
may import this package.  It shares no code with the CUDA path and never imports it.
The arithmetic lives in sssgs_oracle.cpp (plain C++, cited against PAPER.md); this file
only builds it (g++) and marshals numpy arrays.  Scene objects are duck-typed
(attributes as produced by paper_2408_12282_b200.scenes), nothing is imported from there.
"""
from __future__ import annotations

import ctypes
import os
import subprocess
from types import SimpleNamespace

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "sssgs_oracle.cpp")
_LIB = os.path.join(_HERE, "liboracle.so")
_lib = None

GBUF_CH = 16
CXXFLAGS = ["-O2", "-std=c++17", "-ffp-contract=off", "-mfma", "-fopenmp", "-shared", "-fPIC"]


def build(force: bool = False) -> str:
    """Compile liboracle.so if missing or older than its source."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        subprocess.check_call(["g++", *CXXFLAGS, "-o", _LIB, _SRC])
    return _LIB


class OrcCamera(ctypes.Structure):
    _fields_ = [("R", ctypes.c_float * 9), ("t", ctypes.c_float * 3),
                ("fx", ctypes.c_float), ("fy", ctypes.c_float), ("cx", ctypes.c_float),
                ("cy", ctypes.c_float), ("tan_half_fovx", ctypes.c_float),
                ("tan_half_fovy", ctypes.c_float), ("width", ctypes.c_int),
                ("height", ctypes.c_int), ("znear", ctypes.c_float), ("bg", ctypes.c_float * 3)]


def _cam(cam) -> OrcCamera:
    c = OrcCamera()
    c.R[:] = [float(v) for v in np.asarray(cam.R, np.float32).ravel()]
    c.t[:] = [float(v) for v in np.asarray(cam.t, np.float32).ravel()]
    c.fx, c.fy, c.cx, c.cy = cam.fx, cam.fy, cam.cx, cam.cy
    c.tan_half_fovx, c.tan_half_fovy = cam.tan_half_fovx, cam.tan_half_fovy
    c.width, c.height, c.znear = int(cam.width), int(cam.height), cam.znear
    c.bg[:] = [float(v) for v in np.asarray(cam.bg, np.float32).ravel()]
    return c


def lib():
    global _lib
    if _lib is None:
        build()
        _lib = ctypes.CDLL(_LIB)
        _lib.orc_build_lists.restype = ctypes.c_int64
        _lib.orc_num_threads.restype = ctypes.c_int
    return _lib


def num_threads() -> int:
    return int(lib().orc_num_threads())


def _p(a):
    return a.ctypes.data_as(ctypes.c_void_p) if a is not None else None


def _f32(a):
    return np.ascontiguousarray(a, dtype=np.float32)


def mlp_inputs(scene, cam, light_pos) -> np.ndarray:
    """Step 1: [n, 40+F] float64."""
    n = int(scene.n)
    F = int(scene.feat.shape[1]) if scene.feat is not None and scene.feat.ndim == 2 else 0
    x = np.empty((n, 40 + F), np.float64)
    feat = _f32(scene.feat) if F else np.zeros((1,), np.float32)
    lp = _f32(light_pos)
    c = _cam(cam)
    lib().orc_mlp_inputs(ctypes.c_int64(n), _p(_f32(scene.means)), _p(_f32(scene.normals)),
                         _p(_f32(scene.rotations)), _p(_f32(scene.scales)), _p(_f32(scene.vis_sh)),
                         ctypes.c_int(scene.vis_sh_degree), _p(feat), ctypes.c_int(F),
                         ctypes.byref(c), _p(lp), _p(x))
    return x


def round_bf16(x) -> np.ndarray:
    """The oracle's bf16 rounding (float64 in, float64 out), for the pins."""
    x = np.ascontiguousarray(x, np.float64)
    out = np.empty_like(x)
    lib().orc_round_bf16(ctypes.c_int64(x.size), _p(x), _p(out))
    return out


def round_fp16(x) -> np.ndarray:
    """The oracle's binary16 rounding (float64 in, float64 out), for the pins."""
    x = np.ascontiguousarray(x, np.float64)
    out = np.empty_like(x)
    lib().orc_round_fp16(ctypes.c_int64(x.size), _p(x), _p(out))
    return out


def mlp_forward(x, mlp, mode: int = 0) -> np.ndarray:
    """Step 2: x [n, in_dim] float64 -> [n, 4] float64.
    mode 0 = double reference, 1 = bf16-emulating, 2 = fp16-emulating."""
    x = np.ascontiguousarray(x, np.float64)
    n = x.shape[0]
    assert x.shape[1] == mlp.in_dim
    out = np.empty((n, 4), np.float64)
    tw = np.asarray(mlp.trunk_width, np.int32)
    iw = np.asarray(list(mlp.inc_hidden_width) + [0], np.int32)
    params = _f32(mlp.params)
    lib().orc_mlp_forward(ctypes.c_int64(n), _p(x), ctypes.c_int(mlp.in_dim),
                          ctypes.c_int(len(mlp.trunk_width)), _p(tw),
                          ctypes.c_int(len(mlp.inc_hidden_width)), _p(iw),
                          ctypes.c_int(mlp.activation), ctypes.c_double(mlp.leaky_slope),
                          _p(params), ctypes.c_int(mode), _p(out))
    return out


def project(scene, cam, tile=16):
    """Step 3 (Eq. 2), canonical fp32."""
    n = int(scene.n)
    o = SimpleNamespace(
        visible=np.zeros(n, np.int32), pix=np.zeros((n, 2), np.float32),
        depth=np.zeros(n, np.float32), conic=np.zeros((n, 3), np.float32),
        radius=np.zeros(n, np.float32), rect=np.zeros((n, 4), np.int32),
        touched=np.zeros(n, np.int32))
    c = _cam(cam)
    lib().orc_project(ctypes.c_int64(n), _p(_f32(scene.means)), _p(_f32(scene.scales)),
                      _p(_f32(scene.rotations)), ctypes.byref(c), ctypes.c_int(tile),
                      ctypes.c_int(tile), _p(o.visible), _p(o.pix), _p(o.depth), _p(o.conic),
                      _p(o.radius), _p(o.rect), _p(o.touched))
    o.tiles_x = (cam.width + tile - 1) // tile
    o.tiles_y = (cam.height + tile - 1) // tile
    return o


def project_f64(scene, cam):
    n = int(scene.n)
    cov = np.zeros((n, 3), np.float64)
    pix = np.zeros((n, 2), np.float64)
    depth = np.zeros(n, np.float64)
    c = _cam(cam)
    lib().orc_project_f64(ctypes.c_int64(n), _p(_f32(scene.means)), _p(_f32(scene.scales)),
                          _p(_f32(scene.rotations)), ctypes.byref(c), _p(cov), _p(pix), _p(depth))
    return cov, pix, depth


def build_lists(proj):
    """Step 4: (keys u64 [I], vals u32 [I], ranges u32 [tiles, 2])."""
    n = proj.touched.shape[0]
    args = (ctypes.c_int64(n), _p(proj.rect), _p(proj.depth), _p(proj.touched),
            ctypes.c_int(proj.tiles_x), ctypes.c_int(proj.tiles_y))
    total = int(lib().orc_build_lists(*args, None, None, None))
    keys = np.zeros(max(total, 1), np.uint64)
    vals = np.zeros(max(total, 1), np.uint32)
    ranges = np.zeros((proj.tiles_x * proj.tiles_y, 2), np.uint32)
    lib().orc_build_lists(*args, _p(keys), _p(vals), _p(ranges))
    return keys[:total], vals[:total], ranges


def channels(scene, proj, mlp_out) -> np.ndarray:
    """Per-Gaussian channel values [n, 14] in G-buffer order (channels 0..13)."""
    n = int(scene.n)
    ch = np.zeros((n, 14), np.float64)
    ch[:, 0] = proj.depth
    ch[:, 1:4] = scene.normals
    ch[:, 4:7] = scene.base_color
    ch[:, 7] = scene.roughness
    ch[:, 8] = scene.metallic
    ch[:, 9] = scene.subsurface
    ch[:, 10:14] = mlp_out
    return ch


def composite(scene, cam, proj, ch, order, ranges, tile=16):
    """Step 5 (tiled: ranges given) or step 7 (brute force: ranges None); Eq. 3 L68-72."""
    W, H = int(cam.width), int(cam.height)
    gbuf = np.zeros((H, W, GBUF_CH), np.float64)
    unstable = np.zeros((H, W), np.uint8)
    counters = np.zeros(8, np.int64)
    contrib = np.zeros(max(int(scene.n), 1), np.uint8)
    order = np.ascontiguousarray(order, np.uint32)
    rg = np.ascontiguousarray(ranges, np.uint32) if ranges is not None else None
    lib().orc_composite(ctypes.c_int(W), ctypes.c_int(H), ctypes.c_int(tile), ctypes.c_int(tile),
                        _p(proj.pix), _p(proj.conic), _p(_f32(scene.opacities)),
                        _p(np.ascontiguousarray(ch, np.float64)), _p(order),
                        ctypes.c_int64(order.shape[0]), _p(rg), _p(gbuf), _p(unstable),
                        _p(counters), _p(contrib))
    # unstable: True where a skip / stop decision sits within fp32 rounding of its threshold (S7); flags: which
    # rule (bit 0 power ~ 0, bit 1 alpha ~ 1/255, bit 2 T' ~ 1e-4), bits 4-7 = flagged alpha decisions at the pixel
    return SimpleNamespace(gbuf=gbuf, unstable=unstable != 0, flags=unstable, p_eval=int(counters[0]),
                           p_blend=int(counters[1]), n_unstable=int(counters[2]),
                           n_rule_power=int(counters[3]), n_rule_alpha=int(counters[4]), n_rule_T=int(counters[5]),
                           contrib=contrib[:int(scene.n)].astype(bool))


def tile_hits(scene, cam, proj, vals, ranges, tile=16) -> np.ndarray:
    """S5: for every entry of the canonical sorted list, True iff its Gaussian reaches alpha >= 1/255 at some
    pixel of the entry's tile -- the pairs every valid tight tile list must keep."""
    hit = np.zeros(max(len(vals), 1), np.uint8)
    lib().orc_tile_hits(ctypes.c_int(int(cam.width)), ctypes.c_int(int(cam.height)), ctypes.c_int(tile),
                        ctypes.c_int(tile), _p(proj.pix), _p(proj.conic), _p(_f32(scene.opacities)),
                        _p(np.ascontiguousarray(vals, np.uint32)), _p(np.ascontiguousarray(ranges, np.uint32)),
                        ctypes.c_int(proj.tiles_x), ctypes.c_int(proj.tiles_y), _p(hit))
    return hit[:len(vals)].astype(bool)


def brute_order(proj) -> np.ndarray:
    """All visible Gaussians sorted by (depth bits, index) -- the order of step 7."""
    vis = np.nonzero(proj.visible)[0]
    bits = proj.depth.view(np.uint32)[vis].astype(np.uint64)
    key = (bits << np.uint64(32)) | vis.astype(np.uint64)
    return vis[np.argsort(key, kind="stable")].astype(np.uint32)


def shade(cam, light, gbuf, f32: bool = False):
    """Step 6 (Eq. 4, Eq. 7).  Returns (rgb, aov_diffuse, aov_specular)."""
    H, W = gbuf.shape[:2]
    dt = np.float32 if f32 else np.float64
    rgb = np.zeros((H, W, 3), dt)
    ad = np.zeros((H, W, 3), dt)
    as_ = np.zeros((H, W, 3), dt)
    fn = lib().orc_shade_f32 if f32 else lib().orc_shade
    c = _cam(cam)
    fn(ctypes.c_int(W), ctypes.c_int(H), ctypes.byref(c), _p(_f32(light.position)),
       _p(_f32(light.intensity)), _p(np.ascontiguousarray(gbuf, np.float64)), _p(rgb), _p(ad), _p(as_))
    return rgb, ad, as_


def render_frame(scene, view: int = 0, light: int = 0, mlp_mode: int = 0, mlp_out=None, tile=16,
                 geometry=None):
    """Whole path for one (view, light) frame; returns every intermediate.
    `geometry` = a previous result for the same view (re-uses projection and lists)."""
    cam = scene.cameras[view]
    lt = scene.lights[view][light]
    r = SimpleNamespace()
    if geometry is None:
        r.proj = project(scene, cam, tile)
        r.keys, r.vals, r.ranges = build_lists(r.proj)
    else:
        r.proj, r.keys, r.vals, r.ranges = geometry.proj, geometry.keys, geometry.vals, geometry.ranges
    if mlp_out is None:
        r.x = mlp_inputs(scene, cam, lt.position)
        mlp_out = mlp_forward(r.x, scene.mlp, mlp_mode)
    r.mlp_out = np.asarray(mlp_out, np.float64)
    r.ch = channels(scene, r.proj, r.mlp_out)
    r.comp = composite(scene, cam, r.proj, r.ch, r.vals, r.ranges, tile)
    r.gbuf = r.comp.gbuf
    r.rgb, r.aov_diffuse, r.aov_specular = shade(cam, lt, r.gbuf)
    r.n_vis = int(r.proj.visible.sum())
    r.n_instances = int(r.keys.shape[0])
    return r


# -------------------------------------------------------------------------------------------------
# "w/o deferred" variant (Tab. 2 "w/o deferred", Fig. 5; L114 explains what the
# deferred pipeline replaces): Eq. 7 is evaluated per Gaussian and the resulting RGB is splatted.
# Written out in numpy, float64, independently of the C++ pixel shader (which pins it, see
# tests/test_oracle_forward.py).
# -------------------------------------------------------------------------------------------------
def shade_gaussians(scene, cam, light, mlp_out) -> np.ndarray:
    """c_i = intensity * L_out,i with Eq. 7 (L104-106) at the Gaussian's centre mu_i:
        L_out = sss L_SSS + (1 - sss)(f_spec + f_diff) L_in (n . w_in),
    w_in / w_out towards the light / the camera from mu_i, n and the material of the Gaussian itself,
    BRDF of Eq. 4 (L76-80) with the readings S8 (Cook-Torrance with the 4, GGX D with alpha_r = r^2
    floored at 1e-3, Schlick F, Smith-Schlick visibility, k = alpha_r / 2) and the guards of the
    pixel shader (|n| < 1e-8 -> SSS term only; |l + v| < 1e-8 -> h = n; n.v floored at 1e-4).
    mlp_out: [n, 4] (L_SSS rgb, L_in).  Returns [n, 3] float64."""
    f8 = np.float64
    mu = np.asarray(scene.means, f8)
    nrm = np.asarray(scene.normals, f8)
    b = np.asarray(scene.base_color, f8)
    r = np.asarray(scene.roughness, f8)
    m = np.asarray(scene.metallic, f8)
    sss = np.asarray(scene.subsurface, f8)
    mo = np.asarray(mlp_out, f8)
    R = np.asarray(cam.R, f8).reshape(3, 3)
    t = np.asarray(cam.t, f8)
    p_cam = -R.T @ t
    l = np.asarray(light.position, f8)[None, :] - mu
    v = p_cam[None, :] - mu
    l /= np.linalg.norm(l, axis=1, keepdims=True)
    v /= np.linalg.norm(v, axis=1, keepdims=True)
    nn = np.linalg.norm(nrm, axis=1)
    ok = nn >= 1e-8
    n = nrm / np.where(ok, nn, 1.0)[:, None]
    h = l + v
    hl = np.linalg.norm(h, axis=1)
    h = np.where((hl >= 1e-8)[:, None], h / np.where(hl >= 1e-8, hl, 1.0)[:, None], n)
    dot = lambda a, c: np.sum(a * c, axis=1)  # noqa: E731
    nl = np.maximum(0.0, dot(n, l))
    nv = np.maximum(1e-4, dot(n, v))
    nh = np.clip(dot(n, h), 0.0, 1.0)
    vh = np.clip(dot(v, h), 0.0, 1.0)
    ar = np.maximum(1e-3, r * r)
    a2 = ar * ar
    s2 = np.sum(np.cross(n, h) ** 2, axis=1)              # 1 - nh^2 without cancellation (S9)
    D = a2 / (np.pi * np.maximum(1e-12, a2 * nh * nh + s2) ** 2)  # floor: n = -h exactly (see shade_impl)
    k = 0.5 * ar
    V = 1.0 / (4.0 * (nl * (1.0 - k) + k) * (nv * (1.0 - k) + k))
    F0 = 0.04 * (1.0 - m)[:, None] + b * m[:, None]
    F = F0 + (1.0 - F0) * ((1.0 - vh) ** 5)[:, None]
    f_spec = (D * V)[:, None] * F
    f_diff = (1.0 - m)[:, None] * b / np.pi
    brdf = (f_spec + f_diff) * (mo[:, 3] * nl)[:, None]
    brdf = np.where(ok[:, None], brdf, 0.0)
    lout = sss[:, None] * mo[:, :3] + (1.0 - sss)[:, None] * brdf
    return np.asarray(light.intensity, f8)[None, :] * lout


def forward_frame(scene, view: int = 0, light: int = 0, mlp_mode: int = 0, mlp_out=None, geometry=None):
    """Whole "w/o deferred" path for one (view, light): C = sum_i T_i alpha_i c_i + (1 - A) bg (Eq. 3)
    with c_i from shade_gaussians.  The compositor is the one of the deferred path (the per-Gaussian
    colour rides in channels 10-12)."""
    cam = scene.cameras[view]
    lt = scene.lights[view][light]
    r = SimpleNamespace()
    if geometry is None:
        r.proj = project(scene, cam)
        r.keys, r.vals, r.ranges = build_lists(r.proj)
    else:
        r.proj, r.keys, r.vals, r.ranges = geometry.proj, geometry.keys, geometry.vals, geometry.ranges
    if mlp_out is None:
        mlp_out = mlp_forward(mlp_inputs(scene, cam, lt.position), scene.mlp, mlp_mode)
    r.mlp_out = np.asarray(mlp_out, np.float64)
    r.colors = shade_gaussians(scene, cam, lt, r.mlp_out)
    ch = np.zeros((int(scene.n), 14), np.float64)
    ch[:, 10:13] = r.colors
    r.comp = composite(scene, cam, r.proj, ch, r.vals, r.ranges)
    A = r.comp.gbuf[..., 14:15]
    r.rgb = r.comp.gbuf[..., 10:13] + (1.0 - A) * np.asarray(cam.bg, np.float64)
    return r


def bake_visibility(scene, dirs, weights, t_min: float, sh_degree: int = 1, rows=None, positions: bool = False):
    """Ray-traced visibility of every Gaussian towards K directions and its SH projection
    (reading in DESIGN.md section 7d).  Returns (sh [n,(deg+1)^2] float64,
    vis [n,K] float64, unstable [n,K] int32 = number of threshold decisions a float evaluation may flip).
    rows: optional indices of the Gaussians whose rays are traced (outputs then have len(rows) rows).
    positions: `dirs` are points (light positions); rays end there."""
    n = int(scene.n)
    dirs = _f32(dirs).reshape(-1, 3)
    weights = _f32(weights).reshape(-1)
    K = dirs.shape[0]
    assert weights.shape[0] == K and sh_degree in (0, 1)
    nc = (sh_degree + 1) ** 2
    rows_arr = None if rows is None else np.ascontiguousarray(rows, np.int64)
    m = n if rows_arr is None else len(rows_arr)
    sh = np.zeros((m, nc), np.float64)
    vis = np.zeros((m, K), np.float64)
    unstable = np.zeros((m, K), np.int32)
    means, scales, rot, opac = _f32(scene.means), _f32(scene.scales), _f32(scene.rotations), _f32(scene.opacities)
    lib().orc_bake_visibility(ctypes.c_int64(n), _p(means), _p(scales), _p(rot), _p(opac), ctypes.c_int(K),
                              _p(dirs), _p(weights), ctypes.c_float(t_min), ctypes.c_int(sh_degree),
                              ctypes.c_int(1 if positions else 0), ctypes.c_int64(m), _p(rows_arr), _p(sh), _p(vis), _p(unstable))
    return sh, vis, unstable


def relight(frames, weights) -> np.ndarray:
    """Relighting from a precomputed reflectance field ("To speed up generation we can precompute a
    reflectance field assuming white light.  We compute the relit view as the sum over the reflectance field scaled by
    the environment illumination."):  out[p, c] = sum_l weights[l, c] * frames[l, p, c].
    frames [L, H, W, 3]: the OLAT renders of one view under white unit-intensity point lights (on the black background
    of a light stage; with another background every frame carries its (1 - A) bg term and the sum carries it L times
    scaled -- the definition does not remove it); weights [L, 3]: RGB radiance of the environment towards light l.
    Float64, lights added in order.  Pins: tests/test_oracle_forward.py (one-hot weights, brute force, equality with
    shading under coloured lights -- Eq. 7 is linear in the light's intensity, S16)."""
    frames = np.asarray(frames, np.float64)
    weights = np.asarray(weights, np.float64)
    assert frames.ndim == 4 and frames.shape[3] == 3 and weights.shape == (frames.shape[0], 3)
    out = np.zeros(frames.shape[1:], np.float64)
    for l in range(frames.shape[0]):
        out += frames[l] * weights[l][None, None, :]
    return out
