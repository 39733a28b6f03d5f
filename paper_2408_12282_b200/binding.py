"""Thin ctypes binding of libsssgs (include/sssgs.h): argument marshalling only.

Every step of the render path runs in the CUDA kernels behind the C ABI.  The functions
keep the ABI's names (`sssgs_create`, `sssgs_render`, `sssgs_render_host`, `sssgs_destroy`);
`Renderer` is a convenience wrapper that allocates device memory through torch (plumbing) and
hands raw pointers + the current CUDA stream to `sssgs_render`.

Loading fails loudly if libsssgs.so is missing: there is no CPU fallback.
"""
from __future__ import annotations

import ctypes
import os
from typing import Optional, Sequence

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libsssgs.so")

SSSGS_TILE = 16
SSSGS_GBUF_CHANNELS = 16
SSSGS_NCOUNTERS = 8
SSSGS_MAX_TRUNK = 8
SSSGS_MAX_INC_HIDDEN = 2
SSSGS_LIGHTS_PER_CAMERA = 1
SSSGS_SUM_LIGHTS = 2
SSSGS_FORWARD_SHADING = 4
SSSGS_TIGHT_LISTS = 8
SSSGS_BACKWARD_FP32 = 16
SSSGS_F32, SSSGS_BF16 = 0, 1
SSSGS_COMPUTE_FP16, SSSGS_COMPUTE_BF16 = 0, 1
(SSSGS_OK, SSSGS_EINVAL, SSSGS_ECAPACITY, SSSGS_ECUDA, SSSGS_EARCH, SSSGS_EOVERFLOW) = (0, -1, -2, -3, -4, -5)
CNT_NVIS, CNT_INSTANCES, CNT_OVERFLOW, CNT_SORT_ERROR, CNT_MLP_ROWS = 0, 1, 2, 3, 4

EXPORTS = ["sssgs_workspace_bytes", "sssgs_create", "sssgs_destroy", "sssgs_render",
           "sssgs_render_host", "sssgs_last_launch_count", "sssgs_last_error",
           "sssgs_profile_enable", "sssgs_profile_read", "sssgs_bake_visibility", "sssgs_render_backward",
           "sssgs_mlp_eval_static", "sssgs_relight"]
SSSGS_STATIC_SCRATCH_BYTES = 192 * 1024
SSSGS_STATIC_MAX_LIGHTS = 8
STAGES = ["pack", "project", "depth_sort", "emit", "tile_sort", "ranges", "mlp", "raster", "prepass"]

_f = ctypes.c_float
_vp = ctypes.c_void_p


class sssgs_config(ctypes.Structure):
    _fields_ = [("device", ctypes.c_int), ("max_gaussians", ctypes.c_int64),
                ("max_width", ctypes.c_int), ("max_height", ctypes.c_int),
                ("max_instances", ctypes.c_int64), ("max_lights_per_pass", ctypes.c_int),
                ("workspace", _vp), ("workspace_bytes", ctypes.c_size_t), ("flags", ctypes.c_uint32)]


class sssgs_gaussians(ctypes.Structure):
    _fields_ = [("n", ctypes.c_int64), ("means", _vp), ("scales", _vp), ("rotations", _vp),
                ("opacities", _vp), ("normals", _vp), ("base_color", _vp), ("roughness", _vp),
                ("metallic", _vp), ("subsurface", _vp), ("vis_sh", _vp),
                ("vis_sh_degree", ctypes.c_int), ("feat", _vp), ("feat_dim", ctypes.c_int)]


class sssgs_mlp(ctypes.Structure):
    _fields_ = [("in_dim", ctypes.c_int), ("n_trunk", ctypes.c_int),
                ("trunk_width", ctypes.c_int * SSSGS_MAX_TRUNK), ("n_inc_hidden", ctypes.c_int),
                ("inc_hidden_width", ctypes.c_int * SSSGS_MAX_INC_HIDDEN),
                ("activation", ctypes.c_int), ("leaky_slope", _f), ("dtype", ctypes.c_int),
                ("params", _vp), ("params_bytes", ctypes.c_size_t), ("precomputed_out", _vp),
                ("compute", ctypes.c_int)]


class sssgs_camera(ctypes.Structure):
    _fields_ = [("R", _f * 9), ("t", _f * 3), ("fx", _f), ("fy", _f), ("cx", _f), ("cy", _f),
                ("tan_half_fovx", _f), ("tan_half_fovy", _f), ("width", ctypes.c_int),
                ("height", ctypes.c_int), ("znear", _f), ("bg", _f * 3)]


class sssgs_light(ctypes.Structure):
    _fields_ = [("position", _f * 3), ("intensity", _f * 3)]


class sssgs_out(ctypes.Structure):
    _fields_ = [("rgb", _vp), ("gbuffer", _vp), ("aov_diffuse", _vp), ("aov_specular", _vp),
                ("mlp_out", _vp), ("sorted_keys", _vp), ("sorted_vals", _vp), ("tile_ranges", _vp),
                ("counters", _vp)]


class sssgs_grads(ctypes.Structure):
    _fields_ = [(k, _vp) for k in ("grad_rgb", "gbuffer", "grad_gbuffer", "grad_mlp_out", "grad_params",
                                   "grad_opacity", "grad_mean2d", "grad_conic", "grad_depth", "grad_attr",
                                   "grad_means", "grad_scales", "grad_rotations", "grad_feat", "grad_vis_sh",
                                   "grad_gbuffer_in", "counters")]


class sssgs_bake(ctypes.Structure):
    _fields_ = [("n_dirs", ctypes.c_int), ("dirs", _vp), ("weights", _vp), ("t_min", _f),
                ("sh_degree", ctypes.c_int), ("vis_sh_out", _vp), ("vis_out", _vp), ("positions", ctypes.c_int)]


class SssgsError(RuntimeError):
    def __init__(self, code, msg):
        super().__init__(f"libsssgs error {code}: {msg}")
        self.code = code


_lib = None


def lib() -> ctypes.CDLL:
    """Load libsssgs.so (never falls back to anything else)."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise ImportError(f"{LIB_PATH} is missing: build it with `python -m paper_2408_12282_b200.build` "
                              "(libsssgs has no CPU fallback)")
        L = ctypes.CDLL(LIB_PATH)
        L.sssgs_workspace_bytes.restype = ctypes.c_size_t
        L.sssgs_workspace_bytes.argtypes = [ctypes.POINTER(sssgs_config)]
        L.sssgs_create.restype = ctypes.c_int
        L.sssgs_create.argtypes = [ctypes.POINTER(sssgs_config), ctypes.POINTER(_vp)]
        L.sssgs_destroy.restype = None
        L.sssgs_destroy.argtypes = [_vp]
        render_args = [_vp, ctypes.POINTER(sssgs_gaussians), ctypes.POINTER(sssgs_mlp),
                       ctypes.POINTER(sssgs_camera), ctypes.c_int, ctypes.POINTER(sssgs_light),
                       ctypes.c_int, ctypes.POINTER(sssgs_out), ctypes.c_uint32]
        L.sssgs_render.restype = ctypes.c_int
        L.sssgs_render.argtypes = render_args + [_vp]
        L.sssgs_render_host.restype = ctypes.c_int
        L.sssgs_render_host.argtypes = render_args
        L.sssgs_render_backward.restype = ctypes.c_int
        L.sssgs_render_backward.argtypes = [_vp, ctypes.POINTER(sssgs_gaussians), ctypes.POINTER(sssgs_mlp),
                                            ctypes.POINTER(sssgs_camera), ctypes.POINTER(sssgs_light), ctypes.c_int,
                                            ctypes.POINTER(sssgs_grads), ctypes.c_uint32, _vp]
        L.sssgs_bake_visibility.restype = ctypes.c_int
        L.sssgs_bake_visibility.argtypes = [_vp, ctypes.POINTER(sssgs_gaussians), ctypes.POINTER(sssgs_bake), _vp]
        L.sssgs_last_launch_count.restype = ctypes.c_int64
        L.sssgs_last_launch_count.argtypes = [_vp]
        L.sssgs_profile_enable.restype = ctypes.c_int
        L.sssgs_profile_enable.argtypes = [_vp, ctypes.c_int]
        L.sssgs_profile_read.restype = ctypes.c_int
        L.sssgs_profile_read.argtypes = [_vp, ctypes.POINTER(ctypes.c_float), ctypes.POINTER(ctypes.c_int)]
        L.sssgs_mlp_eval_static.restype = ctypes.c_int
        L.sssgs_mlp_eval_static.argtypes = [ctypes.c_int, ctypes.POINTER(sssgs_gaussians), ctypes.POINTER(sssgs_mlp),
                                            ctypes.POINTER(sssgs_camera), ctypes.POINTER(sssgs_light), ctypes.c_int,
                                            _vp, _vp]
        L.sssgs_relight.restype = ctypes.c_int
        L.sssgs_relight.argtypes = [ctypes.c_int, _vp, ctypes.c_int, ctypes.c_int64, _vp, _vp, _vp]
        L.sssgs_last_error.restype = ctypes.c_char_p
        L.sssgs_last_error.argtypes = [_vp]
        _lib = L
    return _lib


# ---- the ABI calls, same names --------------------------------------------------------------
def sssgs_workspace_bytes(cfg: sssgs_config) -> int:
    return int(lib().sssgs_workspace_bytes(ctypes.byref(cfg)))


def sssgs_create(cfg: sssgs_config) -> _vp:
    h = _vp()
    rc = lib().sssgs_create(ctypes.byref(cfg), ctypes.byref(h))
    if rc != SSSGS_OK:
        raise SssgsError(rc, (lib().sssgs_last_error(None) or b"").decode())
    return h


def sssgs_destroy(ctx) -> None:
    lib().sssgs_destroy(ctx)


def _check(ctx, rc):
    if rc != SSSGS_OK:
        raise SssgsError(rc, (lib().sssgs_last_error(ctx) or b"").decode())


def sssgs_render(ctx, g, mlp, cams, n_cam, lights, n_light, out, flags=0, stream=None) -> None:
    _check(ctx, lib().sssgs_render(ctx, ctypes.byref(g), ctypes.byref(mlp), cams, n_cam, lights, n_light,
                                   ctypes.byref(out), flags, _vp(stream or 0)))


def sssgs_render_host(ctx, g, mlp, cams, n_cam, lights, n_light, out, flags=0) -> None:
    _check(ctx, lib().sssgs_render_host(ctx, ctypes.byref(g), ctypes.byref(mlp), cams, n_cam, lights,
                                        n_light, ctypes.byref(out), flags))


def sssgs_render_backward(ctx, g, mlp, cam, lights, n_light, grads, flags=0, stream=None) -> None:
    _check(ctx, lib().sssgs_render_backward(ctx, ctypes.byref(g), ctypes.byref(mlp), ctypes.byref(cam), lights,
                                            n_light, ctypes.byref(grads), flags, _vp(stream or 0)))


def sssgs_bake_visibility(ctx, g, bake, stream=None) -> None:
    _check(ctx, lib().sssgs_bake_visibility(ctx, ctypes.byref(g), ctypes.byref(bake), _vp(stream or 0)))


def sssgs_mlp_eval_static(device, g, mlp, cam, lights, n_light, mlp_out_ptr, stream=None) -> None:
    """The MLP alone, without a context and without any device allocation (include/sssgs.h).

    For callers that cannot call cudaMalloc -- hosts that gave all GPU memory to their own pool, latency-critical
    threads.  mlp_out_ptr: device pointer to [n][n_light][4] floats (Gaussian-major).  The packed weights go through
    one fixed array inside the library (192 KB per GPU, shared by all calls): calls that may overlap on the GPU
    race on it.  Errors are reported through sssgs_last_error(NULL)."""
    rc = lib().sssgs_mlp_eval_static(int(device), ctypes.byref(g), ctypes.byref(mlp), ctypes.byref(cam), lights,
                                     int(n_light), _vp(mlp_out_ptr or 0), _vp(stream or 0))
    if rc != SSSGS_OK:
        raise SssgsError(rc, (lib().sssgs_last_error(None) or b"").decode())


def sssgs_relight(device, frames_ptr, n_light, n_pixels, weights_ptr, out_ptr, stream=None) -> None:
    """out[p][c] = sum_l weights[l][c] * frames[l][p][c]; device pointers, see include/sssgs.h."""
    rc = lib().sssgs_relight(int(device), _vp(frames_ptr or 0), int(n_light), int(n_pixels), _vp(weights_ptr or 0),
                             _vp(out_ptr or 0), _vp(stream or 0))
    if rc != SSSGS_OK:
        raise SssgsError(rc, (lib().sssgs_last_error(None) or b"").decode())


def sssgs_last_launch_count(ctx) -> int:
    return int(lib().sssgs_last_launch_count(ctx))


def sssgs_profile_enable(ctx, enable: bool) -> None:
    _check(ctx, lib().sssgs_profile_enable(ctx, 1 if enable else 0))


def sssgs_profile_read(ctx):
    """-> ({stage: ms}, {stage: kernel launches}) of the last sssgs_render call."""
    ms = (ctypes.c_float * len(STAGES))()
    nl = (ctypes.c_int * len(STAGES))()
    _check(ctx, lib().sssgs_profile_read(ctx, ms, nl))
    return {k: float(ms[i]) for i, k in enumerate(STAGES)}, {k: int(nl[i]) for i, k in enumerate(STAGES)}


# ---- marshalling helpers ------------------------------------------------------------------------
def make_camera(cam) -> sssgs_camera:
    c = sssgs_camera()
    c.R[:] = [float(v) for v in np.asarray(cam.R, np.float32).ravel()]
    c.t[:] = [float(v) for v in np.asarray(cam.t, np.float32).ravel()]
    c.fx, c.fy, c.cx, c.cy = cam.fx, cam.fy, cam.cx, cam.cy
    c.tan_half_fovx, c.tan_half_fovy = cam.tan_half_fovx, cam.tan_half_fovy
    c.width, c.height, c.znear = int(cam.width), int(cam.height), cam.znear
    c.bg[:] = [float(v) for v in np.asarray(cam.bg, np.float32).ravel()]
    return c


def make_light(light) -> sssgs_light:
    l = sssgs_light()
    l.position[:] = [float(v) for v in np.asarray(light.position, np.float32)]
    l.intensity[:] = [float(v) for v in np.asarray(light.intensity, np.float32)]
    return l


def make_mlp(spec, params_ptr, params_bytes, dtype=SSSGS_F32, precomputed_ptr=None,
             compute=SSSGS_COMPUTE_FP16) -> sssgs_mlp:
    m = sssgs_mlp()
    m.in_dim = spec.in_dim
    m.n_trunk = len(spec.trunk_width)
    for i, w in enumerate(spec.trunk_width):
        m.trunk_width[i] = w
    m.n_inc_hidden = len(spec.inc_hidden_width)
    for i, w in enumerate(spec.inc_hidden_width):
        m.inc_hidden_width[i] = w
    m.activation = spec.activation
    m.leaky_slope = spec.leaky_slope
    m.dtype = dtype
    m.params = params_ptr
    m.params_bytes = params_bytes
    m.precomputed_out = precomputed_ptr
    m.compute = compute
    return m


_FIELDS = ("means", "scales", "rotations", "opacities", "normals", "base_color", "roughness",
           "metallic", "subsurface", "vis_sh", "feat")


def make_gaussians(n, ptrs: dict, vis_sh_degree: int, feat_dim: int) -> sssgs_gaussians:
    g = sssgs_gaussians()
    g.n = n
    for f in _FIELDS:
        setattr(g, f, ptrs.get(f))
    g.vis_sh_degree = vis_sh_degree
    g.feat_dim = feat_dim
    return g


class Renderer:
    """Device-resident scene + context.  torch is used for memory and streams only."""

    def __init__(self, scene, max_instances: Optional[int] = None, max_lights_per_pass: int = 0,
                 device: int = 0, max_width: Optional[int] = None, max_height: Optional[int] = None,
                 compute: int = SSSGS_COMPUTE_FP16):
        import torch
        self.torch = torch
        self.scene = scene
        self.compute = compute
        self.device = torch.device("cuda", device)
        self.n = int(scene.n)
        W = max_width or max(c.width for c in scene.cameras)
        H = max_height or max(c.height for c in scene.cameras)
        self.cfg = sssgs_config()
        self.cfg.device = device
        self.cfg.max_gaussians = max(self.n, 1)
        self.cfg.max_width, self.cfg.max_height = W, H
        self.cfg.max_instances = int(max_instances if max_instances is not None else max(16 * self.n, 1 << 16))
        self.cfg.max_lights_per_pass = max_lights_per_pass
        self.ctx = sssgs_create(self.cfg)
        self.t = {}
        for f in _FIELDS:
            a = np.ascontiguousarray(getattr(scene, f), dtype=np.float32)
            if a.size == 0:
                a = np.zeros(4, np.float32)
            self.t[f] = torch.from_numpy(a).to(self.device)
        self.params = torch.from_numpy(np.ascontiguousarray(scene.mlp.params, np.float32)).to(self.device)
        self.feat_dim = int(scene.feat.shape[1]) if scene.feat.ndim == 2 else 0
        self.g = make_gaussians(self.n, {f: self.t[f].data_ptr() for f in _FIELDS}, scene.vis_sh_degree,
                                self.feat_dim)

    def close(self):
        if self.ctx is not None:
            sssgs_destroy(self.ctx)
            self.ctx = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def alloc_outputs(self, n_cam, n_light, W, H, want: Sequence[str]):
        torch = self.torch
        F = n_cam * n_light
        tiles = ((W + 15) // 16) * ((H + 15) // 16)
        cap = int(self.cfg.max_instances)
        shapes = {"rgb": ((F, H, W, 3), torch.float32), "gbuffer": ((F, H, W, 16), torch.float32),
                  "aov_diffuse": ((F, H, W, 3), torch.float32), "aov_specular": ((F, H, W, 3), torch.float32),
                  "mlp_out": ((F, max(self.n, 1), 4), torch.float32),
                  "sorted_keys": ((n_cam, cap), torch.int64), "sorted_vals": ((n_cam, cap), torch.int32),
                  "tile_ranges": ((n_cam, tiles, 2), torch.int32),
                  "counters": ((n_cam, SSSGS_NCOUNTERS), torch.int64)}
        return {k: torch.zeros(shapes[k][0], dtype=shapes[k][1], device=self.device) for k in want}

    def render(self, cams=None, lights=None, want=("rgb",), outputs=None, precomputed=None,
               lights_per_camera=False, stream=None, sum_lights=False, forward=False, tight=False):
        """Enqueue one sssgs_render on the current torch stream.  cams: list of scene cameras;
        lights: list of lights (or list per camera with lights_per_camera).  Returns the dict of
        output tensors (device)."""
        torch = self.torch
        cams = list(cams if cams is not None else self.scene.cameras)
        if lights is None:
            lights = self.scene.lights[0]
        flat = [l for per in lights for l in per] if lights_per_camera else list(lights)
        n_cam = len(cams)
        n_light = (len(lights[0]) if lights else 0) if lights_per_camera else len(flat)
        W, H = cams[0].width, cams[0].height
        if outputs is None:
            outputs = self.alloc_outputs(n_cam, n_light, W, H, want)
            if sum_lights and "rgb" in outputs:   # one frame per camera
                outputs["rgb"] = torch.zeros((n_cam, H, W, 3), dtype=torch.float32, device=self.device)
        o = sssgs_out()
        for k, v in outputs.items():
            setattr(o, k, v.data_ptr())
        carr = (sssgs_camera * max(n_cam, 1))(*[make_camera(c) for c in cams])
        larr = (sssgs_light * max(len(flat), 1))(*[make_light(l) for l in flat])
        pre_ptr = None
        if precomputed is not None:
            self._pre = torch.as_tensor(np.ascontiguousarray(precomputed, np.float32)).to(self.device) \
                if not torch.is_tensor(precomputed) else precomputed
            pre_ptr = self._pre.data_ptr()
        m = make_mlp(self.scene.mlp, self.params.data_ptr(), self.params.numel() * 4, SSSGS_F32, pre_ptr, self.compute)
        st = stream if stream is not None else torch.cuda.current_stream(self.device).cuda_stream
        sssgs_render(self.ctx, self.g, m, carr, n_cam, larr, n_light, o,
                     (SSSGS_LIGHTS_PER_CAMERA if lights_per_camera else 0) | (SSSGS_SUM_LIGHTS if sum_lights else 0) |
                     (SSSGS_FORWARD_SHADING if forward else 0) | (SSSGS_TIGHT_LISTS if tight else 0), st)
        return outputs

    def render_backward(self, cam, lights, grad_rgb, gbuffer, tight=False, stream=None, precomputed=None, fp32=False,
                        through_inputs=False, grad_gbuffer_in=None):
        """Enqueue one sssgs_render_backward: cam one scene camera, lights its lights, grad_rgb [L,H,W,3] and
        gbuffer [L,H,W,16] device tensors (the forward call's G-buffer); grad_gbuffer_in [L,H,W,16]: optional
        upstream gradient on the G-buffer.  Returns the dict of gradient tensors (+ "counters": the list counters of
        the rebuilt tile lists, check SSSGS_CNT_OVERFLOW)."""
        torch = self.torch
        L, n, W, H = len(lights), max(self.n, 1), cam.width, cam.height
        z = lambda *shape: torch.empty(shape, dtype=torch.float32, device=self.device)  # noqa: E731
        out = {"grad_gbuffer": z(L, H, W, 16), "grad_mlp_out": z(L, n, 4), "grad_params": z(self.params.numel()),
               "grad_opacity": z(n), "grad_mean2d": z(n, 2), "grad_conic": z(n, 3), "grad_depth": z(n),
               "grad_attr": z(n, 9), "grad_means": z(n, 3), "grad_scales": z(n, 3), "grad_rotations": z(n, 4)}
        if through_inputs:   # step a1: the gradients through the MLP's inputs (added to means / scales / rotations / normal)
            out["grad_feat"] = z(n, max(self.feat_dim, 1))
            out["grad_vis_sh"] = z(n, (self.scene.vis_sh_degree + 1) ** 2)
        out["counters"] = torch.zeros(SSSGS_NCOUNTERS, dtype=torch.int64, device=self.device)
        gr = sssgs_grads()
        self._bwd_in = (grad_rgb.contiguous(), gbuffer.contiguous(),
                        None if grad_gbuffer_in is None else grad_gbuffer_in.contiguous())
        gr.grad_rgb, gr.gbuffer = self._bwd_in[0].data_ptr(), self._bwd_in[1].data_ptr()
        gr.grad_gbuffer_in = None if self._bwd_in[2] is None else self._bwd_in[2].data_ptr()
        for k, v in out.items():
            setattr(gr, k, v.data_ptr())
        larr = (sssgs_light * max(L, 1))(*[make_light(l) for l in lights])
        pre_ptr = None
        if precomputed is not None:
            self._pre = precomputed
            pre_ptr = precomputed.data_ptr()
        m = make_mlp(self.scene.mlp, self.params.data_ptr(), self.params.numel() * 4, SSSGS_F32, pre_ptr, self.compute)
        st = stream if stream is not None else torch.cuda.current_stream(self.device).cuda_stream
        sssgs_render_backward(self.ctx, self.g, m, make_camera(cam), larr, L, gr,
                              (SSSGS_TIGHT_LISTS if tight else 0) | (SSSGS_BACKWARD_FP32 if fp32 else 0), st)
        return out

    def bake_visibility(self, dirs, weights, t_min: float, sh_degree: int = 1, want_vis: bool = False, stream=None,
                        positions: bool = False):
        """Enqueue one sssgs_bake_visibility on the current torch stream.  dirs [K,3], weights [K] (numpy or
        device tensors).  Returns (vis_sh [n,(deg+1)^2], vis [n,K] or None), device tensors."""
        torch = self.torch
        def dev(a):
            return a if torch.is_tensor(a) else torch.from_numpy(np.ascontiguousarray(a, np.float32)).to(self.device)
        self._bake_in = (dev(dirs).reshape(-1, 3).contiguous(), dev(weights).reshape(-1).contiguous())
        K = int(self._bake_in[0].shape[0])
        nc = (sh_degree + 1) ** 2
        sh = torch.zeros((max(self.n, 1), nc), dtype=torch.float32, device=self.device)
        vis = torch.zeros((max(self.n, 1), K), dtype=torch.float32, device=self.device) if want_vis else None
        b = sssgs_bake()
        b.n_dirs, b.dirs, b.weights = K, self._bake_in[0].data_ptr(), self._bake_in[1].data_ptr()
        b.t_min, b.sh_degree = float(t_min), int(sh_degree)
        b.vis_sh_out, b.vis_out = sh.data_ptr(), (vis.data_ptr() if want_vis else None)
        b.positions = 1 if positions else 0
        st = stream if stream is not None else torch.cuda.current_stream(self.device).cuda_stream
        sssgs_bake_visibility(self.ctx, self.g, b, st)
        return sh[:self.n], (vis[:self.n] if want_vis else None)

    def launch_count(self) -> int:
        return sssgs_last_launch_count(self.ctx)


def render_host(scene, cams=None, lights=None, want=("rgb",), max_instances=None, ctx_holder=None):
    """sssgs_render_host with numpy (host) buffers; returns dict of numpy outputs.
    ctx_holder: optional dict to cache the context between calls."""
    cams = list(cams if cams is not None else scene.cameras)
    lights = list(lights if lights is not None else scene.lights[0])
    n = int(scene.n)
    W, H = cams[0].width, cams[0].height
    n_cam, n_light = len(cams), len(lights)
    key = (n, W, H, max_instances)
    if ctx_holder is not None and ctx_holder.get("key") == key:
        ctx, cfg = ctx_holder["ctx"], ctx_holder["cfg"]
    else:
        cfg = sssgs_config()
        cfg.device = 0
        cfg.max_gaussians = max(n, 1)
        cfg.max_width, cfg.max_height = W, H
        cfg.max_instances = int(max_instances if max_instances is not None else max(16 * n, 1 << 16))
        ctx = sssgs_create(cfg)
        if ctx_holder is not None:
            if ctx_holder.get("ctx") is not None:
                sssgs_destroy(ctx_holder["ctx"])
            ctx_holder.update(key=key, ctx=ctx, cfg=cfg)
    arrs = {f: np.ascontiguousarray(getattr(scene, f), dtype=np.float32) for f in _FIELDS}
    feat_dim = int(scene.feat.shape[1]) if scene.feat.ndim == 2 else 0
    g = make_gaussians(n, {f: arrs[f].ctypes.data if arrs[f].size else None for f in _FIELDS},
                       scene.vis_sh_degree, feat_dim)
    params = np.ascontiguousarray(scene.mlp.params, np.float32)
    m = make_mlp(scene.mlp, params.ctypes.data, params.nbytes)
    F = n_cam * n_light
    tiles = ((W + 15) // 16) * ((H + 15) // 16)
    cap = int(cfg.max_instances)
    shapes = {"rgb": ((F, H, W, 3), np.float32), "gbuffer": ((F, H, W, 16), np.float32),
              "aov_diffuse": ((F, H, W, 3), np.float32), "aov_specular": ((F, H, W, 3), np.float32),
              "mlp_out": ((F, max(n, 1), 4), np.float32), "sorted_keys": ((n_cam, cap), np.uint64),
              "sorted_vals": ((n_cam, cap), np.uint32), "tile_ranges": ((n_cam, tiles, 2), np.uint32),
              "counters": ((n_cam, SSSGS_NCOUNTERS), np.int64)}
    outs = {k: np.zeros(shapes[k][0], shapes[k][1]) for k in want}
    o = sssgs_out()
    for k, v in outs.items():
        setattr(o, k, v.ctypes.data)
    carr = (sssgs_camera * max(n_cam, 1))(*[make_camera(c) for c in cams])
    larr = (sssgs_light * max(n_light, 1))(*[make_light(l) for l in lights])
    try:
        sssgs_render_host(ctx, g, m, carr, n_cam, larr, n_light, o, 0)
    finally:
        if ctx_holder is None:
            sssgs_destroy(ctx)
    return outs


class HostRenderer:
    """sssgs_render_host with PINNED host buffers (torch.pin_memory is used for allocation only).
    Every call crosses host->device with the whole scene and device->host with the outputs."""

    def __init__(self, scene, max_instances: Optional[int] = None, device: int = 0):
        import torch
        self.torch = torch
        self.scene = scene
        self.n = int(scene.n)
        cam = scene.cameras[0]
        self.cfg = sssgs_config()
        self.cfg.device = device
        self.cfg.max_gaussians = max(self.n, 1)
        self.cfg.max_width = max(c.width for c in scene.cameras)
        self.cfg.max_height = max(c.height for c in scene.cameras)
        self.cfg.max_instances = int(max_instances if max_instances is not None else max(16 * self.n, 1 << 16))
        self.ctx = sssgs_create(self.cfg)
        self.t = {}
        for f in _FIELDS:
            a = np.ascontiguousarray(getattr(scene, f), dtype=np.float32)
            if a.size == 0:
                a = np.zeros(4, np.float32)
            self.t[f] = torch.from_numpy(a).pin_memory()
        self.params = torch.from_numpy(np.ascontiguousarray(scene.mlp.params, np.float32)).pin_memory()
        self.feat_dim = int(scene.feat.shape[1]) if scene.feat.ndim == 2 else 0
        self.g = make_gaussians(self.n, {f: self.t[f].data_ptr() for f in _FIELDS}, scene.vis_sh_degree,
                                self.feat_dim)
        self.h2d_bytes = sum(int(getattr(scene, f).nbytes) for f in _FIELDS) + int(scene.mlp.params.nbytes)
        self.out = {}

    def close(self):
        if self.ctx is not None:
            sssgs_destroy(self.ctx)
            self.ctx = None

    def render(self, cams, lights, want=("rgb",), tight=False):
        torch = self.torch
        n_cam, n_light = len(cams), len(lights)
        W, H = cams[0].width, cams[0].height
        F = n_cam * n_light
        shapes = {"rgb": (F, H, W, 3), "gbuffer": (F, H, W, 16), "mlp_out": (F, max(self.n, 1), 4)}
        o = sssgs_out()
        d2h = n_cam * SSSGS_NCOUNTERS * 8
        for k in want:
            if k not in self.out or tuple(self.out[k].shape) != shapes[k]:
                self.out[k] = torch.zeros(shapes[k], dtype=torch.float32).pin_memory()
            setattr(o, k, self.out[k].data_ptr())
            d2h += self.out[k].numel() * 4
        carr = (sssgs_camera * max(n_cam, 1))(*[make_camera(c) for c in cams])
        larr = (sssgs_light * max(n_light, 1))(*[make_light(l) for l in lights])
        m = make_mlp(self.scene.mlp, self.params.data_ptr(), self.params.numel() * 4)
        sssgs_render_host(self.ctx, self.g, m, carr, n_cam, larr, n_light, o, SSSGS_TIGHT_LISTS if tight else 0)
        self.d2h_bytes = d2h
        return {k: self.out[k] for k in want}
