"""Backward pass of hot-path steps a2 / a3 / a7 / a8 -- CPU ORACLE (test infrastructure only).

PAPER.md L11 ("optimize all parameters jointly via raytraced differentiable rendering"), L112 (the
incident-light network is "jointly evaluated" and trained), L343-349 (App. F: the losses are functions
of the rendered image and of the rasterised property images).  The paper trains through the render
path by automatic differentiation of its PyTorch + CUDA implementation (L138) and prints no gradient
formula, so the oracle is the definition itself: the forward steps 2 (MLP), 5 (compositing) and 6
(shading) of SURVEY.md 8(c) are restated here in torch float64 operations, in the order and notation of
oracle/sssgs_oracle.cpp, and differentiated by torch.autograd.  The discontinuous decisions of step 5
(alpha >= 1/255 skip, power > 0 skip, T' < 1e-4 stop, the 0.99 clamp) are constants of the
differentiation, as in every rasteriser of this family.

Pinned (tests/test_oracle_backward.py) by: the forward restatements equal the C++ oracle to 1e-12;
central finite differences of the C++ forward oracle for every gradient; closed forms (one Gaussian
on a pixel centre, two layers).

Loss convention: the caller supplies G_l = dL/d rgb_l [H, W, 3] for every light l of one view; every
gradient below is that of  L = sum_l <G_l, rgb_l>.

Only tests/ (and smoke()) may import this module; it imports nothing from the CUDA path.
"""
from __future__ import annotations

import math
from types import SimpleNamespace

import numpy as np
import torch

F8 = torch.float64
ALPHA_MIN, ALPHA_MAX, T_MIN = 1.0 / 255.0, 0.99, 1e-4


def _t(a):
    return torch.as_tensor(np.ascontiguousarray(a, np.float64))


# ---------------------------------------------------------------------------------------------------
# Step 2: the MLP (orc_mlp_forward, mode 0)
# ---------------------------------------------------------------------------------------------------
def mlp_layers(mlp, params: torch.Tensor):
    """Views of the packed parameter vector: [(W[out,in], b[out], kind)], kinds as scenes.MlpSpec."""
    out, off = [], 0
    for (o, i, kind) in mlp.layer_shapes():
        W = params[off:off + o * i].reshape(o, i)
        off += o * i
        b = params[off:off + o]
        off += o
        out.append((W, b, kind))
    assert off == params.numel()
    return out


def mlp_torch(x: torch.Tensor, mlp, params: torch.Tensor, mode: int = 0) -> torch.Tensor:
    """x [n, in_dim] -> [n, 4] = (sigmoid SSS head (3), relu incident head (1)).
    mode 0: float64.  mode 2: the binary16-operand arithmetic of oracle.mlp_forward(mode 2) (weights rounded once,
    every layer input rounded to binary16, float64 accumulation), the rounding treated as the identity by the
    differentiation (straight-through): the ReLU decisions are then taken in the kernel's precision, which is
    what the tensor-core backward differentiates."""
    if mode == 0:
        rnd = lambda t: t  # noqa: E731
    else:
        rnd = lambda t: t + (t.to(torch.float16).to(F8) - t).detach()  # noqa: E731
    act = (lambda t: torch.where(t > 0, t, mlp.leaky_slope * t)) if mlp.activation == 1 else torch.relu
    h, hi, sss, inc = x, None, None, None
    for W, b, kind in mlp_layers(mlp, params):
        W = rnd(W)
        if kind == "trunk":
            h = act(rnd(h) @ W.T + b)
        elif kind == "sss":
            sss = torch.sigmoid(rnd(h) @ W.T + b)
            hi = h
        elif kind == "inc_hidden":
            hi = act(rnd(hi) @ W.T + b)
        else:
            inc = torch.relu(rnd(hi) @ W.T + b)
    return torch.cat([sss, inc], dim=1)


# ---------------------------------------------------------------------------------------------------
# Step 1: the MLP input row (orc_mlp_inputs: Eq. 6), for the gradients that reach the Gaussians
# through the MLP's inputs
# ---------------------------------------------------------------------------------------------------
Y00, Y1 = 0.2820948, 0.4886025


def mlp_inputs_torch(means, normals, rotations, scales, vis_sh, feat, cam, light_pos, sh_degree: int):
    """[n, 40 + F] float64: n (3), sign-canonical (q_r, q_x) (2), scale (3), w_in (3), w_out (3), light distance,
    SH visibility towards the light clamped to [0, 1], Fourier encoding of mu (24), feature (F).  The clamp and the
    quaternion sign are constants of the differentiation."""
    R, t = _t(cam.R), _t(cam.t)
    pc = -(R.T @ t)
    sgn = torch.where(rotations[:, 0] < 0, -1.0, 1.0).detach()
    wi = _t(light_pos)[None, :] - means
    wo = pc[None, :] - means
    di = torch.linalg.norm(wi, dim=1)
    dn = torch.linalg.norm(wo, dim=1)
    wi = wi / di[:, None]
    wo = wo / dn[:, None]
    v = Y00 * vis_sh[:, 0]
    if sh_degree >= 1:
        v = v + Y1 * (vis_sh[:, 1] * wi[:, 1] + vis_sh[:, 2] * wi[:, 2] + vis_sh[:, 3] * wi[:, 0])
    v = torch.clamp(v, 0.0, 1.0)
    enc = []
    for k in range(4):
        fr = float(1 << k) * math.pi
        enc += [torch.sin(fr * means), torch.cos(fr * means)]
    cols = [normals, (sgn * rotations[:, 0])[:, None], (sgn * rotations[:, 1])[:, None], scales, wi, wo, di[:, None],
            v[:, None]] + enc
    if feat is not None and feat.numel() and feat.shape[1] > 0:
        cols.append(feat)
    return torch.cat(cols, dim=1)


# ---------------------------------------------------------------------------------------------------
# Step 3: EWA projection (orc_project_f64: Eq. 2), for the gradients w.r.t. mean, scale, rotation
# ---------------------------------------------------------------------------------------------------
def project_torch(means, scales, rotations, cam):
    """means [n,3], scales [n,3], rotations [n,4] (r,x,y,z) torch float64 -> (pix [n,2], conic [n,3], depth [n],
    cov2d [n,3]).  Sigma' = J W Sigma W^T J^T + 0.3 I with the frustum clamp of the Jacobian (a constant of the
    differentiation where it clamps), conic = Sigma'^-1.  No culling: the caller masks by the oracle's `visible`."""
    R, t = _t(cam.R), _t(cam.t)
    p = means @ R.T + t
    z = p[:, 2]
    u, w = p[:, 0] / z, p[:, 1] / z
    pix = torch.stack([cam.fx * u + cam.cx, cam.fy * w + cam.cy], dim=1)
    lx, ly = 1.3 * cam.tan_half_fovx, 1.3 * cam.tan_half_fovy
    xc, yc = torch.clamp(u, -lx, lx) * z, torch.clamp(w, -ly, ly) * z
    zero = torch.zeros_like(z)
    J = torch.stack([torch.stack([cam.fx / z, zero, -cam.fx * xc / (z * z)], dim=1),
                     torch.stack([zero, cam.fy / z, -cam.fy * yc / (z * z)], dim=1)], dim=1)       # [n,2,3]
    r, x, y, zq = rotations[:, 0], rotations[:, 1], rotations[:, 2], rotations[:, 3]
    Rq = torch.stack([1 - 2 * (y * y + zq * zq), 2 * (x * y - r * zq), 2 * (x * zq + r * y),
                      2 * (x * y + r * zq), 1 - 2 * (x * x + zq * zq), 2 * (y * zq - r * x),
                      2 * (x * zq - r * y), 2 * (y * zq + r * x), 1 - 2 * (x * x + y * y)], dim=1).reshape(-1, 3, 3)
    M = Rq * scales[:, None, :]
    Sg = M @ M.transpose(1, 2)
    T = J @ R                                                                                     # [n,2,3]
    c2 = T @ Sg @ T.transpose(1, 2)
    a, b, c = c2[:, 0, 0] + 0.3, c2[:, 0, 1], c2[:, 1, 1] + 0.3
    det = a * c - b * b
    conic = torch.stack([c / det, -b / det, a / det], dim=1)
    return pix, conic, z, torch.stack([a, b, c], dim=1)


def project_backward(scene, cam, visible, d_pix, d_conic, d_depth):
    """dL/d(means, scales, rotations) [n,3], [n,3], [n,4] from dL/d(pix, conic, depth) of the visible Gaussians."""
    mu = _t(scene.means).requires_grad_(True)
    sc = _t(scene.scales).requires_grad_(True)
    q = _t(scene.rotations).requires_grad_(True)
    pix, conic, depth, _ = project_torch(mu, sc, q, cam)
    m = torch.as_tensor(np.asarray(visible) != 0)
    loss = (pix[m] * _t(d_pix)[m]).sum() + (conic[m] * _t(d_conic)[m]).sum() + (depth[m] * _t(d_depth)[m]).sum()
    loss.backward()
    return mu.grad.numpy(), sc.grad.numpy(), q.grad.numpy()


# ---------------------------------------------------------------------------------------------------
# Step 5: compositing (orc_composite, tiled mode)
# ---------------------------------------------------------------------------------------------------
def composite_torch(width, height, pix, conic, opac, ch, vals, ranges, tiles_x, tile=16):
    """Eq. 3 (L68-72) per pixel over its tile's list.  pix [n,2], conic [n,3], opac [n], ch [n,14] torch
    float64 (leaf tensors may require grad); vals / ranges numpy.  Returns gbuf [H, W, 16]."""
    gbuf = torch.zeros((height, width, 16), dtype=F8)
    gbuf[..., 15] = 1.0
    n_tiles = ranges.shape[0]
    for t in range(n_tiles):
        b, e = int(ranges[t, 0]), int(ranges[t, 1])
        if e == b:
            continue
        ty, tx = divmod(t, tiles_x)
        ys = torch.arange(ty * tile, min((ty + 1) * tile, height), dtype=F8)
        xs = torch.arange(tx * tile, min((tx + 1) * tile, width), dtype=F8)
        py, px = torch.meshgrid(ys, xs, indexing="ij")
        P = py.numel()
        g = torch.as_tensor(vals[b:e].astype(np.int64))
        dx = px.reshape(P, 1) - pix[g, 0].reshape(1, -1)           # [P, E]
        dy = py.reshape(P, 1) - pix[g, 1].reshape(1, -1)
        ca, cb, cc = conic[g, 0], conic[g, 1], conic[g, 2]
        power = -0.5 * (ca * dx * dx + cc * dy * dy) - cb * dx * dy
        araw = opac[g] * torch.exp(power)
        alpha = torch.clamp(araw, max=ALPHA_MAX)
        with torch.no_grad():                                       # the decisions: constants of the derivative
            passes = (power <= 0.0) & (alpha >= ALPHA_MIN)
            a_eff = torch.where(passes, alpha, torch.zeros_like(alpha))
            t_next = torch.cumprod(1.0 - a_eff, dim=1)              # T' after each entry, ignoring the stop
            stops = passes & (t_next < T_MIN)
            stopped = torch.cumsum(stops.to(torch.int64), dim=1) > 0   # at or after the stopping entry
            blend = passes & ~stopped
        a_b = torch.where(blend, alpha, torch.zeros_like(alpha))
        one_m = 1.0 - a_b
        t_excl = torch.cumprod(torch.cat([torch.ones((P, 1), dtype=F8), one_m[:, :-1]], dim=1), dim=1)
        w = t_excl * a_b                                            # [P, E]
        acc = w @ ch[g]                                             # [P, 14]
        A = w.sum(dim=1)
        T = torch.prod(one_m, dim=1)
        tile_out = torch.cat([acc, A[:, None], T[:, None]], dim=1).reshape(len(ys), len(xs), 16)
        gbuf[ty * tile:ty * tile + len(ys), tx * tile:tx * tile + len(xs)] = tile_out
    return gbuf


# ---------------------------------------------------------------------------------------------------
# Step 6: deferred shading (shade_impl)
# ---------------------------------------------------------------------------------------------------
def shade_torch(cam, light_pos, light_intensity, gbuf: torch.Tensor) -> torch.Tensor:
    """L114, Eq. 4, Eq. 7 L104-106 with the readings S8 / S10; gbuf [H, W, 16] -> rgb [H, W, 3]."""
    H, W = gbuf.shape[:2]
    R = _t(cam.R).reshape(3, 3)
    tt = _t(cam.t)
    pc = -(R.T @ tt)
    bg = _t(cam.bg)
    A = gbuf[..., 14]
    covered = A >= 1e-6
    As = torch.where(covered, A, torch.ones_like(A))
    q = gbuf[..., :14] / As[..., None]
    # uncovered pixels return the background (last line); they get a harmless stand-in here so that autograd
    # does not propagate 0/0 through a branch that is discarded (depth 0 would put the point into the camera)
    safe = torch.zeros(14, dtype=F8)
    safe[0], safe[3] = 1.0, 1.0
    q = torch.where(covered[..., None], q, safe)
    zb, rough, metal, sss, lin = q[..., 0], q[..., 7], q[..., 8], q[..., 9], q[..., 13]
    py, px = torch.meshgrid(torch.arange(H, dtype=F8), torch.arange(W, dtype=F8), indexing="ij")
    xc = torch.stack([(px - cam.cx) / cam.fx * zb, (py - cam.cy) / cam.fy * zb, zb], dim=-1)
    xw = (xc - tt) @ R                                              # R^T (x_c - t), row-vector form
    l = _t(light_pos) - xw
    v = pc - xw
    l = l / torch.linalg.norm(l, dim=-1, keepdim=True)
    v = v / torch.linalg.norm(v, dim=-1, keepdim=True)
    nraw = q[..., 1:4]
    has_n = (nraw.detach() ** 2).sum(-1).sqrt() >= 1e-8
    ex = torch.tensor([1.0, 0.0, 0.0], dtype=F8)
    nraw = torch.where(has_n[..., None], nraw, ex)                  # (|n| < 1e-8: only the SSS term is shaded)
    n = nraw / torch.linalg.norm(nraw, dim=-1, keepdim=True)
    hsum = l + v
    has_h = (hsum.detach() ** 2).sum(-1).sqrt() >= 1e-8
    hsum = torch.where(has_h[..., None], hsum, n)                   # |l + v| < 1e-8: h = n
    h = hsum / torch.linalg.norm(hsum, dim=-1, keepdim=True)
    dot = lambda a, b: (a * b).sum(-1)  # noqa: E731
    nl = torch.clamp(dot(n, l), min=0.0)
    nv = torch.clamp(dot(n, v), min=1e-4)
    nh = torch.clamp(dot(n, h), 0.0, 1.0)
    vh = torch.clamp(dot(v, h), 0.0, 1.0)
    ar = torch.clamp(rough * rough, min=1e-3)
    a2 = ar * ar
    s2 = (torch.linalg.cross(n, h) ** 2).sum(-1)
    dd = torch.clamp(a2 * nh * nh + s2, min=1e-12)
    D = a2 / (math.pi * dd * dd)
    k = 0.5 * ar
    V = 1.0 / (4.0 * (nl * (1.0 - k) + k) * (nv * (1.0 - k) + k))
    om5 = (1.0 - vh) ** 5
    base = q[..., 4:7]
    F0 = 0.04 * (1.0 - metal)[..., None] + base * metal[..., None]
    F = F0 + (1.0 - F0) * om5[..., None]
    fs = (D * V)[..., None] * F
    fd = (1.0 - metal)[..., None] * base / math.pi
    brdf = (fs + fd) * (lin * nl)[..., None]
    brdf = torch.where(has_n[..., None], brdf, torch.zeros_like(brdf))
    lout = sss[..., None] * q[..., 10:13] + (1.0 - sss)[..., None] * brdf
    rgb = _t(light_intensity) * A[..., None] * lout + (1.0 - A)[..., None] * bg
    return torch.where(covered[..., None], rgb, bg.expand_as(rgb))


# ---------------------------------------------------------------------------------------------------
# The gradients
# ---------------------------------------------------------------------------------------------------
def render_backward(scene, proj, vals, ranges, mlp_inputs, grad_rgb, view: int = 0, lights=None, tile=16,
                    given_mlp_out=None, mlp_mode: int = 0, through_projection: bool = False,
                    through_inputs: bool = False, grad_gbuf=None):
    """Gradients of L = sum_l <grad_rgb[l], rgb_l> (+ sum_l <grad_gbuf[l], gbuf_l> when grad_gbuf [L, H, W, 16] is
    given: the losses of PAPER.md L343-349 that act on the rasterised property images directly -- normal / depth
    consistency, mask entropy on A, smoothness of roughness / metalness / sss / base colour, the incident-light
    term) for one view.

    proj / vals / ranges: the oracle's projection and tile lists of the view (oracle.project / build_lists);
    mlp_inputs: [L][n, in_dim] float64 (oracle.mlp_inputs per light); grad_rgb [L, H, W, 3].
    mlp_mode: 0 float64 MLP, 2 its binary16-emulating restatement (mlp_torch).
    through_projection: pix / conic / depth are computed from (means, scales, rotations) by project_torch, and
    d_means [n,3], d_scales [n,3], d_rotations [n,4] are returned too.
    through_inputs (needs through_projection): the MLP inputs are computed from the Gaussians by mlp_inputs_torch
    (step a1) instead of being the constants `mlp_inputs`; d_means / d_scales / d_rotations / d_normals then hold the
    sums over both paths, and d_feat [n,F], d_vis_sh [n,ncoef] are returned.
    given_mlp_out: [L, n, 4] or None: the MLP outputs are these constants instead of mlp(mlp_inputs) (isolates
    the walks: d_params is then zero).
    Returns a namespace of numpy float64 arrays:
      rgb [L,H,W,3], gbuf [L,H,W,16]              forward values of the restatement
      d_gbuf [L,H,W,16]                           step a8 backward (per light), plus grad_gbuf where given
      d_mlp_out [L,n,4]                           what a7 hands to a2
      d_params [P]                                MLP weights and biases, packing of scenes.MlpSpec
      d_opacity [n], d_pix [n,2], d_conic [n,3], d_depth [n]   (depth = G-buffer channel 0's per-Gaussian value)
      d_normals [n,3], d_base [n,3], d_rough [n], d_metal [n], d_sss [n]
    """
    cam = scene.cameras[view]
    lights = scene.lights[view] if lights is None else lights
    L, n = len(lights), int(scene.n)
    params = _t(scene.mlp.params).requires_grad_(True)
    opac = _t(scene.opacities).requires_grad_(True)
    mu = sc = rot = None
    if through_projection:
        mu = _t(scene.means).requires_grad_(True)
        sc = _t(scene.scales).requires_grad_(True)
        rot = _t(scene.rotations).requires_grad_(True)
        tp, tc, td, _ = project_torch(mu, sc, rot, cam)
        vis = torch.as_tensor(np.asarray(proj.visible) != 0)
        pix = torch.where(vis[:, None], tp, _t(proj.pix))
        conic = torch.where(vis[:, None], tc, _t(proj.conic))
        depth = torch.where(vis, td, _t(proj.depth))
        for t_ in (pix, conic, depth):
            t_.retain_grad()
    else:
        pix = _t(proj.pix).requires_grad_(True)
        conic = _t(proj.conic).requires_grad_(True)
        depth = _t(proj.depth).requires_grad_(True)
    normals = _t(scene.normals).requires_grad_(True)
    base = _t(scene.base_color).requires_grad_(True)
    rough = _t(scene.roughness).requires_grad_(True)
    metal = _t(scene.metallic).requires_grad_(True)
    sss = _t(scene.subsurface).requires_grad_(True)
    feat_t = vsh_t = None
    if through_inputs:
        assert through_projection and given_mlp_out is None
        feat_t = _t(scene.feat).requires_grad_(True)
        vsh_t = _t(scene.vis_sh).requires_grad_(True)
    rgbs, gbufs, mlp_outs = [], [], []
    loss = torch.zeros((), dtype=F8)
    for li, lt in enumerate(lights):
        if through_inputs:
            x_in = mlp_inputs_torch(mu, normals, rot, sc, vsh_t, feat_t, cam, lt.position, scene.vis_sh_degree)
            mo = mlp_torch(x_in, scene.mlp, params, mode=mlp_mode)
        elif given_mlp_out is None:
            mo = mlp_torch(_t(mlp_inputs[li]), scene.mlp, params, mode=mlp_mode)
        else:
            mo = _t(given_mlp_out[li]).clone().requires_grad_(True)
        mo.retain_grad()
        ch = torch.cat([depth[:, None], normals, base, rough[:, None], metal[:, None], sss[:, None], mo], dim=1)
        gb = composite_torch(cam.width, cam.height, pix, conic, opac, ch, vals, ranges, proj.tiles_x, tile)
        gb.retain_grad()
        rgb = shade_torch(cam, lt.position, lt.intensity, gb)
        loss = loss + (rgb * _t(grad_rgb[li])).sum()
        if grad_gbuf is not None:
            loss = loss + (gb * _t(grad_gbuf[li])).sum()
        rgbs.append(rgb)
        gbufs.append(gb)
        mlp_outs.append(mo)
    loss.backward()
    z = lambda t: (t.grad if t.grad is not None else torch.zeros_like(t)).detach().numpy()  # noqa: E731
    return SimpleNamespace(
        loss=float(loss.detach()),
        rgb=np.stack([r.detach().numpy() for r in rgbs]), gbuf=np.stack([g.detach().numpy() for g in gbufs]),
        mlp_out=np.stack([m.detach().numpy() for m in mlp_outs]),
        d_gbuf=np.stack([z(g) for g in gbufs]), d_mlp_out=np.stack([z(m) for m in mlp_outs]),
        d_params=z(params), d_opacity=z(opac), d_pix=z(pix), d_conic=z(conic), d_depth=z(depth),
        d_normals=z(normals), d_base=z(base), d_rough=z(rough), d_metal=z(metal), d_sss=z(sss),
        d_means=z(mu) if through_projection else None, d_scales=z(sc) if through_projection else None,
        d_rotations=z(rot) if through_projection else None,
        d_feat=z(feat_t) if through_inputs else None, d_vis_sh=z(vsh_t) if through_inputs else None)
