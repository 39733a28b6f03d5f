"""Pins of the backward oracle (oracle/backward.py: steps a2 / a7 / a8 differentiated; PAPER.md L11, L112,
L343-349): its forward restatements equal the C++ oracle, every gradient equals central finite differences of
the C++ FORWARD oracle, and closed forms of one and two Gaussians on a pixel centre.  CPU only."""
import dataclasses

import numpy as np
import torch

import oracle
from oracle import backward as ob
from paper_2408_12282_b200 import scenes
from util import custom_scene, with_mlp_params


def _setup(scene, view=0):
    cam = scene.cameras[view]
    proj = oracle.project(scene, cam)
    keys, vals, ranges = oracle.build_lists(proj)
    xs = [oracle.mlp_inputs(scene, cam, lt.position) for lt in scene.lights[view]]
    return cam, proj, vals, ranges, xs


def _cpp_loss(scene, proj, vals, ranges, xs, G, view=0):
    """L = sum_l <G_l, rgb_l> through the C++ forward oracle (MLP mode 0, compositing, shading)."""
    cam = scene.cameras[view]
    tot = 0.0
    for li, lt in enumerate(scene.lights[view]):
        mo = oracle.mlp_forward(xs[li], scene.mlp, 0)
        comp = oracle.composite(scene, cam, proj, oracle.channels(scene, proj, mo), vals, ranges)
        rgb = oracle.shade(cam, lt, comp.gbuf)[0]
        tot += float((rgb * G[li]).sum())
    return tot


def _scene():
    s = scenes.make_scene(3, n=400, width=40, height=32, lights=2)
    # moderate opacities: most pixels keep T well above 1e-4, few decisions near a threshold
    return dataclasses.replace(s, opacities=np.clip(s.opacities, 0.05, 0.6).astype(np.float32))


def test_forward_restatements_equal_the_cpp_oracle():
    s = _scene()
    cam, proj, vals, ranges, xs = _setup(s)
    mo_ref = oracle.mlp_forward(xs[0], s.mlp, 0)
    mo = ob.mlp_torch(ob._t(xs[0]), s.mlp, ob._t(s.mlp.params)).numpy()
    np.testing.assert_allclose(mo, mo_ref, rtol=1e-12, atol=1e-13)
    s6 = scenes.make_scene(6, n=50)                                   # paper architecture: split heads, Leaky-ReLU
    x6 = oracle.mlp_inputs(s6, s6.cameras[0], s6.lights[0][0].position)
    np.testing.assert_allclose(ob.mlp_torch(ob._t(x6), s6.mlp, ob._t(s6.mlp.params)).numpy(),
                               oracle.mlp_forward(x6, s6.mlp, 0), rtol=1e-12, atol=1e-13)
    ch = oracle.channels(s, proj, mo_ref)
    comp = oracle.composite(s, cam, proj, ch, vals, ranges)
    gb = ob.composite_torch(cam.width, cam.height, ob._t(proj.pix), ob._t(proj.conic), ob._t(s.opacities), ob._t(ch),
                            vals, ranges, proj.tiles_x).numpy()
    np.testing.assert_allclose(gb, comp.gbuf, rtol=1e-12, atol=1e-13)
    assert comp.p_blend > 1000 and (comp.gbuf[..., 15] < 0.5).any()
    lt = s.lights[0][1]
    rgb = ob.shade_torch(cam, lt.position, lt.intensity, ob._t(comp.gbuf)).numpy()
    np.testing.assert_allclose(rgb, oracle.shade(cam, lt, comp.gbuf)[0], rtol=1e-11, atol=1e-13)


def test_gradients_equal_finite_differences_of_the_cpp_forward():
    s = _scene()
    cam, proj, vals, ranges, xs = _setup(s)
    rng = np.random.default_rng(11)
    G = rng.standard_normal((2, cam.height, cam.width, 3))
    r = ob.render_backward(s, proj, vals, ranges, xs, G)
    np.testing.assert_allclose(r.loss, _cpp_loss(s, proj, vals, ranges, xs, G), rtol=1e-11)

    def fd(apply, h):
        """central difference; apply(delta) -> (scene', proj', actual +delta, actual -delta)"""
        sp, pp, dp = apply(+h)
        sm, pm, dm = apply(-h)
        return (_cpp_loss(sp, pp, vals, ranges, xs, G) - _cpp_loss(sm, pm, vals, ranges, xs, G)) / (dp - dm)

    def pick(g):     # the largest gradients and a few random ones
        flat = np.abs(g).ravel()
        return sorted(set(np.argsort(-flat)[:3].tolist() + rng.choice(flat.size, 3, replace=False).tolist()))

    def check(name, got, ref):
        assert abs(got - ref) <= 2e-5 * max(1.0, abs(ref)) + 1e-7, (name, got, ref)

    # per-Gaussian float32 inputs of the scene
    for name, field, h in [("d_opacity", "opacities", 1e-4), ("d_normals", "normals", 1e-4), ("d_base", "base_color", 1e-4),
                           ("d_rough", "roughness", 1e-4), ("d_metal", "metallic", 1e-4), ("d_sss", "subsurface", 1e-4)]:
        g = getattr(r, name)
        for k in pick(g):
            def apply(d, field=field, k=k):
                a = getattr(s, field).copy()
                a.ravel()[k] = np.float32(a.ravel()[k] + d)
                return dataclasses.replace(s, **{field: a}), proj, float(a.ravel()[k])
            check((name, k), g.ravel()[k], fd(apply, h))
    # projected quantities (inputs of step 5): 2-D mean, conic, depth
    for name, field, h in [("d_pix", "pix", 2e-4), ("d_conic", "conic", 1e-5), ("d_depth", "depth", 1e-4)]:
        g = getattr(r, name)
        for k in pick(g):
            def apply(d, field=field, k=k):
                p2 = type(proj)(**vars(proj))
                a = getattr(proj, field).copy()
                a.ravel()[k] = np.float32(a.ravel()[k] + d)
                setattr(p2, field, a)
                return s, p2, float(a.ravel()[k])
            check((name, k), g.ravel()[k], fd(apply, h))
    # MLP parameters (weights and biases of every layer)
    for k in pick(r.d_params):
        def apply(d, k=k):
            p = s.mlp.params.copy()
            p[k] = np.float32(p[k] + d)
            return with_mlp_params(s, p), proj, float(p[k])
        check(("d_params", k), r.d_params[k], fd(apply, 2e-6))   # small step: a larger one crosses ReLU kinks of some rows
    assert np.abs(r.d_params).max() > 1e-3 and np.abs(r.d_pix).max() > 1e-3 and np.abs(r.d_conic).max() > 1e-3


def test_per_stage_gradients_chain_together():
    # d_gbuf is the shading backward alone (central differences of orc_shade on single G-buffer values), and
    # d_mlp_out is the compositing backward of channels 10-13: sum_p w_i(p) d_gbuf[p, 10 + c]
    s = _scene()
    cam, proj, vals, ranges, xs = _setup(s)
    rng = np.random.default_rng(5)
    G = rng.standard_normal((2, cam.height, cam.width, 3))
    r = ob.render_backward(s, proj, vals, ranges, xs, G)
    lt = s.lights[0][0]
    covered = np.argwhere(r.gbuf[0][..., 14] > 0.3)
    for (y, x) in covered[rng.choice(len(covered), 4, replace=False)]:
        for c in (0, 2, 5, 7, 8, 9, 11, 13, 14):
            gp, gm = r.gbuf[0].copy(), r.gbuf[0].copy()
            h = 1e-6 * max(1.0, abs(gp[y, x, c]))
            gp[y, x, c] += h
            gm[y, x, c] -= h
            d = ((oracle.shade(cam, lt, gp)[0] - oracle.shade(cam, lt, gm)[0]) * G[0]).sum() / (2 * h)
            assert abs(r.d_gbuf[0][y, x, c] - d) <= 1e-6 * max(1.0, abs(d)), (y, x, c)
    assert (r.d_gbuf[..., 15] == 0).all()          # the final transmittance is not an input of the shading
    # weights of Gaussian i at every pixel, from two composites that differ in one channel value of i
    i = int(np.argmax(np.abs(r.d_mlp_out[0]).sum(1)))
    ch0 = oracle.channels(s, proj, r.mlp_out[0])
    ch1 = ch0.copy()
    ch1[i, 10] += 1.0
    w = (oracle.composite(s, cam, proj, ch1, vals, ranges).gbuf - oracle.composite(s, cam, proj, ch0, vals, ranges).gbuf)[..., 10]
    for c in range(4):
        np.testing.assert_allclose(r.d_mlp_out[0][i, c], (w * r.d_gbuf[0][..., 10 + c]).sum(), rtol=1e-9, atol=1e-12)


def test_closed_forms_on_a_pixel_centre():
    # sss = 1, bg = 0: rgb = sum_i T_i alpha_i L_SSS,i (Eq. 7 reduces to the residual, Eq. 3 composites it).
    # One Gaussian whose centre projects onto pixel (32, 32): alpha there = o  =>  d rgb_c / d o = L_SSS_c,
    # d rgb_c / d L_SSS_c = o.  Two Gaussians on that pixel, the first nearer: C = o1 c1 + (1 - o1) o2 c2  =>
    # dC/do1 = c1 - o2 c2, dC/do2 = (1 - o1) c2, dC/dc1 = o1, dC/dc2 = (1 - o1) o2.
    for means, ops in ([[0, 0, 0]], [0.7]), ([[0, -0.5, 0], [0, 0, 0]], [0.6, 0.8]):
        s = custom_scene(means, 0.05, opacities=ops, subsurface=1.0, width=65, height=65)
        cam, proj, vals, ranges, xs = _setup(s)
        G = np.zeros((1, 65, 65, 3))
        G[0, 32, 32] = [1.0, 2.0, -0.5]
        r = ob.render_backward(s, proj, vals, ranges, xs, G)
        c = r.mlp_out[0][:, :3]                                      # L_SSS of each Gaussian
        gvec = G[0, 32, 32]
        if len(ops) == 1:
            np.testing.assert_allclose(r.rgb[0][32, 32], ops[0] * c[0], rtol=1e-6)
            np.testing.assert_allclose(r.d_opacity[0], (gvec * c[0]).sum(), rtol=1e-6)
            np.testing.assert_allclose(r.d_mlp_out[0][0, :3], ops[0] * gvec, rtol=1e-6)
        else:
            o1, o2 = ops
            np.testing.assert_allclose(r.rgb[0][32, 32], o1 * c[0] + (1 - o1) * o2 * c[1], rtol=1e-6)
            np.testing.assert_allclose(r.d_opacity, [(gvec * (c[0] - o2 * c[1])).sum(), (gvec * (1 - o1) * c[1]).sum()], rtol=1e-6)
            np.testing.assert_allclose(r.d_mlp_out[0][:, :3], [o1 * gvec, (1 - o1) * o2 * gvec], rtol=1e-6)
        # on the centre the exponent is stationary: no gradient to the 2-D mean or the conic from this pixel
        # (the fp32 projection puts the centre within ~1e-5 px of the pixel centre, hence the tolerances)
        assert np.abs(r.d_pix).max() < 1e-3 and np.abs(r.d_conic).max() < 1e-8


def test_fp16_emulating_restatement():
    """mode 2 of mlp_torch: forward == the C++ oracle's binary16-emulating mode; its gradient (rounding = identity)
    equals the float64 network's wherever the two take the same ReLU decisions, up to the 2^-11 operand rounding."""
    s = _scene()
    cam, proj, vals, ranges, xs = _setup(s)
    x = ob._t(xs[0])
    y2 = ob.mlp_torch(x, s.mlp, ob._t(s.mlp.params), mode=2).numpy()
    np.testing.assert_allclose(y2, oracle.mlp_forward(xs[0], s.mlp, 2), rtol=1e-12, atol=1e-13)
    assert np.abs(y2 - oracle.mlp_forward(xs[0], s.mlp, 0)).max() > 1e-6      # it does round
    s6 = scenes.make_scene(6, n=50)
    x6 = oracle.mlp_inputs(s6, s6.cameras[0], s6.lights[0][0].position)
    np.testing.assert_allclose(ob.mlp_torch(ob._t(x6), s6.mlp, ob._t(s6.mlp.params), mode=2).numpy(),
                               oracle.mlp_forward(x6, s6.mlp, 2), rtol=1e-12, atol=1e-13)
    # gradient: one row at a time; rows whose hidden pre-activations all stay clear of 0 take the same decisions
    rng = np.random.default_rng(3)
    go = ob._t(rng.standard_normal((len(xs[0]), 4)))
    grads = []
    for mode in (0, 2):
        p = ob._t(s.mlp.params).requires_grad_(True)
        (ob.mlp_torch(x, s.mlp, p, mode=mode) * go).sum().backward()
        grads.append(p.grad.numpy())
    rel = np.abs(grads[1] - grads[0]).max() / np.abs(grads[0]).max()
    assert 0 < rel < 5e-2        # close (a few flipped decisions among 400 x 384 units), not identical
    # a one-row case with every pre-activation far from 0: decisions agree, the difference is rounding only
    w = np.abs(oracle.mlp_forward(xs[0], s.mlp, 0) - oracle.mlp_forward(xs[0], s.mlp, 2)).max(axis=1)
    r = int(np.argmin(w))
    g1 = []
    for mode in (0, 2):
        p = ob._t(s.mlp.params).requires_grad_(True)
        (ob.mlp_torch(x[r:r + 1], s.mlp, p, mode=mode) * go[r:r + 1]).sum().backward()
        g1.append(p.grad.numpy())
    same = (g1[0] != 0) == (g1[1] != 0)
    if same.all():
        assert np.abs(g1[1] - g1[0]).max() <= 5e-3 * np.abs(g1[0]).max()


def test_fp16_emulation_decides_in_the_rounded_arithmetic():
    """Hand-made one-unit net: x = 1 + 2^-12 rounds to 1 in binary16; with W = 1, b = -(1 + 2^-13) (kept in fp32)
    the float64 pre-activation is +2^-13 (ReLU on: dL/dW = x dL/dh) and the emulated one is -2^-13 (off: 0)."""
    x = ob._t(np.array([[1.0 + 2.0 ** -12]]))
    b0 = -(1.0 + 2.0 ** -13)
    params = np.array([1.0, b0,  1.0, 0.0, 0.0,  0.0, 0.0, 0.0,  2.0,  0.5], np.float64)   # trunk, sss 3x1 + b, inc 1x1 + b
    mlp = scenes.MlpSpec(in_dim=1, trunk_width=[1], inc_hidden_width=[], activation=0, leaky_slope=0.01,
                         params=params.astype(np.float32))
    assert float(np.float32(b0)) == b0
    got = {}
    for mode in (0, 2):
        p = ob._t(params).requires_grad_(True)
        y = ob.mlp_torch(x, mlp, p, mode=mode)
        y[0, 3].backward()          # incident head: relu(2 h + 0.5)
        got[mode] = (y.detach().numpy()[0], p.grad.numpy())
    h0 = 2.0 ** -13
    np.testing.assert_allclose(got[0][0][3], 2 * h0 + 0.5, rtol=1e-14)
    np.testing.assert_allclose(got[0][1][0], 2.0 * (1.0 + 2.0 ** -12), rtol=1e-14)   # dL/dW0 = w_inc * x
    np.testing.assert_allclose(got[0][1][8], h0, rtol=1e-12)                            # dL/dw_inc = h
    assert got[2][0][3] == 0.5 and got[2][1][0] == 0.0 and got[2][1][1] == 0.0 and got[2][1][8] == 0.0
    assert got[2][1][9] == 1.0


def test_projection_restatement_and_its_gradient():
    """project_torch == the C++ double projection (orc_project_f64) and, inverted, the canonical fp32 conic;
    its reverse-mode gradient == central finite differences of the C++ function; closed form on the optical axis."""
    s = _scene()
    cam = s.cameras[0]
    proj = oracle.project(s, cam)
    cov, pix, depth = oracle.project_f64(s, cam)
    tp, tc, td, tcov = ob.project_torch(ob._t(s.means), ob._t(s.scales), ob._t(s.rotations), cam)
    np.testing.assert_allclose(tcov.numpy(), cov, rtol=1e-12)
    np.testing.assert_allclose(tp.numpy(), pix, rtol=1e-12)
    np.testing.assert_allclose(td.numpy(), depth, rtol=1e-13)
    vis = proj.visible != 0
    assert vis.sum() > 100
    np.testing.assert_allclose(tc.numpy()[vis], proj.conic[vis], rtol=2e-4, atol=1e-7)
    np.testing.assert_allclose(tp.numpy()[vis], proj.pix[vis], rtol=1e-5, atol=1e-4)
    # finite differences of L = <gp, pix> + <gc, conic(cov)> + <gd, depth> through the C++ function
    rng = np.random.default_rng(5)
    gp, gc, gd = rng.standard_normal((s.n, 2)), rng.standard_normal((s.n, 3)), rng.standard_normal(s.n)
    dm, dsc, dq = ob.project_backward(s, cam, vis, gp, gc, gd)

    def loss(sc_):
        cov_, pix_, dep_ = oracle.project_f64(sc_, cam)
        det = cov_[:, 0] * cov_[:, 2] - cov_[:, 1] ** 2
        con = np.stack([cov_[:, 2] / det, -cov_[:, 1] / det, cov_[:, 0] / det], 1)
        return float((pix_[vis] * gp[vis]).sum() + (con[vis] * gc[vis]).sum() + (dep_[vis] * gd[vis]).sum())

    ids = np.nonzero(vis)[0][:6]
    for field, grad, ncomp in (("means", dm, 3), ("scales", dsc, 3), ("rotations", dq, 4)):
        for i in ids[:3]:
            for k in range(ncomp):
                base = np.array(getattr(s, field), np.float32)
                h = np.float32(2.0 ** -10) * max(1e-3, abs(float(base[i, k])))   # float32 fields: a relative step
                hi, lo = base.copy(), base.copy()
                hi[i, k] += h
                lo[i, k] -= h
                num = (loss(dataclasses.replace(s, **{field: hi})) - loss(dataclasses.replace(s, **{field: lo}))) \
                    / (float(hi[i, k]) - float(lo[i, k]))
                assert abs(num - grad[i, k]) <= 2e-4 * max(1.0, abs(grad[i, k])) + 1e-3 * np.abs(grad[i]).max(), \
                    (field, i, k, num, grad[i, k])
    assert not dm[~vis].any() and not dsc[~vis].any() and not dq[~vis].any()
    # closed form: isotropic Gaussian (sigma) on the optical axis, identity rotation: Sigma' = ((f sigma / z)^2 + 0.3) I
    cam0 = scenes.look_at_camera((0.0, -4.0, 0.0), 64, 64, 40.0)
    sig, z = 0.25, 4.0
    one = custom_scene([[0.0, 0.0, 0.0]], [[sig, sig, sig]], width=64, height=64)
    one = dataclasses.replace(one, cameras=[cam0])
    v = (cam0.fx * sig / z) ** 2 + 0.3
    _, sc1, _ = ob.project_backward(one, cam0, np.ones(1), np.zeros((1, 2)), np.array([[1.0, 0.0, 0.0]]), np.zeros(1))
    # conic_a = 1 / v; the image x axis is fed by one world axis only: d conic_a / d s_k = -(2 f^2 s_k / z^2) / v^2 for that k
    assert np.isclose(np.abs(sc1).sum(), 2 * cam0.fx ** 2 * sig / z ** 2 / v ** 2, rtol=1e-9)


def test_render_backward_through_the_projection_chains():
    """through_projection: dL/d(means, scales, rotations) == project_backward fed the same call's dL/d(pix, conic,
    depth) (chain rule across the two restatements), and the forward image is unchanged to rounding."""
    s = _scene()
    cam, proj, vals, ranges, xs = _setup(s)
    G = np.random.default_rng(13).standard_normal((2, cam.height, cam.width, 3))
    r = ob.render_backward(s, proj, vals, ranges, xs, G, through_projection=True)
    r0 = ob.render_backward(s, proj, vals, ranges, xs, G)
    np.testing.assert_allclose(r.rgb, r0.rgb, rtol=0, atol=2e-5)     # float64 projection vs the canonical fp32 values
    dm, dsc, dq = ob.project_backward(s, cam, proj.visible, r.d_pix, r.d_conic, r.d_depth)
    np.testing.assert_allclose(r.d_means, dm, rtol=1e-9, atol=1e-12)
    np.testing.assert_allclose(r.d_scales, dsc, rtol=1e-9, atol=1e-12)
    np.testing.assert_allclose(r.d_rotations, dq, rtol=1e-9, atol=1e-12)
    assert np.abs(r.d_means).max() > 0 and np.abs(r.d_rotations).max() > 0


def test_mlp_input_restatement_and_its_gradient():
    """mlp_inputs_torch == orc_mlp_inputs (incl. a negative q_r and visibilities clamped at both ends); its
    reverse-mode gradient == central differences of the C++ function."""
    s = _scene()
    rot = np.array(s.rotations, np.float32)
    rot[::3] *= -1.0                                  # q and -q: the sign-canonical pair changes sign
    vsh = np.array(s.vis_sh, np.float32)
    vsh[1::7, 0] += 4.0                               # v > 1: clamped
    vsh[2::7, 0] -= 4.0                               # v < 0: clamped
    s = dataclasses.replace(s, rotations=rot, vis_sh=vsh)
    cam, lt = s.cameras[0], s.lights[0][1]
    x_ref = oracle.mlp_inputs(s, cam, lt.position)
    assert (x_ref[:, 15] == 1.0).any() and (x_ref[:, 15] == 0.0).any() and ((x_ref[:, 15] > 0) & (x_ref[:, 15] < 1)).any()

    def xt(sc_, leaf=None):
        t = {k: ob._t(getattr(sc_, k)) for k in ("means", "normals", "rotations", "scales", "vis_sh", "feat")}
        if leaf:
            t[leaf].requires_grad_(True)
        return t, ob.mlp_inputs_torch(t["means"], t["normals"], t["rotations"], t["scales"], t["vis_sh"], t["feat"], cam,
                                      lt.position, sc_.vis_sh_degree)
    np.testing.assert_allclose(xt(s)[1].numpy(), x_ref, rtol=1e-12, atol=1e-13)
    rng = np.random.default_rng(9)
    gx = rng.standard_normal(x_ref.shape)
    for field in ("means", "normals", "rotations", "scales", "vis_sh", "feat"):
        t, x = xt(s, field)
        (x * ob._t(gx)).sum().backward()
        grad = t[field].grad.numpy()
        base = np.array(getattr(s, field), np.float32)
        for i in (0, 1, 2, 3, 7):
            for k in range(min(base.shape[1], 4)):
                h = np.float32(2.0 ** -10) * max(1e-2, abs(float(base[i, k])))
                hi, lo = base.copy(), base.copy()
                hi[i, k] += h
                lo[i, k] -= h
                if field == "rotations" and (hi[i, 0] < 0) != (lo[i, 0] < 0):
                    continue                              # the canonical sign flips inside the step
                f = lambda b: float((oracle.mlp_inputs(dataclasses.replace(s, **{field: b}), cam, lt.position) * gx).sum())  # noqa: E731
                num = (f(hi) - f(lo)) / (float(hi[i, k]) - float(lo[i, k]))
                assert abs(num - grad[i, k]) <= 1e-4 * max(1.0, np.abs(grad[i]).max()), (field, i, k, num, grad[i, k])


def test_render_backward_through_the_inputs_equals_finite_differences():
    """through_inputs: dL/d(feat, vis_sh, normals) of the WHOLE chain (inputs -> MLP -> compositing -> shading) ==
    central differences of the C++ forward oracle with the inputs recomputed by orc_mlp_inputs."""
    s = _scene()
    cam, proj, vals, ranges, xs = _setup(s)
    rng = np.random.default_rng(21)
    G = rng.standard_normal((2, cam.height, cam.width, 3))
    r = ob.render_backward(s, proj, vals, ranges, xs, G, through_projection=True, through_inputs=True)
    r0 = ob.render_backward(s, proj, vals, ranges, xs, G, through_projection=True)
    np.testing.assert_allclose(r.rgb, r0.rgb, rtol=0, atol=1e-12)
    assert np.abs(r.d_means - r0.d_means).max() > 0            # the inputs add their share

    def loss(sc_):
        xs_ = [oracle.mlp_inputs(sc_, cam, lt.position) for lt in sc_.lights[0]]
        return _cpp_loss(sc_, proj, vals, ranges, xs_, G)

    for field, grad in (("feat", r.d_feat), ("vis_sh", r.d_vis_sh), ("normals", r.d_normals)):
        flat = np.abs(grad).ravel()
        for j in np.argsort(-flat)[:4]:
            i, k = np.unravel_index(j, grad.shape)
            base = np.array(getattr(s, field), np.float32)
            h = np.float32(2.0 ** -8) * max(1e-2, abs(float(base[i, k])))
            hi, lo = base.copy(), base.copy()
            hi[i, k] += h
            lo[i, k] -= h
            num = (loss(dataclasses.replace(s, **{field: hi})) - loss(dataclasses.replace(s, **{field: lo}))) \
                / (float(hi[i, k]) - float(lo[i, k]))
            assert abs(num - grad[i, k]) <= 2e-3 * abs(grad[i, k]) + 1e-6, (field, i, k, num, grad[i, k])


def test_shading_backward_of_the_back_projection_at_an_off_centre_pixel():
    # The pixel term ((px - cx) / fx) z of the back-projection enters the shading backward through
    # d(world point) / d(depth) = f + a r + b d.  Pin: the restatement's value at pixel (41, 17) of a 64 x 48 frame
    # equals the closed form built from the camera's basis vectors (tests/test_oracle_shading.py), and its reverse-mode
    # gradient w.r.t. the accumulated depth channel equals the central difference of that closed form in z.
    import test_oracle_shading as tos
    cam, light, basis, eye = tos._off_centre_setup()
    px, py, z, A = 41, 17, 3.3, 0.8
    n = tos._unit((0.3, -0.8, 0.4))
    b = np.array([0.8, 0.4, 0.1])
    g = torch.tensor(tos._gbuf_with_pixel(cam, px, py, z, n, b, 1.7, A=A), dtype=torch.float64, requires_grad=True)
    rgb = ob.shade_torch(cam, light.position, light.intensity, g)
    want = tos._lambert_at(cam, light, basis, eye, px, py, z, n, b, 1.7, A=A)
    np.testing.assert_allclose(rgb[py, px].detach().numpy(), want, rtol=1e-9)
    w = np.array([0.7, -1.3, 0.45])
    (rgb[py, px] * torch.tensor(w)).sum().backward()
    h = 1e-5
    fd = (tos._lambert_at(cam, light, basis, eye, px, py, z + h, n, b, 1.7, A=A) -
          tos._lambert_at(cam, light, basis, eye, px, py, z - h, n, b, 1.7, A=A)) @ w / (2 * h)
    got = float(g.grad[py, px, 0]) * A            # channel 0 holds A z: d/dz = A d/d(channel)
    assert abs(fd) > 1e-3 and abs(got - fd) <= 1e-7 * abs(fd) + 1e-10, (got, fd)
    # teeth: with px and py swapped the derivative is a different number
    fd_swapped = (tos._lambert_at(cam, light, basis, eye, py, px, z + h, n, b, 1.7, A=A) -
                  tos._lambert_at(cam, light, basis, eye, py, px, z - h, n, b, 1.7, A=A)) @ w / (2 * h)
    assert abs(fd_swapped - fd) > 1e-2 * abs(fd)
    # no other pixel's G-buffer received a gradient
    gg = g.grad.clone()
    gg[py, px] = 0
    assert float(gg.abs().max()) == 0.0


def test_upstream_gradient_on_the_gbuffer_equals_finite_differences():
    # L = sum_l <G_rgb, rgb_l> + <G_gb, gbuf_l>: the losses on the rasterised property images
    # reach the Gaussians through the compositing alone.  All 16 channels carry a gradient, the final
    # transmittance (15) included.  Reference: central differences of the C++ forward oracle.
    s = _scene()
    cam, proj, vals, ranges, xs = _setup(s)
    rng = np.random.default_rng(23)
    G = 0.3 * rng.standard_normal((2, cam.height, cam.width, 3))
    Gg = rng.standard_normal((2, cam.height, cam.width, 16))

    def cpp_loss(scene, pr):
        tot = 0.0
        for li, lt in enumerate(scene.lights[0]):
            mo = oracle.mlp_forward(xs[li], scene.mlp, 0)
            comp = oracle.composite(scene, cam, pr, oracle.channels(scene, pr, mo), vals, ranges)
            tot += float((oracle.shade(cam, lt, comp.gbuf)[0] * G[li]).sum() + (comp.gbuf * Gg[li]).sum())
        return tot

    r = ob.render_backward(s, proj, vals, ranges, xs, G, grad_gbuf=Gg)
    np.testing.assert_allclose(r.loss, cpp_loss(s, proj), rtol=1e-11)
    r0 = ob.render_backward(s, proj, vals, ranges, xs, G)
    np.testing.assert_allclose(r.d_gbuf, r0.d_gbuf + Gg, rtol=1e-12, atol=1e-13)     # a8 backward + the upstream term
    assert np.abs(r.d_opacity - r0.d_opacity).max() > 1e-2                          # and it reaches the Gaussians

    def pick(g):
        flat = np.abs(g).ravel()
        return sorted(set(np.argsort(-flat)[:3].tolist() + rng.choice(flat.size, 2, replace=False).tolist()))

    def check(name, got, ref):
        assert abs(got - ref) <= 2e-5 * max(1.0, abs(ref)) + 1e-7, (name, got, ref)

    for name, field, h in [("d_opacity", "opacities", 1e-4), ("d_normals", "normals", 1e-4), ("d_rough", "roughness", 1e-4),
                           ("d_sss", "subsurface", 1e-4)]:
        g = getattr(r, name)
        for k in pick(g):
            a = getattr(s, field)
            ap, am = a.copy(), a.copy()
            ap.ravel()[k] = np.float32(a.ravel()[k] + h)
            am.ravel()[k] = np.float32(a.ravel()[k] - h)
            fd = (cpp_loss(dataclasses.replace(s, **{field: ap}), proj) - cpp_loss(dataclasses.replace(s, **{field: am}), proj)) \
                / (float(ap.ravel()[k]) - float(am.ravel()[k]))
            check((name, k), g.ravel()[k], fd)
    for name, field, h in [("d_pix", "pix", 2e-4), ("d_conic", "conic", 1e-5), ("d_depth", "depth", 1e-4)]:
        g = getattr(r, name)
        for k in pick(g):
            vals_pm = []
            for sgn in (+1, -1):
                p2 = type(proj)(**vars(proj))
                a = getattr(proj, field).copy()
                a.ravel()[k] = np.float32(a.ravel()[k] + sgn * h)
                setattr(p2, field, a)
                vals_pm.append((cpp_loss(s, p2), float(a.ravel()[k])))
            fd = (vals_pm[0][0] - vals_pm[1][0]) / (vals_pm[0][1] - vals_pm[1][1])
            check((name, k), g.ravel()[k], fd)
    # a loss on the final transmittance alone: dL/d opacity of a Gaussian = -sum_p dT(p) T(p) alpha_i(p) / (o_i (1 - alpha_i(p)))
    # has the sign of -dT: more opacity, less transmittance
    Gt = np.zeros_like(Gg)
    Gt[..., 15] = 1.0
    rt = ob.render_backward(s, proj, vals, ranges, xs, np.zeros_like(G), grad_gbuf=Gt)
    assert (rt.d_opacity <= 1e-15).all() and rt.d_opacity.min() < -1e-2
