"""Pins of the oracle's compositing (steps 5, 7; Eq. 3) against closed
forms, invariants and the tile-free brute force.  CPU only."""
import numpy as np

import oracle
from paper_2408_12282_b200 import scenes
from util import custom_scene


def _frame(s, mlp_out=None, **kw):
    if mlp_out is None:
        mlp_out = np.tile(np.array([0.2, 0.4, 0.6, 1.5]), (s.n, 1))
    return oracle.render_frame(s, mlp_out=mlp_out, **kw)


def test_single_gaussian_centre_alpha_and_profile():
    # one isotropic Gaussian projecting exactly onto a pixel centre: alpha there = opacity,
    # profile o exp(-r^2 / (2 sigma'^2)), sigma'^2 = (f sigma / z)^2 + 0.3
    o = 0.7
    s = custom_scene([[0, 0, 0]], 0.05, opacities=o, width=65, height=65)
    cam = s.cameras[0]
    r = _frame(s)
    np.testing.assert_allclose(r.proj.pix[0], [32, 32], atol=1e-4)
    A = r.gbuf[..., 14]
    assert abs(A[32, 32] - o) < 1e-6
    var = (cam.fx * 0.05 / 4.0) ** 2 + 0.3
    ys, xs = np.mgrid[0:65, 0:65]
    ref = o * np.exp(-((xs - 32.0) ** 2 + (ys - 32.0) ** 2) / (2 * var))
    ref[ref < 1 / 255.0] = 0
    mask = np.abs(ref - 1 / 255.0) > 1e-4  # exclude the threshold ring
    np.testing.assert_allclose(A[mask], ref[mask], atol=2e-5)
    # channels = weight x value
    np.testing.assert_allclose(r.gbuf[32, 32, 0], o * 4.0, rtol=1e-6)      # depth
    np.testing.assert_allclose(r.gbuf[32, 32, 10:14], o * np.array([0.2, 0.4, 0.6, 1.5]), rtol=1e-6)


def test_alpha_clamp_099():
    s = custom_scene([[0, 0, 0]], 0.05, opacities=1.0, width=33, height=33)
    r = _frame(s)
    assert abs(r.gbuf[16, 16, 14] - 0.99) < 1e-9


def test_zero_opacity_returns_background():
    s = scenes.make_scene(1, n=300, width=48, height=48)
    s.opacities[:] = 0
    s.cameras[0].bg[:] = [0.1, 0.2, 0.3]
    r = oracle.render_frame(s)
    assert (r.gbuf[..., :15] == 0).all() and (r.gbuf[..., 15] == 1).all()
    np.testing.assert_allclose(r.rgb, np.broadcast_to(np.float32([0.1, 0.2, 0.3]), r.rgb.shape), atol=1e-7)


def test_weights_plus_transmittance_sum_to_one():
    s = scenes.make_scene(1, width=96, height=96)
    r = oracle.render_frame(s)
    np.testing.assert_allclose(r.gbuf[..., 14] + r.gbuf[..., 15], 1.0, atol=1e-12)
    assert (r.gbuf[..., 14] > 0.5).sum() > 100  # the scene actually covers pixels


def test_coincident_gaussians():
    # K identical coincident Gaussians: A = 1 - (1-o)^K at the centre
    K, o = 5, 0.3
    s = custom_scene(np.zeros((K, 3)), 0.05, opacities=o, width=33, height=33)
    r = _frame(s)
    assert abs(r.gbuf[16, 16, 14] - (1 - (1 - o) ** K)) < 1e-6


def test_two_layers():
    # front layer (nearer the camera at y=-4) then back: o1 c1 + (1-o1) o2 c2
    o1, o2 = 0.6, 0.8
    s = custom_scene([[0, 0.5, 0], [0, -0.5, 0]], 0.2, opacities=[o2, o1], width=33, height=33)
    mlp_out = np.array([[0.1, 0.2, 0.3, 2.0], [0.9, 0.8, 0.7, 1.0]])  # index 0 = back, 1 = front
    r = _frame(s, mlp_out)
    ctr = r.gbuf[16, 16]
    # alpha at the centre pixel: both project to the centre
    a1 = o1 * np.exp(0.0)
    a2 = o2 * np.exp(0.0)
    np.testing.assert_allclose(ctr[10:14], a1 * mlp_out[1] + (1 - a1) * a2 * mlp_out[0], rtol=1e-6)
    np.testing.assert_allclose(ctr[0], a1 * 3.5 + (1 - a1) * a2 * 4.5, rtol=1e-6)
    np.testing.assert_allclose(ctr[15], (1 - a1) * (1 - a2), rtol=1e-6)


def test_stop_rule_does_not_blend_last():
    # T' < 1e-4 stops BEFORE blending: with alpha = 0.99 each, T goes 1 -> 1e-2 -> (1e-4 is not
    # < 1e-4 in exact arithmetic, but 0.01*0.01 rounds to just above) -> third would give 1e-6: stop
    s = custom_scene(np.zeros((4, 3)), 0.3, opacities=1.0, width=17, height=17)
    r = _frame(s)
    A, T = r.gbuf[8, 8, 14], r.gbuf[8, 8, 15]
    assert abs(T - 1e-4) < 1e-9 and abs(A - (1 - 1e-4)) < 1e-9


def test_permutation_invariance_distinct_depths():
    s = scenes.make_scene(1, n=800, width=64, height=64)
    d0 = oracle.project(s, s.cameras[0]).depth
    _, first = np.unique(d0, return_index=True)  # keep one Gaussian per distinct depth
    s = scenes.subset(s, np.sort(first))
    perm = np.random.default_rng(5).permutation(s.n)
    s2 = scenes.subset(s, perm)
    r1 = oracle.render_frame(s)
    r2 = oracle.render_frame(s2)
    vis = r1.proj.visible.astype(bool)
    assert len(set(r1.proj.depth[vis].tolist())) == vis.sum()
    np.testing.assert_array_equal(r1.gbuf, r2.gbuf)
    np.testing.assert_array_equal(r1.rgb, r2.rgb)


def test_tiled_equals_brute_force():
    # S3: the tile machinery must not change the image (brute force over ALL Gaussians per pixel)
    for cfg, n, w, h in ((1, 200, 64, 64), (1, 1500, 50, 37), (2, 3000, 64, 48)):
        s = scenes.make_scene(cfg, n=n, width=w, height=h)
        r = oracle.render_frame(s)
        b = oracle.composite(s, s.cameras[0], r.proj, r.ch, oracle.brute_order(r.proj), None)
        np.testing.assert_array_equal(r.gbuf, b.gbuf)
        assert b.p_blend == r.comp.p_blend


def test_interpenetrating_layers_and_ragged_image():
    # two interpenetrating shells on an image that is not a multiple of the tile size
    rng = np.random.default_rng(7)
    d = rng.standard_normal((400, 3))
    d /= np.linalg.norm(d, axis=1, keepdims=True)
    means = np.concatenate([d[:200] * 0.8, d[200:] * 0.8 + [0.3, 0.0, 0.0]])
    s = custom_scene(means, 0.06, opacities=0.6, width=50, height=37)
    r = _frame(s)
    b = oracle.composite(s, s.cameras[0], r.proj, r.ch, oracle.brute_order(r.proj), None)
    np.testing.assert_array_equal(r.gbuf, b.gbuf)
    np.testing.assert_allclose(r.gbuf[..., 14] + r.gbuf[..., 15], 1.0, atol=1e-12)


def test_counters():
    s = scenes.make_scene(1, n=500, width=64, height=64)
    r = oracle.render_frame(s)
    assert r.comp.p_blend <= r.comp.p_eval
    lens = (r.ranges[:, 1].astype(np.int64) - r.ranges[:, 0])
    assert r.comp.p_eval <= int(lens.sum()) * 256
    assert r.comp.contrib.sum() <= r.n_vis


# ---- tight tile lists: the minimal set of (tile, Gaussian) pairs --------------------------
def _hits_of(s):
    cam = s.cameras[0]
    proj = oracle.project(s, cam)
    keys, vals, ranges = oracle.build_lists(proj)
    return proj, keys, vals, ranges, oracle.tile_hits(s, cam, proj, vals, ranges)


def test_tile_hits_closed_form_isotropic():
    # One isotropic Gaussian: alpha(p) = o exp(-|p - c|^2 / 2 s^2) with s^2 = (f sigma / z)^2 + 0.3 (low-pass; the
    # x^2 / z^2 terms of the Jacobian change s by < 0.3 % this close to the axis), so alpha >= 1/255 inside the disc
    # of radius R = s sqrt(2 ln(255 o)) ~ 11 px.  A tile is hit iff its nearest pixel CENTRE (coordinates 16 t ..
    # 16 t + 15) lies within R of the projected centre c ~ (27, 32): tile column 0 is in the canonical rectangle
    # (27 - 3.33 s = 15.7 < 16) but its nearest pixel centre, x = 15, is 12 px away: not hit.
    s = custom_scene([[-0.224, 0, 0]], 0.15, opacities=0.8, width=65, height=65)
    cam = s.cameras[0]
    proj, keys, vals, ranges, hit = _hits_of(s)
    cx, cy = float(proj.pix[0, 0]), float(proj.pix[0, 1])
    var = (cam.fx * 0.15 / float(proj.depth[0])) ** 2 + 0.3
    R = np.sqrt(var * 2 * np.log(255 * 0.8))
    assert 26.0 < cx < 28.0 and abs(cy - 32) < 1e-3 and 10.5 < R < 11.5
    tiles = (keys >> np.uint64(32)).astype(int)
    seen = []
    for t, h in zip(tiles, hit):
        ty, tx = divmod(int(t), proj.tiles_x)
        nx = min(max(cx, 16 * tx), min(16 * tx + 15, 64))   # nearest point of the tile's pixel-centre box
        ny = min(max(cy, 16 * ty), min(16 * ty + 15, 64))
        # the nearest pixel CENTRE is the nearest integer point: on the axes through c it is the rounding of c
        nx, ny = (round(nx) if 16 * tx <= cx <= 16 * tx + 15 else nx), (round(ny) if 16 * ty <= cy <= 16 * ty + 15 else ny)
        d = np.hypot(nx - cx, ny - cy)
        assert abs(d - R) > 0.3                               # no borderline tile in this construction
        assert bool(h) == (d <= R), (tx, ty, d, R)
        seen.append((tx, ty, bool(h)))
    assert (0, 2, False) in seen and (1, 2, True) in seen and (2, 2, True) in seen
    assert 0 < hit.sum() < len(hit)


def test_tile_hits_equal_what_each_tile_blends_without_saturation():
    # With low opacities no pixel ever stops (T stays far above 1e-4), so within ONE tile the Gaussians the
    # compositor blends somewhere are exactly the tile's entries with a pixel at alpha >= 1/255: orc_tile_hits
    # against orc_composite (pinned on its own) restricted to one tile at a time.
    s = scenes.make_scene(2, n=3000, width=96, height=80)
    s.opacities[:] = np.minimum(s.opacities, 0.02)
    cam = s.cameras[0]
    proj, keys, vals, ranges, hit = _hits_of(s)
    ch = np.zeros((s.n, 14))
    checked = 0
    for t in range(proj.tiles_x * proj.tiles_y):
        b, e = int(ranges[t, 0]), int(ranges[t, 1])
        if e == b:
            continue
        one = np.zeros_like(ranges)
        one[t] = ranges[t]
        comp = oracle.composite(s, cam, proj, ch, vals, one)
        assert comp.gbuf[..., 15].min() > 0.05                       # nothing saturates
        blended = set(np.nonzero(comp.contrib)[0].tolist())
        assert blended == set(vals[b:e][hit[b:e]].tolist()), t
        checked += 1
    assert checked > 20 and 0 < hit.sum() < len(hit)


def test_tile_hits_zero_below_threshold_opacity():
    s = custom_scene([[0, 0, 0], [0.2, 0, 0.1]], 0.05, opacities=[1.0 / 300, 0.5], width=64, height=64)
    proj, keys, vals, ranges, hit = _hits_of(s)
    assert not hit[vals == 0].any() and hit[vals == 1].any()
