"""Pins of the oracle's "w/o deferred" variant (oracle.shade_gaussians / forward_frame, PAPER.md L283
Tab. 2): the per-Gaussian evaluation of Eq. 7 written in numpy must agree with the (separately
pinned) C++ pixel shader on one-pixel G-buffers, and with closed forms."""
import dataclasses

import numpy as np

import oracle
from paper_2408_12282_b200 import scenes
from util import custom_scene


def _one_pixel_reference(scene, cam, light, mlp_out, i):
    """Shade Gaussian i with the C++ pixel shader: a 1x1 image whose pixel back-projects to mu_i and
    whose G-buffer holds the Gaussian's own attributes at coverage 1."""
    R = np.asarray(cam.R, np.float64).reshape(3, 3)
    pc = R @ scene.means[i].astype(np.float64) + np.asarray(cam.t, np.float64)
    c1 = dataclasses.replace(cam, width=1, height=1, cx=float(-cam.fx * pc[0] / pc[2]),
                             cy=float(-cam.fy * pc[1] / pc[2]), bg=np.zeros(3, np.float32))
    g = np.zeros((1, 1, 16))
    g[0, 0, 0] = pc[2]
    g[0, 0, 1:4] = scene.normals[i]
    g[0, 0, 4:7] = scene.base_color[i]
    g[0, 0, 7], g[0, 0, 8], g[0, 0, 9] = scene.roughness[i], scene.metallic[i], scene.subsurface[i]
    g[0, 0, 10:14] = mlp_out[i]
    g[0, 0, 14], g[0, 0, 15] = 1.0, 0.0
    return oracle.shade(c1, light, g)[0][0, 0]


def test_per_gaussian_shading_equals_pixel_shader_on_one_pixel_gbuffers():
    scene = scenes.make_scene(1, n=400, width=64, height=64)
    cam = scene.cameras[0]
    light = dataclasses.replace(scene.lights[0][0], intensity=np.float32([0.7, 1.1, 0.4]))
    rng = np.random.default_rng(3)
    mlp_out = np.concatenate([rng.uniform(0, 1, (scene.n, 3)), rng.uniform(0, 3, (scene.n, 1))], axis=1)
    got = oracle.shade_gaussians(scene, cam, light, mlp_out)
    for i in range(0, scene.n, 7):
        ref = _one_pixel_reference(scene, cam, light, mlp_out, i)
        # cx, cy of the one-pixel camera pass through fp32, so the back-projected point is mu_i to ~1e-7
        np.testing.assert_allclose(got[i], ref, rtol=2e-5, atol=1e-7)


def test_closed_forms():
    n = 5
    means = np.zeros((n, 3), np.float32)
    s = custom_scene(means, 0.05, normals=(0, -1, 0), base_color=(0.2, 0.5, 0.8), roughness=1.0, metallic=0.0,
                     subsurface=0.0, eye=(0, -4, 0), lights=((0, -3, 0),))
    cam, light = s.cameras[0], s.lights[0][0]
    mo = np.tile(np.float64([0.3, 0.6, 0.9, 2.0]), (n, 1))
    # n = l = v: r = 1, m = 0 -> D = 1/pi, k = 1/2, V = 1/((1+1)(1+1)) = 1/4, F = F0 = 0.04 (vh = 1)
    c = oracle.shade_gaussians(s, cam, light, mo)
    want = (0.04 / np.pi / 4.0 + np.float64(s.base_color[0]) / np.pi) * 2.0 * 1.0
    np.testing.assert_allclose(c[0], want, rtol=1e-12)
    # sss = 1 -> c = intensity * L_SSS whatever the BRDF
    s1 = dataclasses.replace(s, subsurface=np.ones(n, np.float32))
    l2 = dataclasses.replace(light, intensity=np.float32([2.0, 0.5, 1.0]))
    np.testing.assert_allclose(oracle.shade_gaussians(s1, cam, l2, mo)[0], np.float64([0.6, 0.3, 0.9]), rtol=1e-12)
    # light behind the surface (n . w_in <= 0) and sss = 0 -> black
    s2 = custom_scene(means, 0.05, normals=(0, 1, 0), subsurface=0.0, eye=(0, -4, 0), lights=((0, -3, 0),))
    assert np.abs(oracle.shade_gaussians(s2, s2.cameras[0], s2.lights[0][0], mo)).max() == 0.0


def test_forward_frame_of_one_gaussian():
    # a single Gaussian on a pixel centre: C(centre) = o c + (1 - o) bg  (Eq. 3 with one term)
    s = custom_scene([[0, 0, 0]], 0.05, opacities=0.6, width=65, height=65, bg=(0.1, 0.2, 0.3), subsurface=1.0)
    mo = np.float64([[0.2, 0.4, 0.8, 1.0]])
    r = oracle.forward_frame(s, mlp_out=mo)
    np.testing.assert_allclose(r.rgb[32, 32], 0.6 * mo[0, :3] + 0.4 * np.float64([0.1, 0.2, 0.3]), rtol=1e-6)
    assert np.allclose(r.rgb[0, 0], [0.1, 0.2, 0.3])


# ---- oracle.relight: the reflectance-field sum of PAPER.md L301 ----------------------------------------------------
def test_relight_one_hot_and_brute_force():
    rng = np.random.default_rng(4)
    L, H, W = 5, 3, 7
    frames = rng.uniform(0.0, 2.0, (L, H, W, 3))
    w = rng.uniform(0.0, 3.0, (L, 3))
    for l in range(L):       # a single white light of the field switched on: that frame, exactly
        e = np.zeros((L, 3))
        e[l] = 1.0
        np.testing.assert_array_equal(oracle.relight(frames, e), frames[l])
    e = np.zeros((L, 3))
    e[2, 1] = 0.5            # only the green channel of light 2
    want = np.zeros((H, W, 3))
    want[..., 1] = 0.5 * frames[2, ..., 1]
    np.testing.assert_array_equal(oracle.relight(frames, e), want)
    got = oracle.relight(frames, w)
    for y in range(H):       # brute force, element by element
        for x in range(W):
            for c in range(3):
                s = 0.0
                for l in range(L):
                    s += w[l, c] * frames[l, y, x, c]
                assert abs(got[y, x, c] - s) <= 1e-14 * max(1.0, abs(s))
    assert oracle.relight(np.zeros((0, H, W, 3)), np.zeros((0, 3))).shape == (H, W, 3)


def test_relight_equals_shading_under_coloured_lights():
    # Eq. 7 (L104-106) is linear in the light's RGB intensity (S16) and a point-light sum is a sum of frames
    # (L301, App. D): on a black background, relighting the white-light OLAT frames with weights w_l equals the sum of
    # the frames shaded under lights of intensity w_l -- a statement about the separately pinned shader.
    import dataclasses
    s = scenes.make_scene(3, n=300, width=24, height=20, lights=4)
    cam = s.cameras[0]
    assert not np.any(cam.bg)
    r0 = oracle.render_frame(s, 0, 0)
    rng = np.random.default_rng(9)
    w = rng.uniform(0.1, 2.0, (4, 3))
    white, coloured = [], np.zeros((cam.height, cam.width, 3))
    for l, lt in enumerate(s.lights[0]):
        r = oracle.render_frame(s, 0, l, geometry=r0)
        assert np.all(lt.intensity == 1.0)
        white.append(r.rgb)
        lc = dataclasses.replace(lt, intensity=w[l].astype(np.float32))
        coloured += oracle.shade(cam, lc, r.comp.gbuf)[0]
    got = oracle.relight(np.stack(white), w.astype(np.float32))
    assert np.abs(coloured).max() > 1e-2
    np.testing.assert_allclose(got, coloured, rtol=1e-12, atol=1e-15)
