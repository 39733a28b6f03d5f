"""Pins of the oracle's deferred shading (step 6; Eq. 4, Eq. 7
L104-106, AOVs L320) against closed forms and BRDF invariants.  CPU only."""
import numpy as np

import oracle
from paper_2408_12282_b200 import scenes


def _unit(v):
    v = np.asarray(v, np.float64)
    return v / np.linalg.norm(v)


def shade_point(n, l_dir, v_dir, base=(0.5, 0.5, 0.5), rough=0.5, metal=0.0, sss=0.0,
                lsss=(0.0, 0.0, 0.0), lin=1.0, A=1.0, intensity=(1, 1, 1), bg=(0, 0, 0), f32=False,
                n_scale=1.0):
    """Shade ONE pixel whose back-projection is the world origin, with unit light / view
    directions l_dir, v_dir (from the surface point) and normal n."""
    l_dir, v_dir, n = _unit(l_dir), _unit(v_dir), _unit(n)
    up = (0, 0, 1) if abs(v_dir[2]) < 0.9 else (1, 0, 0)
    cam = scenes.look_at_camera(4.0 * v_dir, 1, 1, 40.0, up=up, bg=bg)
    light = scenes.Light((3.0 * l_dir).astype(np.float32), np.asarray(intensity, np.float32))
    g = np.zeros((1, 1, 16))
    g[0, 0, 0] = 4.0
    g[0, 0, 1:4] = n * n_scale
    g[0, 0, 4:7] = base
    g[0, 0, 7], g[0, 0, 8], g[0, 0, 9] = rough, metal, sss
    g[0, 0, 10:13] = lsss
    g[0, 0, 13] = lin
    g[0, 0, :14] *= A
    g[0, 0, 14], g[0, 0, 15] = A, 1 - A
    rgb, ad, asp = oracle.shade(cam, light, g, f32=f32)
    return rgb[0, 0].astype(np.float64), ad[0, 0].astype(np.float64), asp[0, 0].astype(np.float64)


def test_sss_one_gives_residual_only():
    rgb, ad, asp = shade_point((0, 0, 1), (0.3, 0.2, 1), (-0.4, 0.1, 1), sss=1.0, lsss=(0.2, 0.5, 0.9), A=0.6)
    np.testing.assert_allclose(rgb, 0.6 * np.array([0.2, 0.5, 0.9]), atol=1e-7)
    assert (ad == 0).all() and (asp == 0).all()


def test_lambertian_closed_form():
    # sss=0, m=0, r=1: alpha_r = 1 -> D = 1/pi, k = 1/2, V = 1/((1+nl)(1+nv)), F0 = 0.04:
    # rgb = [ b/pi + F/(pi (1+nl)(1+nv)) ] L_in nl;  diffuse AOV x b = Lambert b/pi L_in nl
    n = _unit((0.1, -0.2, 1))
    l = _unit((0.5, 0.3, 1.0))
    v = _unit((-0.3, 0.6, 0.8))
    b = np.array([0.8, 0.4, 0.1])
    lin = 1.7
    rgb, ad, asp = shade_point(n, l, v, base=b, rough=1.0, metal=0.0, lin=lin)
    nl, nv = n @ l, n @ v
    h = _unit(l + v)
    F = 0.04 + 0.96 * (1 - v @ h) ** 5
    lambert = b / np.pi * lin * nl
    spec = F / (np.pi * (1 + nl) * (1 + nv)) * lin * nl
    np.testing.assert_allclose(ad * b, lambert, rtol=1e-6)
    np.testing.assert_allclose(asp, np.full(3, spec), rtol=1e-6)
    np.testing.assert_allclose(rgb, lambert + spec, rtol=1e-6)
    np.testing.assert_allclose(rgb - asp, lambert, rtol=1e-6)


def test_mirror_configuration_peak():
    # n = l = v: nh = 1 -> D = 1/(pi alpha_r^2), F = F0 (vh = 1), nl = nv = 1 -> V = 1/4
    for r in (0.3, 0.7):
        for m, b in ((0.0, 0.5), (1.0, 0.9)):
            rgb, ad, asp = shade_point((0, 0, 1), (0, 0, 1), (0, 0, 1), base=(b, b, b), rough=r, metal=m, lin=1.0)
            a = r * r
            F0 = 0.04 * (1 - m) + b * m
            np.testing.assert_allclose(asp, np.full(3, F0 / (np.pi * a * a) / 4), rtol=2e-5)
            np.testing.assert_allclose(rgb, asp + (1 - m) * b / np.pi, rtol=2e-5)


def test_fresnel_grazing_goes_to_one():
    # l = -v mirrored about n at grazing angle: vh -> 0, F -> 1 for any F0
    th = np.radians(89.9)
    l = (np.sin(th), 0, np.cos(th))
    v = (-np.sin(th), 0, np.cos(th))
    a = shade_point((0, 0, 1), l, v, base=(0.2, 0.2, 0.2), rough=0.6, metal=0.0)[2]
    b = shade_point((0, 0, 1), l, v, base=(0.2, 0.2, 0.2), rough=0.6, metal=1.0)[2]
    np.testing.assert_allclose(a, b, rtol=1e-2)  # F0 = 0.04 vs 0.2 no longer matters


def test_brdf_reciprocity():
    rng = np.random.default_rng(0)
    for _ in range(20):
        n = _unit(rng.standard_normal(3))
        l = _unit(n + 0.8 * rng.standard_normal(3))
        v = _unit(n + 0.8 * rng.standard_normal(3))
        if n @ l < 0.05 or n @ v < 0.05:
            continue
        kw = dict(base=(0.7, 0.5, 0.3), rough=float(rng.uniform(0.2, 0.9)), metal=float(rng.uniform()))
        r1 = shade_point(n, l, v, **kw)[0] / (n @ l)
        r2 = shade_point(n, v, l, **kw)[0] / (n @ v)
        np.testing.assert_allclose(r1, r2, rtol=1e-5)


def test_ggx_normalisation_integral():
    # int_hemisphere D(h) (n.h) dw_h = 1.  With l = v = h: spec = D F V L_in nh, F = 1 (m=1,b=1),
    # V = 1/(4 (nh(1-k)+k)^2)  ->  D = spec / (V nh)
    for r in (0.4, 0.8):
        a = r * r
        k = a / 2
        th = (np.arange(400) + 0.5) / 400 * (np.pi / 2)
        total = 0.0
        for t in th:
            h = (np.sin(t), 0.0, np.cos(t))
            spec = shade_point((0, 0, 1), h, h, base=(1, 1, 1), rough=r, metal=1.0)[2][0]
            nh = np.cos(t)
            V = 1 / (4 * (nh * (1 - k) + k) ** 2)
            D = spec / (V * nh)
            total += D * nh * np.sin(t) * 2 * np.pi * (np.pi / 2 / 400)
        assert abs(total - 1) < 2e-3


def test_white_furnace_albedo_below_one():
    # directional albedo of the specular lobe (F = 1) under uniform incoming light stays <= 1
    rng = np.random.default_rng(1)
    v = _unit((0.3, 0.0, 1.0))
    for r in (0.3, 0.6, 1.0):
        d = rng.standard_normal((1500, 3))
        d /= np.linalg.norm(d, axis=1, keepdims=True)
        d[:, 2] = np.abs(d[:, 2])
        acc = 0.0
        for l in d:
            acc += shade_point((0, 0, 1), l, v, base=(1, 1, 1), rough=r, metal=1.0)[2][0]  # f_spec * nl
        albedo = acc / len(d) * 2 * np.pi
        assert albedo <= 1.02


def test_coverage_background_and_intensity():
    bg = (0.2, 0.3, 0.4)
    rgb_full = shade_point((0, 0, 1), (0, 0.3, 1), (0.2, 0, 1), A=1.0, bg=bg)[0]
    rgb_half = shade_point((0, 0, 1), (0, 0.3, 1), (0.2, 0, 1), A=0.5, bg=bg)[0]
    np.testing.assert_allclose(rgb_half, 0.5 * rgb_full + 0.5 * np.array(bg), rtol=1e-6)
    rgb_none = shade_point((0, 0, 1), (0, 0.3, 1), (0.2, 0, 1), A=0.0, bg=bg)[0]
    np.testing.assert_allclose(rgb_none, np.float32(bg), atol=1e-7)
    tint = shade_point((0, 0, 1), (0, 0.3, 1), (0.2, 0, 1), intensity=(2.0, 0.5, 0.0))[0]
    np.testing.assert_allclose(tint, rgb_full * [2.0, 0.5, 0.0], rtol=1e-6)


def test_normal_is_renormalised_and_backfacing_light():
    a = shade_point((0, 0, 1), (0.3, 0, 1), (0, 0.2, 1), n_scale=1.0)[0]
    b = shade_point((0, 0, 1), (0.3, 0, 1), (0, 0.2, 1), n_scale=0.37)[0]
    np.testing.assert_allclose(a, b, rtol=1e-6)
    # light below the surface: nl = 0 -> only the SSS residual survives
    c = shade_point((0, 0, 1), (0.3, 0, -1), (0, 0.2, 1), sss=0.25, lsss=(0.4, 0.4, 0.4))[0]
    np.testing.assert_allclose(c, 0.25 * 0.4 * np.ones(3), atol=1e-7)


def test_fp32_shading_tracks_double():
    rng = np.random.default_rng(2)
    for _ in range(50):
        n = _unit(rng.standard_normal(3))
        l = _unit(n + rng.standard_normal(3))
        v = _unit(n + rng.standard_normal(3))
        kw = dict(base=tuple(rng.uniform(size=3)), rough=float(rng.uniform(0.3, 1)), metal=float(rng.uniform()),
                  sss=float(rng.uniform()), lsss=tuple(rng.uniform(size=3)), lin=float(rng.uniform(0, 3)))
        a = shade_point(n, l, v, **kw)[0]
        b = shade_point(n, l, v, f32=True, **kw)[0]
        np.testing.assert_allclose(a, b, rtol=2e-4, atol=2e-5)


# ---- the pixel -> world back-projection ("The image space surface position is projected back to
# the 3D space") at a pixel that is NOT the image centre.  Every pin above shades a 1x1 image (px = py = 0), where
# the pixel term ((px - cx) / fx) z of the back-projection is a constant; here it is pinned against a world point
# built from the camera's basis vectors alone. -----------------------------------------------------------------
def _off_centre_setup():
    from paper_2408_12282_b200.scenes import Camera, Light
    W, H = 64, 48
    eye = np.array([0.7, -3.1, 0.4])
    f = _unit(np.array([0.1, 0.3, -0.2]) - eye)             # forward (+z of the camera)
    r = _unit(np.cross(f, (0.0, 0.0, 1.0)))                 # right   (+x)
    d = np.cross(f, r)                                      # down    (+y)
    R = np.stack([r, d, f]).astype(np.float32)              # p_c = R p + t   (include/sssgs.h, sssgs_camera)
    t = (-(R.astype(np.float64) @ eye)).astype(np.float32)
    # anisotropic focal lengths and a principal point off the image centre: fx/fy, cx/cy mix-ups change the answer
    cam = Camera(R=R, t=t, fx=61.0, fy=47.0, cx=29.25, cy=25.5, tan_half_fovx=W / 2 / 61.0, tan_half_fovy=H / 2 / 47.0,
                 width=W, height=H, znear=0.2, bg=np.array([0.05, 0.1, 0.2], np.float32), position=eye.astype(np.float32))
    light = Light(np.array([0.9, -1.2, 1.1], np.float32), np.array([1.0, 0.8, 0.6], np.float32))  # close: directions vary over the image
    return cam, light, (r, d, f), eye


def _world_point(cam, basis, eye, px, py, z):
    """The point whose camera coordinates are (a z, b z, z), written with the basis vectors -- no R^T, no t."""
    r, d, f = basis
    # the camera the shader sees holds float32 R and t: use the same rounded basis / eye so that the comparison
    # is at rounding level (the convention, not the rounding, is what is pinned)
    Rm = cam.R.astype(np.float64)
    r, d, f = Rm[0], Rm[1], Rm[2]
    eye = -(Rm.T @ cam.t.astype(np.float64))
    a, b = (px - cam.cx) / cam.fx, (py - cam.cy) / cam.fy
    return eye + z * (f + a * r + b * d), eye


def _lambert_at(cam, light, basis, eye, px, py, z, n, b, lin, A=1.0):
    """Closed form of test_lambertian_closed_form (sss = 0, m = 0, r = 1) at the world point of pixel (px, py)."""
    X, eye = _world_point(cam, basis, eye, px, py, z)
    l = _unit(light.position.astype(np.float64) - X)
    v = _unit(eye - X)
    nl, nv = max(0.0, n @ l), max(1e-4, n @ v)
    h = _unit(l + v)
    F = 0.04 + 0.96 * (1 - v @ h) ** 5
    # alpha_r = 1: D = 1 / (pi (nh^2 + |n x h|^2)^2) = 1 / pi, except where the viewer is behind the surface and
    # n.h < 0 is clamped to 0 (then only |n x h|^2 = 1 - (n.h)^2 is left)
    nh = n @ h
    D = 1.0 / (np.pi * (max(0.0, nh) ** 2 + 1.0 - nh * nh) ** 2)
    lout = (b / np.pi + D * F / ((1 + nl) * (1 + nv))) * lin * nl
    return light.intensity.astype(np.float64) * A * lout + (1 - A) * cam.bg.astype(np.float64)


def _gbuf_with_pixel(cam, px, py, z, n, b, lin, A=1.0):
    g = np.zeros((cam.height, cam.width, 16))
    g[..., 15] = 1.0
    q = np.zeros(16)
    q[0], q[1:4], q[4:7], q[7], q[8], q[9], q[13] = z, n, b, 1.0, 0.0, 0.0, lin
    q[:14] *= A
    q[14], q[15] = A, 1 - A
    g[py, px] = q
    return g


def test_back_projection_off_centre_pixel():
    cam, light, basis, eye = _off_centre_setup()
    px, py, z = 41, 17, 3.3
    n = _unit((0.3, -0.8, 0.4))
    b = np.array([0.8, 0.4, 0.1])
    g = _gbuf_with_pixel(cam, px, py, z, n, b, 1.7, A=0.8)
    rgb = oracle.shade(cam, light, g)[0]
    want = _lambert_at(cam, light, basis, eye, px, py, z, n, b, 1.7, A=0.8)
    np.testing.assert_allclose(rgb[py, px], want, rtol=1e-9)
    # every other pixel is background
    mask = np.ones((cam.height, cam.width), bool)
    mask[py, px] = False
    np.testing.assert_allclose(rgb[mask], np.broadcast_to(cam.bg.astype(np.float64), (mask.sum(), 3)), atol=0)
    # the pin has teeth: each plausible slip of the pixel term moves the closed form far beyond the tolerance
    X, e = _world_point(cam, basis, eye, px, py, z)
    slips = {
        "px <-> py": _lambert_at(cam, light, basis, eye, py, px, z, n, b, 1.7, A=0.8),
        "x sign": _lambert_at(cam, light, basis, eye, 2 * cam.cx - px, py, z, n, b, 1.7, A=0.8),
        "y sign": _lambert_at(cam, light, basis, eye, px, 2 * cam.cy - py, z, n, b, 1.7, A=0.8),
        "no pixel term": _lambert_at(cam, light, basis, eye, cam.cx, cam.cy, z, n, b, 1.7, A=0.8),
        "fx <-> fy": _lambert_at(cam, light, basis, eye, cam.cx + (px - cam.cx) * cam.fx / cam.fy,
                                 cam.cy + (py - cam.cy) * cam.fy / cam.fx, z, n, b, 1.7, A=0.8),
        "cx <-> cy": _lambert_at(cam, light, basis, eye, px + cam.cx - cam.cy, py + cam.cy - cam.cx, z, n, b, 1.7, A=0.8),
        "pixel term not scaled by z": _lambert_at(cam, light, basis, eye, cam.cx + (px - cam.cx) / z,
                                                  cam.cy + (py - cam.cy) / z, z, n, b, 1.7, A=0.8),
    }
    for name, val in slips.items():
        assert np.abs(val - want).max() > 1e-3 * np.abs(want).max(), name
    # the fp32 evaluation of the same text (the calibration arm of S9) follows
    np.testing.assert_allclose(oracle.shade(cam, light, g, f32=True)[0][py, px], want, rtol=2e-5)


def test_back_projection_inverts_the_projection():
    # the world point of pixel (px, py) at depth z, pushed through the (separately pinned) EWA projection of
    # step 3, lands on (px, py) with depth z: the two halves of the path use one pixel convention
    cam, light, basis, eye = _off_centre_setup()
    pts = [(41, 17, 3.3), (5, 40, 2.1), (60, 3, 4.0)]
    X = np.stack([_world_point(cam, basis, eye, px, py, z)[0] for px, py, z in pts])
    from types import SimpleNamespace
    sc = SimpleNamespace(n=len(pts), means=X.astype(np.float32), scales=np.full((len(pts), 3), 0.05, np.float32),
                         rotations=np.tile(np.array([1, 0, 0, 0], np.float32), (len(pts), 1)))
    proj = oracle.project(sc, cam)
    assert proj.visible.all()
    for k, (px, py, z) in enumerate(pts):
        np.testing.assert_allclose(proj.pix[k], (px, py), atol=2e-4)
        np.testing.assert_allclose(proj.depth[k], z, rtol=1e-6)


def test_shading_every_pixel_of_a_frame_against_the_closed_form():
    # all pixels of a 64 x 48 frame at varying depth / normal: no pixel-dependent term escapes
    cam, light, basis, eye = _off_centre_setup()
    rng = np.random.default_rng(3)
    H, W = cam.height, cam.width
    g = np.zeros((H, W, 16))
    want = np.zeros((H, W, 3))
    b = np.array([0.6, 0.5, 0.3])
    for py in range(H):
        for px in range(W):
            z = 2.0 + 2.0 * rng.random()
            n = _unit(rng.standard_normal(3))
            g[py, px] = _gbuf_with_pixel(cam, px, py, z, n, b, 1.0)[py, px]
            want[py, px] = _lambert_at(cam, light, basis, eye, px, py, z, n, b, 1.0)
    rgb = oracle.shade(cam, light, g)[0]
    np.testing.assert_allclose(rgb, want, rtol=1e-8, atol=1e-12)
