"""Pins of the oracle's projection / list building (steps 3-4) against closed forms,
an independent double evaluation, invariants and brute force.  CPU only."""
import numpy as np

import oracle
from paper_2408_12282_b200 import scenes
from util import custom_scene


def _inv2(con):
    a, b, c = con[..., 0].astype(np.float64), con[..., 1].astype(np.float64), con[..., 2].astype(np.float64)
    det = a * c - b * b
    return np.stack([c / det, -b / det, a / det], -1)


def test_isotropic_closed_form():
    # Isotropic Gaussian sigma at camera-space (x,y,z) (Eq. 2):
    # Sigma' = sigma^2 f^2 / z^2 [[1+x^2/z^2, xy/z^2],[xy/z^2, 1+y^2/z^2]] + 0.3 I.
    rng = np.random.default_rng(0)
    n = 200
    means = rng.uniform(-0.6, 0.6, size=(n, 3))
    sig = rng.uniform(0.01, 0.05, size=n)
    q = rng.standard_normal((n, 4))
    q /= np.linalg.norm(q, axis=1, keepdims=True)
    s = custom_scene(means, np.repeat(sig[:, None], 3, 1), rotations=q, width=128, height=96)
    cam = s.cameras[0]
    p = oracle.project(s, cam)
    assert p.visible.all()
    pc = s.means.astype(np.float64) @ cam.R.astype(np.float64).T + cam.t.astype(np.float64)
    x, y, z = pc[:, 0], pc[:, 1], pc[:, 2]
    k = (sig * cam.fx / z) ** 2
    ref = np.stack([k * (1 + x * x / z / z) + 0.3, k * x * y / z / z, k * (1 + y * y / z / z) + 0.3], -1)
    cov = _inv2(p.conic)
    np.testing.assert_allclose(cov, ref, rtol=2e-4, atol=1e-5)
    np.testing.assert_allclose(p.depth, z, rtol=1e-6)
    np.testing.assert_allclose(p.pix[:, 0], cam.fx * x / z + cam.cx, rtol=1e-5, atol=1e-4)
    np.testing.assert_allclose(p.pix[:, 1], cam.fy * y / z + cam.cy, rtol=1e-5, atol=1e-4)
    # radius = 3.33 sqrt(lambda_max)
    mid = 0.5 * (ref[:, 0] + ref[:, 2])
    lam = mid + np.sqrt(np.maximum(0.1, mid * mid - (ref[:, 0] * ref[:, 2] - ref[:, 1] ** 2)))
    np.testing.assert_allclose(p.radius, 3.33 * np.sqrt(lam), rtol=1e-4)


def test_on_axis_isotropic():
    # on the optical axis: (f sigma / z)^2 + 0.3 on the diagonal, 0 off it
    s = custom_scene([[0, 0, 0]], 0.03, width=65, height=65)
    cam = s.cameras[0]
    p = oracle.project(s, cam)
    cov = _inv2(p.conic)[0]
    d = (cam.fx * 0.03 / 4.0) ** 2 + 0.3
    np.testing.assert_allclose(cov, [d, 0.0, d], rtol=1e-5, atol=1e-6)
    np.testing.assert_allclose(p.pix[0], [32.0, 32.0], atol=1e-4)


def test_rotation_invariance_isotropic():
    rng = np.random.default_rng(1)
    means = rng.uniform(-0.5, 0.5, size=(50, 3))
    q = rng.standard_normal((50, 4))
    q /= np.linalg.norm(q, axis=1, keepdims=True)
    a = oracle.project(custom_scene(means, 0.04), custom_scene(means, 0.04).cameras[0])
    sb = custom_scene(means, 0.04, rotations=q)
    b = oracle.project(sb, sb.cameras[0])
    np.testing.assert_allclose(_inv2(a.conic), _inv2(b.conic), rtol=2e-5, atol=1e-6)


def test_canonical_fp32_vs_double():
    # the canonical text evaluated in fp32 agrees with a direct double evaluation of Eq. 2
    s = scenes.make_scene(2, n=5000)
    cam = s.cameras[0]
    p = oracle.project(s, cam)
    cov64, pix64, depth64 = oracle.project_f64(s, cam)
    v = p.visible.astype(bool)
    assert v.sum() > 4000
    cov = _inv2(p.conic[v])
    np.testing.assert_allclose(cov, cov64[v], rtol=5e-5, atol=1e-5)
    np.testing.assert_allclose(p.pix[v], pix64[v], rtol=1e-5, atol=2e-4)
    np.testing.assert_allclose(p.depth[v], depth64[v], rtol=1e-6)


def test_anisotropic_rotated_vs_numpy():
    # anisotropic Gaussian: Sigma = R S S^T R^T via an independent numpy construction
    rng = np.random.default_rng(2)
    n = 100
    means = rng.uniform(-0.5, 0.5, size=(n, 3))
    sc = np.exp(rng.normal(-3.5, 0.6, size=(n, 3)))
    q = rng.standard_normal((n, 4))
    q /= np.linalg.norm(q, axis=1, keepdims=True)
    s = custom_scene(means, sc, rotations=q, width=96, height=96)
    cam = s.cameras[0]
    p = oracle.project(s, cam)
    Rw = cam.R.astype(np.float64)
    for i in range(n):
        w, x, y, z = s.rotations[i].astype(np.float64)
        Rq = np.array([[1 - 2 * (y * y + z * z), 2 * (x * y - w * z), 2 * (x * z + w * y)],
                       [2 * (x * y + w * z), 1 - 2 * (x * x + z * z), 2 * (y * z - w * x)],
                       [2 * (x * z - w * y), 2 * (y * z + w * x), 1 - 2 * (x * x + y * y)]])
        Sg = Rq @ np.diag(s.scales[i].astype(np.float64) ** 2) @ Rq.T
        pc = Rw @ s.means[i].astype(np.float64) + cam.t
        J = np.array([[cam.fx / pc[2], 0, -cam.fx * pc[0] / pc[2] ** 2],
                      [0, cam.fy / pc[2], -cam.fy * pc[1] / pc[2] ** 2]])
        c2 = J @ Rw @ Sg @ Rw.T @ J.T + 0.3 * np.eye(2)
        np.testing.assert_allclose(_inv2(p.conic[i]), [c2[0, 0], c2[0, 1], c2[1, 1]], rtol=2e-4, atol=1e-5)


def test_culling_cases():
    # behind the camera, straddling z_near, far off-screen, degenerate scale (low-pass keeps det > 0)
    means = [[0, -5, 0],      # behind the camera (camera at y = -4 looking +y)
             [0, -3.85, 0],   # z = 0.15 < znear 0.2
             [0, -3.75, 0],   # z = 0.25 > znear
             [50, 0, 0],      # far off-screen
             [0, 0, 0]]       # degenerate scale
    sc = [[0.05] * 3, [0.05] * 3, [0.001] * 3, [0.05] * 3, [1e-8, 0.05, 0.05]]
    s = custom_scene(means, sc)
    p = oracle.project(s, s.cameras[0])
    assert list(p.visible) == [0, 0, 1, 0, 1]
    assert p.touched[0] == 0 and p.touched[3] == 0
    assert np.isfinite(p.conic).all()


def test_full_image_gaussian_rect_clamps():
    s = custom_scene([[0, 0, 0]], 5.0, width=50, height=37)
    p = oracle.project(s, s.cameras[0])
    assert list(p.rect[0]) == [0, 0, 4, 3] and p.touched[0] == 12


def test_rect_covers_alpha_support():
    # S3: every pixel with alpha >= 1/255 lies inside the tile rectangle (K_R = 3.33,
    # inclusive upper bound), so the image does not depend on the tile lists.
    s = scenes.make_scene(1, n=600, width=96, height=80)
    cam = s.cameras[0]
    p = oracle.project(s, cam)
    ys, xs = np.mgrid[0:cam.height, 0:cam.width]
    for g in np.nonzero(p.visible)[0]:
        dx = xs - np.float64(p.pix[g, 0])
        dy = ys - np.float64(p.pix[g, 1])
        a, b, c = p.conic[g].astype(np.float64)
        alpha = s.opacities[g] * np.exp(-0.5 * (a * dx * dx + c * dy * dy) - b * dx * dy)
        yy, xx = np.nonzero(alpha >= 1.0 / 255.0)
        if len(yy) == 0:
            continue
        x0, y0, x1, y1 = p.rect[g]
        assert (xx // 16 >= x0).all() and (xx // 16 < x1).all()
        assert (yy // 16 >= y0).all() and (yy // 16 < y1).all()


def test_lists_sorted_and_ranges_partition():
    s = scenes.make_scene(1, width=100, height=70)
    cam = s.cameras[0]
    p = oracle.project(s, cam)
    keys, vals, ranges = oracle.build_lists(p)
    I = int(p.touched.sum())
    assert keys.shape[0] == I and vals.shape[0] == I
    assert (np.diff(keys.astype(np.uint64)) >= 0).all() if I > 1 else True
    # ranges partition [0, I) in tile order
    assert ranges[0, 0] == 0 and ranges[-1, 1] == I
    assert (ranges[1:, 0] == ranges[:-1, 1]).all()
    tiles = (keys >> np.uint64(32)).astype(np.int64)
    for t in range(ranges.shape[0]):
        b, e = ranges[t]
        assert (tiles[b:e] == t).all()
    # per tile: depth ascending, index ascending among equal depths; values match rects
    dbits = (keys & np.uint64(0xFFFFFFFF)).astype(np.uint32)
    assert (dbits == p.depth.view(np.uint32)[vals]).all()
    cnt = np.bincount(vals, minlength=s.n)
    assert (cnt == p.touched).all()
    tx = tiles % p.tiles_x
    ty = tiles // p.tiles_x
    r = p.rect[vals]
    assert ((tx >= r[:, 0]) & (tx < r[:, 2]) & (ty >= r[:, 1]) & (ty < r[:, 3])).all()


def test_equal_depth_tie_break_by_index():
    # many Gaussians at IDENTICAL depth: order within a tile must be ascending index
    n = 40
    means = np.zeros((n, 3), np.float32)
    means[:, 0] = np.linspace(-0.05, 0.05, n)  # same camera-space z (camera looks along +y)
    s = custom_scene(means, 0.03, width=32, height=32)
    p = oracle.project(s, s.cameras[0])
    assert len(set(p.depth.view(np.uint32))) == 1
    keys, vals, ranges = oracle.build_lists(p)
    for t in range(ranges.shape[0]):
        b, e = ranges[t]
        assert (np.diff(vals[b:e].astype(np.int64)) > 0).all()


def test_permutation_gives_same_key_multiset():
    s = scenes.make_scene(1, n=500, width=64, height=64)
    perm = np.random.default_rng(3).permutation(s.n)
    s2 = scenes.subset(s, perm)
    p1 = oracle.project(s, s.cameras[0])
    p2 = oracle.project(s2, s2.cameras[0])
    k1, v1, _ = oracle.build_lists(p1)
    k2, v2, _ = oracle.build_lists(p2)
    assert (np.sort(k1) == np.sort(k2)).all()
    if len(set(p1.depth[p1.visible.astype(bool)])) == p1.visible.sum():
        assert (perm[v2] == v1).all()


def test_empty_scene():
    s = custom_scene(np.zeros((0, 3)), 0.05)
    p = oracle.project(s, s.cameras[0])
    keys, vals, ranges = oracle.build_lists(p)
    assert keys.shape[0] == 0 and (ranges == 0).all()
