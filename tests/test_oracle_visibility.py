"""Pins of oracle.bake_visibility (ray-traced per-Gaussian visibility + SH fit, PAPER.md L110-112,
reading in DESIGN.md section 7d) against closed forms, an independent numpy restatement that uses
scipy's quaternion convention and a different formula for the ray-Gaussian distance, a dense search
over the ray parameter, invariances and a physical half-space case."""
from types import SimpleNamespace

import numpy as np
from scipy.spatial.transform import Rotation

import oracle

Y00, Y1 = 0.2820948, 0.4886025


def _scene(means, scales, rotations, opacities):
    means = np.asarray(means, np.float32).reshape(-1, 3)
    n = len(means)
    return SimpleNamespace(n=n, means=means, scales=np.asarray(scales, np.float32).reshape(n, 3),
                           rotations=np.asarray(rotations, np.float32).reshape(n, 4),
                           opacities=np.asarray(opacities, np.float32).reshape(n))


def _fib(K):
    k = np.arange(K) + 0.5
    z = 1 - 2 * k / K
    phi = k * np.pi * (3 - np.sqrt(5))
    r = np.sqrt(1 - z * z)
    return np.stack([r * np.cos(phi), r * np.sin(phi), z], 1).astype(np.float32), np.full(K, 4 * np.pi / K, np.float32)


IDQ = [1, 0, 0, 0]


def test_single_isotropic_occluder_closed_form():
    # occluder of std sigma at distance 2 along +x, offset b sideways: m2 = b^2 / sigma^2 at the closest point
    sigma, o = 0.1, 0.8
    for b in (0.0, 0.05, 0.13, 0.25):
        sc = _scene([[0, 0, 0], [2, b, 0]], [[1e-3] * 3, [sigma] * 3], [IDQ, IDQ], [0.0, o])
        sh, vis, _ = oracle.bake_visibility(sc, [[1, 0, 0], [-1, 0, 0]], [1, 1], t_min=0.01)
        a = o * np.exp(-0.5 * b * b / sigma**2)
        want = 1 - a if a >= 1 / 255 else 1.0
        assert abs(vis[0, 0] - want) < 1e-6   # inputs are fp32
        # looking away: the closest point of the ray is its start, 2 units from the occluder: nothing
        assert vis[0, 1] == 1.0
        # the occluder's own rays see the (transparent) first Gaussian only
        assert vis[1, 0] == 1.0 and vis[1, 1] == 1.0


def test_ray_start_offset_clamps_the_closest_point():
    # occluder centred between mu_i and the ray start: the minimiser t* < 0 is clamped to the start
    sigma, o, t_min = 0.2, 0.9, 0.3
    sc = _scene([[0, 0, 0], [0.1, 0, 0]], [[1e-3] * 3, [sigma] * 3], [IDQ, IDQ], [0.0, o])
    _, vis, _ = oracle.bake_visibility(sc, [[1, 0, 0]], [1], t_min=t_min)
    d = t_min - 0.1
    assert abs(vis[0, 0] - (1 - o * np.exp(-0.5 * d * d / sigma**2))) < 1e-6


def test_cap_threshold_product_and_floor():
    sig = 0.05
    # three occluders on the ray: a capped one (o = 1 -> 0.99), a thin one, one below 1/255 (ignored)
    sc = _scene([[0, 0, 0], [1, 0, 0], [2, 0, 0], [3, 0, 0]], [[1e-3] * 3] + [[sig] * 3] * 3, [IDQ] * 4,
                [0.0, 1.0, 0.3, 0.003])
    _, vis, _ = oracle.bake_visibility(sc, [[1, 0, 0]], [1], t_min=0.01)
    assert abs(vis[0, 0] - (1 - 0.99) * (1 - 0.3)) < 1e-7
    # three capped occluders: 1e-6 < 1e-4 -> exactly 0
    sc = _scene([[0, 0, 0], [1, 0, 0], [2, 0, 0], [3, 0, 0]], [[1e-3] * 3] + [[sig] * 3] * 3, [IDQ] * 4,
                [0.0, 1.0, 1.0, 1.0])
    _, vis, _ = oracle.bake_visibility(sc, [[1, 0, 0]], [1], t_min=0.01)
    assert vis[0, 0] == 0.0


def _numpy_vis(sc, dirs, t_min):
    """Independent restatement: whitened cross-product form of the line-point Mahalanobis distance,
    rotation matrices from scipy (quaternion given as x, y, z, w there)."""
    n, K = sc.n, len(dirs)
    q = sc.rotations.astype(np.float64)
    R = Rotation.from_quat(np.stack([q[:, 1], q[:, 2], q[:, 3], q[:, 0]], 1)).as_matrix()  # [n,3,3]
    out = np.ones((n, K))
    for i in range(n):
        for k in range(K):
            w = dirs[k].astype(np.float64)
            o = sc.means[i].astype(np.float64) + np.float64(np.float32(t_min)) * w
            T = 1.0
            for j in range(n):
                if j == i:
                    continue
                Minv = (R[j] / sc.scales[j].astype(np.float64)[None, :]).T   # S^-1 R^T
                dp, wp = Minv @ (o - sc.means[j].astype(np.float64)), Minv @ w
                t = -(dp @ wp) / (wp @ wp)
                if t >= 0:
                    m2 = np.sum(np.cross(dp, wp) ** 2) / (wp @ wp)
                else:
                    m2 = dp @ dp
                a = float(sc.opacities[j]) * np.exp(-0.5 * m2)
                if a >= 1 / 255:
                    T *= 1 - min(a, 0.99)
            out[i, k] = T if T >= 1e-4 else 0.0
    return out


def _random_scene(rng, n, spread=1.0, scale=0.15):
    q = rng.normal(size=(n, 4))
    q /= np.linalg.norm(q, axis=1, keepdims=True)
    return _scene(rng.normal(size=(n, 3)) * spread, np.exp(rng.normal(np.log(scale), 0.5, size=(n, 3))), q,
                  rng.uniform(0.05, 1.0, size=n))


def test_matches_independent_numpy_restatement():
    rng = np.random.default_rng(5)
    sc = _random_scene(rng, 40)
    dirs, wts = _fib(12)
    _, vis, unstable = oracle.bake_visibility(sc, dirs, wts, t_min=0.05)
    ref = _numpy_vis(sc, dirs, 0.05)
    ok = unstable == 0
    assert ok.mean() > 0.95
    np.testing.assert_allclose(vis[ok], ref[ok], rtol=2e-6, atol=1e-9)   # scipy renormalises the fp32 quaternions
    assert (vis < 1).mean() > 0.3   # the case is not trivial


def test_minimum_over_the_ray_by_dense_search():
    rng = np.random.default_rng(6)
    sc = _random_scene(rng, 2, spread=0.8, scale=0.3)
    sc.opacities[:] = [0.0, 0.7]
    dirs, wts = _fib(16)
    t_min = 0.02
    _, vis, _ = oracle.bake_visibility(sc, dirs, wts, t_min=t_min)
    q = sc.rotations[1].astype(np.float64)
    R = Rotation.from_quat([q[1], q[2], q[3], q[0]]).as_matrix()
    Sinv = R @ np.diag(1.0 / sc.scales[1].astype(np.float64) ** 2) @ R.T
    t = np.linspace(0, 12, 240001)
    for k in range(16):
        w = dirs[k].astype(np.float64)
        x = sc.means[0].astype(np.float64) + (np.float64(np.float32(t_min)) + t)[:, None] * w - sc.means[1].astype(np.float64)
        m2 = np.einsum("ta,ab,tb->t", x, Sinv, x).min()
        a = 0.7 * np.exp(-0.5 * m2)
        want = 1 - a if a >= 1 / 255 else 1.0
        assert abs(vis[0, k] - want) < 1e-6


def test_rigid_motion_and_permutation_invariance():
    rng = np.random.default_rng(7)
    sc = _random_scene(rng, 30)
    dirs, wts = _fib(10)
    _, vis, unstable = oracle.bake_visibility(sc, dirs, wts, t_min=0.05)
    G = Rotation.from_rotvec([0.3, -0.8, 0.5])
    q = sc.rotations.astype(np.float64)
    q2 = (G * Rotation.from_quat(np.stack([q[:, 1], q[:, 2], q[:, 3], q[:, 0]], 1))).as_quat()
    sc2 = _scene(G.apply(sc.means.astype(np.float64)) + [0.4, -1.0, 2.0], sc.scales,
                 np.stack([q2[:, 3], q2[:, 0], q2[:, 1], q2[:, 2]], 1), sc.opacities)
    _, vis2, unstable2 = oracle.bake_visibility(sc2, G.apply(dirs.astype(np.float64)), wts, t_min=0.05)
    ok = (unstable == 0) & (unstable2 == 0)
    np.testing.assert_allclose(vis2[ok], vis[ok], atol=2e-5)   # inputs are rounded to fp32 after the motion
    perm = rng.permutation(30)
    sc3 = _scene(sc.means[perm], sc.scales[perm], sc.rotations[perm], sc.opacities[perm])
    sh3, vis3, _ = oracle.bake_visibility(sc3, dirs, wts, t_min=0.05)
    np.testing.assert_allclose(vis3, vis[perm], rtol=1e-12, atol=1e-15)


def test_sh_projection_of_full_and_half_space_visibility():
    dirs, wts = _fib(4000)
    # nothing occludes: V = 1, c0 = 4 pi Y00 = sqrt(4 pi), the degree-1 coefficients vanish
    sc = _scene([[0, 0, 0], [5, 5, 5]], [[0.01] * 3] * 2, [IDQ] * 2, [0.5, 0.0])
    sh, vis, _ = oracle.bake_visibility(sc, dirs, wts, t_min=0.05)
    assert np.all(vis[0] == 1.0)
    assert abs(sh[0, 0] - np.sqrt(4 * np.pi)) < 1e-5 and np.abs(sh[0, 1:]).max() < 2e-3
    sh0, _, _ = oracle.bake_visibility(sc, dirs, wts, t_min=0.05, sh_degree=0)
    assert sh0.shape == (2, 1) and abs(sh0[0, 0] - sh[0, 0]) < 1e-12
    # an opaque slab just below the point, normal n: the lower half space is blocked.
    # c0 -> 2 pi Y00, (c3, c1, c2) -> pi Y1 n   (integral of w over the upper hemisphere = pi n)
    nrm = np.array([0.36, 0.48, 0.8])
    Rn = Rotation.align_vectors([nrm], [[0, 0, 1]])[0]   # maps z to n
    qx, qy, qz, qw = Rn.as_quat()
    sc = _scene([[0, 0, 0], -0.2 * nrm], [[0.01] * 3, [50, 50, 0.02]], [IDQ, [qw, qx, qy, qz]], [0.0, 1.0])
    sh, vis, _ = oracle.bake_visibility(sc, dirs, wts, t_min=0.01)
    up = dirs.astype(np.float64) @ nrm
    assert np.all(vis[0][up > 0.05] == 1.0)
    assert np.all(vis[0][up < -0.05] <= 0.0100001)   # one capped occluder: 1 - 0.99
    assert abs(sh[0, 0] - (2 * np.pi * Y00 * (1 + 0.01))) < 0.03
    got = np.array([sh[0, 3], sh[0, 1], sh[0, 2]])
    np.testing.assert_allclose(got, np.pi * Y1 * nrm * (1 - 0.01), atol=0.03)


def test_row_subset_equals_rows_of_the_full_result():
    rng = np.random.default_rng(8)
    sc = _random_scene(rng, 25)
    dirs, wts = _fib(6)
    sh, vis, un = oracle.bake_visibility(sc, dirs, wts, t_min=0.05)
    rows = [3, 17, 4]
    sh2, vis2, un2 = oracle.bake_visibility(sc, dirs, wts, t_min=0.05, rows=rows)
    np.testing.assert_array_equal(sh2, sh[rows])
    np.testing.assert_array_equal(vis2, vis[rows])
    np.testing.assert_array_equal(un2, un[rows])


def test_positions_mode_segment_ends_at_the_light():
    sigma, o = 0.1, 0.8
    # occluder between the Gaussian and the light: same as the direction ray; occluder behind the light: free
    sc = _scene([[0, 0, 0], [2, 0.05, 0], [6, 0.05, 0]], [[1e-3] * 3, [sigma] * 3, [sigma] * 3], [IDQ] * 3, [0.0, o, 0.0])
    _, vis_dir, _ = oracle.bake_visibility(sc, [[1, 0, 0]], [1], t_min=0.01)
    _, vis_pos, _ = oracle.bake_visibility(sc, [[4, 0, 0]], [1], t_min=0.01, positions=True)
    assert abs(vis_pos[0, 0] - vis_dir[0, 0]) < 1e-12 and vis_pos[0, 0] < 0.5
    sc.opacities[:] = [0.0, 0.0, o]
    _, vis_pos, _ = oracle.bake_visibility(sc, [[4, 0, 0]], [1], t_min=0.01, positions=True)
    # the closest point of the segment is its end (4, 0, 0), 2 units from the occluder: nothing
    assert vis_pos[0, 0] == 1.0
    # occluder just behind the light: acts at the segment's end, m2 = (0.15^2 + 0.05^2) / sigma^2
    sc.means[2] = [4.15, 0.05, 0]
    _, vis_pos, _ = oracle.bake_visibility(sc, [[4, 0, 0]], [1], t_min=0.01, positions=True)
    want = 1 - o * np.exp(-0.5 * (0.15**2 + 0.05**2) / sigma**2)
    assert abs(vis_pos[0, 0] - want) < 1e-6
    # light closer than the ray start: no segment, nothing occludes; SH uses the direction to the light
    sh, vis_pos, _ = oracle.bake_visibility(sc, [[0, 0.005, 0]], [2.0], t_min=0.01, positions=True)
    assert vis_pos[0, 0] == 1.0
    np.testing.assert_allclose(sh[0], [2 * Y00, 2 * Y1, 0, 0], atol=1e-6)   # w = +y


def test_positions_mode_matches_directions_for_far_lights():
    rng = np.random.default_rng(9)
    sc = _random_scene(rng, 30)
    dirs, wts = _fib(8)
    _, vis_dir, un1 = oracle.bake_visibility(sc, dirs, wts, t_min=0.05)
    _, vis_pos, un2 = oracle.bake_visibility(sc, dirs.astype(np.float64) * 1e6, wts, t_min=0.05, positions=True)
    ok = (un1 == 0) & (un2 == 0)
    np.testing.assert_allclose(vis_pos[ok], vis_dir[ok], atol=2e-5)
