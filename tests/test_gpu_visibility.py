"""Parity of sssgs_bake_visibility (BVH ray-traced per-Gaussian visibility + SH fit,
PAPER.md L110-112) against the brute-force oracle, through the C ABI.

Bars: visibilities within 5e-5 on rays the oracle calls stable (no pair within 1e-4
relative of the 1/255 threshold, product not within 1e-2 relative of 1e-4), within 1e-2 on the others (one
flipped pair changes V by at most 1/255 of itself per flip... bounded by flips * 0.4 % + 1e-4); SH
coefficients within the quadrature-weighted sum of those bounds."""
import copy

import numpy as np
import pytest

import oracle
from paper_2408_12282_b200 import scenes

pytestmark = pytest.mark.gpu

Y00, Y1 = 0.2820948, 0.4886025


def fib(K):
    k = np.arange(K) + 0.5
    z = 1 - 2 * k / K
    phi = k * np.pi * (3 - np.sqrt(5))
    r = np.sqrt(1 - z * z)
    return np.stack([r * np.cos(phi), r * np.sin(phi), z], 1).astype(np.float32), np.full(K, 4 * np.pi / K, np.float32)


def gpu_bake(scene, dirs, wts, t_min, sh_degree=1, positions=False):
    import torch
    from paper_2408_12282_b200 import binding
    r = binding.Renderer(scene)
    try:
        sh, vis = r.bake_visibility(dirs, wts, t_min, sh_degree=sh_degree, want_vis=True, positions=positions)
        torch.cuda.synchronize()
        out = sh.cpu().numpy(), vis.cpu().numpy(), r.launch_count()
    finally:
        r.close()
    return out


def check(scene, dirs, wts, t_min, sh_degree=1, min_occluded=0.0, positions=False):
    sh, vis, launches = gpu_bake(scene, dirs, wts, t_min, sh_degree, positions)
    sh_ref, vis_ref, unstable = oracle.bake_visibility(scene, dirs, wts, t_min, sh_degree, positions=positions)
    assert launches >= 9 or scene.n < 2
    tol = np.where(unstable == 0, 5e-5, 1e-4 + 5e-3 * unstable)
    err = np.abs(vis.astype(np.float64) - vis_ref)
    bad = err > tol
    assert not bad.any(), f"{bad.sum()} rays off, worst {err[bad].max():.3e} (stable worst {err[unstable == 0].max():.3e})"
    assert (vis_ref < 0.999).mean() >= min_occluded, "case is trivial"
    basis = [np.full(len(dirs), Y00)] + ([Y1 * dirs[:, 1], Y1 * dirs[:, 2], Y1 * dirs[:, 0]] if sh_degree else [])
    if positions:   # per-Gaussian directions: bound every basis function by its maximum
        basis = [np.full(len(dirs), Y00)] + ([np.full(len(dirs), Y1)] * 3 if sh_degree else [])
    for m, b in enumerate(basis):
        bound = (tol * np.abs(wts * b)[None, :]).sum(1) + 2e-5
        assert (np.abs(sh[:, m] - sh_ref[:, m]) <= bound).all(), f"SH coefficient {m}"
    return vis, vis_ref, unstable


def scaled(scene, f):
    s = copy.copy(scene)
    s.scales = (scene.scales * f).astype(np.float32)
    return s


@pytest.mark.parametrize("name,scene,t_min,K", [
    ("cfg1", scaled(scenes.make_scene(1), 3.0), 0.1, 24),
    ("cfg2_small", scaled(scenes.make_scene(2, n=6000, width=64, height=64), 3.0), 0.03, 16),
    ("cfg3_small", scaled(scenes.make_scene(3, n=3000, width=64, height=64, lights=1), 4.0), 0.05, 32),
])
def test_visibility_matches_oracle(name, scene, t_min, K):
    dirs, wts = fib(K)
    vis, vis_ref, unstable = check(scene, dirs, wts, t_min, min_occluded=0.2)
    # rays that leave a closed surface outwards are mostly free, inward ones mostly blocked
    assert vis_ref.min() < 0.05 and vis_ref.max() > 0.9


def test_degree_zero_and_determinism():
    scene = scaled(scenes.make_scene(1), 6.0)
    dirs, wts = fib(12)
    check(scene, dirs, wts, 0.05, sh_degree=0)
    a = gpu_bake(scene, dirs, wts, 0.05)
    b = gpu_bake(scene, dirs, wts, 0.05)
    np.testing.assert_array_equal(a[0].view(np.uint32), b[0].view(np.uint32))
    np.testing.assert_array_equal(a[1].view(np.uint32), b[1].view(np.uint32))


def _tiny(means, scales, opac):
    base = scenes.make_scene(1)
    n = len(means)
    idx = np.arange(n) % base.n
    s = scenes.subset(base, idx)
    s.means = np.asarray(means, np.float32)
    s.scales = np.asarray(scales, np.float32)
    s.opacities = np.asarray(opac, np.float32)
    s.rotations = np.tile(np.array([1, 0, 0, 0], np.float32), (n, 1))
    return s


def test_edge_cases():
    dirs, wts = fib(16)
    # one Gaussian: nothing can occlude it
    s1 = _tiny([[0, 0, 0]], [[0.1] * 3], [0.9])
    sh, vis, _ = gpu_bake(s1, dirs, wts, 0.01)
    assert np.all(vis == 1.0) and abs(sh[0, 0] - np.sqrt(4 * np.pi)) < 1e-5
    # two Gaussians; coincident centres (equal Morton codes); a chain on one line (degenerate extent);
    # transparent and sub-threshold Gaussians that never occlude
    check(_tiny([[0, 0, 0], [0.5, 0, 0]], [[0.1] * 3] * 2, [0.9, 0.9]), dirs, wts, 0.01)
    check(_tiny([[0, 0, 0]] * 5 + [[0.3, 0.1, 0]], [[0.1] * 3] * 6, [0.5] * 6), dirs, wts, 0.01)
    check(_tiny([[0.1 * k, 0, 0] for k in range(40)], [[0.03] * 3] * 40, [0.7] * 40),
          np.array([[1, 0, 0], [-1, 0, 0], [0, 1, 0], [0.6, 0.8, 0]], np.float32), np.ones(4, np.float32), 0.01)
    rng = np.random.default_rng(3)
    opac = np.where(rng.random(300) < 0.5, rng.uniform(0, 1 / 255, 300), rng.uniform(0.3, 1, 300))
    opac[:10] = 0.0
    check(_tiny(rng.normal(size=(300, 3)), np.full((300, 3), 0.2), opac), dirs, wts, 0.05, min_occluded=0.1)


def test_bake_then_render_leaves_the_renderer_intact():
    """The tree lives in workspace regions a render rewrites: a render after a bake equals one before."""
    import torch
    from paper_2408_12282_b200 import binding
    scene = scenes.make_scene(2, n=20000, width=128, height=96)
    dirs, wts = fib(8)
    r = binding.Renderer(scene)
    try:
        a = r.render(want=("rgb",))["rgb"].cpu().numpy()
        r.bake_visibility(dirs, wts, 0.02)
        b = r.render(want=("rgb",))["rgb"].cpu().numpy()
        torch.cuda.synchronize()
    finally:
        r.close()
    np.testing.assert_array_equal(a.view(np.uint32), b.view(np.uint32))


def test_invalid_arguments():
    import torch
    from paper_2408_12282_b200 import binding
    scene = scenes.make_scene(1)
    dirs, wts = fib(8)
    r = binding.Renderer(scene)
    try:
        with pytest.raises(binding.SssgsError):
            r.bake_visibility(dirs, wts, -1.0)
        with pytest.raises(binding.SssgsError):
            r.bake_visibility(dirs, wts, float("nan"))
        with pytest.raises(binding.SssgsError):
            r.bake_visibility(dirs, wts, 0.01, sh_degree=2)
        with pytest.raises(binding.SssgsError):
            r.bake_visibility(np.zeros((0, 3), np.float32), np.zeros(0, np.float32), 0.01)
        torch.cuda.synchronize()
    finally:
        r.close()


@pytest.mark.parametrize("cfg,K,n_rows,t_min", [(2, 32, 192, 0.05), (3, 16, 96, 0.05)])
def test_full_size_sampled_rows(cfg, K, n_rows, t_min):
    """BASELINE-size scenes as they are (no rescaling): the oracle traces the rays of a seeded sample of
    Gaussians against ALL Gaussians; the GPU result of those rows must match."""
    scene = scenes.make_scene(cfg, views=1, lights=1)
    dirs, wts = fib(K)
    sh, vis, _ = gpu_bake(scene, dirs, wts, t_min)
    assert np.isfinite(sh).all() and (vis >= 0).all() and (vis <= 1).all()
    rows = np.sort(np.random.default_rng(50 + cfg).choice(scene.n, size=n_rows, replace=False))
    sh_ref, vis_ref, unstable = oracle.bake_visibility(scene, dirs, wts, t_min, rows=rows)
    tol = np.where(unstable == 0, 5e-5, 1e-4 + 5e-3 * unstable)
    err = np.abs(vis[rows].astype(np.float64) - vis_ref)
    assert (err <= tol).all(), f"worst {err.max():.3e}"
    assert (vis_ref < 0.999).mean() > 0.05 and vis_ref.max() > 0.5
    bound = (tol * np.abs(wts * Y00)[None, :]).sum(1) + 1e-5
    assert (np.abs(sh[rows, 0] - sh_ref[:, 0]) <= bound).all()


def test_positions_mode_matches_oracle():
    """Rays towards known light positions: the OLAT lights of config 3 around the object, and
    points inside the scene's bounding box (segments that end between the Gaussians)."""
    scene = scaled(scenes.make_scene(3, n=3000, width=64, height=64, lights=24), 4.0)
    lights = np.stack([np.asarray(l.position, np.float32) for l in scene.lights[0]])
    wts = np.full(len(lights), 4 * np.pi / len(lights), np.float32)
    vis, vis_ref, _ = check(scene, lights, wts, 0.05, min_occluded=0.2, positions=True)
    assert vis_ref.min() < 0.05 and vis_ref.max() > 0.9
    rng = np.random.default_rng(11)
    inner = rng.uniform(-1.0, 1.0, size=(12, 3)).astype(np.float32)
    check(scene, inner, np.ones(12, np.float32), 0.05, min_occluded=0.2, positions=True)
    # a light on top of a Gaussian (closer than the ray start): nothing occludes
    on_top = scene.means[:4] + np.float32(0.01)
    sh, vis, _ = gpu_bake(scene, on_top, np.ones(4, np.float32), 0.05, positions=True)
    assert vis[0, 0] == 1.0 and vis[1, 1] == 1.0 and vis[3, 3] == 1.0
