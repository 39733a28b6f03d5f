"""Parity at BASELINE.json's full sizes, in the launch configuration bench.py times (one view of the
workload per sssgs_render call, all lights of a step in that call).

The oracle composites a whole 1-2 Mpix frame of a 1-3 M Gaussian scene in seconds, but not every light
of a 64-light sweep, so:
  * counters, sort keys, tile lists and tile ranges are compared in full, bit-exact (the oracle's
    projection and stable sort do run at full size);
  * MLP outputs are compared on a seeded sample of Gaussians (a row depends on its Gaussian only):
    all four outputs within 1e-2 of the float64 reference, 3e-3 of the fp16-emulating oracle;
  * the G-buffer of the first checked light of every (config, view) is compared on EVERY pixel, element by
    element; the other checked lights on a seeded sample of >= 32 whole tiles per frame (the longest list,
    the median one, tiles of every partial edge row / column the image has, random non-empty tiles):
    the oracle composites from the full sorted list, in the original pixel coordinates, fed the GPU's
    own MLP outputs (so that the 1e-4 bar isolates compositing);
  * RGB / AOVs are compared over the whole frame against the oracle's shading of the GPU's
    G-buffer (per-pixel work the oracle does at full size);
  * A + T = 1 and finiteness are checked on every pixel of every checked frame.
Two calls are checked per (config, view): the full-output call (every output requested: the list walks
render it) and the call shape bench.py times (no MLP outputs requested: from 4 lights per view on the
visibility pre-pass, the row-skipping MLP and the cached walks render it).  The second one's frames must
equal the first one's bit for bit, and its G-buffer is compared with the oracle directly, on the first,
second and last light batch (the later batches run the MLP-channels-only cached walk).
"""
import numpy as np
import pytest

import oracle
from paper_2408_12282_b200 import scenes
from test_gpu_parity import check_gbuffer, check_lists, check_shading, check_tight_lists

pytestmark = pytest.mark.gpu

N_TILES = 32
N_ROWS = 4096


def _render_both(scene, view, lights_checked):
    """-> (full, bench): numpy outputs of the full-output call and of the benchmarked call shape; the per-frame
    outputs only for the lights in `lights_checked` (a 64-light G-buffer is 2.6 GB)."""
    import torch
    from paper_2408_12282_b200 import binding
    R = binding.Renderer(scene, max_instances=int(20 * scene.n))
    cams, lights = [scene.cameras[view]], scene.lights[view]
    sel = torch.tensor(sorted(lights_checked), device="cuda")
    per_frame = ("rgb", "gbuffer", "aov_diffuse", "aov_specular", "mlp_out")
    try:
        out = R.render(cams=cams, lights=lights,
                       want=per_frame + ("sorted_keys", "sorted_vals", "tile_ranges", "counters"))
        torch.cuda.synchronize()
        full = {k: (v.index_select(0, sel) if k in per_frame else v).cpu().numpy() for k, v in out.items()}
        full["rgb_all"] = out["rgb"].cpu().numpy()
        del out
        # the call bench.py times asks for frames and counters only, over TIGHT tile lists: in a sweep (>= 4 lights)
        # the MLP then runs on the rows a visibility pre-pass keeps and the walks stream the weight cache
        out = R.render(cams=cams, lights=lights, want=("rgb", "gbuffer", "aov_diffuse", "aov_specular", "counters"),
                       tight=True)
        torch.cuda.synchronize()
        bench = {k: (v.index_select(0, sel) if k in per_frame else v).cpu().numpy() for k, v in out.items()}
        bench["rgb_all"] = out["rgb"].cpu().numpy()
        bench["launches"] = R.launch_count()
        del out
        # the tight lists themselves, exported by a geometry-only call
        out = R.render(cams=cams, lights=lights[:1], want=("sorted_keys", "sorted_vals", "tile_ranges", "counters"),
                       tight=True, precomputed=torch.zeros((1, scene.n, 4), device="cuda"))
        torch.cuda.synchronize()
        bench["tight"] = {k: v.cpu().numpy() for k, v in out.items()}
        del out
    finally:
        R.close()
    return full, bench


def _sample_tiles(rng, ranges, tiles_x, tiles_y, width, height):
    length = (ranges[:, 1].astype(np.int64) - ranges[:, 0].astype(np.int64))
    nonempty = np.nonzero(length > 0)[0]
    picks = [int(np.argmax(length)), int(nonempty[np.argsort(length[nonempty])[len(nonempty) // 2]])]

    def add_from(cands, k):
        cands = cands[length[cands] > 0]
        if len(cands):
            order = cands[np.argsort(-length[cands])]
            for t in list(order[:1]) + list(rng.permutation(order[1:])[:k - 1]):   # the longest + random others
                if int(t) not in picks:
                    picks.append(int(t))
    if height % 16:   # partial last tile row (1080 = 67.5 tiles): 8 of its tiles
        add_from(np.arange((tiles_y - 1) * tiles_x, tiles_y * tiles_x), 8)
    if width % 16:    # partial last tile column
        add_from(np.arange(tiles_x - 1, tiles_x * tiles_y, tiles_x), 8)
    for t in rng.permutation(nonempty):
        if len(picks) >= N_TILES:
            break
        if int(t) not in picks:
            picks.append(int(t))
    return picks


# (config, view, lights of the step, lights whose frames are checked against the oracle)
CASES = [
    (3, 0, 64, (0, 7, 8, 15, 56, 63)),   # first / second / last light batch of the 64-light sweep
    (4, 0, 1, (0,)),
    (4, 5, 1, (0,)),                      # a second view of the orbit
    (5, 0, 16, (0, 15)),                  # both light batches
    (5, 11, 16, (7, 8)),
]


@pytest.mark.parametrize("cfg,view,n_lights,checked", CASES)
def test_full_size_config(cfg, view, n_lights, checked):
    scene = scenes.make_scene(cfg, lights=n_lights)
    cam = scene.cameras[view]
    full, bench = _render_both(scene, view, checked)

    # the benchmarked call shape renders the same frames, bit for bit (all lights)
    np.testing.assert_array_equal(bench["rgb_all"].view(np.uint32), full["rgb_all"].view(np.uint32))
    if n_lights >= 4:
        assert 0 < bench["counters"][0][4] < scene.n       # the MLP really ran on the kept rows only
    for k in ("gbuffer", "aov_diffuse", "aov_specular"):
        np.testing.assert_array_equal(bench[k].view(np.uint32), full[k].view(np.uint32))

    # ---- lists, ranges, counters: full, bit-exact ------------------------------------------------
    proj = oracle.project(scene, cam)
    keys, vals, ranges = oracle.build_lists(proj)
    ref = type("R", (), dict(n_vis=int(proj.visible.sum()), n_instances=len(keys), keys=keys, vals=vals,
                             ranges=ranges))
    check_lists(scene, full, ref, 0)

    rng = np.random.default_rng(1000 + 10 * cfg + view)
    # ---- the tight lists of the benchmarked call: S5 conditions, the minimal set on 256 sampled tiles --------
    nonempty = np.nonzero(ranges[:, 1] > ranges[:, 0])[0]
    t_sel = np.sort(rng.choice(nonempty, size=min(256, len(nonempty)), replace=False))
    masked_r = np.zeros_like(ranges)
    masked_r[t_sel] = ranges[t_sel]
    hit = oracle.tile_hits(scene, cam, proj, vals, masked_r)
    It, _ = check_tight_lists(bench["tight"], keys, vals, ranges, hit, tiles_checked=t_sel)
    assert It == bench["counters"][0][1] and It < len(keys)
    print(f"cfg {cfg} view {view}: canonical {len(keys)} instances, tight {It} ({It / len(keys):.3f})")
    # ---- MLP on a sample of Gaussians --------------------------------------------------------------
    idx = np.sort(rng.choice(scene.n, size=N_ROWS, replace=False))
    sub = scenes.subset(scene, idx)
    for f, l in enumerate(sorted(checked)):
        x = oracle.mlp_inputs(sub, cam, scene.lights[view][l].position)
        y_em = oracle.mlp_forward(x, scene.mlp, 2)
        y_ref = oracle.mlp_forward(x, scene.mlp, 0)
        got = full["mlp_out"][f][idx].astype(np.float64)
        e_em = np.abs(got - y_em)
        assert (e_em <= 1e-3).mean() >= 0.999 and e_em.max() <= 3e-3, f"light {l}: max {e_em.max():.3e}"
        assert np.abs(got - y_ref).max() <= 1e-2, f"light {l}: MLP vs float64 {np.abs(got - y_ref).max():.3e} (north_star 1e-2)"

    # ---- sampled tiles of the G-buffer, from the call shape bench.py times -------------------------
    picks = _sample_tiles(rng, ranges, proj.tiles_x, proj.tiles_y, cam.width, cam.height)
    assert len(picks) >= N_TILES
    masked = np.zeros_like(ranges)
    masked[picks] = ranges[picks]
    pix_mask = np.zeros((cam.height, cam.width), bool)
    for t in picks:
        ty, tx = divmod(t, proj.tiles_x)
        pix_mask[ty * 16:(ty + 1) * 16, tx * 16:(tx + 1) * 16] = True
    for f, l in enumerate(sorted(checked)):
        ch = oracle.channels(scene, proj, full["mlp_out"][f].astype(np.float64))
        # the first checked light: EVERY pixel of the frame, element by element (the oracle composites a whole
        # 1-2 Mpix frame of these scenes in seconds on the box's cores); the other lights: the sampled tiles
        whole = f == 0
        comp = oracle.composite(scene, cam, proj, ch, vals, ranges if whole else masked)
        mask = np.ones_like(pix_mask) if whole else pix_mask
        assert (mask & ~comp.unstable).sum() > 0
        check_gbuffer(bench["gbuffer"][f], None, mask=mask, comp=comp, ch=ch[proj.visible != 0],
                      label=f"cfg {cfg} view {view} light {l} ({'whole frame' if whole else f'{len(picks)} tiles'}):")

    # ---- every pixel of every checked frame: A + T = 1, finite; shading of the GPU's own G-buffer --
    g = bench["gbuffer"]
    assert np.isfinite(g).all() and np.isfinite(bench["rgb_all"]).all()
    np.testing.assert_allclose(g[..., 14] + g[..., 15], 1.0, atol=3e-6)
    for f, l in enumerate(sorted(checked)):
        check_shading(scene, bench, f, view, l)
