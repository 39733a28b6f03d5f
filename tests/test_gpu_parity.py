"""Parity of the CUDA path (through the C ABI) against the CPU oracle, element by element on
the same seeded inputs.  Needs a B200: every test is marked gpu.

Bars (BASELINE.json north_star):
  * sort keys, tile lists, tile ranges, counters: bit-exact;
  * G-buffer and RGB: 1e-4 absolute on stable pixels (pixels whose skip/stop decisions sit within
    fp32 rounding of a threshold are flagged by the oracle, S7, and compared at 2e-2);
    RGB at ill-conditioned highlights: max(1e-4 max(1,|ref|), 4 |ref32 - ref64|) (S9);
  * MLP (default: binary16 layer inputs): all four outputs within 1e-2 of the fp64 reference, and within 3e-3
    of the fp16-emulating oracle; compute = bf16: max <= 2e-2 vs the bf16-emulating oracle, L_SSS <= 1e-2 vs fp64.
"""
import numpy as np
import pytest

import oracle
from paper_2408_12282_b200 import scenes
from util import custom_scene

pytestmark = pytest.mark.gpu

ALL = ("rgb", "gbuffer", "aov_diffuse", "aov_specular", "mlp_out", "sorted_keys", "sorted_vals",
       "tile_ranges", "counters")


def gpu_render(scene, want=ALL, precomputed=None, cams=None, lights=None, tight=False, **kw):
    import torch
    from paper_2408_12282_b200 import binding
    r = binding.Renderer(scene, **kw)
    try:
        out = r.render(cams=cams, lights=lights, want=want, precomputed=precomputed, tight=tight)
        torch.cuda.synchronize()
        res = {k: v.cpu().numpy() for k, v in out.items()}
        res["launches"] = r.launch_count()
    finally:
        r.close()
    return res


def check_lists(scene, res, ref, view=0):
    cnt = res["counters"][view]
    assert cnt[3] == 0, "look-back bound tripped"
    assert cnt[2] == 0, "instance overflow"
    assert cnt[0] == ref.n_vis
    I = ref.n_instances
    assert cnt[1] == I
    keys = res["sorted_keys"][view].view(np.uint64)[:I]
    vals = res["sorted_vals"][view].view(np.uint32)[:I]
    np.testing.assert_array_equal(keys, ref.keys)
    np.testing.assert_array_equal(vals, ref.vals)
    np.testing.assert_array_equal(res["tile_ranges"][view].view(np.uint32), ref.ranges)


def check_tight_lists(res, keys, vals, ranges, hit, view=0, tiles_checked=None):
    """SURVEY S5 conditions of a tight tile list (SSSGS_TIGHT_LISTS) against the oracle's canonical list
    (keys, vals, ranges) and its minimal set `hit` (oracle.tile_hits): the tight list is a sub-sequence of the
    canonical one (same pairs, same order), keeps every pair with alpha >= 1/255 at some pixel of its tile, and
    its ranges / instance counter describe it.  tiles_checked: `hit` was only computed for these tiles."""
    cnt = res["counters"][view]
    It = int(cnt[1])
    assert cnt[2] == 0 and cnt[3] == 0
    tk = res["sorted_keys"][view].view(np.uint64)[:It]
    tv = res["sorted_vals"][view].view(np.uint32)[:It]
    assert It <= len(keys)
    # position of every tight pair in the canonical list: equal keys (same tile, same depth bits) are rare
    lo = np.searchsorted(keys, tk, "left")
    hi = np.searchsorted(keys, tk, "right")
    assert (hi > lo).all(), "a tight pair's key is not in the canonical list"
    pos = lo.copy()
    for j in np.nonzero(hi - lo > 1)[0]:
        m = np.nonzero(vals[lo[j]:hi[j]] == tv[j])[0]
        assert len(m) == 1
        pos[j] = lo[j] + m[0]
    assert (vals[pos] == tv).all(), "a tight pair is not in the canonical list"
    assert (np.diff(pos.astype(np.int64)) > 0).all(), "tight list is not in canonical order"
    kept = np.zeros(len(keys), bool)
    kept[pos] = True
    must = hit if tiles_checked is None else hit & np.isin((keys >> np.uint64(32)).astype(np.int64), tiles_checked)
    assert kept[must].all(), f"{int((must & ~kept).sum())} pairs with alpha >= 1/255 in their tile were dropped"
    # ranges of the tight list
    tt = (tk >> np.uint64(32)).astype(np.int64)
    n_tiles = ranges.shape[0]
    want = np.stack([np.searchsorted(tt, np.arange(n_tiles), "left"), np.searchsorted(tt, np.arange(n_tiles), "right")], 1)
    np.testing.assert_array_equal(res["tile_ranges"][view].view(np.uint32).astype(np.int64), want)
    return It, int(hit.sum())


def unstable_bound(ref_gbuf, flags, ch):
    """What the flagged decisions of a pixel can move a G-buffer value by (S7).
    ch: [n, 14] per-Gaussian channel values (M_c = max |ch_c|; 1 for the A and T channels).
      * an alpha ~ 1/255 decision flipped: the entry is blended or not with weight <= 1/255, and every later
        weight (and the final T) scales by (1 - 1/255): |delta| <= (M_c + |ref|) / 255 per flagged decision;
      * the T' ~ 1e-4 stop flipped: the stopping entry is blended or not; T' = T (1 - alpha) ~ 1e-4 with
        alpha <= 0.99 means T <= 1e-2, so its weight T alpha and the final T move by <= 1e-2, the entries
        behind it carry <= 1e-4 in total: |delta| <= 1.02e-2 M_c;
      * power ~ 0 (pixel on the centre of a Gaussian whose exponent rounds either side of 0): the entry is
        skipped or blended with alpha = o: |delta| <= M_c.
    5 % slack for the fp32 evaluation on top, plus the 1e-4 bar of stable pixels."""
    M = np.concatenate([np.abs(ch).max(axis=0) if len(ch) else np.zeros(14), [1.0, 1.0]])
    n_alpha = (flags >> 4).astype(np.float64)[..., None]
    t_rule = ((flags & 4) != 0).astype(np.float64)[..., None]
    p_rule = ((flags & 1) != 0).astype(np.float64)[..., None]
    return 1e-4 + 1.05 * (n_alpha / 255.0 * (M + np.abs(ref_gbuf)) + t_rule * 1.02e-2 * M + p_rule * M)


def check_gbuffer(gpu_gbuf, ref, atol=1e-4, mask=None, comp=None, ch=None, label=""):
    """G-buffer vs the oracle: 1e-4 on stable pixels, the derived bound of the flagged decisions on the others.
    mask restricts the comparison to sampled pixels; comp / ch default to ref.comp / ref.ch."""
    comp = comp if comp is not None else ref.comp
    ch = ch if ch is not None else ref.ch
    d = np.abs(gpu_gbuf.astype(np.float64) - comp.gbuf)
    stable = ~comp.unstable if mask is None else (mask & ~comp.unstable)
    unst = comp.unstable if mask is None else (mask & comp.unstable)
    worst = d[stable].max() if stable.any() else 0.0
    assert worst <= atol, f"{label} stable-pixel G-buffer error {worst:.3e} > {atol}"
    if unst.any():
        bound = unstable_bound(comp.gbuf, comp.flags, ch)
        bad = unst[..., None] & (d > bound)
        assert not bad.any(), f"{label} unstable-pixel error beyond the flagged decisions' reach: {d[bad].max():.3e}"
    f = comp.flags[unst] if unst.any() else np.zeros(0, np.uint8)
    print(f"{label} G-buffer: stable worst {worst:.2e}; unstable pixels {int(unst.sum())} "
          f"(power ~ 0: {int(((f & 1) != 0).sum())}, alpha ~ 1/255: {int(((f & 2) != 0).sum())}, "
          f"T' ~ 1e-4: {int(((f & 4) != 0).sum())})")
    return worst, int(unst.sum())


def check_shading(scene, gpu, frame, view, light):
    """RGB/AOVs of the GPU vs the oracle's shading of the GPU's OWN G-buffer (isolates step a8)."""
    cam, lt = scene.cameras[view], scene.lights[view][light]
    g64 = gpu["gbuffer"][frame].astype(np.float64)
    rgb64, ad64, as64 = oracle.shade(cam, lt, g64)
    rgb32, ad32, as32 = oracle.shade(cam, lt, g64, f32=True)
    for name, got, r64, r32 in (("rgb", gpu["rgb"][frame], rgb64, rgb32),
                                ("aov_diffuse", gpu["aov_diffuse"][frame], ad64, ad32),
                                ("aov_specular", gpu["aov_specular"][frame], as64, as32)):
        tol = np.maximum(1e-4 * np.maximum(1.0, np.abs(r64)), 4.0 * np.abs(r32.astype(np.float64) - r64))
        err = np.abs(got.astype(np.float64) - r64)
        bad = err > tol
        assert not bad.any(), f"{name}: {bad.sum()} values off, worst {err[bad].max():.3e}"


def _small_scenes():
    yield "cfg1", scenes.make_scene(1)
    yield "cfg2_small", scenes.make_scene(2, n=20000, width=256, height=192)
    yield "cfg3_small", scenes.make_scene(3, n=30000, width=200, height=200, lights=3)
    yield "cfg4_small", scenes.make_scene(4, n=40000, width=240, height=135, views=2)
    yield "cfg5_small", scenes.make_scene(5, n=30000, width=128, height=128, views=1, lights=2)
    yield "cfg6_paper_arch", scenes.make_scene(6, n=5000, width=128, height=128)


@pytest.mark.parametrize("name,scene", list(_small_scenes()))
def test_lists_bit_exact(name, scene):
    res = gpu_render(scene, want=("sorted_keys", "sorted_vals", "tile_ranges", "counters"),
                     precomputed=np.zeros((len(scene.cameras) * len(scene.lights[0]), scene.n, 4), np.float32))
    for v in range(len(scene.cameras)):
        cam = scene.cameras[v]
        proj = oracle.project(scene, cam)
        keys, vals, ranges = oracle.build_lists(proj)
        ref = type("R", (), dict(n_vis=int(proj.visible.sum()), n_instances=len(keys), keys=keys, vals=vals, ranges=ranges))
        check_lists(scene, res, ref, v)


@pytest.mark.parametrize("name,scene", list(_small_scenes()))
def test_gbuffer_and_shading_with_reference_mlp(name, scene):
    # rasteriser + shading fed the ORACLE's MLP outputs (fp64 reference rounded to fp32)
    nv, nl = len(scene.cameras), len(scene.lights[0])
    refs, pre = {}, np.zeros((nv * nl, scene.n, 4), np.float32)
    for v in range(nv):
        geo = None
        for l in range(nl):
            r = oracle.render_frame(scene, v, l, geometry=geo)
            geo = geo or r
            pre[v * nl + l] = r.mlp_out.astype(np.float32)
    # the oracle composites exactly what the GPU is given (fp32-rounded MLP outputs)
    for v in range(nv):
        geo = None
        for l in range(nl):
            r = oracle.render_frame(scene, v, l, mlp_out=pre[v * nl + l].astype(np.float64), geometry=geo)
            geo = geo or r
            refs[(v, l)] = r
    lights = [scene.lights[v] for v in range(nv)]
    import torch
    from paper_2408_12282_b200 import binding
    R = binding.Renderer(scene)
    try:
        out = R.render(cams=scene.cameras, lights=lights, want=ALL, precomputed=pre, lights_per_camera=True)
        torch.cuda.synchronize()
        gpu = {k: t.cpu().numpy() for k, t in out.items()}
    finally:
        R.close()
    for (v, l), r in refs.items():
        f = v * nl + l
        check_lists(scene, gpu, r, v)
        worst, nun = check_gbuffer(gpu["gbuffer"][f], r)
        np.testing.assert_allclose(gpu["gbuffer"][f][..., 14] + gpu["gbuffer"][f][..., 15], 1.0, atol=2e-6)
        check_shading(scene, gpu, f, v, l)
        # end to end against the oracle's own RGB on stable pixels: north_star's 1e-4 bar (HDR highlights scale it:
        # S9); measured <= 0.23 of it on these scenes, so no conditioning term is needed here
        tol = 1e-4 * np.maximum(1.0, np.abs(r.rgb))
        err = np.abs(gpu["rgb"][f] - r.rgb)
        st = ~r.comp.unstable
        assert (err[st] <= tol[st]).all(), f"rgb vs oracle: worst {err[st].max():.3e}"
        np.testing.assert_array_equal(gpu["mlp_out"][f], pre[f])


# MLP bars.  Default compute = binary16 layer inputs: every output within 1e-2 of the float64
# reference (BASELINE north_star) and within 3e-3 of the fp16-emulating oracle (same rounding points, double instead
# of fp32 accumulation: a rare rounding flip of a hidden activation moves an output by <= 2^-11 x |activation| x
# |weight path| ~ 1e-3).  compute = bf16: the kernel-correctness bar against the bf16-emulating oracle (2e-2, flips
# are 8x larger) and the L_SSS bar against float64; the unbounded ReLU output L_in exceeds 1e-2 there -- which is why
# bf16 is not the default -- and is reported.
@pytest.mark.parametrize("compute", ["fp16", "bf16"])
@pytest.mark.parametrize("name,scene", list(_small_scenes()))
def test_mlp_outputs(name, scene, compute):
    nv, nl = len(scene.cameras), len(scene.lights[0])
    import torch
    from paper_2408_12282_b200 import binding
    R = binding.Renderer(scene, compute=binding.SSSGS_COMPUTE_FP16 if compute == "fp16" else binding.SSSGS_COMPUTE_BF16)
    try:
        out = R.render(cams=scene.cameras, lights=[scene.lights[v] for v in range(nv)],
                       want=("mlp_out", "rgb"), lights_per_camera=True)
        torch.cuda.synchronize()
        got = out["mlp_out"].cpu().numpy().astype(np.float64)
    finally:
        R.close()
    for v in range(nv):
        for l in range(nl):
            x = oracle.mlp_inputs(scene, scene.cameras[v], scene.lights[v][l].position)
            y_em = oracle.mlp_forward(x, scene.mlp, 2 if compute == "fp16" else 1)
            y_ref = oracle.mlp_forward(x, scene.mlp, 0)
            e_em = np.abs(got[v * nl + l] - y_em)
            e_ref = np.abs(got[v * nl + l] - y_ref)
            frac = (e_em <= 1e-3).mean()
            print(f"{name} {compute} v{v} l{l}: vs emulating oracle max {e_em.max():.3e} frac<=1e-3 {frac:.5f}; "
                  f"vs fp64 L_SSS max {e_ref[:, :3].max():.3e} L_in max {e_ref[:, 3].max():.3e} "
                  f"L_in frac>1e-2 {(e_ref[:, 3] > 1e-2).mean():.5f}")
            assert frac >= 0.999, f"only {frac:.5f} of MLP outputs within 1e-3 of the emulating oracle"
            if compute == "fp16":
                assert e_em.max() <= 3e-3
                assert e_ref.max() <= 1e-2, f"MLP vs float64: {e_ref.max():.3e} > 1e-2 (north_star)"
            else:
                assert e_em.max() <= 2e-2
                assert e_ref[:, :3].max() <= 1e-2


def test_end_to_end_rgb_cfg1():
    # whole path on the GPU (its own MLP, binary16 layer inputs) vs the oracle with the fp16-emulating MLP
    scene = scenes.make_scene(1)
    gpu = gpu_render(scene)
    r = oracle.render_frame(scene, mlp_mode=2)
    check_lists(scene, gpu, r)
    st = ~r.comp.unstable
    err = np.abs(gpu["rgb"][0] - r.rgb)
    # the fp16 MLP outputs differ from the emulating oracle's by <= 3e-3 on rare rows: measured p99.9 8e-6, max 6e-5
    assert np.percentile(err[st], 99.9) <= 1e-4 and err[st].max() <= 1e-3
    assert np.abs(gpu["gbuffer"][0][..., :10] - r.gbuf[..., :10])[st].max() <= 1e-4


def test_light_batching_is_consistent():
    scene = scenes.make_scene(3, n=20000, width=160, height=160, lights=6)
    a = gpu_render(scene, want=("rgb", "gbuffer"), lights=scene.lights[0])
    b = gpu_render(scene, want=("rgb", "gbuffer"), lights=scene.lights[0], max_lights_per_pass=1)
    c = gpu_render(scene, want=("rgb", "gbuffer"), lights=scene.lights[0], max_lights_per_pass=4)
    # the accumulations are bit-identical whatever the batch width; the shading epilogue is a
    # different template instantiation per width (fp32 contraction may differ by an ulp)
    np.testing.assert_array_equal(a["gbuffer"], b["gbuffer"])
    np.testing.assert_array_equal(a["gbuffer"], c["gbuffer"])
    np.testing.assert_allclose(a["rgb"], b["rgb"], rtol=2e-6, atol=1e-6)
    np.testing.assert_allclose(a["rgb"], c["rgb"], rtol=2e-6, atol=1e-6)


# 169 tiles -> several entry slots per warp; 1681 tiles -> 1.  19 lights = three light batches: the first
# cached walk blends all channels, the next two (8 and 3 lights) only the MLP channels
@pytest.mark.parametrize("width,n_lights", [(200, 6), (656, 6), (656, 19), (200, 12)])
def test_sweep_row_skipping_changes_nothing(width, n_lights):
    # From 4 lights per view on, a visibility pre-pass restricts the MLP to the Gaussians that are
    # blended somewhere (unless the MLP outputs of all Gaussians are requested).  Frames must be
    # bit-identical with and without it, and the skipped rows must really be skippable.
    scene = scenes.make_scene(3, n=40000, width=width, height=width, lights=n_lights)
    on = gpu_render(scene, want=("rgb", "gbuffer", "aov_diffuse", "aov_specular", "counters"), lights=scene.lights[0])
    off = gpu_render(scene, want=("rgb", "gbuffer", "aov_diffuse", "aov_specular", "counters", "mlp_out"),
                     lights=scene.lights[0])
    assert on["launches"] > off["launches"]          # pre-pass + compaction were launched
    assert off["counters"][0][4] == scene.n
    for k in ("rgb", "gbuffer", "aov_diffuse", "aov_specular"):
        if width > 640:   # same one-slot walk order with and without the pre-pass: bit-identical
            np.testing.assert_array_equal(on[k].view(np.uint32), off[k].view(np.uint32))
        else:             # small images walk 2 entries per warp step without the pre-pass: the per-slot
            # partial sums are added in another order than the cached one-slot walk (both within 1e-4)
            np.testing.assert_allclose(on[k], off[k], rtol=5e-5, atol=2e-6)
    r = oracle.render_frame(scene, 0, 0, mlp_out=off["mlp_out"][0].astype(np.float64))
    # the rows the pre-pass keeps are the Gaussians the oracle blends at some pixel (pixels whose
    # skip / stop decisions sit within rounding of a threshold may add or drop a few)
    kept, ref = int(on["counters"][0][4]), int(r.comp.contrib.sum())
    assert 0 < kept < scene.n and abs(kept - ref) <= max(8, int(2e-3 * ref)), (kept, ref)


@pytest.mark.parametrize("width,n_lights", [(96, 3), (128, 11), (656, 9)])
def test_sum_lights_is_the_sum_of_the_frames(width, n_lights):
    # SSSGS_SUM_LIGHTS (image-based lighting as a sum of point lights, App. D): one frame
    # per camera = sum_l intensity_l A L_out,l + (1 - A) bg, formed in the rasteriser's epilogue.
    import dataclasses
    import torch
    from paper_2408_12282_b200 import binding
    scene = scenes.make_scene(3, n=30000, width=width, height=width, lights=n_lights)
    rng = np.random.default_rng(5)
    lights = [dataclasses.replace(l, intensity=rng.uniform(0.2, 1.5, 3).astype(np.float32)) for l in scene.lights[0]]
    cam = dataclasses.replace(scene.cameras[0], bg=np.float32([0.3, 0.1, 0.2]))
    R = binding.Renderer(scene)
    try:
        per = R.render(cams=[cam], lights=lights, want=("rgb", "gbuffer", "mlp_out"))
        torch.cuda.synchronize()
        per = {k: v.cpu().numpy() for k, v in per.items()}
        tot = R.render(cams=[cam], lights=lights, want=("rgb",), sum_lights=True)
        torch.cuda.synchronize()
        tot = tot["rgb"].cpu().numpy()
    finally:
        R.close()
    assert tot.shape == (1, width, width, 3)
    A = per["gbuffer"][0][..., 14:15].astype(np.float64)
    bg_term = (1.0 - np.where(A >= 1e-6, A, 0.0)) * cam.bg.astype(np.float64)
    # every per-light frame carries the background term once: remove the extra copies
    want = per["rgb"].astype(np.float64).sum(axis=0) - (n_lights - 1) * bg_term
    np.testing.assert_allclose(tot[0], want, rtol=2e-5, atol=2e-5)
    # and against the oracle: shading of the GPU's G-buffers, summed in float64
    ref = np.zeros_like(want)
    for l, lt in enumerate(lights):
        ref += oracle.shade(cam, lt, per["gbuffer"][l].astype(np.float64))[0]
    ref -= (n_lights - 1) * bg_term
    rgb32 = np.zeros_like(want)
    for l, lt in enumerate(lights):
        rgb32 += oracle.shade(cam, lt, per["gbuffer"][l].astype(np.float64), f32=True)[0].astype(np.float64)
    rgb32 -= (n_lights - 1) * bg_term
    tol = np.maximum(1e-4 * np.maximum(1.0, np.abs(ref)), 4.0 * np.abs(rgb32 - ref) + 1e-5)
    assert (np.abs(tot[0] - ref) <= tol).all()


@pytest.mark.parametrize("width,n_lights", [(128, 1), (160, 6), (656, 3)])
def test_forward_shading_variant_matches_oracle(width, n_lights):
    # "w/o deferred" (Tab. 2): Eq. 7 per Gaussian, RGB composited (SSSGS_FORWARD_SHADING).
    # The rasteriser is fed the oracle's MLP outputs so that the 1e-4 bar applies to the frames.
    import dataclasses
    import torch
    from paper_2408_12282_b200 import binding
    scene = scenes.make_scene(3, n=20000, width=width, height=width, lights=n_lights)
    cam = dataclasses.replace(scene.cameras[0], bg=np.float32([0.05, 0.1, 0.2]))
    scene = dataclasses.replace(scene, cameras=[cam])
    lights = scene.lights[0]
    pre = np.zeros((n_lights, scene.n, 4), np.float32)
    for l in range(n_lights):
        x = oracle.mlp_inputs(scene, cam, lights[l].position)
        pre[l] = oracle.mlp_forward(x, scene.mlp, 0).astype(np.float32)
    R = binding.Renderer(scene)
    try:
        out = R.render(cams=[cam], lights=lights, want=("rgb",), precomputed=pre, forward=True)
        torch.cuda.synchronize()
        got = out["rgb"].cpu().numpy()
        # and with the library's own MLP: same frames up to the fp16 MLP tolerance
        own = R.render(cams=[cam], lights=lights, want=("rgb",), forward=True)
        torch.cuda.synchronize()
        own = own["rgb"].cpu().numpy()
        with pytest.raises(binding.SssgsError):
            R.render(cams=[cam], lights=lights, want=("rgb", "gbuffer"), forward=True)
    finally:
        R.close()
    geo = None
    for l in range(n_lights):
        r = oracle.forward_frame(scene, 0, l, mlp_out=pre[l].astype(np.float64), geometry=geo)
        geo = geo or r
        st = ~r.comp.unstable
        # per-Gaussian shading runs in fp32 on the GPU: colours carry ~1e-6 relative error, and a
        # specular highlight at a Gaussian's centre can be large (HDR): scale the bar with the value
        tol = 1e-4 * np.maximum(1.0, np.abs(r.rgb))
        err = np.abs(got[l] - r.rgb)
        assert (err[st] <= tol[st]).all(), f"light {l}: worst {err[st].max():.3e}"
        # pixels with a flagged decision: what those decisions can move the composited colour (channels 10-12) and
        # the coverage (times the background) by -- the derived bound of the deferred path, not a flat figure
        ch = np.zeros((int(scene.n), 14))
        ch[:, 10:13] = r.colors
        ub = unstable_bound(r.comp.gbuf, r.comp.flags, ch)
        bound = ub[..., 10:13] + ub[..., 14:15] * np.asarray(cam.bg, np.float64) + tol
        assert (err[~st] <= bound[~st]).all(), f"light {l}: unstable pixels beyond their decisions' reach"
        assert np.percentile(np.abs(own[l] - r.rgb)[st], 99.9) <= 1e-3   # own fp16 MLP vs the float64 MLP's frames


def test_weight_cache_overflow_falls_back_to_the_list_walks(monkeypatch):
    # In a sweep the visibility pre-pass caches the compositing weights and the per-light walks stream
    # the cache.  The pool is bounded: when it runs out the list walks run instead.  Same frames.
    scene = scenes.make_scene(3, n=40000, width=656, height=656, lights=6)
    want = ("rgb", "gbuffer", "counters")
    cached = gpu_render(scene, want=want, lights=scene.lights[0])
    monkeypatch.setenv("SSSGS_WC_CHUNKS", "16")       # 512 cached entries for a frame that needs ~1e5
    fallback = gpu_render(scene, want=want, lights=scene.lights[0])
    monkeypatch.delenv("SSSGS_WC_CHUNKS")
    full = gpu_render(scene, want=want + ("mlp_out",), lights=scene.lights[0])  # no pre-pass at all
    for k in ("rgb", "gbuffer"):
        np.testing.assert_array_equal(cached[k].view(np.uint32), full[k].view(np.uint32))
        np.testing.assert_array_equal(fallback[k].view(np.uint32), full[k].view(np.uint32))


@pytest.mark.parametrize("cfg,n,width,height", [
    (2, 50000, 320, 240),
    (1, 50000, 656, 200),   # dense small image: more long tile lists than the long-list CTAs of the mixed kernel
])
def test_run_to_run_determinism(cfg, n, width, height):
    scene = scenes.make_scene(cfg, n=n, width=width, height=height)
    a = gpu_render(scene)
    for _ in range(3):
        b = gpu_render(scene)
        for k in ("rgb", "gbuffer", "sorted_vals", "tile_ranges", "mlp_out"):
            np.testing.assert_array_equal(a[k].view(np.uint32) if a[k].dtype == np.float32 else a[k],
                                          b[k].view(np.uint32) if b[k].dtype == np.float32 else b[k])
    # and the same frame when other outputs are requested
    c = gpu_render(scene, want=("rgb", "counters"))
    np.testing.assert_array_equal(a["rgb"].view(np.uint32), c["rgb"].view(np.uint32))


def _tight_scenes():
    yield from _small_scenes()
    yield "full_image", custom_scene([[0, 0, 0]], 5.0, width=50, height=37)
    yield "huge_near_plane", custom_scene([[0, -3.7, 0], [0.1, 0, 0]], [[2.0, 0.01, 2.0], [0.05] * 3], width=96, height=64)
    yield "sub_threshold_opacity", custom_scene(np.random.default_rng(2).uniform(-0.5, 0.5, (200, 3)), 0.08,
                                                opacities=np.random.default_rng(3).choice([0.002, 1.0 / 255, 0.004, 0.5], 200))
    yield "dense_1080_like", scenes.make_scene(4, n=20000, width=200, height=120, views=1)
    yield "one_slot_walk", scenes.make_scene(3, n=30000, width=672, height=640, lights=2)   # 1680 tiles: bit-identical


@pytest.mark.parametrize("name,scene", list(_tight_scenes()))
def test_tight_lists_satisfy_s5_and_render_the_same_frames(name, scene):
    # SSSGS_TIGHT_LISTS: sub-sequence of the canonical list, superset of the pairs with
    # alpha >= 1/255 at a pixel of the tile, same order, identical image (bit for bit).
    want = ("rgb", "gbuffer", "sorted_keys", "sorted_vals", "tile_ranges", "counters")
    cam = scene.cameras[0]
    lights = scene.lights[0]
    canon = gpu_render(scene, want=want, cams=[cam], lights=lights)
    tight = gpu_render(scene, want=want, cams=[cam], lights=lights, tight=True)
    proj = oracle.project(scene, cam)
    keys, vals, ranges = oracle.build_lists(proj)
    hit = oracle.tile_hits(scene, cam, proj, vals, ranges)
    It, n_hit = check_tight_lists(tight, keys, vals, ranges, hit)
    print(f"{name}: canonical {len(keys)}, tight {It}, minimal {n_hit}")
    assert canon["counters"][0][1] == len(keys) and tight["counters"][0][0] == canon["counters"][0][0]
    assert n_hit <= It <= len(keys)
    if len(keys) > 2000:
        assert It < len(keys)       # it really is tighter
    # the blended (pixel, entry) pairs are the same; with one entry slot per warp (> 1600 tiles) so is the order of
    # every sum: bit-identical frames.  The 2- and 4-slot walks of small images group the entries of a staged batch
    # by position, so another list changes which partial sum an entry joins (last-bit differences).
    tiles = proj.tiles_x * proj.tiles_y
    for k in ("rgb", "gbuffer"):
        if tiles > 1600:
            np.testing.assert_array_equal(tight[k].view(np.uint32), canon[k].view(np.uint32))
        else:
            np.testing.assert_allclose(tight[k], canon[k], rtol=5e-5, atol=2e-6)


def test_tight_lists_in_a_sweep_render_the_same_frames():
    # the call shape bench.py times: sweep (pre-pass, row-skipping MLP, cached walks) over tight lists
    scene = scenes.make_scene(3, n=40000, width=656, height=656, lights=11)
    want = ("rgb", "gbuffer", "counters")
    a = gpu_render(scene, want=want, lights=scene.lights[0])
    b = gpu_render(scene, want=want, lights=scene.lights[0], tight=True)
    assert 0 < b["counters"][0][1] < a["counters"][0][1] and b["counters"][0][4] == a["counters"][0][4]
    for k in ("rgb", "gbuffer"):
        np.testing.assert_array_equal(a[k].view(np.uint32), b[k].view(np.uint32))


def test_empty_scene_and_zero_opacity():
    s = custom_scene(np.zeros((0, 3)), 0.05, width=40, height=24, bg=(0.1, 0.2, 0.3))
    g = gpu_render(s, want=("rgb", "gbuffer", "counters", "tile_ranges"))
    assert (g["gbuffer"][0][..., :15] == 0).all() and (g["gbuffer"][0][..., 15] == 1).all()
    np.testing.assert_allclose(g["rgb"][0], np.broadcast_to(np.float32([0.1, 0.2, 0.3]), g["rgb"][0].shape))
    assert (g["counters"][0][:3] == 0).all() and (g["tile_ranges"] == 0).all()
    s = scenes.make_scene(1, n=500, width=64, height=64)
    s.opacities[:] = 0
    g = gpu_render(s, want=("rgb", "gbuffer"))
    assert (g["gbuffer"][0][..., :15] == 0).all() and (g["rgb"] == 0).all()


def test_edge_scenes_match_oracle():
    cases = {
        "pixel_centre": custom_scene([[0, 0, 0]], 0.05, opacities=0.7, width=65, height=65),
        "behind_and_near": custom_scene([[0, -5, 0], [0, -3.85, 0], [0, -3.75, 0], [50, 0, 0], [0, 0, 0]],
                                        [[0.05] * 3, [0.05] * 3, [0.001] * 3, [0.05] * 3, [1e-8, 0.05, 0.05]]),
        "full_image": custom_scene([[0, 0, 0]], 5.0, width=50, height=37),
        "equal_depth": custom_scene(np.stack([np.linspace(-0.05, 0.05, 40), np.zeros(40), np.zeros(40)], 1), 0.03,
                                    width=32, height=32),
        "coincident": custom_scene(np.zeros((5, 3)), 0.05, opacities=0.3, width=33, height=33),
        "ragged_1080_like": scenes.make_scene(4, n=5000, width=96, height=54, views=1),
    }
    for name, s in cases.items():
        r = oracle.render_frame(s)
        pre = r.mlp_out.astype(np.float32)[None]
        r = oracle.render_frame(s, mlp_out=pre[0].astype(np.float64))
        g = gpu_render(s, precomputed=pre)
        check_lists(s, g, r)
        check_gbuffer(g["gbuffer"][0], r)
        check_shading(s, g, 0, 0, 0)


def test_instance_overflow_sets_flag_and_host_call_reports_it():
    from paper_2408_12282_b200 import binding
    s = scenes.make_scene(1, n=1000, width=64, height=64)
    I = int(oracle.project(s, s.cameras[0]).touched.sum())
    g = gpu_render(s, want=("rgb", "counters"), max_instances=I)       # exactly at capacity: fine
    assert g["counters"][0][1] == I and g["counters"][0][2] == 0
    g = gpu_render(s, want=("rgb", "counters"), max_instances=I - 1)   # one short: flagged
    assert g["counters"][0][1] == I and g["counters"][0][2] == 1
    with pytest.raises(binding.SssgsError) as ei:
        binding.render_host(s, max_instances=I - 1)
    assert ei.value.code == binding.SSSGS_EOVERFLOW


def test_render_host_equals_render():
    from paper_2408_12282_b200 import binding
    s = scenes.make_scene(2, n=10000, width=128, height=128)
    a = gpu_render(s)
    b = binding.render_host(s, want=ALL)
    for k in ("rgb", "gbuffer", "mlp_out", "tile_ranges"):
        np.testing.assert_array_equal(a[k].view(np.uint8), b[k].view(np.uint8))


def test_invalid_arguments_fail_cleanly():
    from paper_2408_12282_b200 import binding
    cfg = binding.sssgs_config()
    cfg.max_gaussians, cfg.max_width, cfg.max_height, cfg.max_instances = 10, 0, 16, 100
    with pytest.raises(binding.SssgsError):
        binding.sssgs_create(cfg)
    s = scenes.make_scene(1, n=100, width=32, height=32)
    r = binding.Renderer(s)
    try:
        big = scenes.look_at_camera((0, -4, 0), 64, 64, 40.0)
        with pytest.raises(binding.SssgsError) as ei:
            r.render(cams=[big])
        assert ei.value.code == binding.SSSGS_ECAPACITY
        # one image size per call: frames are laid out [F][H][W]
        small = scenes.look_at_camera((0, -4, 0), 16, 32, 40.0)
        with pytest.raises(binding.SssgsError) as ei:
            r.render(cams=[s.cameras[0], small])
        assert ei.value.code == binding.SSSGS_EINVAL
    finally:
        r.close()


def test_full_size_cfg2_matches_oracle():
    # BASELINE configs[1] at full size, in the launch configuration bench.py times
    scene = scenes.make_scene(2)
    gpu = gpu_render(scene)
    r = oracle.render_frame(scene, mlp_mode=2)
    check_lists(scene, gpu, r)
    e = np.abs(gpu["mlp_out"][0] - r.mlp_out)
    assert (e <= 1e-3).mean() >= 0.999 and e.max() <= 3e-3
    y_ref = oracle.mlp_forward(r.x, scene.mlp, 0)
    assert np.abs(gpu["mlp_out"][0] - y_ref).max() <= 1e-2   # north_star's bar, all four outputs
    # light-independent channels do not depend on the MLP: 1e-4 on stable pixels
    st = ~r.comp.unstable
    assert np.abs(gpu["gbuffer"][0][..., :10] - r.gbuf[..., :10])[st].max() <= 1e-4
    assert np.abs(gpu["gbuffer"][0][..., 14:] - r.gbuf[..., 14:])[st].max() <= 1e-4
    check_shading(scene, gpu, 0, 0, 0)
    err = np.abs(gpu["rgb"][0] - r.rgb)[st]
    assert np.percentile(err, 99.9) <= 1e-4 and err.max() <= 1e-3     # measured 1.8e-5 / 1.0e-4


@pytest.mark.parametrize("seed", range(10))
def test_random_scenes(seed):
    """Seeded random (config, size, image, lights) draws: lists bit-exact, the frames of the benchmarked call
    shape (RGB only: row skipping and weight cache from 4 lights on) equal those of the full-output call
    (bit for bit where both walk one entry per warp step), RGB within the S9 bound of the oracle."""
    rng = np.random.default_rng(7000 + seed)
    cfg = int(rng.choice([1, 2, 3, 4, 5]))
    n = int(rng.integers(500, 60000))
    w, h = int(rng.choice([96, 200, 333, 656, 700])), int(rng.choice([64, 200, 333, 656]))
    scene = scenes.make_scene(cfg, n=n, width=w, height=h, lights=int(rng.choice([1, 3, 4, 5, 8, 9, 13, 16])), views=1)
    nl = len(scene.lights[0])
    on = gpu_render(scene, want=("rgb", "counters", "sorted_keys", "sorted_vals", "tile_ranges"), lights=scene.lights[0])
    off = gpu_render(scene, want=("rgb", "counters", "mlp_out"), lights=scene.lights[0])
    cam = scene.cameras[0]
    proj = oracle.project(scene, cam)
    keys, vals, ranges = oracle.build_lists(proj)
    ref = type("R", (), dict(n_vis=int(proj.visible.sum()), n_instances=len(keys), keys=keys, vals=vals, ranges=ranges))
    check_lists(scene, on, ref, 0)
    tiles = ((w + 15) // 16) * ((h + 15) // 16)
    if tiles > 1600 or nl < 4:
        np.testing.assert_array_equal(on["rgb"].view(np.uint32), off["rgb"].view(np.uint32))
    else:
        np.testing.assert_allclose(on["rgb"], off["rgb"], rtol=5e-5, atol=2e-6)
    for l in sorted({0, nl - 1}):
        r = oracle.render_frame(scene, 0, l, mlp_out=off["mlp_out"][l].astype(np.float64))
        d = np.abs(off["rgb"][l].astype(np.float64) - r.rgb)
        tol = np.where(r.comp.unstable[..., None], 5e-2, 1e-4) * np.maximum(1.0, np.abs(r.rgb))
        assert (d <= tol).all(), f"light {l}: worst {d.max():.3e}"
