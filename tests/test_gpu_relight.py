"""Parity of sssgs_relight (second half; the relit view as the sum over a precomputed
reflectance field scaled by the environment illumination) with oracle.relight, element by element.

Bar: the kernel accumulates the L products in fp32 in light order with fused multiply-adds; the oracle in float64.
|got - ref| <= L 2^-23 sum_l |w_l f_l| per element (one rounding of at most 2^-24 relative per partial sum, doubled
for slack), written in `_check`.
"""
import dataclasses

import numpy as np
import pytest

import oracle
from paper_2408_12282_b200 import binding, scenes

pytestmark = pytest.mark.gpu


def _relight_gpu(frames, w):
    import torch
    L, H, W = frames.shape[:3]
    f = torch.from_numpy(np.ascontiguousarray(frames, np.float32)).cuda() if L else torch.zeros(4, device="cuda")
    wt = torch.from_numpy(np.ascontiguousarray(w, np.float32)).cuda() if L else torch.zeros(4, device="cuda")
    out = torch.full((H, W, 3), float("nan"), device="cuda")
    binding.sssgs_relight(0, f.data_ptr() if L else None, L, H * W, wt.data_ptr() if L else None, out.data_ptr(),
                          torch.cuda.current_stream().cuda_stream)
    torch.cuda.synchronize()
    return out.cpu().numpy()


def _check(got, frames, w):
    f64, w64 = frames.astype(np.float32).astype(np.float64), w.astype(np.float32).astype(np.float64)
    ref = oracle.relight(f64, w64)
    mag = oracle.relight(np.abs(f64), np.abs(w64))
    L = frames.shape[0]
    tol = max(L, 1) * 2.0 ** -23 * mag + 1e-37
    err = np.abs(got.astype(np.float64) - ref)
    assert np.isfinite(got).all()
    assert (err <= tol).all(), f"worst {err.max():.3e} (tolerance there {tol.flat[np.argmax(err)]:.3e})"
    return float((err / np.maximum(tol, 1e-37)).max())


# vector path: pixel counts that are multiples of 4 (whole warp units, a ragged last unit, less than one unit);
# scalar path: pixel counts that are not (later frames are then not 16-byte aligned); empty stack
@pytest.mark.parametrize("L,H,W", [(1, 16, 16), (7, 33, 20), (3, 2, 6), (5, 17, 19), (2, 1, 1), (64, 200, 200), (9, 128, 96), (0, 8, 8)])
def test_relight_matches_oracle(L, H, W):
    rng = np.random.default_rng(100 * L + H)
    frames = rng.uniform(0.0, 2.0, (L, H, W, 3)).astype(np.float32)
    frames[rng.random(frames.shape) < 0.1] *= 50.0                     # HDR highlights
    w = rng.uniform(-0.5, 3.0, (L, 3)).astype(np.float32)               # an asymmetric [L, 3]: a transposed read fails
    got = _relight_gpu(frames, w)
    if L == 0:
        assert not got.any()
        return
    r = _check(got, frames, w)
    print(f"relight L={L} {W}x{H}: worst error / tolerance {r:.3f}")


def test_relight_of_a_rendered_olat_stack_equals_the_summed_render():
    # the two halves of (f).1 meet: the OLAT frames of the library (white lights, black background), relit with
    # weights w_l, equal ONE SSSGS_SUM_LIGHTS render under lights of intensity w_l (Eq. 7 is linear in the intensity)
    import torch
    s = scenes.make_scene(3, n=30000, width=160, height=160, lights=6)
    cam = s.cameras[0]
    assert not np.any(cam.bg)
    rng = np.random.default_rng(12)
    w = rng.uniform(0.2, 1.5, (6, 3)).astype(np.float32)
    coloured = [dataclasses.replace(l, intensity=w[i]) for i, l in enumerate(s.lights[0])]
    R = binding.Renderer(s)
    try:
        olat = R.render(cams=[cam], lights=s.lights[0], want=("rgb",))["rgb"]
        tot = R.render(cams=[cam], lights=coloured, want=("rgb",), sum_lights=True)["rgb"]
        wt = torch.from_numpy(w).cuda()
        out = torch.empty((cam.height, cam.width, 3), device="cuda")
        binding.sssgs_relight(0, olat.data_ptr(), 6, cam.height * cam.width, wt.data_ptr(), out.data_ptr(),
                              torch.cuda.current_stream().cuda_stream)
        torch.cuda.synchronize()
        olat, tot, out = olat.cpu().numpy(), tot.cpu().numpy()[0], out.cpu().numpy()
    finally:
        R.close()
    _check(out, olat, w)                                                # the kernel against the oracle on the GPU's frames
    ref = oracle.relight(olat.astype(np.float64), w.astype(np.float64))
    assert np.abs(ref).max() > 0.05
    np.testing.assert_allclose(tot, ref, rtol=2e-5, atol=2e-5)         # and against the summed render (fp32 shading twice)


def test_relight_full_size_stack():
    # configs[4]'s frame shape: 16 frames of 1024 x 1024 (201 MB in, 12.6 MB out), every output element checked
    rng = np.random.default_rng(3)
    L, H, W = 16, 1024, 1024
    frames = rng.random((L, H, W, 3), dtype=np.float32) * 2.0
    w = rng.uniform(0.0, 2.0, (L, 3)).astype(np.float32)
    got = _relight_gpu(frames, w)
    ref = np.zeros((H, W, 3))
    mag = np.zeros((H, W, 3))
    for l in range(L):
        t = frames[l].astype(np.float64) * w[l].astype(np.float64)
        ref += t
        mag += np.abs(t)
    assert (np.abs(got - ref) <= L * 2.0 ** -23 * mag).all()


def test_relight_rejects_bad_arguments():
    import torch
    f = torch.zeros((2, 8, 8, 3), device="cuda")
    w = torch.ones((2, 3), device="cuda")
    with pytest.raises(binding.SssgsError):       # out inside the stack
        binding.sssgs_relight(0, f.data_ptr(), 2, 64, w.data_ptr(), f.data_ptr() + 64 * 12)
    with pytest.raises(binding.SssgsError):       # misaligned output
        binding.sssgs_relight(0, f.data_ptr(), 1, 64, w.data_ptr(), f.data_ptr() + 64 * 12 + 4)
    with pytest.raises(binding.SssgsError):
        binding.sssgs_relight(0, None, 2, 64, w.data_ptr(), f.data_ptr())
    with pytest.raises(binding.SssgsError):
        binding.sssgs_relight(0, f.data_ptr(), -1, 64, w.data_ptr(), f.data_ptr())
    binding.sssgs_relight(0, None, 0, 0, None, None)   # nothing to do
