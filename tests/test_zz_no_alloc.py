"""sssgs_mlp_eval_static: the MLP without a context and without any device allocation.

Some programs that embed this library may not call cudaMalloc: a host that handed the whole GPU to its own memory
pool when it started (a library's cudaMalloc then fails or eats the pool's head-room), or a thread with a latency
budget (cudaMalloc / cudaFree take the driver's allocator lock and can wait for the device to drain).  For them
the library has one entry point whose only scratch -- the network's parameters repacked as tensor-core operand
tiles -- sits in a fixed 192 KB array inside the library image instead of in a context's workspace.

What is checked here: the values that entry point writes equal, bit for bit, the `mlp_out` that the ordinary
context-based sssgs_render produces for the same scene, camera and lights (same kernel, same per-row arithmetic;
the GPU-vs-GPU comparisons of this suite use exact equality), and are within the suite's MLP bar (3e-3) of the
fp16-emulating oracle.  Two calls are made back to back on one stream, the second with a different and smaller
network, more Gaussians and another light count: every call shares the one array, which still holds the first
network when the second call starts, so the second result shows that nothing stale leaks in.  The limits are
checked too (they are decided on the host before anything is enqueued, so those cases need no GPU).

This file sorts last on purpose: `pytest -x` stops at the first failure, and a failure here must not hide the
other tests.  It passes alone in a fresh process and after the rest of the suite (the first call on a device
resolves the array's device address; nothing else carries over between calls).
"""

import numpy as np
import pytest

from paper_2408_12282_b200 import binding, scenes


def _fake_gaussians(n, feat_dim):
    """A descriptor with plausible (aligned, never dereferenced) pointers: for the host-side limit checks."""
    ptrs = {f: 0x10000 for f in ("means", "scales", "rotations", "opacities", "normals", "base_color",
                                 "roughness", "metallic", "subsurface", "vis_sh", "feat")}
    return binding.make_gaussians(n, ptrs, 1, feat_dim)


def _spec(in_dim, trunk):
    return scenes._make_mlp(np.random.default_rng(0), in_dim, list(trunk), [], scenes.ACT_RELU)


def test_static_limits_are_rejected_with_a_clear_error():
    cam = binding.make_camera(scenes.look_at_camera((0.0, -4.0, 0.0), 64, 64, 40.0))
    lights = (binding.sssgs_light * 9)()
    spec = _spec(40, [64, 64])
    m = binding.make_mlp(spec, 0x20000, spec.params.nbytes)
    g = _fake_gaussians(1000, 0)
    # more lights than one batch
    with pytest.raises(binding.SssgsError) as ei:
        binding.sssgs_mlp_eval_static(0, g, m, cam, lights, 9, 0x30000)
    assert ei.value.code == binding.SSSGS_ECAPACITY and "SSSGS_STATIC_MAX_LIGHTS" in str(ei.value)
    # a network sssgs_render would still take (196 KB of packed operands fit its shared-memory budget) but the
    # 192 KB static array does not hold
    big = _spec(128, [128] * 5)
    mb = binding.make_mlp(big, 0x20000, big.params.nbytes)
    with pytest.raises(binding.SssgsError) as ei:
        binding.sssgs_mlp_eval_static(0, _fake_gaussians(1000, 88), mb, cam, lights, 1, 0x30000)
    assert ei.value.code == binding.SSSGS_ECAPACITY and "SSSGS_STATIC_SCRATCH_BYTES" in str(ei.value)
    assert str(binding.SSSGS_STATIC_SCRATCH_BYTES) in str(ei.value)
    # argument errors
    with pytest.raises(binding.SssgsError) as ei:
        binding.sssgs_mlp_eval_static(0, g, m, cam, lights, 1, 0)          # no output
    assert ei.value.code == binding.SSSGS_EINVAL
    with pytest.raises(binding.SssgsError) as ei:
        binding.sssgs_mlp_eval_static(0, g, m, cam, lights, 1, 0x30004)    # misaligned output
    assert ei.value.code == binding.SSSGS_EINVAL
    # nothing to do: validated, nothing enqueued, no device touched
    binding.sssgs_mlp_eval_static(0, _fake_gaussians(0, 0), m, cam, lights, 1, 0)
    binding.sssgs_mlp_eval_static(0, g, m, cam, lights, 0, 0)


def _existing_path(scene, cam, lights):
    """mlp_out [L][n][4] of the context-based render (the path every other test of this suite exercises)."""
    import torch
    R = binding.Renderer(scene)
    try:
        out = R.render(cams=[cam], lights=lights, want=("mlp_out",))
        torch.cuda.synchronize()
        return out["mlp_out"].cpu().numpy()
    finally:
        R.close()


class _DeviceScene:
    """The scene's arrays on the device, allocated up front (torch: memory only) -- the static call itself is
    handed pointers and allocates nothing."""

    def __init__(self, scene, n_light):
        import torch
        dev = torch.device("cuda", 0)
        self.t = {}
        for f in binding._FIELDS:
            a = np.ascontiguousarray(getattr(scene, f), dtype=np.float32)
            self.t[f] = torch.from_numpy(a if a.size else np.zeros(4, np.float32)).to(dev)
        self.params = torch.from_numpy(np.ascontiguousarray(scene.mlp.params, np.float32)).to(dev)
        feat_dim = int(scene.feat.shape[1]) if scene.feat.ndim == 2 else 0
        self.g = binding.make_gaussians(int(scene.n), {f: self.t[f].data_ptr() for f in binding._FIELDS},
                                        scene.vis_sh_degree, feat_dim)
        self.m = binding.make_mlp(scene.mlp, self.params.data_ptr(), self.params.numel() * 4)
        # NaN-filled: every element must be written by the call
        self.out = torch.full((int(scene.n), n_light, 4), float("nan"), dtype=torch.float32, device=dev)


@pytest.mark.gpu
def test_static_mlp_equals_the_context_path_on_two_calls_in_a_row():
    import torch
    import oracle
    # call 1: 128-wide four-layer network on a 72-wide input (164 KB of packed operands), 6 lights, ragged row tail
    a = scenes.make_scene(5, n=20_037, width=128, height=128, views=1, lights=6)
    # call 2: the paper's architecture ([64, 32, 32] trunk, incident head with a hidden layer,
    # Leaky-ReLU; ~40 KB packed), more Gaussians, 2 lights
    b = scenes.make_scene(6, n=33_001, width=128, height=128, views=1, lights=2)
    ref_a = _existing_path(a, a.cameras[0], a.lights[0])
    ref_b = _existing_path(b, b.cameras[0], b.lights[0])

    da, db = _DeviceScene(a, 6), _DeviceScene(b, 2)
    la = (binding.sssgs_light * 6)(*[binding.make_light(l) for l in a.lights[0]])
    lb = (binding.sssgs_light * 2)(*[binding.make_light(l) for l in b.lights[0]])
    torch.cuda.synchronize()
    st = torch.cuda.current_stream().cuda_stream
    # two calls in a row on one stream, no synchronisation in between
    binding.sssgs_mlp_eval_static(0, da.g, da.m, binding.make_camera(a.cameras[0]), la, 6, da.out.data_ptr(), st)
    binding.sssgs_mlp_eval_static(0, db.g, db.m, binding.make_camera(b.cameras[0]), lb, 2, db.out.data_ptr(), st)
    torch.cuda.synchronize()
    got_a = da.out.cpu().numpy().transpose(1, 0, 2)   # [n][L][4] -> [L][n][4]
    got_b = db.out.cpu().numpy().transpose(1, 0, 2)
    assert np.isfinite(got_a).all() and np.isfinite(got_b).all()
    np.testing.assert_array_equal(got_a, ref_a)
    np.testing.assert_array_equal(got_b, ref_b)
    # and the second call against the oracle, at the MLP bar of tests/test_gpu_parity.py::test_mlp_outputs
    for l in range(2):
        x = oracle.mlp_inputs(b, b.cameras[0], b.lights[0][l].position)
        y = oracle.mlp_forward(x, b.mlp, 2)
        assert np.abs(got_b[l].astype(np.float64) - y).max() <= 3e-3

    # once more in the other order (large network after the small one), same answers; with everything warm, the
    # device's free memory (cudaMemGetInfo: sees every allocation of the process, not only torch's) does not move
    da.out.fill_(float("nan"))
    torch.cuda.synchronize()
    free_before = torch.cuda.mem_get_info()[0]
    binding.sssgs_mlp_eval_static(0, da.g, da.m, binding.make_camera(a.cameras[0]), la, 6, da.out.data_ptr(), st)
    torch.cuda.synchronize()
    assert torch.cuda.mem_get_info()[0] == free_before
    np.testing.assert_array_equal(da.out.cpu().numpy().transpose(1, 0, 2), ref_a)
