"""Two contexts alive in one process: per-(kernel, device) attribute cache, device guard.
Each context renders a different scene with a different MLP shape (different dynamic shared memory sizes for the
same kernels); calls are interleaved; every frame must equal, bit for bit, the frame of a context that lived
alone."""
import numpy as np
import pytest

from paper_2408_12282_b200 import scenes

pytestmark = pytest.mark.gpu


def _alone(scene, **kw):
    import torch
    from paper_2408_12282_b200 import binding
    R = binding.Renderer(scene)
    try:
        out = R.render(cams=scene.cameras[:1], lights=scene.lights[0], want=("rgb", "gbuffer"), **kw)
        torch.cuda.synchronize()
        return {k: v.cpu().numpy() for k, v in out.items()}
    finally:
        R.close()


def test_two_contexts_interleaved():
    import torch
    from paper_2408_12282_b200 import binding
    a = scenes.make_scene(1, lights=2)                          # 64-wide trunk
    b = scenes.make_scene(3, n=20000, width=200, height=120, lights=5)   # 128-wide trunk, sweep path (>= 4 lights)
    ref_a, ref_b = _alone(a), _alone(b, tight=True)
    Ra, Rb = binding.Renderer(a), binding.Renderer(b)
    try:
        s1, s2 = torch.cuda.Stream(), torch.cuda.Stream()
        outs = []
        for it in range(3):
            with torch.cuda.stream(s1):
                oa = Ra.render(cams=a.cameras[:1], lights=a.lights[0], want=("rgb", "gbuffer"))
            with torch.cuda.stream(s2):
                ob = Rb.render(cams=b.cameras[:1], lights=b.lights[0], want=("rgb", "gbuffer"), tight=True)
            outs.append((oa, ob))
        torch.cuda.synchronize()
        for oa, ob in outs:
            for k in ("rgb", "gbuffer"):
                np.testing.assert_array_equal(oa[k].cpu().numpy().view(np.uint32), ref_a[k].view(np.uint32))
                np.testing.assert_array_equal(ob[k].cpu().numpy().view(np.uint32), ref_b[k].view(np.uint32))
        # destroying one context leaves the other usable
        Ra.close()
        ob = Rb.render(cams=b.cameras[:1], lights=b.lights[0], want=("rgb",), tight=True)
        torch.cuda.synchronize()
        np.testing.assert_array_equal(ob["rgb"].cpu().numpy().view(np.uint32), ref_b["rgb"].view(np.uint32))
    finally:
        Ra.close()
        Rb.close()


def test_context_restores_the_callers_device():
    import torch
    from paper_2408_12282_b200 import binding
    s = scenes.make_scene(1, lights=1)
    before = torch.cuda.current_device()
    R = binding.Renderer(s, device=0)
    try:
        R.render(cams=s.cameras[:1], lights=s.lights[0], want=("rgb",))
        torch.cuda.synchronize()
        assert torch.cuda.current_device() == before
    finally:
        R.close()
