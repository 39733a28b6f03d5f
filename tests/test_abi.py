"""CPU checks of the boundary: libsssgs.so builds, loads, exports every symbol that
include/sssgs.h declares, validates its configuration on the host, and fails loudly (no CPU
fallback) when there is no CUDA device.  No compute is launched here."""
import ctypes
import os
import re

import pytest

from paper_2408_12282_b200 import binding, build

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def libpath():
    return build.build()


def _declared_functions():
    src = open(os.path.join(ROOT, "include", "sssgs.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(sssgs_[a-z_]+)\s*\(", src)))


def test_header_symbols_are_exported(libpath):
    names = _declared_functions()
    assert set(names) == set(binding.EXPORTS), names
    L = ctypes.CDLL(libpath)
    for n in names:
        assert hasattr(L, n), f"{n} declared in sssgs.h but not exported"


def test_struct_layouts_match_header(libpath):
    # sizes implied by the header's field lists on LP64
    assert ctypes.sizeof(binding.sssgs_camera) == 4 * (9 + 3 + 6) + 8 + 4 + 12
    assert ctypes.sizeof(binding.sssgs_light) == 24
    assert ctypes.sizeof(binding.sssgs_out) == 9 * 8
    assert ctypes.sizeof(binding.sssgs_gaussians) == 8 + 10 * 8 + 8 + 8 + 8
    assert ctypes.sizeof(binding.sssgs_config) == 64
    assert ctypes.sizeof(binding.sssgs_mlp) == 4 * (2 + 8 + 1 + 2 + 3) + 3 * 8 + 8   # ints/float, 3 pointers/size_t, compute + pad
    assert binding.sssgs_mlp.compute.offset == 88 and binding.sssgs_mlp.params.offset == 64


def test_workspace_bytes_and_config_validation(libpath):
    cfg = binding.sssgs_config()
    cfg.max_gaussians, cfg.max_width, cfg.max_height, cfg.max_instances = 100000, 512, 512, 2_000_000
    a = binding.sssgs_workspace_bytes(cfg)
    assert a > 100000 * (48 + 44) + 2_000_000 * 16
    cfg.max_instances = 4_000_000
    assert binding.sssgs_workspace_bytes(cfg) > a
    cfg.max_width = 0
    assert binding.sssgs_workspace_bytes(cfg) == 0
    cfg.max_width = 512
    cfg.max_lights_per_pass = 3
    assert binding.sssgs_workspace_bytes(cfg) == 0
    cfg.max_lights_per_pass = 4
    cfg.max_instances = 1 << 30
    assert binding.sssgs_workspace_bytes(cfg) == 0


def test_create_fails_loudly_without_gpu(libpath):
    import torch
    if torch.cuda.is_available():
        pytest.skip("a CUDA device is present")
    cfg = binding.sssgs_config()
    cfg.max_gaussians, cfg.max_width, cfg.max_height, cfg.max_instances = 10, 16, 16, 100
    with pytest.raises(binding.SssgsError) as ei:
        binding.sssgs_create(cfg)
    assert ei.value.code in (binding.SSSGS_ECUDA, binding.SSSGS_EARCH)
    assert "fallback" in str(ei.value) or "CUDA" in str(ei.value)


def test_destroy_is_null_safe(libpath):
    binding.sssgs_destroy(None)


def test_product_does_not_import_oracle():
    pkg = os.path.join(ROOT, "paper_2408_12282_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                txt = open(os.path.join(dirpath, f)).read()
                assert "import oracle" not in txt and "from oracle" not in txt and "liboracle" not in txt, f
