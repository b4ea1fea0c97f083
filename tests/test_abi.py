"""Host-side checks that need no GPU: the C-ABI library builds, loads, exports every symbol that
include/vs.h declares, validates arguments, and fails loudly (no CPU fallback) without a device."""
import ctypes as C
import os
import re

import numpy as np
import pytest

from paper_2409_02482_b200 import binding

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def test_library_exports_every_declared_symbol():
    lib = binding.load_library()
    header = open(os.path.join(ROOT, "include", "vs.h")).read()
    header = re.sub(r"/\*.*?\*/", "", header, flags=re.S)
    declared = set(re.findall(r"\b(vs_[a-z_]+)\s*\(", header))
    assert declared == set(binding.EXPORTS)
    for name in declared:
        assert hasattr(lib, name), name
    assert "sm_100a" in binding.vs_version()


def test_struct_layouts_match_header():
    assert C.sizeof(binding.vs_camera) == 64
    assert C.sizeof(binding.vs_render_params) == 36
    assert C.sizeof(binding.vs_layer_desc) == 56
    assert C.sizeof(binding.vs_scene_desc) == 24
    assert C.sizeof(binding.vs_render_stats) == 104
    assert C.sizeof(binding.vs_layer_desc_banded) == 104      # 5 geometry fields (40) + 4 pointers + 2 x 4 uint32
    assert C.sizeof(binding.vs_scene_desc_banded) == 32
    assert C.sizeof(binding.vs_aov_buffers) == 32


def test_argument_validation_happens_before_any_cuda_work():
    lib = binding.load_library()
    h = C.c_void_p(123)
    assert lib.vs_scene_create(None, None, C.byref(h)) == binding.VS_ERR_INVALID_ARG and h.value is None
    layer = binding.vs_layer_desc()
    for k, deg in ((0, 1), (10, 1), (3, 4)):
        desc = binding.vs_scene_desc(k, deg, 0, 0, (binding.vs_layer_desc * 1)(layer))
        assert lib.vs_scene_create(C.byref(desc), None, C.byref(h)) == binding.VS_ERR_INVALID_ARG
        assert lib.vs_last_error() != b""
    p = binding.make_params(8, 8)
    assert lib.vs_render(None, None, 0, C.byref(p), None, None, None) == binding.VS_ERR_INVALID_ARG
    lib.vs_scene_destroy(None)  # NULL is a no-op


def test_no_cpu_fallback_without_a_device():
    import torch
    if torch.cuda.is_available():
        pytest.skip("a GPU is present")
    import types
    ly = types.SimpleNamespace(positions=np.zeros((3, 3), np.float32), uvs=np.zeros((3, 2), np.float32),
                               indices=np.array([[0, 1, 2]], np.uint32), texture=np.zeros((2, 2, 1, 4), np.float32))
    with pytest.raises(binding.VsError) as e:
        binding.vs_scene_create([ly], 0, stream=types.SimpleNamespace(cuda_stream=0))
    assert e.value.status == binding.VS_ERR_CUDA and "no CPU fallback" in str(e.value)


def test_product_path_does_not_touch_the_oracle():
    """Nothing under the package imports, links or reads oracle/ (and vice versa)."""
    pkg = os.path.join(ROOT, "paper_2409_02482_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                src = open(os.path.join(dirpath, f)).read()
                assert "import oracle" not in src and "from oracle" not in src and "vs_oracle" not in src, f
    for f in os.listdir(os.path.join(ROOT, "oracle")):
        if f.endswith((".py", ".c")):
            src = open(os.path.join(ROOT, "oracle", f)).read()
            assert "binding" not in src.replace("binding.py", "") and "libvs_b200" not in src and "csrc/" not in src.replace("paper_2409_02482_b200/csrc", ""), f
