"""CPU-side checks of the boundary: the C-ABI library loads, exports every symbol include/ggt.h declares,
and fails loudly (no CPU fallback) without a CUDA device.  No compute calls here."""
import ctypes
import os
import re

import pytest

from paper_2505_18932_b200 import binding, build

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _declared():
    src = open(os.path.join(ROOT, "include", "ggt.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(ggt_[a-z_]+)\s*\(", src)))


def test_header_symbols_all_exported():
    build.build()
    lib = ctypes.CDLL(binding.LIB_PATH)
    names = _declared()
    assert len(names) >= 15
    for n in names:
        assert hasattr(lib, n), n
    assert sorted(binding.EXPORTS) == names


def test_struct_sizes_match_header():
    assert ctypes.sizeof(binding.ggt_camera) == 4 * 4 + 9 * 4 + 3 * 4 + 2 * 4
    assert ctypes.sizeof(binding.ggt_refine_params) == 20
    assert ctypes.sizeof(binding.ggt_volume_desc) == 56
    assert ctypes.sizeof(binding.ggt_raymarch_params) == 40


def test_volume_bytes_layout():
    import numpy as np
    lib = binding.load_library()
    z = np.linspace(0.5, 5, 128).astype(np.float32)
    for dtype, per_voxel in ((binding.GGT_F32, 8), (binding.GGT_F16, 4)):
        d = binding.ggt_volume_desc(1920, 1080, 128, z.ctypes.data_as(ctypes.POINTER(ctypes.c_float)), 2.0, 0.0,
                                    0.001, 0.02, 7, 64.0, 1.0, dtype)
        n = lib.ggt_volume_bytes(ctypes.byref(d))
        # table header (2 x 128 floats) + the two planes + one 32-bit search range per ray, each block 256-B aligned
        assert n == 1024 + 1920 * 1080 * 128 * per_voxel + 1920 * 1080 * 4
    # ragged bin count pads to the 128-bit group
    d = binding.ggt_volume_desc(10, 10, 33, z.ctypes.data_as(ctypes.POINTER(ctypes.c_float)), 2.0, 0.0, 0.001, 0.02,
                                7, 64.0, 1.0, binding.GGT_F16)
    assert lib.ggt_volume_bytes(ctypes.byref(d)) == 512 + 16128 + 512      # 33 bins -> 5 groups of 8: 16000 B of voxels (rounded up to 256), 400 B of hints
    assert lib.ggt_workspace_bytes(4, 1920, 1080) == 4 * (-(-(1921 * 1081 * 8) // 256) * 256)


def test_no_cpu_fallback():
    import torch
    if torch.cuda.is_available():
        pytest.skip("GPU present")
    lib = binding.load_library()
    h = ctypes.c_void_p()
    assert lib.ggt_create(ctypes.byref(h)) == -4          # GGT_ERR_CUDA
    assert b"no CPU path" in lib.ggt_last_error(None)
    with pytest.raises(binding.GgtError):
        binding.Context()
