"""Host-side checks that need no GPU: the C-ABI library loads and exports every function include/legs.h declares,
the ctypes structs mirror the header, and the binding fails loudly without the library."""
import ctypes
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def declared_functions():
    text = open(os.path.join(ROOT, "include", "legs.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(legs_[a-z0-9_]+)\s*\(", text)))


@pytest.fixture(scope="module")
def lib():
    from paper_2311_18482_b200 import build
    return ctypes.CDLL(build.build())


def test_every_declared_symbol_is_exported(lib):
    names = declared_functions()
    assert len(names) >= 18 and "legs_render_backward" in names
    for n in names:
        assert hasattr(lib, n), n
    from paper_2311_18482_b200 import binding
    assert sorted(binding.EXPORTS) == names


def test_pure_host_entry_points(lib):
    assert lib.legs_record_stride(8) == 20 and lib.legs_record_stride(16) == 28
    assert lib.legs_pixel_channels(8) == 16 and lib.legs_pixel_channels(16) == 24
    lib.legs_status_string.restype = ctypes.c_char_p
    assert b"capacity" in lib.legs_status_string(-4)
    lib.legs_sort_workspace_bytes.restype = ctypes.c_size_t
    small = lib.legs_sort_workspace_bytes(ctypes.c_int64(1000), ctypes.c_uint64(4096), 64, 64)
    big = lib.legs_sort_workspace_bytes(ctypes.c_int64(1000000), ctypes.c_uint64(40000000), 1600, 1064)
    assert 0 < small < big < (2 << 30)
    lib.legs_backward_workspace_bytes.restype = ctypes.c_size_t
    assert lib.legs_backward_workspace_bytes(ctypes.c_int64(1000), 8) >= 1000 * 8 * 4


def test_struct_sizes_match_header():
    from paper_2311_18482_b200 import binding
    assert ctypes.sizeof(binding.CCamera) == 4 * 2 + 4 * 4 + 48 + 4 + 12
    assert ctypes.sizeof(binding.CGaussians) == 8 + 4 * 3 + 4 + 8 * 7     # 4 bytes of padding before the pointers
    assert ctypes.sizeof(binding.CFrame) == 8 * 10
    assert ctypes.sizeof(binding.CGrads) == 8 * 8
    assert ctypes.sizeof(binding.CDecoder) == 4 * 5 + 4 + 8 * 6


def test_no_gpu_means_loud_failure(lib):
    import torch
    if torch.cuda.is_available():
        pytest.skip("a GPU is present")
    from paper_2311_18482_b200 import binding
    with pytest.raises(binding.LegsError):
        binding.Context(0)      # legs_create fails: no device, and there is no CPU fallback to drop to


def test_product_path_never_imports_the_oracle():
    pkg = os.path.join(ROOT, "paper_2311_18482_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                text = open(os.path.join(dirpath, f)).read()
                assert not re.search(r"(import\s+.*oracle|from\s+oracle|legs_oracle|liblegs_oracle)", text), f
