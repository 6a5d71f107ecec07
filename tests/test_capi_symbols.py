"""CPU checks of the boundary: the C-ABI library builds, loads without a GPU, and exports every symbol
include/bvh_b200.h declares; host-only entry points (sizes, argument checks) behave as documented."""
from __future__ import annotations

import ctypes
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    from paper_2402_00665_b200 import build

    build.build()
    from paper_2402_00665_b200 import binding

    return binding.load_library()


def _declared():
    text = open(os.path.join(ROOT, "include", "bvh_b200.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\bint\s+(bvh_\w+)\s*\(", text)))


def test_header_symbols_exported_and_bound(lib):
    from paper_2402_00665_b200 import binding

    names = _declared()
    assert len(names) >= 15
    for name in names:
        assert hasattr(lib, name), name
        assert name in binding.SYMBOLS, f"{name} not bound"
        assert callable(getattr(binding, name)), name
    assert sorted(binding.SYMBOLS) == names


def test_sizes_and_errors_host_only(lib):
    from paper_2402_00665_b200 import binding

    assert binding.bvh_version() >= 1
    nb, sb = binding.bvh_sizes(1000, 30)
    assert nb == 64 + 32 * 1999      # 64-byte header + (n-1) internal + n leaf records at their larger size
    assert sb >= 1000 * (4 + 2 * 4 + 2 * 4)
    nb63, sb63 = binding.bvh_sizes(1000, 63)
    assert nb63 == nb and sb63 > sb
    assert binding.bvh_sizes(0, 30)[0] == 64 + 32
    with pytest.raises(binding.BvhError, match="MORTON_BITS"):
        binding.bvh_sizes(10, 32)
    with pytest.raises(binding.BvhError, match="TOO_LARGE"):
        binding.bvh_sizes(1 << 30, 63)
    with pytest.raises(binding.BvhError, match="INVALID_ARGUMENT"):
        binding.bvh_sizes(-1, 63)
    assert binding.bvh_scan_sizes(0) >= 8 and binding.bvh_scan_sizes(1 << 24) >= 8 * ((1 << 24) // 4096)
    # argument checks return before anything is enqueued, so they are safe without a GPU
    f = lib.bvh_build_points
    assert f(None, 10, 30, None, None, 0, None) == -1           # null pointers
    assert f(None, 10, 31, None, None, 0, None) == -2
    assert f(None, 1 << 30, 30, None, None, 0, None) == -3
    assert f(None, 0, 30, None, None, 0, None) == 0             # n = 0 is a valid no-op
    assert f(ctypes.c_void_p(16), 10, 30, ctypes.c_void_p(64), ctypes.c_void_p(256), 16, None) == -4   # scratch too small
    assert f(ctypes.c_void_p(8), 10, 30, ctypes.c_void_p(64), ctypes.c_void_p(256), 1 << 30, None) == -1  # misaligned
    assert lib.bvh_query_spheres_count(None, 5, None, -1, None, None, None) == -1
    assert lib.bvh_query_spheres_count(None, 5, None, 0, None, None, None) == 0
    assert binding.bvh_query_order_sizes(1000) >= 1000 * 16
    assert lib.bvh_query_order_spheres(None, 5, None, 0, None, None, 0, None) == 0
    assert lib.bvh_query_order_spheres(None, 5, None, 7, None, None, 0, None) == -1


def test_binding_refuses_cpu_tensors(lib):
    import torch
    from paper_2402_00665_b200 import binding

    with pytest.raises(binding.BvhError, match="device memory"):
        binding.bvh_build_points(torch.zeros(4, 3), 4, 30, torch.zeros(8), torch.zeros(8))
