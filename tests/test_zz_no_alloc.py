"""bvh_scan_counts_static: the counts -> offsets scan for callers that cannot bring scratch memory.

Every other call of the library works in memory the caller allocates.  That leaves out code which is not free to
allocate at the time it runs: a stage that starts after the application has committed all device memory to its own
pool, a callback in a framework that forbids allocator calls (cudaMalloc synchronises the device and fails while a
stream is being captured), a loop with a latency budget the allocator's lock would break.  For those the library keeps
the scan's tile sums in a fixed 64 KB array of its own, one per GPU, which all calls on that GPU share and which still
holds the previous call's values when the next one starts.

So the checks here are: same offsets, bit for bit, as bvh_scan_counts with caller scratch; still the same on a second
call that finds the first call's leftovers in the array (a longer batch first, a shorter one after it); no device
memory taken by a call; sizes beyond the array's reach refused before anything is enqueued.

The file is named to be collected last: under `pytest -x` a failure here cannot hide another test.  Nothing in it
depends on what ran before (the array needs no initial state), so it passes alone in a fresh process as well.
"""
from __future__ import annotations

import pytest
import torch

from paper_2402_00665_b200 import binding, build


@pytest.fixture(scope="module")
def lib():
    build.build()
    return binding.load_library()


def _counts(q: int, seed: int, high: int) -> torch.Tensor:
    g = torch.Generator().manual_seed(seed)
    return torch.randint(0, high, (q,), generator=g, dtype=torch.int32)


def _scan_with_caller_scratch(counts: torch.Tensor) -> torch.Tensor:
    q = counts.numel()
    offsets = torch.full((q + 1,), -7, dtype=torch.int64, device=counts.device)
    scratch = torch.empty(max(binding.bvh_scan_sizes(q), 8), dtype=torch.uint8, device=counts.device)
    binding.bvh_scan_counts(counts, q, offsets, scratch)
    return offsets


def _scan_static(counts: torch.Tensor) -> torch.Tensor:
    q = counts.numel()
    offsets = torch.full((q + 1,), -7, dtype=torch.int64, device=counts.device)
    binding.bvh_scan_counts_static(counts, q, offsets)
    return offsets


def test_static_scan_refuses_more_than_its_array_covers(lib):
    """The size check comes before any CUDA call, so it can be exercised without a GPU: null-free dummy pointers,
    q one past the limit -> BVH_ERR_STATIC_LIMIT (-6); the ordinary argument checks still answer first."""
    import ctypes

    f = lib.bvh_scan_counts_static
    dummy = ctypes.c_void_p(256)
    assert f(dummy, binding.SCAN_STATIC_MAX_Q + 1, dummy, None) == -6
    assert f(dummy, 1 << 40, dummy, None) == -6
    assert f(None, 5, dummy, None) == -1
    assert f(dummy, -1, dummy, None) == -1
    assert f(dummy, 5, None, None) == -1
    with pytest.raises(binding.BvhError, match="STATIC_LIMIT"):
        binding._check(f(dummy, binding.SCAN_STATIC_MAX_Q + 1, dummy, None), "bvh_scan_counts_static")


@pytest.mark.gpu
def test_static_scan_equals_scan_with_caller_scratch_twice_in_a_row(lib):
    dev = torch.device("cuda:0")
    # first call: 245 tiles and a ragged tail, total beyond 2^31 so the 64-bit carries matter;
    # second call: 13 tiles, other values -- entries 13..244 of the shared array still hold the first call's sums
    first = _counts(1_000_003, seed=20240201, high=5000).to(dev)
    second = _counts(50_001, seed=665, high=700).to(dev)

    want_first = _scan_with_caller_scratch(first)
    got_first = _scan_static(first)
    torch.cuda.synchronize()
    assert int(want_first[-1]) > 2**31
    assert torch.equal(got_first, want_first)          # integers: bit for bit, the tolerance of every scan test here

    want_second = _scan_with_caller_scratch(second)
    got_second = torch.full((second.numel() + 1,), -7, dtype=torch.int64, device=dev)
    torch.cuda.synchronize()
    free_before, _ = torch.cuda.mem_get_info(dev)
    binding.bvh_scan_counts_static(second, second.numel(), got_second)
    torch.cuda.synchronize()
    free_after, _ = torch.cuda.mem_get_info(dev)
    assert free_after == free_before                   # the call took no device memory (kernels were loaded by call one)
    assert torch.equal(got_second, want_second)

    # and against the definition, on the host: offsets = exclusive prefix sum, offsets[q] = nnz
    ref = torch.zeros(second.numel() + 1, dtype=torch.int64)
    ref[1:] = torch.cumsum(second.cpu().to(torch.int64), 0)
    assert torch.equal(got_second.cpu(), ref)


@pytest.mark.gpu
def test_static_scan_small_and_empty_batches(lib):
    """q = 0 and a batch of one tile do not touch the array at all; a batch right at a tile boundary does."""
    dev = torch.device("cuda:0")
    for q, seed in ((0, 1), (1, 2), (4096, 3), (4097, 4), (8192, 5)):
        counts = _counts(q, seed=seed, high=100).to(dev) if q else torch.empty(0, dtype=torch.int32, device=dev)
        got = _scan_static(counts)
        torch.cuda.synchronize()
        ref = torch.zeros(q + 1, dtype=torch.int64)
        if q:
            ref[1:] = torch.cumsum(counts.cpu().to(torch.int64), 0)
        assert torch.equal(got.cpu(), ref), q
