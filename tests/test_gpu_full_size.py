"""GPU parity at BASELINE.json's FULL sizes, in the launch configuration bench.py times (Morton-ordered
queries through a QueryWorkspace, count -> scan -> fill).

Build: every exported array bit-equal to the oracle's (the serial oracle builds 10^7 primitives in a few
seconds).  Queries: the whole batch runs on the GPU; what is compared is
  * EVERY row of C2 and C4, and a seeded sample of 50 000 rows of C3 and C5, against the oracle's tree search
    (row lengths and row contents in traversal order),
  * a smaller sample against the oracle's brute force over all n primitives,
  * properties that hold at any size: offsets non-decreasing, offsets[q] = nnz, every stored index < n,
  * the single-pass path (collect -> scan -> rows_to_csr -> fill_overflow) against the two-pass result, every
    byte, on the device.
The construction-only sweep of configs[4] (n = 2^14 .. 2^27) is covered bit for bit at every size, 2^27 included
(the oracle builds it in about half a minute), and by the size-independent invariants (P3) at 2^27 as well.
"""
from __future__ import annotations

import numpy as np
import pytest

from helpers import csr_rows_sorted
from paper_2402_00665_b200 import workloads as W
from test_gpu_parity import _dev, assert_build_equal, export_np, gpu_build

torch = pytest.importorskip("torch")
pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def B():
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    from paper_2402_00665_b200 import binding

    binding.load_library()
    return binding


def _sample(q: int, k: int, seed: int) -> np.ndarray:
    """k distinct query indices, seeded, always including the first and the last query."""
    rng = np.random.default_rng(seed)
    s = rng.choice(q, size=min(k, q), replace=False)
    s[0], s[-1] = 0, q - 1
    return np.unique(s)


def _rows(off, idx, sel):
    return [idx[off[j]:off[j + 1]] for j in sel]


def _check_queries(B, oracle_lib, w, bvh, o, n_tree=50_000, n_brute=48):
    ws = B.QueryWorkspace(w.q)
    dq = _dev(w.queries)
    off, idx = B.query(bvh, dq, ws, ordered=True)
    torch.cuda.synchronize()
    # ---- the single-pass path gives the same bytes (capacity from this batch's own counts; one that makes a few
    # per cent of the rows overflow; both on the device) ----------------------------------------------------------
    cnt = (off[1:] - off[:-1])
    cap_all = (int(cnt.max()) + 7) // 8 * 8
    cap_some = max(8, int(torch.quantile(cnt[:: max(1, w.q // 100_000)].float(), 0.97)) // 8 * 8)
    off0, idx0 = off.clone(), idx
    for cap in (cap_all, cap_some):
        off1, idx1 = B.query(bvh, dq, ordered=True, row_capacity=cap)
        torch.cuda.synchronize()
        assert torch.equal(off1, off0) and torch.equal(idx1[: int(off0[-1])], idx0[: int(off0[-1])]), f"single pass, cap {cap}"
        del off1, idx1
    off = off0
    # ---- properties at full size, on the device --------------------------------------------------------
    nnz = int(off[-1])
    assert idx.numel() >= nnz and nnz > 0
    assert bool((off[1:] >= off[:-1]).all()) and int(off[0]) == 0
    assert int(idx[:nnz].min()) >= 0 and int(idx[:nnz].max()) < w.n
    off = off.cpu().numpy()
    # ---- sampled rows against the oracle's tree search -------------------------------------------------
    sel = _sample(w.q, n_tree, seed=11)
    tree = oracle_lib.query_spheres_tree if w.query_kind == "spheres" else oracle_lib.query_boxes_tree
    ooff, oidx = tree(o, np.ascontiguousarray(w.queries[sel]))
    assert np.array_equal(off[sel + 1] - off[sel], np.diff(ooff)), "row lengths"
    # gather the sampled rows on the device (the full index array of C3/C5 is 2 GB; do not copy it)
    d_off = torch.from_numpy(off).cuda()
    lens = torch.from_numpy(np.diff(ooff)).cuda()
    starts = d_off[torch.from_numpy(sel).cuda()]
    base = torch.repeat_interleave(starts - torch.from_numpy(ooff[:-1]).cuda(), lens)
    got = idx[base + torch.arange(int(ooff[-1]), device="cuda")].cpu().numpy()
    assert np.array_equal(got, oidx), "row contents in traversal order"
    # ---- a smaller sample against brute force over all n primitives -------------------------------------
    selb = sel[:: max(1, len(sel) // n_brute)][:n_brute]
    brute = oracle_lib.query_spheres_brute if w.query_kind == "spheres" else oracle_lib.query_boxes_brute
    boff, bidx = brute(w.prims, np.ascontiguousarray(w.queries[selb]))
    pos = np.searchsorted(sel, selb)
    sub_off = np.concatenate([[0], np.cumsum(np.diff(ooff)[pos])])
    sub_idx = np.concatenate([got[ooff[p]:ooff[p + 1]] for p in pos]) if len(pos) else got[:0]
    assert np.array_equal(sub_off, boff)
    assert np.array_equal(csr_rows_sorted(sub_off, sub_idx), bidx), "rows = brute force"
    return nnz


FULL = [("C2", 1 << 20, 1 << 20), ("C3", 10_000_000, 1_000_000), ("C4", 4_000_000, 4_000_000), ("C5", 1 << 24, 1 << 24)]


@pytest.mark.parametrize("name,n,q", FULL)
def test_full_size_config(B, oracle_lib, name, n, q):
    assert W.FULL_SIZES[name] == (n, q)
    w = W.make(name)
    o = oracle_lib.build_bvh(w.prims, w.morton_bits)
    bvh = gpu_build(B, w.prims, w.morton_bits)
    assert_build_equal(export_np(bvh), o, name)
    # C2, C4: every row against the oracle (1.7e7 / 1.4e7 hits: seconds for the serial oracle); C3, C5: 50 000 rows
    nnz = _check_queries(B, oracle_lib, w, bvh, o, n_tree=q if name in ("C2", "C4") else 50_000)
    expected_hits = {"C2": 16.7, "C3": 590.0, "C4": 3.4, "C5": 30.5}[name]   # SURVEY.md 8(d) Monte Carlo figures
    assert 0.8 * expected_hits < nnz / q < 1.25 * expected_hits


@pytest.mark.parametrize("log2n", [14, 15, 16, 17, 18, 19, 20, 21, 22, 23, 25, 26, 27])
def test_c5_sweep_build(B, oracle_lib, log2n):
    """configs[4] construction-only sweep, bit for bit at every size (2^24 is in test_full_size_config).  The arrays of
    the largest sizes are compared one at a time (2^27: 6.4 GB of boxes on each side)."""
    w = W.make("C5", n=1 << log2n, q=0)
    o = oracle_lib.build_bvh(w.prims, w.morton_bits)
    bvh = gpu_build(B, w.prims, w.morton_bits)
    if log2n < 25:
        assert_build_equal(export_np(bvh), o, f"2^{log2n}")
        return
    ex = bvh.export()
    n = w.n
    assert np.array_equal(ex.pop("scene_bounds").cpu().numpy().view(np.uint32), o.scene_bounds.view(np.uint32))
    assert np.array_equal(ex.pop("sorted_codes").cpu().numpy().view(np.uint64), o.sorted_codes), "sorted codes"
    assert np.array_equal(ex.pop("perm").cpu().numpy().view(np.uint32), o.perm), "perm"
    assert np.array_equal(ex.pop("left_child").cpu().numpy(), o.left_child), "left_child"
    assert np.array_equal(ex.pop("rope").cpu().numpy(), o.rope), "rope"
    aabb = ex.pop("aabb")
    assert aabb.shape[0] == 2 * n - 1
    step = 1 << 24
    for a in range(0, 2 * n - 1, step):                      # the boxes in slices: bit patterns, not float compares
        assert np.array_equal(aabb[a:a + step].cpu().numpy().view(np.uint32), o.aabb[a:a + step].view(np.uint32)), f"aabb [{a}, ...)"


def test_c5_sweep_largest_invariants(B, oracle_lib):
    """n = 2^27, the largest size of the sweep: the size-independent properties (P3) of the GPU output, and the
    sorted codes / permutation against numpy's stable sort of the GPU's own codes."""
    n = 1 << 27
    pts = W.hollow_shell(n, seed=5)
    bvh = gpu_build(B, pts, 63)
    lb = n - 1
    ex = bvh.export()
    codes = ex["sorted_codes"].view(torch.int64)
    perm = ex["perm"].view(torch.int32).to(torch.int64)
    assert bool((codes[1:] >= codes[:-1]).all())
    assert bool((perm[1:][codes[1:] == codes[:-1]] > perm[:-1][codes[1:] == codes[:-1]]).all())   # stable
    seen = torch.zeros(n, dtype=torch.uint8, device="cuda")
    seen[perm] = 1
    assert int(seen.sum()) == n                                                                    # a permutation
    del seen, codes
    left = ex["left_child"].cpu().numpy()
    rope = ex["rope"].cpu().numpy()
    order = oracle_lib.walk_all(left, rope, n)
    assert len(order) == 2 * n - 1 and np.array_equal(order[order >= lb] - lb, np.arange(n))
    del order
    assert rope[0] == -1 and rope[-1] == -1
    il = left[:lb]
    sib = rope[il]
    assert np.all(np.where(sib >= lb, sib - lb, sib) == np.where(il >= lb, il - lb, il) + 1)       # siblings consecutive
    aabb = ex["aabb"]
    assert np.array_equal(aabb[0].cpu().numpy(), np.concatenate([pts.min(axis=0), pts.max(axis=0)]))
    assert np.array_equal(ex["scene_bounds"].cpu().numpy(), aabb[0].cpu().numpy())
    # leaf boxes = permuted input; every internal box = union of its two children
    d_pts = _dev(pts)
    assert bool((aabb[lb:, :3] == d_pts[perm]).all()) and bool((aabb[lb:, 3:] == d_pts[perm]).all())
    d_left = ex["left_child"][:lb].to(torch.int64)
    d_right = ex["rope"].to(torch.int64)[d_left]
    assert bool((aabb[:lb, :3] == torch.minimum(aabb[d_left, :3], aabb[d_right, :3])).all())
    assert bool((aabb[:lb, 3:] == torch.maximum(aabb[d_left, 3:], aabb[d_right, 3:])).all())
