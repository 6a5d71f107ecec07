"""GPU parity: the CUDA path (through the C ABI) against the CPU oracle, element by element, tolerance 0.

Bit-exact on: scene bounds, sorted codes, permutation, left_child, rope, AABBs, CSR offsets and sorted
rows (rows are sets, G13; the raw traversal order is additionally checked to be ascending Morton
position).  Sizes span several sort tiles (4096 / 3072 keys) plus a ragged tail.
"""
from __future__ import annotations

import os

import numpy as np
import pytest

from helpers import csr_rows_sorted
from paper_2402_00665_b200 import workloads as W

torch = pytest.importorskip("torch")
pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def B():
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    from paper_2402_00665_b200 import binding

    binding.load_library()  # must exist on a GPU box: no fallback
    return binding


def _dev(a):
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


def gpu_build(B, prims, bits):
    bvh = B.Bvh(prims.shape[0], bits)
    bvh.build(_dev(prims))
    torch.cuda.synchronize()
    return bvh


def export_np(bvh):
    e = {k: v.cpu().numpy() for k, v in bvh.export().items()}
    e["sorted_codes"] = e["sorted_codes"].view(np.uint32 if bvh.morton_bits == 30 else np.uint64).astype(np.uint64)
    e["perm"] = e["perm"].view(np.uint32)
    return e


def assert_build_equal(e, o, ctx=""):
    n = o.n
    assert np.array_equal(e["scene_bounds"].view(np.uint32), o.scene_bounds.view(np.uint32)), ctx + " scene bounds"
    assert np.array_equal(e["sorted_codes"], o.sorted_codes), ctx + " sorted codes"
    assert np.array_equal(e["perm"], o.perm), ctx + " perm"
    assert np.array_equal(e["left_child"], o.left_child), ctx + " left_child"
    assert np.array_equal(e["rope"], o.rope), ctx + " rope"
    assert np.array_equal(e["aabb"].view(np.uint32), o.aabb.view(np.uint32)), ctx + " aabb"
    assert e["left_child"].shape[0] == 2 * n - 1


def gpu_query(B, bvh, queries):
    off, idx = B.query(bvh, _dev(queries))
    torch.cuda.synchronize()
    return off.cpu().numpy(), idx.cpu().numpy()


def assert_query_equal(B, bvh, o, oracle_lib, queries, ctx=""):
    goff, gidx = gpu_query(B, bvh, queries)
    if queries.shape[1] == 4:
        ooff, oidx = oracle_lib.query_spheres_tree(o, queries)
    else:
        ooff, oidx = oracle_lib.query_boxes_tree(o, queries)
    assert np.array_equal(goff, ooff), ctx + " offsets"
    gidx = gidx[: goff[-1]]
    assert np.array_equal(csr_rows_sorted(goff, gidx), csr_rows_sorted(ooff, oidx)), ctx + " rows"
    # stronger: raw order = traversal order = ascending Morton position, which is also the oracle's DFS order
    assert np.array_equal(gidx, oidx), ctx + " raw order"
    return goff, gidx


CASES = [
    # name, n, q, radius: small enough for the oracle, several sort tiles + ragged tail
    ("C1", 4096, 4096, None),
    ("C2", 50_000, 20_000, 0.05),
    ("C2", 4096 * 3 + 1, 1000, 0.05),
    ("C3", 120_001, 5_000, 0.004),
    ("C4", 70_003, 30_000, 4e-3),
    ("C5", 65_537, 10_000, 0.04),
]


@pytest.mark.parametrize("name,n,q,radius", CASES)
def test_build_and_query_parity(B, oracle_lib, name, n, q, radius):
    w = W.make(name, n=n, q=q, radius=radius)
    o = oracle_lib.build_bvh(w.prims, w.morton_bits)
    bvh = gpu_build(B, w.prims, w.morton_bits)
    assert_build_equal(export_np(bvh), o, name)
    goff, gidx = assert_query_equal(B, bvh, o, oracle_lib, w.queries, name)
    assert goff[-1] > 0


def test_c1_brute_force(B, oracle_lib):
    """configs[0]: GPU result = O(n*q) brute force."""
    w = W.make("C1")
    bvh = gpu_build(B, w.prims, w.morton_bits)
    goff, gidx = gpu_query(B, bvh, w.queries)
    boff, bidx = oracle_lib.query_spheres_brute(w.prims, w.queries)
    assert np.array_equal(goff, boff)
    assert np.array_equal(csr_rows_sorted(goff, gidx[: goff[-1]]), bidx)


@pytest.mark.parametrize("n", [1, 2, 3, 4, 5, 7, 31, 32, 33, 255, 256, 257, 511, 513, 1024, 1025, 2047, 2048, 2049, 4095,
                               4096, 4097, 8191, 8192, 8193, 16383, 16384, 16385])
@pytest.mark.parametrize("bits", [30, 63])
def test_tiny_and_boundary_sizes(B, oracle_lib, n, bits):
    """Sizes around every switch of the build: one leaf, one group of 32, one level-1 window of 256, and the cluster sizes
    and pairs per thread of the one-launch front of a small build (small_build.cu: 256 x {1, 2, 4, 8} pairs x {1 .. 8}
    blocks, up to 16384; above that the one-sweep pipeline)."""
    pts = W.uniform_cube(n, seed=100 + n)
    o = oracle_lib.build_bvh(pts, bits)
    bvh = gpu_build(B, pts, bits)
    assert_build_equal(export_np(bvh), o, f"n={n}")
    qs = W.spheres_at(W.uniform_cube(64, seed=7), 0.3)
    assert_query_equal(B, bvh, o, oracle_lib, qs, f"n={n}")


@pytest.mark.parametrize("bits", [30, 63])
@pytest.mark.parametrize("n", [700, 3000, 6000, 12_000])
def test_small_build_boxes_and_ties(B, oracle_lib, n, bits):
    """The one-launch front of a small build on box primitives and on inputs with many equal codes (a coarse lattice:
    the stable order of equal codes is the original index, G5/G6), bit for bit against the oracle."""
    w = W.make("C4", n=n, q=0)
    o = oracle_lib.build_bvh(w.prims, bits)
    assert_build_equal(export_np(gpu_build(B, w.prims, bits)), o, f"boxes n={n}")
    rng = np.random.default_rng(n)
    pts = (rng.integers(0, 5, size=(n, 3)).astype(np.float32) * np.float32(0.25)) + np.float32(0.0)
    o = oracle_lib.build_bvh(pts, bits)
    e = export_np(gpu_build(B, pts, bits))
    assert_build_equal(e, o, f"lattice n={n}")
    assert len(np.unique(o.sorted_codes)) <= 125


@pytest.mark.parametrize("frame", ["unit", "odd", "tiny", "huge", "flat"])
def test_30bit_cells_on_and_next_to_cell_boundaries(B, oracle_lib, frame):
    """30-bit codes where D2's arithmetic is most fragile: coordinates exactly on cell boundaries, one and two ulps to
    either side, and random ones, in frames whose extent is a power of two, an odd number, tiny, huge, or zero on one
    axis: every code must be the oracle's.  (Written for a division-free quantisation that was measured and not kept:
    profiles/r02_experiments.md; it pins the kernel's rounding all the same.)"""
    rng = np.random.default_rng(abs(hash(frame)) % (1 << 31))
    lo, hi = {"unit": (0.0, 1.0), "odd": (0.1, 0.7), "tiny": (1.0, 1.0 + 3e-5), "huge": (-3.0e7, 5.0e8),
              "flat": (0.25, 0.8)}[frame]
    lo32, hi32 = np.float32(lo), np.float32(hi)
    e = np.float32(hi32 - lo32)
    k = rng.integers(0, 1025, size=(30_000, 3))
    on = (lo32 + (k.astype(np.float32) / np.float32(1024)) * e).astype(np.float32)       # on (or within an ulp of) a boundary
    parts = [on]
    for steps in (1, 2):
        up, dn = on.copy(), on.copy()
        for _ in range(steps):
            up = np.nextafter(up, np.float32(np.inf)).astype(np.float32)
            dn = np.nextafter(dn, np.float32(-np.inf)).astype(np.float32)
        parts += [up, dn]
    parts.append((lo32 + rng.random((60_000, 3)).astype(np.float32) * e).astype(np.float32))
    pts = np.clip(np.concatenate(parts), lo32, hi32).astype(np.float32)
    pts = np.concatenate([np.array([[lo32] * 3, [hi32] * 3], np.float32), pts]) + np.float32(0.0)
    if frame == "flat":
        pts[:, 1] = np.float32(0.5)                      # zero extent on y: t = 0 there (G7)
    o = oracle_lib.build_bvh(pts, 30)
    e_gpu = export_np(gpu_build(B, pts, 30))
    assert_build_equal(e_gpu, o, frame)


@pytest.mark.parametrize("pattern", ["pairs", "short", "serial_limit", "medium", "tile_edge", "long", "mixed", "coincident_blocks"])
def test_two_stage_sort_of_63bit_codes(B, oracle_lib, pattern):
    """63-bit builds sort by the upper 32 bits of the code and then order every run of equal upper bits by the lower 31
    (csrc/tie_fixup.cu).  Inputs whose primitives share 32-bit cells in runs of every size class: pairs, runs up to the
    one-thread limit (32) and just past it, runs of hundreds (block path), runs that straddle the 2048-position tiles,
    runs too long for a block (the conditional eight-pass sort takes over), exact duplicates inside runs (stability).
    The hierarchy must be the oracle's bit for bit in every case."""
    rng = np.random.default_rng(abs(hash(pattern)) % (1 << 31))
    def cluster(m, side):                      # m points inside one tiny cube: same upper bits, different lower bits
        c = rng.random(3) * 0.9 + 0.05
        return (c + rng.random((m, 3)) * side).astype(np.float32)
    bg = rng.random((40_000, 3)).astype(np.float32)
    corners = np.array([[0, 0, 0], [1, 1, 1]], np.float32)
    if pattern == "pairs":
        parts = [cluster(2, 1e-6) for _ in range(3000)]
    elif pattern == "short":
        parts = [cluster(int(rng.integers(2, 20)), 1e-6) for _ in range(1500)]
    elif pattern == "serial_limit":
        parts = [cluster(m, 1e-6) for m in (31, 32, 33, 34, 32, 33) * 40]
    elif pattern == "medium":
        parts = [cluster(int(rng.integers(100, 900)), 2e-6) for _ in range(40)]
    elif pattern == "tile_edge":
        parts = [cluster(int(rng.integers(1500, 2040)), 2e-6) for _ in range(12)]
    elif pattern == "long":
        parts = [cluster(9000, 2e-6), cluster(300, 1e-6)]
    elif pattern == "mixed":
        parts = [cluster(int(m), 2e-6) for m in rng.integers(2, 400, 300)] + [cluster(5000, 2e-6)]
    else:                                      # runs made of exact duplicates: the original index decides
        parts = [np.repeat(cluster(7, 1e-6), 9, axis=0) for _ in range(200)]
    pts = np.concatenate([corners, bg] + parts).astype(np.float32)
    pts = pts[rng.permutation(len(pts))] + np.float32(0.0)
    o = oracle_lib.build_bvh(pts, 63)
    runs = np.diff(np.flatnonzero(np.diff(np.concatenate([[-1], (o.sorted_codes >> np.uint64(31)).astype(np.int64), [-2]])) != 0))
    if pattern in ("long", "mixed"):
        assert runs.max() > 4096               # the fix-up cannot hold it: the second sort must run
    elif pattern in ("medium", "tile_edge"):
        assert 33 < runs.max() <= 2048 + 64
    bvh = gpu_build(B, pts, 63)
    assert_build_equal(export_np(bvh), o, pattern)
    bvh2 = gpu_build(B, pts, 63)               # a second build into fresh buffers: flags and work list start from zero again
    assert_build_equal(export_np(bvh2), o, pattern + " again")
    bvh2.build(_dev(pts))                      # and a third into USED buffers: the second sort finds its own histograms and
    torch.cuda.synchronize()                   # status words as the last build left them and has to clear them itself
    assert_build_equal(export_np(bvh2), o, pattern + " into used scratch")


def test_two_stage_sort_fallback_at_scale(B, oracle_lib):
    """The conditional second sort with a persistent grid (more tiles than resident blocks) and grid-wide barriers: 2.5 M
    points of which 200 000 sit inside ONE of the 2^32 cells, and a second dense cell of 30 000."""
    rng = np.random.default_rng(77)
    bg = rng.random((2_270_000, 3)).astype(np.float32)
    c1 = (np.array([0.3, 0.6, 0.2]) + rng.random((200_000, 3)) * 5e-5).astype(np.float32)
    c2 = (np.array([0.8, 0.1, 0.7]) + rng.random((30_000, 3)) * 5e-5).astype(np.float32)
    pts = np.concatenate([np.array([[0, 0, 0], [1, 1, 1]], np.float32), bg, c1, c2]).astype(np.float32)
    pts = pts[rng.permutation(len(pts))] + np.float32(0.0)
    o = oracle_lib.build_bvh(pts, 63)
    runs = np.diff(np.flatnonzero(np.diff(np.concatenate([[-1], (o.sorted_codes >> np.uint64(31)).astype(np.int64), [-2]])) != 0))
    assert runs.max() > 20_000
    assert_build_equal(export_np(gpu_build(B, pts, 63)), o, "fallback at scale")


def test_second_device_in_the_same_process(B, oracle_lib):
    """What a kernel needs set once (the opt-in to more than 48 KB of dynamic shared memory, the occupancy of the
    cooperative sort, the SM count) is remembered per device: after builds on cuda:0, the same builds on cuda:1 in the
    same process must work and give the same bits.  63-bit codes with n > 16384 go through tie_long_kernel (83 KB of
    shared memory) and the cooperative second sort; 30-bit through the one-sweep passes and the merge kernel."""
    if torch.cuda.device_count() < 2:
        pytest.skip("needs two CUDA devices")
    for name, n in (("C4", 70_003), ("C3", 120_001)):
        w = W.make(name, n=n, q=16)
        o = oracle_lib.build_bvh(w.prims, w.morton_bits)
        for dev in ("cuda:0", "cuda:1", "cuda:0"):
            with torch.cuda.device(dev):
                bvh = B.Bvh(n, w.morton_bits, device=dev)
                bvh.build(torch.from_numpy(w.prims).to(dev))
                torch.cuda.synchronize(dev)
                assert_build_equal(export_np(bvh), o, f"{name} on {dev}")


@pytest.mark.parametrize("bits", [30, 63])
@pytest.mark.parametrize("n", [1, 2, 5, 1000, 10_000])
def test_all_points_coincident(B, oracle_lib, n, bits):
    """Every code equal: the tree comes from the index tie-break alone (P4); zero scene extent on every axis."""
    pts = np.full((n, 3), 0.25, np.float32)
    o = oracle_lib.build_bvh(pts, bits)
    bvh = gpu_build(B, pts, bits)
    e = export_np(bvh)
    assert_build_equal(e, o)
    assert np.array_equal(e["perm"], np.arange(n, dtype=np.uint32))
    qs = np.array([[0.25, 0.25, 0.25, 0.0], [0.5, 0.25, 0.25, 0.25], [0.5, 0.25, 0.25, 0.2499]], np.float32)
    goff, gidx = assert_query_equal(B, bvh, o, oracle_lib, qs)
    assert list(np.diff(goff)) == [n, n, 0]


def test_t_corner_63bit(B, oracle_lib):
    """G14: codes 0 and 2^63-1; delta* = INT64_MAX must stay below +infinity."""
    pts = np.array([[0, 0, 0], [1, 1, 1]], np.float32)
    bvh = gpu_build(B, pts, 63)
    e = export_np(bvh)
    assert list(e["sorted_codes"]) == [0, (1 << 63) - 1]
    assert list(e["left_child"][:1]) == [1] and list(e["rope"]) == [-1, 2, -1]
    assert_build_equal(e, oracle_lib.build_bvh(pts, 63))


def test_points_equal_degenerate_boxes(B):
    w = W.make("C2", n=30_000, q=0)
    a = export_np(gpu_build(B, w.prims, 63))
    b = export_np(gpu_build(B, np.concatenate([w.prims, w.prims], axis=1), 63))
    for k in a:
        assert np.array_equal(a[k].view(np.uint8), b[k].view(np.uint8)), k


def test_plane_and_negative_coordinates(B, oracle_lib):
    """A zero-extent axis (no NaN from 0/0) and negative coordinates (float atomic min/max)."""
    pts = W.uniform_cube(20_000, seed=5) * np.float32(8.0) - np.float32(6.0)
    pts[:, 2] = np.float32(-3.5)
    for bits in (30, 63):
        o = oracle_lib.build_bvh(pts, bits)
        bvh = gpu_build(B, pts, bits)
        assert_build_equal(export_np(bvh), o)
    boxes = W.boxes_around(pts, 0.05)
    o = oracle_lib.build_bvh(boxes, 63)
    bvh = gpu_build(B, boxes, 63)
    assert_build_equal(export_np(bvh), o)
    assert_query_equal(B, bvh, o, oracle_lib, W.boxes_around(pts[:2000] + np.float32(0.01), 0.08))
    assert_query_equal(B, bvh, o, oracle_lib, W.spheres_at(pts[:2000], 0.1))


def test_schedule_independence(B):
    """P8: 20 builds of the same input give identical bytes (nodes and exported arrays)."""
    w = W.make("C3", n=200_000, q=0)
    d = _dev(w.prims)
    ref = None
    for _ in range(20):
        bvh = B.Bvh(w.n, w.morton_bits)
        bvh.nodes.zero_()
        bvh.build(d)
        torch.cuda.synchronize()
        cur = bvh.nodes.cpu().numpy().tobytes()
        if ref is None:
            ref = cur
        assert cur == ref


def test_structural_invariants_large(B, oracle_lib):
    """Properties that hold at any size (P3), checked on the GPU output at n = 2^20 without the oracle tree."""
    w = W.make("C2", n=1 << 20, q=0)
    bvh = gpu_build(B, w.prims, w.morton_bits)
    e = export_np(bvh)
    n, lb = w.n, w.n - 1
    assert np.array_equal(np.sort(e["perm"]), np.arange(n, dtype=np.uint32))
    d = np.diff(e["sorted_codes"].astype(np.int64))
    assert np.all(d >= 0) and np.all(np.diff(e["perm"].astype(np.int64))[d == 0] > 0)
    order = oracle_lib.walk_all(e["left_child"], e["rope"], n)
    assert len(order) == 2 * n - 1 and np.array_equal(order[order >= lb] - lb, np.arange(n))
    assert e["rope"][0] == -1
    # root box = scene bounds = numpy min/max of the input
    assert np.array_equal(e["aabb"][0, :3], w.prims.min(axis=0)) and np.array_equal(e["aabb"][0, 3:], w.prims.max(axis=0))
    assert np.array_equal(e["scene_bounds"], e["aabb"][0])
    assert np.array_equal(e["aabb"][lb:, :3], w.prims[e["perm"]])
    # rope of a left child is its sibling: consecutive Karras indices
    left = e["left_child"][:lb]
    sib = e["rope"][left]
    gl = np.where(left >= lb, left - lb, left)
    gs = np.where(sib >= lb, sib - lb, sib)
    assert np.all(gs == gl + 1)


def test_query_order_is_a_permutation_and_does_not_change_results(B):
    w = W.make("C3", n=150_000, q=40_000, radius=0.004)
    bvh = gpu_build(B, w.prims, w.morton_bits)
    dq = _dev(w.queries)
    ws = B.QueryWorkspace(w.q)
    o1, i1 = B.query(bvh, dq, ws, ordered=True)
    torch.cuda.synchronize()
    order = ws.order.cpu().numpy().view(np.uint32)
    assert np.array_equal(np.sort(order), np.arange(w.q, dtype=np.uint32))
    o1, i1 = o1.cpu().numpy().copy(), i1.cpu().numpy().copy()
    o2, i2 = B.query(bvh, dq, ws, ordered=False)
    torch.cuda.synchronize()
    assert np.array_equal(o1, o2.cpu().numpy()) and np.array_equal(i1, i2.cpu().numpy())
    # box queries too, including queries whose centroid lies outside the scene box (clamped for ordering only)
    wb = W.make("C4", n=60_000, q=20_000, radius=4e-3)
    bvh = gpu_build(B, wb.prims, wb.morton_bits)
    qs = wb.queries.copy()
    qs[:100] += np.float32(3.0)
    qs[100:200, 3:] += np.float32(5.0)
    dq = _dev(qs)
    o1, i1 = B.query(bvh, dq, ordered=True)
    o2, i2 = B.query(bvh, dq, ordered=False)
    torch.cuda.synchronize()
    assert torch.equal(o1, o2) and torch.equal(i1, i2)
    assert int(o1[100]) == 0 and int(o1[-1]) > 0


def _oracle_csr(oracle_lib, o, queries):
    fn = {4: oracle_lib.query_spheres_tree, 6: oracle_lib.query_boxes_tree, 8: oracle_lib.query_rays_tree}[queries.shape[1]]
    return fn(o, queries)


@pytest.mark.parametrize("name,n,q,radius", [("C1", 4096, 4096, None), ("C3", 120_001, 5_000, 0.004),
                                             ("C4", 70_003, 30_000, 4e-3), ("C5", 65_537, 10_000, 0.04)])
def test_single_pass_query_equals_oracle(B, oracle_lib, name, n, q, radius):
    """NEXT-3: collect (one traversal into rows of `cap` entries + exact counts) -> scan -> rows_to_csr -> fill_overflow
    gives the oracle's CSR byte for byte, whatever the capacity: every row fits / some rows overflow / almost all do."""
    w = W.make(name, n=n, q=q, radius=radius)
    o = oracle_lib.build_bvh(w.prims, w.morton_bits)
    bvh = gpu_build(B, w.prims, w.morton_bits)
    ooff, oidx = _oracle_csr(oracle_lib, o, w.queries)
    counts = np.diff(ooff)
    mx = int(counts.max())
    caps = sorted({(mx + 7) // 8 * 8, max(8, int(np.median(counts)) // 8 * 8), 8})
    dq = _dev(w.queries)
    for cap in caps:
        for ordered in (True, False):
            off, idx = B.query(bvh, dq, ordered=ordered, row_capacity=cap)
            torch.cuda.synchronize()
            assert np.array_equal(off.cpu().numpy(), ooff), (name, cap, "offsets")
            assert np.array_equal(idx.cpu().numpy()[: ooff[-1]], oidx), (name, cap, "indices in traversal order")
    # the rows themselves: the first min(count, cap) hits of every query, counts exact
    cap = caps[len(caps) // 2]
    rows = torch.full((w.q * cap,), -7, dtype=torch.int32, device="cuda")
    cnt = torch.empty(w.q, dtype=torch.int32, device="cuda")
    B.bvh_query_collect(bvh.nodes, bvh.n, dq, B.QUERY_KINDS[w.queries.shape[1]], w.q, None, cap, rows, cnt)
    torch.cuda.synchronize()
    assert np.array_equal(cnt.cpu().numpy(), counts)
    r = rows.cpu().numpy().reshape(w.q, cap)
    for j in np.random.default_rng(3).choice(w.q, 200, replace=False):
        k = min(int(counts[j]), cap)
        assert np.array_equal(r[j, :k], oidx[ooff[j]: ooff[j] + k]) and np.all(r[j, k:] == -7), j


@pytest.mark.parametrize("name,n,q,radius", [("C1", 4096, 4096, None), ("C1", 4096, 1, None), ("C3", 120_001, 5_000, 0.004),
                                             ("C2", 50_000, 8_192, 0.03), ("C4", 70_003, 30_000, 4e-3),
                                             ("C5", 65_537, 10_000, 0.04)])
def test_one_call_query_csr_equals_oracle(B, oracle_lib, name, n, q, radius):
    """bvh_query_csr: order + collect + scan + rows -> CSR + overflow rows enqueued by ONE call (small batches: input
    order, the scan and the row copy in one kernel, queries spread over the warps) = the oracle's CSR byte for byte,
    whatever the row capacity; a result buffer that is too small is never overrun, and the documented completion
    (bvh_rows_to_csr + bvh_query_fill_overflow into a larger buffer) yields the same bytes."""
    w = W.make(name, n=n, q=q, radius=radius)
    o = oracle_lib.build_bvh(w.prims, w.morton_bits)
    bvh = gpu_build(B, w.prims, w.morton_bits)
    ooff, oidx = _oracle_csr(oracle_lib, o, w.queries)
    counts = np.diff(ooff)
    nnz = int(ooff[-1])
    mx = int(counts.max())
    dq = _dev(w.queries)
    kind = B.QUERY_KINDS[w.queries.shape[1]]
    ws = B.QueryWorkspace(w.q)
    for cap in sorted({max(8, (mx + 7) // 8 * 8), max(8, int(np.median(counts)) // 8 * 8), 8}):
        ind = torch.full((nnz + 16,), -7, dtype=torch.int32, device="cuda")
        off, _ = B.query_csr(bvh, dq, cap, ind, ws=ws)
        torch.cuda.synchronize()
        assert np.array_equal(off.cpu().numpy(), ooff), (name, cap, "offsets")
        got = ind.cpu().numpy()
        assert np.array_equal(got[:nnz], oidx) and np.all(got[nnz:] == -7), (name, cap, "indices")
        # a buffer that holds only part of the result: rows that end inside it are complete, nothing past it is touched
        short = max(1, nnz // 2)
        buf = torch.full((short + 64,), -7, dtype=torch.int32, device="cuda")
        rows = torch.empty(w.q * cap, dtype=torch.int32, device="cuda")
        B.bvh_query_csr(bvh.nodes, bvh.n, dq, kind, w.q, cap, rows, ws.order, ws.counts, ws.offsets, buf, short, ws.order_scratch)
        torch.cuda.synchronize()
        assert int(ws.offsets[w.q].item()) == nnz                      # the caller learns that it did not fit
        got = buf.cpu().numpy()
        assert np.all(got[short:] == -7), (name, cap, "written past the capacity")
        fits = ooff[1:] <= short
        last = int(ooff[1:][fits].max()) if fits.any() else 0          # rows are in offset order: a prefix fits
        assert np.array_equal(got[:last], oidx[:last]), (name, cap, "rows inside the capacity")
        # completion into a buffer that is large enough
        full = torch.full((nnz + 8,), -7, dtype=torch.int32, device="cuda")
        order = ws.order if w.q > 8192 else None
        B.bvh_rows_to_csr(rows, cap, ws.counts, ws.offsets, w.q, full)
        B.bvh_query_fill_overflow(bvh.nodes, bvh.n, dq, kind, w.q, order, cap, ws.counts, ws.offsets, full)
        torch.cuda.synchronize()
        assert np.array_equal(full.cpu().numpy()[:nnz], oidx), (name, cap, "completion")
    # capacity 0, empty batch, empty hierarchy
    B.bvh_query_csr(bvh.nodes, bvh.n, dq, kind, w.q, 8, rows, ws.order, ws.counts, ws.offsets, buf, 0, ws.order_scratch)
    torch.cuda.synchronize()
    assert np.array_equal(ws.offsets.cpu().numpy()[: w.q + 1], ooff)
    offs = torch.full((1,), 5, dtype=torch.int64, device="cuda")
    B.bvh_query_csr(bvh.nodes, bvh.n, dq, kind, 0, 8, None, None, None, offs, None, 0, None)
    torch.cuda.synchronize()
    assert int(offs[0].item()) == 0
    B.bvh_query_csr(None, 0, dq, kind, w.q, 8, rows, ws.order, ws.counts, ws.offsets, buf, short, ws.order_scratch)
    torch.cuda.synchronize()
    assert not ws.offsets[: w.q + 1].any()


def test_single_pass_rays_and_argument_checks(B, oracle_lib):
    w = W.make("C4", n=30_000, q=0)
    bvh = gpu_build(B, w.prims, w.morton_bits)
    rays = _rays_through(w.prims, 4000, seed=31, tmax=4.0)
    o = oracle_lib.build_bvh(w.prims, w.morton_bits)
    ooff, oidx = oracle_lib.query_rays_tree(o, rays)
    off, idx = B.query(bvh, _dev(rays), row_capacity=16)
    torch.cuda.synchronize()
    assert np.array_equal(off.cpu().numpy(), ooff) and np.array_equal(idx.cpu().numpy()[: ooff[-1]], oidx)
    dq = _dev(rays)
    cnt = torch.empty(4000, dtype=torch.int32, device="cuda")
    rows = torch.empty(4000 * 16 + 8, dtype=torch.int32, device="cuda")
    for bad_cap, bad_rows in ((12, rows), (0, rows), (16, rows[1:])):     # not a multiple of 8 / zero / rows misaligned
        with pytest.raises(B.BvhError):
            B.bvh_query_collect(bvh.nodes, bvh.n, dq, 2, 4000, None, bad_cap, bad_rows, cnt)
    with pytest.raises(B.BvhError):
        B.bvh_query_collect(bvh.nodes, bvh.n, dq, 3, 4000, None, 16, rows, cnt)      # unknown query kind
    with pytest.raises(B.BvhError):
        B.query(B.Bvh(100, 30), _dev(W.spheres_at(W.uniform_cube(4, seed=1), 0.1)))    # never built


def test_stale_or_mismatched_nodes_buffer_is_not_traversed(B):
    """The query kernels check the header the build wrote (magic, n) on the device: a buffer that was never built, was
    built for another n or was overwritten gives counts of 0 and stores nothing, instead of a walk over garbage."""
    pts = W.uniform_cube(5000, seed=9)
    bvh = gpu_build(B, pts, 30)
    qs = _dev(W.spheres_at(pts[:512], 0.2))
    cnt = torch.full((512,), -1, dtype=torch.int32, device="cuda")
    B.bvh_query_spheres_count(bvh.nodes, 5000, qs, 512, None, cnt)
    torch.cuda.synchronize()
    assert int(cnt.min()) > 0
    # wrong n for this buffer
    cnt.fill_(-1)
    B.bvh_query_spheres_count(bvh.nodes, 4999, qs, 512, None, cnt)
    torch.cuda.synchronize()
    assert cnt.cpu().tolist() == [0] * 512
    # garbage where the hierarchy should be
    junk = torch.randint(0, 255, (bvh.nodes.numel(),), dtype=torch.uint8, device="cuda")
    junk[:4] = 0
    cnt.fill_(-1)
    B.bvh_query_spheres_count(junk, 5000, qs, 512, None, cnt)
    rows = torch.full((512 * 8,), -7, dtype=torch.int32, device="cuda")
    cnt2 = torch.full((512,), -1, dtype=torch.int32, device="cuda")
    B.bvh_query_collect(junk, 5000, qs, 0, 512, None, 8, rows, cnt2)
    idx = torch.full((64,), -7, dtype=torch.int32, device="cuda")
    off = torch.zeros(513, dtype=torch.int64, device="cuda")
    B.bvh_query_spheres_fill(junk, 5000, qs, 512, None, off, idx)
    torch.cuda.synchronize()
    assert cnt.cpu().tolist() == [0] * 512 and cnt2.cpu().tolist() == [0] * 512
    assert int((rows != -7).sum()) == 0 and int((idx != -7).sum()) == 0
    with pytest.raises(B.BvhError):                      # 256-bit node loads: 32-byte alignment
        B.bvh_query_spheres_count(bvh.nodes[16:], 5000, qs, 512, None, cnt)


def test_touching_counts_as_intersecting_boxes_and_rays(B, oracle_lib):
    """G12: closed comparisons.  Box queries that share exactly a face / an edge / a corner with a primitive box hit
    it, one ulp away they miss; rays that graze a face or end exactly on it (tmax) hit, one ulp short they miss."""
    f = np.float32
    prims = np.array([[0.25, 0.25, 0.25, 0.5, 0.5, 0.5], [0.75, 0.75, 0.75, 0.875, 0.875, 0.875],
                      [-1.0, -1.0, -1.0, -0.5, -0.5, -0.5]], f)
    up, dn = (lambda x: np.nextafter(f(x), f(np.inf))), (lambda x: np.nextafter(f(x), f(-np.inf)))
    qb = np.array([
        [0.5, 0.25, 0.25, 0.625, 0.5, 0.5],              # shares the face x = 0.5
        [up(0.5), 0.25, 0.25, 0.625, 0.5, 0.5],          # one ulp off
        [0.5, 0.5, 0.25, 0.625, 0.625, 0.5],             # shares an edge
        [0.5, 0.5, 0.5, 0.75, 0.75, 0.75],               # corner of the first, corner of the second
        [0.5, 0.5, up(0.5), 0.75, 0.75, dn(0.75)],       # neither
        [-0.5, -0.5, -0.5, 0.25, 0.25, 0.25],            # corner of the third and of the first
    ], f)
    o = oracle_lib.build_bvh(prims, 63)
    bvh = gpu_build(B, prims, 63)
    goff, gidx = assert_query_equal(B, bvh, o, oracle_lib, qb, "touching boxes")
    assert list(np.diff(goff)) == [1, 0, 1, 2, 0, 2]
    rays = np.array([
        [0.0, 0.5, 0.375, 1, 0, 0, 0.0, 8.0],            # runs in the face y = 0.5 of the first box
        [0.0, up(0.5), 0.375, 1, 0, 0, 0.0, 8.0],        # one ulp above it
        [0.0, 0.375, 0.375, 1, 0, 0, 0.0, 0.25],         # ends exactly on the face x = 0.25 (tmax)
        [0.0, 0.375, 0.375, 1, 0, 0, 0.0, dn(0.25)],     # ends one ulp short
        [1.0, 0.375, 0.375, -1, 0, 0, 0.5, 8.0],         # starts exactly on the face x = 0.5 (tmin)
        [0.0, 0.0, 0.0, 1, 1, 1, 0.0, 8.0],              # through the corners of the first two boxes
    ], f)
    ooff, oidx = oracle_lib.query_rays_tree(o, rays)
    off, idx = B.query(bvh, _dev(rays))
    torch.cuda.synchronize()
    assert np.array_equal(off.cpu().numpy(), ooff) and np.array_equal(idx.cpu().numpy()[: ooff[-1]], oidx)
    assert list(np.diff(ooff)) == [1, 0, 1, 0, 1, 2]


def test_containment_shortcut_large_queries(B, oracle_lib):
    """A subtree whose box lies inside the query is reported without walking it (traverse.cu, contains_box).  The result
    must not change: queries that swallow whole subtrees (up to the whole scene), queries for which the farthest-corner
    distance of a node equals r*r exactly, and one ulp less -- on a dyadic lattice, where that arithmetic is exact."""
    f = np.float32
    g = np.arange(32, dtype=f) / f(32.0)
    pts = np.stack(np.meshgrid(g, g, g, indexing="ij"), axis=-1).reshape(-1, 3).astype(f)     # 32768 lattice points
    for bits in (30, 63):
        o = oracle_lib.build_bvh(pts, bits)
        bvh = gpu_build(B, pts, bits)
        c = f(0.5) - f(1.0 / 64.0)                      # centre of the lattice
        # farthest corner of the whole scene from the centre: (31/64)^2 * 3, exactly representable
        r2 = f(3.0) * f(31.0 / 64.0) * f(31.0 / 64.0)
        r = f(np.sqrt(np.float64(r2)))
        qs = [[c, c, c, 2.0], [c, c, c, r], [c, c, c, np.nextafter(r, f(0))], [c, c, c, np.nextafter(r, f(2))],
              [0.25, 0.25, 0.25, 0.25], [0.25, 0.25, 0.25, np.nextafter(f(0.25), f(0))], [0.0, 0.0, 0.0, 0.5],
              [0.75, 0.5, 0.25, 0.3], [5.0, 5.0, 5.0, 1.0]]
        # spheres whose radius is exactly the farthest-corner distance of an octant [0, 15/32]^3 from its own centre
        h = f(15.0 / 64.0)
        rr = f(np.sqrt(np.float64(f(3.0) * h * h)))
        for dr in (rr, np.nextafter(rr, f(0)), np.nextafter(rr, f(1))):
            qs.append([h, h, h, dr])
        qs = np.array(qs, f)
        goff, gidx = assert_query_equal(B, bvh, o, oracle_lib, qs, f"containment {bits}")
        assert np.diff(goff)[0] == len(pts) and np.diff(goff)[-4] == 0
        off, idx = B.query(bvh, _dev(qs), row_capacity=32768)
        torch.cuda.synchronize()
        assert np.array_equal(off.cpu().numpy(), goff) and np.array_equal(idx.cpu().numpy()[: goff[-1]], gidx)
        off, idx = B.query(bvh, _dev(qs), row_capacity=1024)            # contained subtrees larger than the row: truncated, refilled
        torch.cuda.synchronize()
        assert np.array_equal(off.cpu().numpy(), goff) and np.array_equal(idx.cpu().numpy()[: goff[-1]], gidx)
    # box queries and box leaves
    boxes = W.boxes_around(pts[::2], 1.0 / 256.0)
    o = oracle_lib.build_bvh(boxes, 63)
    bvh = gpu_build(B, boxes, 63)
    lo, hi = boxes[:, :3].min(axis=0), boxes[:, 3:].max(axis=0)
    qb = np.array([[*lo, *hi], [*np.nextafter(lo, f(1)), *hi], [-1, -1, -1, 2, 2, 2], [*lo, 0.5, 0.5, 0.5],
                   [0.25, 0.25, 0.25, 0.75, 0.75, 0.75], [*lo, *lo]], f)
    goff, gidx = assert_query_equal(B, bvh, o, oracle_lib, qb, "containment boxes")
    assert np.diff(goff)[0] == len(boxes) and np.diff(goff)[2] == len(boxes)
    assert_query_equal(B, bvh, o, oracle_lib, np.array([[0.5, 0.5, 0.5, 0.45], [0.5, 0.5, 0.5, 5.0]], f), "containment sphere/box leaves")


# ---- NEXT-1: operations at the leaf (D10 nearest, D11 first hit, any hit) -----------------------------------------

@pytest.mark.parametrize("name,n,q,radius", [("C1", 4096, 4096, None), ("C3", 120_001, 6_000, 0.004),
                                             ("C5", 65_537, 6_000, 0.04), ("C4", 70_003, 6_000, None)])
def test_nearest_within_radius_equals_oracle(B, oracle_lib, name, n, q, radius):
    w = W.make(name, n=n, q=q, radius=radius)
    spheres = w.queries if w.queries.shape[1] == 4 else W.spheres_at(w.queries[:, :3], 0.01)   # C4: box leaves
    spheres = spheres.copy()
    spheres[::7, 3] = 0.0                                     # some queries that (almost surely) find nothing
    o = oracle_lib.build_bvh(w.prims, w.morton_bits)
    oi, od = oracle_lib.nearest_spheres_tree(o, spheres)
    bvh = gpu_build(B, w.prims, w.morton_bits)
    for ordered in (True, False):
        gi, gd = B.reduce_query(bvh, _dev(spheres), "nearest", ordered=ordered)
        torch.cuda.synchronize()
        assert np.array_equal(gi.cpu().numpy(), oi), name
        assert np.array_equal(gd.cpu().numpy().view(np.uint32), od.view(np.uint32)), name     # distances: same bits
    assert (oi >= 0).sum() > q // 4 and (name == "C1" or (oi < 0).sum() > 0)   # (C1's queries sit on the points)
    hit = B.reduce_query(bvh, _dev(spheres), "any_hit")
    torch.cuda.synchronize()
    assert np.array_equal(hit.cpu().numpy(), (oi >= 0).astype(np.int32))


def test_nearest_ties_and_duplicates(B, oracle_lib):
    """Coincident primitives and lattice points at equal distance: the smallest ORIGINAL index wins, whatever the tree
    order; zero radius; the radius exactly at a point (closed)."""
    f = np.float32
    g = np.arange(8, dtype=f) / f(8.0)
    pts = np.stack(np.meshgrid(g, g, g, indexing="ij"), axis=-1).reshape(-1, 3).astype(f)
    pts = np.concatenate([pts, pts[::3], pts[::5]])           # duplicates with larger indices
    rng = np.random.default_rng(5)
    pts = pts[rng.permutation(len(pts))]
    qc = (np.stack(np.meshgrid(g, g, g, indexing="ij"), axis=-1).reshape(-1, 3) + f(1.0 / 16.0)).astype(f)   # cell centres: 8 equidistant corners
    qs = np.concatenate([W.spheres_at(qc, 0.25), W.spheres_at(pts[:200], 0.0), W.spheres_at(qc[:100], float(np.sqrt(3.0) / 16.0))])
    for bits in (30, 63):
        o = oracle_lib.build_bvh(pts, bits)
        bi, bd = oracle_lib.nearest_spheres_brute(pts, qs)
        bvh = gpu_build(B, pts, bits)
        gi, gd = B.reduce_query(bvh, _dev(qs), "nearest")
        torch.cuda.synchronize()
        assert np.array_equal(gi.cpu().numpy(), bi) and np.array_equal(gd.cpu().numpy().view(np.uint32), bd.view(np.uint32))
        assert (bi[:512] >= 0).all() and (bi[512:712] >= 0).all()


@pytest.mark.parametrize("name,n", [("C4", 60_000), ("C2", 40_000)])
def test_first_hit_and_any_hit_rays_equal_oracle(B, oracle_lib, name, n):
    w = W.make(name, n=n, q=0, radius=0.02 if name == "C4" else None)      # C4: boxes large enough to be hit often
    prims = w.prims if w.prims.shape[1] == 6 else W.boxes_around(w.prims, 0.004)
    rays = _rays_through(prims, 8000, seed=41, tmax=4.0)
    rays[::9, 6] = np.float32(-0.5)                            # negative tmin: entry parameters may be negative
    o = oracle_lib.build_bvh(prims, 63)
    oi, ot = oracle_lib.first_hit_rays_tree(o, rays)
    bvh = gpu_build(B, prims, 63)
    for ordered in (True, False):
        gi, gt = B.reduce_query(bvh, _dev(rays), "first_hit", ordered=ordered)
        torch.cuda.synchronize()
        assert np.array_equal(gi.cpu().numpy(), oi), name
        assert np.array_equal(gt.cpu().numpy(), ot), name      # numeric equality (-0.0 == +0.0)
    assert (oi >= 0).sum() > 500
    hit = B.reduce_query(bvh, _dev(rays), "any_hit")
    torch.cuda.synchronize()
    assert np.array_equal(hit.cpu().numpy(), (oi >= 0).astype(np.int32))
    # any hit with box queries = "the row is not empty"
    qb = W.boxes_around(W.uniform_cube(5000, seed=3) * np.float32(2.4) - np.float32(1.2), 0.01)
    ooff, _ = oracle_lib.query_boxes_tree(o, qb)
    hit = B.reduce_query(bvh, _dev(qb), "any_hit")
    torch.cuda.synchronize()
    assert np.array_equal(hit.cpu().numpy(), (np.diff(ooff) > 0).astype(np.int32))
    with pytest.raises(B.BvhError):
        B.reduce_query(bvh, _dev(qb), "nearest")


def test_reduce_modes_empty_and_stale(B):
    bvh = B.Bvh(0, 30)
    bvh.build(torch.zeros((0, 3), dtype=torch.float32, device="cuda"))
    qs = _dev(np.array([[0.5, 0.5, 0.5, 1.0], [0, 0, 0, 2.0]], np.float32))
    i, d = B.reduce_query(bvh, qs, "nearest")
    h = B.reduce_query(bvh, qs, "any_hit")
    torch.cuda.synchronize()
    assert i.cpu().tolist() == [-1, -1] and bool(torch.isinf(d).all()) and h.cpu().tolist() == [0, 0]
    pts = W.uniform_cube(3000, seed=2)
    bvh = gpu_build(B, pts, 30)
    idx = torch.zeros(2, dtype=torch.int32, device="cuda")
    key = torch.zeros(2, dtype=torch.float32, device="cuda")
    B.bvh_query_spheres_nearest(bvh.nodes, 2999, qs, 2, None, idx, key)      # n does not match the buffer's header
    torch.cuda.synchronize()
    assert idx.cpu().tolist() == [-1, -1] and bool(torch.isinf(key).all())


def test_query_to_host_pipeline_equals_query(B, oracle_lib):
    """End-to-end helper: pinned host queries -> chunked single-pass search -> CSR in pinned host memory, copies
    overlapped with the search of the next chunk.  Same CSR as the oracle, whatever the chunking."""
    w = W.make("C3", n=150_000, q=30_001, radius=0.004)
    o = oracle_lib.build_bvh(w.prims, w.morton_bits)
    ooff, oidx = oracle_lib.query_spheres_tree(o, w.queries)
    bvh = gpu_build(B, w.prims, w.morton_bits)
    hq = torch.from_numpy(w.queries).pin_memory()
    cap = (int(np.diff(ooff).max()) + 7) // 8 * 8
    for chunks, c in ((1, cap), (7, cap), (8, 8)):
        out = B.HostCsr(w.q, int(ooff[-1]))
        B.query_to_host(bvh, hq, out, row_capacity=c, chunks=chunks)
        assert out.nnz == int(ooff[-1])
        assert np.array_equal(out.offsets.numpy(), ooff) and np.array_equal(out.indices.numpy()[: out.nnz], oidx)
    with pytest.raises(B.BvhError):
        B.query_to_host(bvh, hq, B.HostCsr(w.q, 10), row_capacity=cap)          # too small for the result


def test_empty_inputs(B):
    bvh = B.Bvh(0, 30)
    bvh.build(torch.zeros((0, 3), dtype=torch.float32, device="cuda"))
    qs = _dev(np.array([[0.5, 0.5, 0.5, 1.0]], np.float32))
    off, idx = B.query(bvh, qs)
    torch.cuda.synchronize()
    assert off.cpu().tolist() == [0, 0]
    bvh = gpu_build(B, W.uniform_cube(100, seed=1), 30)
    off, idx = B.query(bvh, torch.zeros((0, 4), dtype=torch.float32, device="cuda"))
    torch.cuda.synchronize()
    assert off.cpu().tolist() == [0]
    # queries that hit nothing
    off, idx = B.query(bvh, _dev(np.array([[5, 5, 5, 0.1], [-5, 0, 0, 0.1]], np.float32)))
    torch.cuda.synchronize()
    assert off.cpu().tolist() == [0, 0, 0]


def test_deep_skewed_hierarchy(B, oracle_lib):
    """Heavy-tailed coordinates (u^12): a deep, lopsided radix tree with long runs of equal codes near the origin, so
    windows of the bottom-up pass hand over many subtrees and the upper windows see long chains."""
    u = W.uniform_cube(300_000, seed=77).astype(np.float64)
    pts = (u ** 12).astype(np.float32) + np.float32(0.0)
    for bits in (30, 63):
        o = oracle_lib.build_bvh(pts, bits)
        bvh = gpu_build(B, pts, bits)
        assert_build_equal(export_np(bvh), o, f"skewed {bits}")
    assert_query_equal(B, bvh, o, oracle_lib, W.spheres_at(pts[:3000], 1e-3), "skewed")


def test_merge_windows_multipass_reduced_capacity(B, oracle_lib, tmp_path):
    """The upper windows of the bottom-up pass shorten an item list that does not fit their shared memory by passes
    compacted in place.  With the product's capacity (1024 items per window) few inputs get there, so
    this test compiles the same sources with the smallest legal capacity (384 items, 128 threads) and checks the
    result of that build bit for bit: 64 hand-overs of ~8 subtrees each overflow 384 on ordinary data."""
    import shutil

    from paper_2402_00665_b200 import build as cuda_build

    if shutil.which("nvcc") is None and not __import__("os").path.exists("/usr/local/cuda/bin/nvcc"):
        pytest.skip("no nvcc on this box")
    lib = cuda_build.build(out=str(tmp_path / "libbvh_small_windows.so"),
                           extra=["-DBVH_MERGE_MAX_ITEMS=384", "-DBVH_MERGE_THREADS=128"])
    saved = (B._lib, B.LIB_PATH)
    try:
        B._lib, B.LIB_PATH = None, lib
        B.load_library()
        for name, n in (("C3", 1_200_000), ("C5", 700_001)):
            w = W.make(name, n=n, q=0)
            o = oracle_lib.build_bvh(w.prims, w.morton_bits)
            assert_build_equal(export_np(gpu_build(B, w.prims, w.morton_bits)), o, name)
    finally:
        B._lib, B.LIB_PATH = saved


# ---- NEXT-1: ray queries (D9) ---------------------------------------------------------------------------------

def _rays_through(prims, q, seed, tmax):
    lo, hi = prims[:, :3].min(axis=0), prims[:, -3:].max(axis=0)
    origins = W.uniform_cube(q, seed=seed) * (hi - lo) * np.float32(1.2) + lo - (hi - lo) * np.float32(0.1)
    rays = W.rays_at(origins.astype(np.float32), W.sphere_surface(q, seed=seed + 1), 0.0, tmax)
    rays[: q // 5, 3] = 0.0                        # parallel to the x slabs
    rays[q // 5: q // 4, 4:6] = 0.0                # along the x axis
    rays[q // 5: q // 4, 3] = -1.0
    rays[q // 4: q // 3, 6] = np.float32(0.05)     # tmin > 0
    return rays


@pytest.mark.parametrize("name,n,q,half,tmax", [("C2", 60_001, 20_000, 0.004, 0.5), ("C4", 80_000, 20_000, 0.01, 3.0),
                                               ("C3", 100_000, 8_000, 0.0005, 0.3)])
def test_ray_queries_parity(B, oracle_lib, name, n, q, half, tmax):
    """Ray predicate through the same Algorithm 1 kernel: CSR bit-equal to the oracle's stack traversal, raw order
    included; box leaves (32-byte records)."""
    w = W.make(name, n=n, q=0, radius=half if name == "C4" else None)
    prims = w.prims if name == "C4" else W.boxes_around(w.prims, half)
    rays = _rays_through(prims, q, seed=31, tmax=tmax)
    if name == "C3":                               # clustered: start the rays inside the clusters
        rays[:, :3] = w.prims[:q] + np.float32(0.0003)
    o = oracle_lib.build_bvh(prims, w.morton_bits)
    bvh = gpu_build(B, prims, w.morton_bits)
    goff, gidx = gpu_query(B, bvh, rays)
    ooff, oidx = oracle_lib.query_rays_tree(o, rays)
    assert np.array_equal(goff, ooff) and ooff[-1] > q // 2
    assert np.array_equal(gidx[: goff[-1]], oidx)


def test_ray_queries_point_leaves_and_brute_force(B, oracle_lib):
    """Point leaves (16-byte records): a ray hits a point only if it passes exactly through it, so the rays start AT
    primitives and run along an axis or towards another primitive's coordinates; checked against brute force."""
    pts = (W.uniform_cube(20_000, seed=12) * np.float32(64.0)).round().astype(np.float32) / np.float32(64.0)  # a lattice: many exact hits
    q = 3000
    d = np.zeros((q, 3), np.float32)
    d[np.arange(q), np.arange(q) % 3] = np.float32(1.0)
    d[::7] = np.float32([1.0, 1.0, 0.0])
    d[::11] = np.float32([-2.0, 1.0, 0.5])
    rays = W.rays_at(pts[:q], d, 0.0, 0.75)
    bvh = gpu_build(B, pts, 63)
    goff, gidx = gpu_query(B, bvh, rays)
    boff, bidx = oracle_lib.query_rays_brute(pts, rays)
    assert np.array_equal(goff, boff) and np.all(np.diff(goff) >= 1) and goff[-1] > 3 * q
    assert np.array_equal(csr_rows_sorted(goff, gidx[: goff[-1]]), bidx)
    # unordered = ordered
    o2, i2 = B.query(bvh, _dev(rays), ordered=False)
    torch.cuda.synchronize()
    assert np.array_equal(o2.cpu().numpy(), goff) and np.array_equal(i2.cpu().numpy(), gidx[: goff[-1]])


@pytest.mark.parametrize("n", [65_536 + 77, 5_000])
def test_cuda_graph_capture_and_replay(B, n):
    """The C ABI only enqueues work (no allocation, no synchronisation, no host read): a whole build + ordered
    count / scan / fill can be captured in a CUDA graph and replayed; the replay reproduces the eager result on the
    captured inputs and follows the inputs when their contents change.  Both forms of the build: the pipeline (with its
    cooperative launch of the conditional second sort) and the one-cluster front of a small build."""
    w = W.make("C5", n=n, q=4096, radius=0.02)
    d, dq = _dev(w.prims), _dev(w.queries)
    bvh, ws = B.Bvh(w.n, w.morton_bits), B.QueryWorkspace(w.q)
    bvh.nodes.zero_()
    bvh.build(d)
    off, idx = B.query(bvh, dq, ws)
    torch.cuda.synchronize()
    ref_nodes, ref_off, ref_idx = bvh.nodes.clone(), off.clone(), idx.clone()
    indices = torch.empty(2 * idx.numel() + 16, dtype=torch.int32, device="cuda")
    g, s = torch.cuda.CUDAGraph(), torch.cuda.Stream()
    with torch.cuda.stream(s):
        bvh.build(d)                                   # warm-up on the capture stream
        B.query(bvh, dq, ws, indices=indices)
        torch.cuda.synchronize()
        with torch.cuda.graph(g, stream=s):
            bvh.build(d)
            B.query(bvh, dq, ws, indices=indices)      # indices passed in: no nnz read-back inside the capture
    for _ in range(3):
        bvh.nodes.zero_(); indices.zero_(); ws.offsets.zero_()
        g.replay()
        torch.cuda.synchronize()
        assert torch.equal(bvh.nodes, ref_nodes)
        assert torch.equal(ws.offsets[: w.q + 1], ref_off) and torch.equal(indices[: ref_idx.numel()], ref_idx)
    # new contents in the captured buffers: the replay builds and queries the new scene
    w2 = W.make("C2", n=w.n, q=w.q, radius=0.02)
    d.copy_(_dev(w2.prims)); dq.copy_(_dev(w2.queries))
    g.replay()
    torch.cuda.synchronize()
    got_off, got_nodes = ws.offsets[: w.q + 1].clone(), bvh.nodes.clone()
    nnz = int(got_off[-1])
    got_idx = indices[:nnz].clone()
    bvh2 = B.Bvh(w.n, w.morton_bits)
    bvh2.nodes.zero_()
    bvh2.build(d)
    off2, idx2 = B.query(bvh2, dq)
    torch.cuda.synchronize()
    assert nnz <= indices.numel() and torch.equal(got_off, off2) and torch.equal(got_idx, idx2)
    assert torch.equal(got_nodes, bvh2.nodes)


@pytest.mark.parametrize("name,n", [("C1", 4096), ("C2", 100_001), ("C3", 300_000), ("C4", 120_000), ("C5", 70_000)])
def test_variant_karras_topdown(B, oracle_lib, name, n):
    """NEXT-2: Karras' top-down construction + Algorithm 2 + a separate box pass gives the same bytes as the single
    bottom-up pass ("identical hierarchy structure"), and both equal the oracle."""
    w = W.make(name, n=n, q=0)
    is_box = int(w.prims.shape[1] == 6)
    a = B.Bvh(w.n, w.morton_bits)
    a.nodes.zero_()
    a.build(_dev(w.prims))
    v = B.Bvh(w.n, w.morton_bits)
    v.scratch = torch.empty(B.bvh_variant_sizes(w.n, w.morton_bits, 1), dtype=torch.uint8, device="cuda")
    v.nodes.zero_()
    B.bvh_build_variant(_dev(w.prims), is_box, w.n, w.morton_bits, v.nodes, v.scratch, 1)
    torch.cuda.synchronize()
    assert torch.equal(a.nodes, v.nodes)
    assert_build_equal(export_np(v), oracle_lib.build_bvh(w.prims, w.morton_bits), name)
    for tiny in (1, 2, 3, 5):
        pts = W.uniform_cube(tiny, seed=tiny)
        t = B.Bvh(tiny, 63)
        t.scratch = torch.empty(B.bvh_variant_sizes(tiny, 63, 1), dtype=torch.uint8, device="cuda")
        B.bvh_build_variant(_dev(pts), 0, tiny, 63, t.nodes, t.scratch, 1)
        torch.cuda.synchronize()
        assert_build_equal(export_np(t), oracle_lib.build_bvh(pts, 63), f"tiny {tiny}")


def _variant2(B, prims, bits):
    n = prims.shape[0]
    v = B.Bvh(n, bits)
    v.scratch = torch.empty(B.bvh_variant_sizes(n, bits, 2), dtype=torch.uint8, device="cuda")
    v.nodes.zero_()
    B.bvh_build_variant(_dev(prims), int(prims.shape[1] == 6), n, bits, v.nodes, v.scratch, 2)
    out = {"left": torch.zeros(max(n - 1, 1), dtype=torch.int32, device="cuda"),
           "right": torch.zeros(max(n - 1, 1), dtype=torch.int32, device="cuda"),
           "rope": torch.zeros(2 * n - 1, dtype=torch.int32, device="cuda"),
           "aabb": torch.zeros((2 * n - 1, 6), dtype=torch.float32, device="cuda"),
           "root": torch.zeros(1, dtype=torch.int32, device="cuda")}
    B.bvh_variant_export(v.nodes, v.scratch, n, bits, 2, **out)
    torch.cuda.synchronize()
    return v, {k: t.cpu().numpy() for k, t in out.items()}


@pytest.mark.parametrize("name,n", [("C1", 4096), ("C2", 60_001), ("C3", 200_000), ("C4", 50_000), ("C5", 70_000)])
def test_variant_apetrei_algorithm3(B, oracle_lib, name, n):
    """NEXT-2 (a): the unmodified Algorithm 3 + a separate skip-connection pass builds the same tree with Apetrei's node
    numbering (index = split, stored root): every array equals the oracle's serial Algorithm 3 (which is pinned to the
    top-down tree renamed node-to-split), boxes bit for bit; the product's queries refuse the buffer."""
    w = W.make(name, n=n, q=0)
    o = oracle_lib.build_bvh(w.prims, w.morton_bits)
    t = oracle_lib.apetrei_tree(w.prims, o)
    v, g = _variant2(B, w.prims, w.morton_bits)
    assert int(g["root"][0]) == t.root
    assert np.array_equal(g["left"][: n - 1], t.left) and np.array_equal(g["right"][: n - 1], t.right)
    assert np.array_equal(g["rope"], t.rope)
    assert np.array_equal(g["aabb"].view(np.uint32), t.aabb.view(np.uint32))
    # the same tree as the product's: the always-true walk from the stored root visits the leaves in order
    lb = n - 1
    node, seen = t.root, []
    lc = np.concatenate([g["left"][: n - 1], np.zeros(n, np.int32)])
    for _ in range(2 * n):
        if node < 0:
            break
        if node >= lb:
            seen.append(node - lb)
            node = g["rope"][node]
        else:
            node = lc[node]
    assert seen == list(range(n))
    cnt = torch.full((4,), -1, dtype=torch.int32, device="cuda")
    B.bvh_query_spheres_count(v.nodes, n, _dev(W.spheres_at(W.uniform_cube(4, seed=1), 0.5)), 4, None, cnt)
    torch.cuda.synchronize()
    assert cnt.cpu().tolist() == [0, 0, 0, 0]                  # not a Karras-ordered hierarchy: refused
    for tiny in (1, 2, 3, 5):
        pts = W.uniform_cube(tiny, seed=tiny)
        ot = oracle_lib.apetrei_tree(pts, oracle_lib.build_bvh(pts, 63))
        _, gt = _variant2(B, pts, 63)
        assert np.array_equal(gt["rope"], ot.rope) and np.array_equal(gt["aabb"].view(np.uint32), ot.aabb.view(np.uint32))
        if tiny >= 2:
            assert int(gt["root"][0]) == ot.root and np.array_equal(gt["left"][: tiny - 1], ot.left)
            assert np.array_equal(gt["right"][: tiny - 1], ot.right)


# ---- the paper's worked example and the equal-codes case, straight through the CUDA path ---------------------------
# (tests/golden/*.txt are hand-derived from PAPER.md:120, :166, :101, :75; the oracle is not involved here)

def _gold_rows(name):
    with open(os.path.join(os.path.dirname(__file__), "golden", name)) as f:
        return [ln.split("#")[0].strip() for ln in f if ln.split("#")[0].strip()]


def _gold_arrays(name):
    return {t[0]: [int(v) for v in t[1:]] for t in (ln.split() for ln in _gold_rows(name)) if t[0] not in ("keys", "internal")}


def _p1_points():
    """Eight points on the x axis whose 10-bit x cells are c = 0, 64, 128, 160, 608, 768, 800, 1023 (x = c / 1024 and x = 1
    in the frame [0, 1]): c / 32 = 0, 2, 4, 5, 19, 24, 25, 31 has the same highest differing bit between neighbours
    (1, 2, 0, 4, 3, 0, 2) as the golden's 5-bit keys, and interleaving with the zero bits of y and z keeps that order, so the
    hierarchy is the one PAPER.md:120 describes.  Given in a shuffled order: the sort has to find the Morton order."""
    c = np.array([0, 64, 128, 160, 608, 768, 800, 1024], np.float32) / np.float32(1024)
    given = np.array([5, 2, 7, 0, 3, 6, 1, 4])
    pts = np.zeros((8, 3), np.float32)
    pts[:, 0] = c[given]
    return pts, np.argsort(given)                      # perm[i] = where the i-th smallest x was given


@pytest.mark.parametrize("bits", [30, 63])
def test_paper_worked_example_p1_through_the_cuda_path(B, bits):
    g = _gold_arrays("p1_worked_example.txt")
    pts, perm = _p1_points()
    bvh = gpu_build(B, pts, bits)
    e = export_np(bvh)
    assert e["perm"].tolist() == perm.tolist()
    assert e["left_child"][:7].tolist() == g["left_child"]          # I_3 -> I_1, I_2;  I_4 -> L_4, I_5
    assert e["rope"].tolist() == g["rope"]                          # right-most path -> sentinel
    d = np.diff(e["sorted_codes"].astype(np.int64))
    x = e["sorted_codes"][:-1] ^ e["sorted_codes"][1:]
    assert (d > 0).all() and np.array_equal(np.argsort(x, kind="stable"), np.argsort(np.array(g["delta_star"]), kind="stable"))
    # Algorithm 1 with an always-true predicate over the arrays the GPU built
    node, walk = 0, []
    while node != -1:
        walk.append(node)
        node = int(e["left_child"][node]) if node < 7 else int(e["rope"][node])
        assert len(walk) <= 15
    assert walk == g["walk"]
    # and the GPU's own traversal: a sphere around everything reports every leaf, in leaf order
    off, idx = gpu_query(B, bvh, np.array([[0.5, 0, 0, 2.0], [0.0625, 0, 0, 1.0 / 1024]], np.float32))
    assert off.tolist() == [0, 8, 9] and idx[:8].tolist() == perm.tolist() and idx[8] == perm[1]


def test_paper_worked_example_p1_apetrei_numbering_through_variant_2(B):
    """Algorithm 3 unmodified: nodes named by their split, root stored; "the children of I_0 have a
    gap of 3": root 3 with children 1 and 4."""
    g = _gold_arrays("p1_apetrei_numbering.txt")
    pts, _ = _p1_points()
    _, v = _variant2(B, pts, 30)
    assert int(v["root"][0]) == g["root"][0] == 3
    assert v["left"][:7].tolist() == g["left"] and v["right"][:7].tolist() == g["right"]
    assert (int(v["left"][3]), int(v["right"][3])) == (1, 4)
    assert v["rope"].tolist() == g["rope"]


@pytest.mark.parametrize("bits", [30, 63])
def test_equal_codes_p4_goldens_through_the_cuda_path(B, bits):
    """All codes equal: the augmented keys (code, i) decide; n = 1..5 against the hand-derived arrays."""
    for line in _gold_rows("p4_equal_codes.txt"):
        head, lc, rp = line.split("|")
        n = int(head.split()[1])
        e = export_np(gpu_build(B, np.full((n, 3), 0.25, np.float32), bits))
        assert e["left_child"][: n - 1].tolist() == [int(t) for t in lc.split()], n
        assert e["rope"].tolist() == [int(t) for t in rp.split()], n
        assert e["perm"].tolist() == list(range(n))


@pytest.mark.parametrize("cap", [128, 136, 1024])
def test_rows_to_csr_wide_copy_every_alignment_and_length(B, cap):
    """bvh_rows_to_csr on its own ("Store the result"): rows of 128 entries and more are copied by a warp with
    128-bit accesses whose destination starts at any 4-byte offset.  Every row length 0 .. cap + 3 occurs, next to rows of
    every other length, so every (alignment, length, head, tail) combination does; rows longer than cap are left alone."""
    rng = np.random.default_rng(cap)
    lengths = np.concatenate([np.arange(cap + 4), rng.integers(0, cap + 4, 3000), np.arange(cap + 4)[::-1], [cap] * 9])
    rng.shuffle(lengths[cap + 4: -9])
    q = len(lengths)
    rows = rng.integers(0, 1 << 30, (q, cap)).astype(np.int32)
    offsets = np.concatenate([[0], np.cumsum(lengths)]).astype(np.int64)
    want = np.full(int(offsets[-1]) + 8, -5, np.int32)
    for j in range(q):
        if lengths[j] <= cap:
            want[offsets[j]: offsets[j] + lengths[j]] = rows[j, : lengths[j]]
    got = torch.full((len(want),), -5, dtype=torch.int32, device="cuda")
    B.bvh_rows_to_csr(_dev(rows.reshape(-1)), cap, _dev(lengths.astype(np.int32)), _dev(offsets), q, got)
    torch.cuda.synchronize()
    assert np.array_equal(got.cpu().numpy(), want)


@pytest.mark.parametrize("name,n", [("C1", 4096), ("C2", 100_001), ("C3", 300_000), ("C4", 120_000), ("C5", 70_000)])
def test_variant_algorithm4_as_written(B, oracle_lib, name, n):
    """NEXT-2, third arm: Algorithm 4 in the plain form the paper gives it (one thread per leaf, global
    `store`, ATOMICCAS) produces the same bytes as the product's windowed single pass, and both equal the oracle."""
    w = W.make(name, n=n, q=0)
    is_box = int(w.prims.shape[1] == 6)
    a = B.Bvh(w.n, w.morton_bits)
    a.nodes.zero_()
    a.build(_dev(w.prims))
    v = B.Bvh(w.n, w.morton_bits)
    v.scratch = torch.empty(B.bvh_variant_sizes(w.n, w.morton_bits, 3), dtype=torch.uint8, device="cuda")
    v.nodes.zero_()
    for _ in range(2):                                  # twice into the same scratch: `store` is re-initialised per build
        B.bvh_build_variant(_dev(w.prims), is_box, w.n, w.morton_bits, v.nodes, v.scratch, 3)
        torch.cuda.synchronize()
        assert torch.equal(a.nodes, v.nodes)
    assert_build_equal(export_np(v), oracle_lib.build_bvh(w.prims, w.morton_bits), name)
    for tiny in (1, 2, 3, 4, 5):
        pts = W.uniform_cube(tiny, seed=tiny)
        t = B.Bvh(tiny, 63)
        t.scratch = torch.empty(B.bvh_variant_sizes(tiny, 63, 3), dtype=torch.uint8, device="cuda")
        B.bvh_build_variant(_dev(pts), 0, tiny, 63, t.nodes, t.scratch, 3)
        torch.cuda.synchronize()
        assert_build_equal(export_np(t), oracle_lib.build_bvh(pts, 63), f"tiny {tiny}")
    # the paper's worked example and the equal-codes case, against the hand-derived goldens
    g = _gold_arrays("p1_worked_example.txt")
    pts, perm = _p1_points()
    t = B.Bvh(8, 30)
    t.scratch = torch.empty(B.bvh_variant_sizes(8, 30, 3), dtype=torch.uint8, device="cuda")
    B.bvh_build_variant(_dev(pts), 0, 8, 30, t.nodes, t.scratch, 3)
    torch.cuda.synchronize()
    e = export_np(t)
    assert e["left_child"][:7].tolist() == g["left_child"] and e["rope"].tolist() == g["rope"] and e["perm"].tolist() == perm.tolist()
    for line in _gold_rows("p4_equal_codes.txt"):
        head, lc, rp = line.split("|")
        m = int(head.split()[1])
        t = B.Bvh(m, 30)
        t.scratch = torch.empty(B.bvh_variant_sizes(m, 30, 3), dtype=torch.uint8, device="cuda")
        B.bvh_build_variant(_dev(np.full((m, 3), 0.25, np.float32)), 0, m, 30, t.nodes, t.scratch, 3)
        torch.cuda.synchronize()
        e = export_np(t)
        assert e["left_child"][: m - 1].tolist() == [int(x) for x in lc.split()] and e["rope"].tolist() == [int(x) for x in rp.split()]
