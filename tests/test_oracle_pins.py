"""Pins for the CPU oracle (P1-P7 of DESIGN.md): what the paper and the mathematics fix.

None of these compares the oracle with itself or with the CUDA path: expected values are the paper's
facts (tests/golden/*.txt, hand-derived, cited), closed forms, numpy library routines, brute force in
exact arithmetic, or the test-side transliteration of Algorithm 4 in tests/helpers.py.
"""
from __future__ import annotations

import os
from fractions import Fraction

import numpy as np
import pytest

from helpers import alg4_serial, csr_rows_sorted
from paper_2402_00665_b200 import workloads as W

GOLD = os.path.join(os.path.dirname(__file__), "golden")


def _read_gold(name):
    rows = []
    with open(os.path.join(GOLD, name)) as f:
        for line in f:
            line = line.split("#")[0].strip()
            if line:
                rows.append(line)
    return rows


# ---- P1: worked example -----------------------------------------------------------------------------

def _p1():
    g = {"internal": {}}
    for line in _read_gold("p1_worked_example.txt"):
        tok = line.split()
        if tok[0] == "keys":
            g["keys"] = np.array([int(t, 2) for t in tok[1:]], np.uint64)
        elif tok[0] == "internal":
            g["internal"][int(tok[1])] = tuple(int(t) for t in tok[2:])
        else:
            g[tok[0]] = np.array([int(t) for t in tok[1:]], np.int64)
    return g


def test_p1_worked_example_states_the_papers_facts():
    """The fixture itself must say what PAPER.md:120 and PAPER.md:166 say."""
    g = _p1()
    n, lb = 8, 7
    f, l, split, left, right = g["internal"][3]
    assert (f, l, split, left, right) == (0, 3, 1, 1, 2)          # I3: [0,3], gamma=1, children I1, I2
    f, l, split, left, right = g["internal"][4]
    assert (f, l, split, left, right) == (4, 7, 4, lb + 4, 5)     # I4: [4,7], gamma=4, children L4, I5
    # Apetrei numbering = each node's own split; root's children have splits 1 and 4: gap 3
    _, _, _, rl, rr = g["internal"][0]
    assert g["internal"][rr][2] - g["internal"][rl][2] == 3
    # XOR form of delta*
    k = g["keys"]
    assert list(k[:-1] ^ k[1:]) == list(g["delta_star"])
    assert len(g["left_child"]) == n - 1 and len(g["rope"]) == 2 * n - 1


def test_p1_worked_example(oracle_lib):
    g = _p1()
    n = 8
    left, right, first, last = oracle_lib.hierarchy(g["keys"])
    for k, (f, l, split, lc, rc) in g["internal"].items():
        assert (first[k], last[k], left[k], right[k]) == (f, l, lc, rc), k
    assert list(left) == list(g["left_child"])
    rope = oracle_lib.ropes(left, right, n)
    assert list(rope) == list(g["rope"])
    assert list(oracle_lib.ropes_alg2(g["keys"], first, last)) == list(g["rope"])
    assert list(oracle_lib.walk_all(np.concatenate([left, np.zeros(n, np.int32)]), rope, n)) == list(g["walk"])


def test_p1_alg4_transliteration_reproduces_example():
    """The test-side Algorithm 4 (the second route used below) also lands on the paper's example."""
    g = _p1()
    left, rope = alg4_serial(g["keys"])
    assert list(left) == list(g["left_child"])
    assert list(rope) == list(g["rope"])


# ---- P4: closed forms -------------------------------------------------------------------------------

def test_p4_equal_codes(oracle_lib):
    for line in _read_gold("p4_equal_codes.txt"):
        head, lc, rp = line.split("|")
        n = int(head.split()[1])
        exp_left = [int(t) for t in lc.split()]
        exp_rope = [int(t) for t in rp.split()]
        codes = np.full(n, 12345, np.uint64)
        left, right, first, last = oracle_lib.hierarchy(codes)
        assert list(left) == exp_left, n
        assert list(oracle_lib.ropes(left, right, n)) == exp_rope, n
        # through the whole build: coincident points
        b = oracle_lib.build_bvh(np.full((n, 3), 0.25, np.float32), 30)
        assert list(b.left_child[: n - 1]) == exp_left
        assert list(b.rope) == exp_rope
        assert list(b.perm) == list(range(n))


@pytest.mark.parametrize("n", [2, 4, 64, 1024])
def test_p4_perfect_tree(oracle_lib, n):
    """codes = 0..n-1, n a power of two: perfect tree of depth log2 n; node covering [f,l] splits in the middle."""
    left, right, first, last = oracle_lib.hierarchy(np.arange(n, dtype=np.uint64))
    lb = n - 1
    for k in range(n - 1):
        f, l = int(first[k]), int(last[k])
        size = l - f + 1
        assert size & (size - 1) == 0 and f % size == 0
        gamma = f + size // 2 - 1
        assert left[k] == (lb + gamma if size == 2 else gamma)
        assert right[k] == (lb + gamma + 1 if size == 2 else gamma + 1)
    rope = oracle_lib.ropes(left, right, n)
    order = oracle_lib.walk_all(np.concatenate([left, np.zeros(n, np.int32)]), rope, n)
    assert len(order) == 2 * n - 1
    assert list(order[order >= lb] - lb) == list(range(n))


def test_p4_t_corner(oracle_lib):
    """G14: codes 0 and 2^63-1 (opposite scene corners, 63-bit): XOR = INT64_MAX must still be < +inf."""
    b = oracle_lib.build_bvh(np.array([[0, 0, 0], [1, 1, 1]], np.float32), 63)
    assert list(b.sorted_codes) == [0, (1 << 63) - 1]
    assert list(b.left_child[:1]) == [1]
    assert list(b.rope) == [-1, 2, -1]
    left, rope = alg4_serial(b.sorted_codes)
    assert list(left) == [1] and list(rope) == [-1, 2, -1]


def test_p4_points_equal_degenerate_boxes(oracle_lib):
    w = W.make("C2", n=3000, q=0)
    a = oracle_lib.build_bvh(w.prims, 63)
    b = oracle_lib.build_bvh(np.concatenate([w.prims, w.prims], axis=1), 63)
    for f in ("sorted_codes", "perm", "left_child", "rope", "aabb", "scene_bounds"):
        assert np.array_equal(getattr(a, f).view(np.uint8), getattr(b, f).view(np.uint8)), f


def test_p4_zero_extent_axis(oracle_lib):
    pts = W.uniform_cube(500, seed=77)
    pts[:, 1] = 0.5
    b = oracle_lib.build_bvh(pts, 30)
    y_bits = sum(1 << (3 * k + 1) for k in range(10))
    assert not np.any(b.sorted_codes & np.uint64(y_bits))
    assert np.all(np.isfinite(b.aabb))


# ---- P7: Morton ---------------------------------------------------------------------------------------

def _interleave_str(cx, cy, cz, b):
    """x most significant within each triple; written with strings, not shifts."""
    sx, sy, sz = (format(c, f"0{b}b") for c in (cx, cy, cz))
    return int("".join(x + y + z for x, y, z in zip(sx, sy, sz)), 2)


@pytest.mark.parametrize("bits", [30, 63])
def test_p7_morton_corners(oracle_lib, bits):
    b = bits // 3
    scene = np.array([0, 0, 0, 1, 1, 1], np.float32)
    pts = np.array([[0, 0, 0], [1, 1, 1], [0.5, 0.5, 0.5], [1, 0, 0], [0, 1, 0], [0, 0, 1]], np.float32)
    codes = oracle_lib.morton(pts, scene, bits)
    ones = (1 << b) - 1
    assert codes[0] == 0
    assert codes[1] == (1 << bits) - 1                       # clamp path
    assert codes[2] == 0b111 << (3 * (b - 1))                # centre: cell 2^(b-1) on each axis
    assert codes[3] == _interleave_str(ones, 0, 0, b)
    assert codes[4] == _interleave_str(0, ones, 0, b)
    assert codes[5] == _interleave_str(0, 0, ones, b)
    assert codes[3] > codes[4] > codes[5]                     # x most significant


@pytest.mark.parametrize("bits", [30, 63])
def test_p7_morton_exact_grid(oracle_lib, bits):
    """Points at k / 2^b in a [0,1] frame: (k/2^b - 0)/1 * 2^b = k exactly, so cell = k on every axis."""
    b = bits // 3
    rng = np.random.default_rng(7)
    cells = rng.integers(0, 1 << b, size=(2000, 3))
    pts = (cells.astype(np.float64) / (1 << b)).astype(np.float32)   # exact: b <= 21 < 24 bits
    pts = np.concatenate([pts, [[0, 0, 0], [1, 1, 1]]]).astype(np.float32)
    scene = oracle_lib.scene_bounds(pts)
    assert list(scene) == [0, 0, 0, 1, 1, 1]
    codes = oracle_lib.morton(pts, scene, bits)
    for i in range(0, 2000, 37):
        assert int(codes[i]) == _interleave_str(*[int(c) for c in cells[i]], b), i


def test_p7_morton_box_centroid_and_frame(oracle_lib):
    """Centroid of a box, frame not at the origin (exactly representable numbers throughout)."""
    scene = np.array([-2, -2, -2, 2, 2, 2], np.float32)
    box = np.array([[-1.5, 0.0, 1.0, -0.5, 1.0, 2.0]], np.float32)    # centroid (-1, 0.5, 1.5)
    # t = (c + 2) / 4 = 0.25, 0.625, 0.875 ; cell = t * 1024 = 256, 640, 896
    code = oracle_lib.morton(box, scene, 30)[0]
    assert int(code) == _interleave_str(256, 640, 896, 10)


@pytest.mark.parametrize("bits", [30, 63])
def test_p7_morton_monotone_and_matches_exact_rational(oracle_lib, bits):
    """cell = floor(t * 2^b) where t is the fp32 quotient; check against exact rational arithmetic on the
    fp32 operands wherever the exact value is further from a cell boundary than the fp32 rounding error."""
    b = bits // 3
    pts = W.uniform_cube(4000, seed=11) * np.float32(3.0) - np.float32(1.0)
    scene = oracle_lib.scene_bounds(pts)
    codes = oracle_lib.morton(pts, scene, bits)
    # de-interleave
    cells = np.zeros((len(pts), 3), np.int64)
    for k in range(b):
        for a in range(3):
            cells[:, a] |= ((codes >> np.uint64(3 * k + 2 - a)) & np.uint64(1)).astype(np.int64) << k
    checked = 0
    for i in range(0, len(pts), 13):
        for a in range(3):
            c, lo, hi = (Fraction(float(v)) for v in (pts[i, a], scene[a], scene[3 + a]))
            t = (c - lo) / (hi - lo) * (1 << b)
            margin = t * Fraction(1, 1 << 22)                    # two fp32 roundings (numerator, quotient)
            if abs(t - round(t)) > margin:
                assert cells[i, a] == min(int(t), (1 << b) - 1), (i, a)
                checked += 1
    assert checked > 300
    order = np.argsort(pts[:, 0], kind="stable")
    assert np.all(np.diff(cells[order, 0]) >= 0)             # moving along +x never decreases cell_x


# ---- D1 / P6 ----------------------------------------------------------------------------------------

def test_d1_scene_bounds_vs_numpy(oracle_lib):
    w = W.make("C4", n=5000, q=0)
    s = oracle_lib.scene_bounds(w.prims)
    assert np.array_equal(s[:3], w.prims[:, :3].min(axis=0)) and np.array_equal(s[3:], w.prims[:, 3:].max(axis=0))
    assert s[0] < 0 < s[3]
    p = W.make("C2", n=5000, q=0).prims
    s = oracle_lib.scene_bounds(p)
    assert np.array_equal(s[:3], p.min(axis=0)) and np.array_equal(s[3:], p.max(axis=0))


def test_p6_sort_vs_numpy_stable(oracle_lib):
    rng = np.random.default_rng(3)
    codes = rng.integers(0, 50, size=20000).astype(np.uint64) << np.uint64(40)   # many ties
    s, perm = oracle_lib.sort_codes(codes)
    ref = np.argsort(codes, kind="stable")
    assert np.array_equal(perm, ref.astype(np.uint32))
    assert np.array_equal(s, codes[ref])


# ---- P2 / P3 / Algorithm 4 on random inputs ------------------------------------------------------------

def _random_sorted_codes(rng, n, kind):
    if kind == "distinct":
        c = rng.choice(1 << 20, size=n, replace=False).astype(np.uint64)
    elif kind == "ties":
        c = rng.integers(0, max(2, n // 4), size=n).astype(np.uint64)
    elif kind == "wide":
        c = rng.integers(0, 1 << 62, size=n).astype(np.uint64) * np.uint64(2) + rng.integers(0, 2, size=n).astype(np.uint64)
        c &= np.uint64((1 << 63) - 1)
    else:
        c = np.full(n, 9, np.uint64)
    return np.sort(c)


@pytest.mark.parametrize("kind", ["distinct", "ties", "wide", "equal"])
def test_alg4_any_schedule_equals_karras_topdown(oracle_lib, kind):
    """PAPER.md:33 'identical hierarchy structure' + Section 4: Algorithm 4 in any thread order gives the
    Karras numbering, left children and ropes the top-down oracle gives."""
    rng = np.random.default_rng(hash(kind) % 1000)
    for trial in range(120):
        n = int(rng.integers(1, 40))
        codes = _random_sorted_codes(rng, n, kind)
        left, right, first, last = oracle_lib.hierarchy(codes)
        rope = oracle_lib.ropes(left, right, n)
        a_left, a_rope = alg4_serial(codes, order=rng.permutation(n))
        assert list(a_left) == list(left), (kind, trial, list(codes))
        assert list(a_rope) == list(rope), (kind, trial, list(codes))


@pytest.mark.parametrize("name,n", [("C1", 4096), ("C2", 20000), ("C3", 30000), ("C4", 20000), ("C5", 20000)])
def test_p2_p3_invariants(oracle_lib, name, n):
    w = W.make(name, n=n, q=0)
    b = oracle_lib.build_bvh(w.prims, w.morton_bits)
    lb = n - 1
    left, right, first, last = oracle_lib.hierarchy(b.sorted_codes)
    assert np.array_equal(left, b.left_child[:lb])
    # P2: Algorithm 2 closed form == stack-walk ropes
    assert np.array_equal(oracle_lib.ropes_alg2(b.sorted_codes, first, last), b.rope)
    # sort invariants
    assert np.array_equal(np.sort(b.perm), np.arange(n, dtype=np.uint32))
    d = np.diff(b.sorted_codes.astype(np.int64))
    assert np.all(d >= 0)
    assert np.all(np.diff(b.perm.astype(np.int64))[d == 0] > 0)
    # root and right-most path
    assert first[0] == 0 and last[0] == n - 1 and b.rope[0] == -1
    node = 0
    while node < lb:
        assert b.rope[node] == -1
        node = right[node]
    assert b.rope[node] == -1 and node == lb + n - 1
    # Karras index = a range bound; siblings consecutive; rope of a left child = sibling
    k = np.arange(lb)
    assert np.all((first == k) | (last == k))
    gl = np.where(left >= lb, left - lb, left)
    gr = np.where(right >= lb, right - lb, right)
    assert np.all(gr == gl + 1)
    assert np.array_equal(b.rope[left], right)
    # always-true traversal: every node once, leaves in order
    order = oracle_lib.walk_all(b.left_child, b.rope, n)
    assert len(order) == 2 * n - 1 and len(np.unique(order)) == 2 * n - 1
    assert np.array_equal(order[order >= lb] - lb, np.arange(n))
    # boxes: internal = union of leaf boxes in its range (checked by prefix-free direct reduction on a sample);
    # root box = scene bounds bit for bit
    assert np.array_equal(b.aabb[0].view(np.uint32), b.scene_bounds.view(np.uint32))
    leaf = b.aabb[lb:]
    rng = np.random.default_rng(0)
    for kk in rng.integers(0, lb, size=200):
        f, l = first[kk], last[kk]
        assert np.array_equal(b.aabb[kk, :3], leaf[f:l + 1, :3].min(axis=0))
        assert np.array_equal(b.aabb[kk, 3:], leaf[f:l + 1, 3:].max(axis=0))
    src = w.prims if w.prims.shape[1] == 6 else np.concatenate([w.prims, w.prims], axis=1)
    assert np.array_equal(leaf, src[b.perm])
    assert np.array_equal(b.left_child[lb:], b.perm.astype(np.int32))


# ---- P5: queries --------------------------------------------------------------------------------------

def _exact_sphere_rows(prims6, xyzr, margin=1e-5):
    """fp64 distance test; returns (surely_in, surely_out) boolean matrices, leaving a band around the
    threshold undecided (fp32 rounding of d2 and r*r is ~1e-7 relative)."""
    lo, hi = prims6[:, :3].astype(np.float64), prims6[:, 3:].astype(np.float64)
    c = xyzr[:, None, :3].astype(np.float64)
    d = np.maximum(np.maximum(lo[None] - c, c - hi[None]), 0.0)
    d2 = (d * d).sum(axis=2)
    r2 = (xyzr[:, 3].astype(np.float64) ** 2)[:, None]
    return d2 < r2 * (1 - margin), d2 > r2 * (1 + margin)


def test_p5_c1_brute_force_and_exact(oracle_lib):
    w = W.make("C1")
    b = oracle_lib.build_bvh(w.prims, w.morton_bits)
    to, ti = oracle_lib.query_spheres_tree(b, w.queries)
    bo, bi = oracle_lib.query_spheres_brute(w.prims, w.queries)
    assert np.array_equal(to, bo)
    assert np.array_equal(csr_rows_sorted(to, ti), bi)
    assert 9.5 < to[-1] / w.q < 11.5                          # ~10 neighbours each (BASELINE.json configs[0])
    # every query is centred on its own point: d2 = 0
    for j in range(0, w.q, 97):
        assert j in bi[bo[j]:bo[j + 1]]
    # exact arithmetic outside the rounding band
    sure_in, sure_out = _exact_sphere_rows(w.prims[:, :6], w.queries[:256])
    member = np.zeros_like(sure_in)
    for j in range(256):
        member[j, bi[bo[j]:bo[j + 1]]] = True
    assert np.all(member[sure_in]) and not np.any(member[sure_out])


@pytest.mark.parametrize("name,n,q", [("C2", 30000, 400), ("C3", 40000, 300), ("C5", 30000, 400)])
def test_p5_sphere_tree_equals_brute(oracle_lib, name, n, q):
    w = W.make(name, n=n, q=q, radius={"C2": 0.05, "C3": 0.004, "C5": 0.05}[name])
    b = oracle_lib.build_bvh(w.prims, w.morton_bits)
    to, ti = oracle_lib.query_spheres_tree(b, w.queries)
    bo, bi = oracle_lib.query_spheres_brute(w.prims, w.queries)
    assert to[-1] > q
    assert np.array_equal(to, bo) and np.array_equal(csr_rows_sorted(to, ti), bi)
    p6 = np.concatenate([w.prims, w.prims], axis=1)
    sure_in, sure_out = _exact_sphere_rows(p6, w.queries[:64])
    member = np.zeros_like(sure_in)
    for j in range(64):
        member[j, bi[bo[j]:bo[j + 1]]] = True
    assert np.all(member[sure_in]) and not np.any(member[sure_out])


def test_p5_box_tree_equals_brute_and_numpy(oracle_lib):
    w = W.make("C4", n=30000, q=500, radius=1e-2)
    b = oracle_lib.build_bvh(w.prims, w.morton_bits)
    to, ti = oracle_lib.query_boxes_tree(b, w.queries)
    bo, bi = oracle_lib.query_boxes_brute(w.prims, w.queries)
    assert to[-1] > 500
    assert np.array_equal(to, bo) and np.array_equal(csr_rows_sorted(to, ti), bi)
    # box-box overlap has no arithmetic: numpy comparison is the definition
    P, Q = w.prims, w.queries
    for j in range(0, 500, 7):
        hit = np.all((Q[j, :3] <= P[:, 3:]) & (P[:, :3] <= Q[j, 3:]), axis=1)
        assert np.array_equal(np.nonzero(hit)[0].astype(np.int32), bi[bo[j]:bo[j + 1]])


def test_p5_touching_counts(oracle_lib):
    """G12 closed comparisons: a sphere of radius exactly the distance, a box sharing a face."""
    prim = np.array([[1, 0, 0, 2, 1, 1]], np.float32)
    o, i = oracle_lib.query_spheres_brute(prim, np.array([[0, 0.5, 0.5, 1.0]], np.float32))
    assert list(i) == [0]
    o, i = oracle_lib.query_spheres_brute(prim, np.array([[0, 0.5, 0.5, 0.99999994]], np.float32))
    assert list(i) == []
    o, i = oracle_lib.query_boxes_brute(prim, np.array([[0, 0, 0, 1, 1, 1]], np.float32))
    assert list(i) == [0]
    o, i = oracle_lib.query_boxes_brute(prim, np.array([[0, 0, 0, 0.99999994, 1, 1]], np.float32))
    assert list(i) == []


# ---- D9 (NEXT-1): ray predicate -----------------------------------------------------------------------------

def test_d9_ray_closed_forms(oracle_lib):
    """Axis-aligned and diagonal rays against boxes on a lattice: hits known by inspection; touching counts (G12);
    a ray parallel to a slab is inside it or never enters it; [tmin, tmax] clips the ray."""
    boxes = np.array([[0, 0, 0, 1, 1, 1], [2, 0, 0, 3, 1, 1], [0, 2, 0, 1, 3, 1], [2, 2, 2, 3, 3, 3]], np.float32)
    rays = np.array([
        [-1, .5, .5, 1, 0, 0, 0, 10],      # +x through boxes 0 and 1
        [-1, .5, .5, 1, 0, 0, 0, 2.5],     # stops at x = 1.5: box 0 only
        [-1, .5, .5, 1, 0, 0, 2.5, 10],    # starts at x = 1.5: box 1 only
        [-1, .5, .5, -1, 0, 0, 0, 10],     # points away
        [.5, -1, .5, 0, 1, 0, 0, 10],      # +y through boxes 0 and 2
        [-1, 1, .5, 1, 0, 0, 0, 10],       # grazes the face y = 1: touching counts
        [-1, 1.5, .5, 1, 0, 0, 0, 10],     # between the rows: nothing
        [-1, -1, -1, 1, 1, 1, 0, 10],      # the diagonal: boxes 0 and 3
        [-1, -1, -1, 1, 1, 1, 0, 3],       # ... clipped at (2,2,2): reaches the corner of box 3 (touching)
        [-1, -1, -1, 1, 1, 1, 0, 2.5],     # ... clipped before box 3
        [-1, .5, .5, 2, 0, 0, 0, 1],       # faster ray: t in [0,1] covers x in [-1,1]: box 0
    ], np.float32)
    off, idx = oracle_lib.query_rays_brute(boxes, rays)
    rows = [sorted(idx[off[j]:off[j + 1]].tolist()) for j in range(len(rays))]
    assert rows == [[0, 1], [0], [1], [], [0, 2], [0, 1], [], [0, 3], [0, 3], [0], [0]]


def test_d9_ray_matches_exact_rational(oracle_lib):
    """Inputs on which every fp32 operation of D9 is exact (coordinates and t in multiples of 1/8, direction
    components 0, +-1/2, +-1, +-2): the oracle must equal the slab test evaluated in exact rational arithmetic."""
    from fractions import Fraction as F

    rng = np.random.default_rng(9)
    nb, nr = 60, 400
    lo = rng.integers(-40, 40, size=(nb, 3))
    ext = rng.integers(0, 24, size=(nb, 3))
    boxes = (np.concatenate([lo, lo + ext], axis=1) / 8.0).astype(np.float32)
    o = rng.integers(-48, 48, size=(nr, 3)) / 8.0
    d = rng.choice([0.0, 0.5, -0.5, 1.0, -1.0, 2.0, -2.0], size=(nr, 3))
    tmin = rng.integers(0, 16, size=nr) / 8.0
    tmax = tmin + rng.integers(0, 80, size=nr) / 8.0
    rays = np.concatenate([o, d, tmin[:, None], tmax[:, None]], axis=1).astype(np.float32)
    off, idx = oracle_lib.query_rays_brute(boxes, rays)
    for j in range(nr):
        expect = []
        for i in range(nb):
            tn, tf, ok = F(float(tmin[j])), F(float(tmax[j])), True
            for a in range(3):
                oa, da = F(float(o[j, a])), F(float(d[j, a]))
                l, h = F(float(boxes[i, a])), F(float(boxes[i, 3 + a]))
                if da == 0:
                    ok = ok and (l <= oa <= h)
                else:
                    t1, t2 = (l - oa) / da, (h - oa) / da
                    tn, tf = max(tn, min(t1, t2)), min(tf, max(t1, t2))
            if ok and tn <= tf:
                expect.append(i)
        assert idx[off[j]:off[j + 1]].tolist() == expect, j


def _ray_case(name, n, q):
    """Boxes a ray has a chance to hit, and rays through them: (prims [n,6], rays [q,8])."""
    if name == "C2":
        prims = W.boxes_around(W.make("C2", n=n, q=0).prims, 0.01)
        origins = W.uniform_cube(q, seed=77)
    else:
        prims = W.make("C4", n=n, q=0, radius=0.02).prims
        origins = W.uniform_cube(q, seed=78) * np.float32(3.0) - np.float32(1.5)
    rays = W.rays_at(origins, W.sphere_surface(q, seed=55), 0.0, 0.4 if name == "C2" else 3.0)
    rays[: q // 4, 3] = 0.0                       # some rays parallel to the x slabs
    rays[q // 4: q // 3, 4:6] = 0.0               # some along the x axis
    rays[q // 4: q // 3, 3] = 1.0
    return prims, rays


@pytest.mark.parametrize("name,n,q", [("C2", 30000, 300), ("C4", 30000, 300)])
def test_d9_ray_tree_equals_brute(oracle_lib, name, n, q):
    """The hit set does not depend on the tree (every step of D9 is monotone in the box, so a hit leaf implies hit
    ancestors): stack traversal of the oracle tree = brute force over all primitives."""
    prims, rays = _ray_case(name, n, q)
    o = oracle_lib.build_bvh(prims, 63)
    toff, tidx = oracle_lib.query_rays_tree(o, rays)
    boff, bidx = oracle_lib.query_rays_brute(prims, rays)
    assert np.array_equal(toff, boff) and toff[-1] > q
    assert np.array_equal(csr_rows_sorted(toff, tidx), bidx)


# ---- NEXT-2 (a): Algorithm 3, Apetrei's numbering ----------------------------------------------------------------

def _renumber_karras_to_apetrei(o_left, o_right, o_last, n):
    """Test-side renaming of a Karras-ordered tree: every internal node takes its split position as its index
    (PAPER.md:164).  Returns (root, left, right) in unified indices."""
    lb = n - 1
    split = np.array([(o_left[k] - lb) if o_left[k] >= lb else o_last[o_left[k]] for k in range(n - 1)], np.int64)
    ren = lambda c: c if c >= lb else split[c]  # noqa: E731
    left, right = np.empty(n - 1, np.int32), np.empty(n - 1, np.int32)
    for k in range(n - 1):
        left[split[k]] = ren(o_left[k])
        right[split[k]] = ren(o_right[k])
    assert sorted(split.tolist()) == list(range(n - 1))       # every boundary is the split of exactly one node
    return int(split[0]), left, right, split


def test_apetrei_p1_numbering(oracle_lib):
    """Algorithm 3 on the worked example: the root's children sit at 1 and 4, a gap of 3."""
    g = {ln.split()[0]: [int(x) for x in ln.split()[1:]] for ln in _read_gold("p1_apetrei_numbering.txt")}
    keys = _p1()["keys"]
    pts = np.zeros((8, 3), np.float32)                         # boxes are not looked at here

    class O:                                                   # the part of a Bvh that apetrei_tree reads
        sorted_codes = keys
        perm = np.arange(8, dtype=np.uint32)

    t = oracle_lib.apetrei_tree(pts, O)
    assert t.root == g["root"][0] == 3
    assert list(t.left) == g["left"] and list(t.right) == g["right"]
    assert list(t.rope) == g["rope"]
    assert (t.left[t.root], t.right[t.root]) == (1, 4) and t.right[t.root] - t.left[t.root] == 3


@pytest.mark.parametrize("kind", ["distinct", "ties", "wide", "equal"])
def test_apetrei_equals_renumbered_karras(oracle_lib, kind):
    """Karras' and Apetrei's constructions "result in an identical hierarchy structure"; only the node
    indices differ.  Algorithm 3 run serially = the top-down tree with every node renamed to its split."""
    rng = np.random.default_rng(17)
    for n in (2, 3, 5, 8, 33, 257, 2000):
        codes = _random_sorted_codes(rng, n, kind)
        left, right, first, last = oracle_lib.hierarchy(codes)
        root, a_left, a_right, split = _renumber_karras_to_apetrei(left, right, last, n)
        class O:
            sorted_codes = codes
            perm = np.arange(n, dtype=np.uint32)

        pts = rng.random((n, 3)).astype(np.float32)
        t = oracle_lib.apetrei_tree(pts, O)
        assert t.root == root and np.array_equal(t.left, a_left) and np.array_equal(t.right, a_right), (kind, n)
        # skip-connections and boxes: the Karras tree's, renamed
        rope_k = oracle_lib.ropes(left, right, n)
        box_k = oracle_lib.boxes(pts, O.perm, left, right)
        lb = n - 1
        ren = lambda c: c if (c >= lb or c < 0) else split[c]  # noqa: E731
        for k in range(n - 1):
            assert t.rope[split[k]] == ren(rope_k[k])
            assert np.array_equal(t.aabb[split[k]], box_k[k])
        assert np.array_equal(t.rope[lb:], np.array([ren(c) for c in rope_k[lb:]], np.int32))
        assert np.array_equal(t.aabb[lb:], box_k[lb:])


# ---- D10 / D11: operations at the leaf -----------------------------------------------------------------

def test_d10_nearest_closed_forms(oracle_lib):
    """Cases whose answer is known by inspection (coordinates and radii are dyadic: every fp32 step is exact)."""
    f = np.float32
    pts = np.array([[0, 0, 0], [1, 0, 0], [3, 0, 0], [1, 0, 0]], f)           # primitives 1 and 3 coincide
    qs = np.array([
        [0.875, 0, 0, 1.0],      # nearest is primitive 1 (d2 = 1/64); 3 is as near: the smaller index wins
        [0.5, 0, 0, 1.0],        # 0 and 1 (and 3) at d2 = 1/4: smallest index 0
        [2.0, 0, 0, 0.125],      # nothing within the radius
        [2.0, 0, 0, 1.0],        # primitives 1, 2, 3 exactly AT the radius (closed, G12): smallest index 1
        [3.0, 0.5, 0, 0.5],      # only primitive 2, at the radius
        [0, 0, 0, 0.0],          # zero radius on a primitive: d2 = 0 <= 0
    ], f)
    idx, d2 = oracle_lib.nearest_spheres_brute(pts, qs)
    assert idx.tolist() == [1, 0, -1, 1, 2, 0]
    assert d2[[0, 1, 3, 4, 5]].tolist() == [1 / 64, 0.25, 1.0, 0.25, 0.0] and np.isposinf(d2[2])
    # box primitives: distance to the box, not to its centre
    boxes = np.array([[0, 0, 0, 1, 1, 1], [2, 0, 0, 4, 1, 1]], f)
    idx, d2 = oracle_lib.nearest_spheres_brute(boxes, np.array([[1.5, 0.5, 0.5, 1], [1.75, 0.5, 0.5, 1], [0.5, 0.5, 0.5, 0]], f))
    assert idx.tolist() == [0, 1, 0] and d2.tolist() == [0.25, 1 / 16, 0.0]


@pytest.mark.parametrize("name,n,q", [("C1", 4096, 300), ("C3", 30000, 300), ("C4", 20000, 300)])
def test_d10_nearest_tree_equals_brute_and_is_the_row_minimum(oracle_lib, name, n, q):
    w = W.make(name, n=n, q=q, radius=(0.02 if name == "C4" else None))
    spheres = w.queries if w.queries.shape[1] == 4 else W.spheres_at(w.queries[:, :3], 0.02)
    o = oracle_lib.build_bvh(w.prims, w.morton_bits)
    bi, bd = oracle_lib.nearest_spheres_brute(w.prims, spheres)
    ti, td = oracle_lib.nearest_spheres_tree(o, spheres)
    assert np.array_equal(bi, ti) and np.array_equal(bd.view(np.uint32), td.view(np.uint32))
    # the definition again, in numpy on the CSR rows of the range search: minimum of (d2, index) over the row
    off, idx = oracle_lib.query_spheres_brute(w.prims, spheres)
    prim6 = w.prims if w.prims.shape[1] == 6 else np.concatenate([w.prims, w.prims], axis=1)
    some = 0
    for j in range(q):
        row = idx[off[j]:off[j + 1]]
        if len(row) == 0:
            assert bi[j] == -1 and np.isposinf(bd[j])
            continue
        c = spheres[j, :3]
        d = np.maximum(np.maximum(prim6[row, :3] - c, c - prim6[row, 3:]), np.float32(0))
        s = d * d
        d2 = (s[:, 0] + s[:, 1]) + s[:, 2]
        k = np.lexsort((row, d2))[0]
        assert bi[j] == row[k] and bd[j] == d2[k]
        some += 1
    assert some > q // 2


def test_d11_first_hit_closed_forms(oracle_lib):
    f = np.float32
    boxes = np.array([[4, -1, -1, 5, 1, 1], [1, -1, -1, 2, 1, 1], [1, -1, -1, 3, 1, 1], [7, 2, 2, 8, 3, 3]], f)
    rays = np.array([
        [0, 0, 0, 1, 0, 0, 0, 100],        # enters boxes 1 and 2 at t = 1 (smaller index wins), box 0 at t = 4
        [0, 0, 0, 1, 0, 0, 2.5, 100],      # tmin inside box 2 only: t_enter = tmin = 2.5; box 1 is behind, box 0 at 4
        [6, 0, 0, -1, 0, 0, 0, 100],       # from the other side: box 0 first, at t = 1
        [0, 0, 0, 1, 0, 0, 0, 0.5],        # too short
        [0, 5, 0, 1, 0, 0, 0, 100],        # misses everything
        [0, 0, 0, 2, 0, 0, 0, 100],        # direction not normalised: t in units of |d|: box 1 at t = 0.5
        [1.5, 0, 0, 0, 0, 1, 0, 100],      # starts inside boxes 1 and 2, parallel to two slabs: t_enter = tmin = 0
    ], f)
    idx, t = oracle_lib.first_hit_rays_brute(boxes, rays)
    assert idx.tolist() == [1, 2, 0, -1, -1, 1, 1]
    assert t[[0, 1, 2, 5, 6]].tolist() == [1.0, 2.5, 1.0, 0.5, 0.0] and np.isposinf(t[3]) and np.isposinf(t[4])


@pytest.mark.parametrize("name,n,q", [("C2", 30000, 300), ("C4", 30000, 300)])
def test_d11_first_hit_tree_equals_brute_and_is_the_row_minimum(oracle_lib, name, n, q):
    prims, rays = _ray_case(name, n, q)
    o = oracle_lib.build_bvh(prims, 63)
    bi, bt = oracle_lib.first_hit_rays_brute(prims, rays)
    ti, tt = oracle_lib.first_hit_rays_tree(o, rays)
    assert np.array_equal(bi, ti) and np.array_equal(bt.view(np.uint32), tt.view(np.uint32))
    off, idx = oracle_lib.query_rays_brute(prims, rays)
    assert np.array_equal(bi >= 0, np.diff(off) > 0)                      # "any hit" = the row is not empty
    for j in range(q):                                                     # the winner is a member of the row
        assert bi[j] == -1 or bi[j] in idx[off[j]:off[j + 1]]
    assert (bi >= 0).sum() > 10
