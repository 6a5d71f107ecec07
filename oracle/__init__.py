"""CPU oracle for the linear-BVH hot path -- TEST INFRASTRUCTURE ONLY.

Thin ctypes loader around ``oracle/bvh_oracle.cpp`` (serial C++, fp32, no contraction), which states
what the path computes, written from PAPER.md (see the header of that file for the passage each
function follows).  Only ``tests/``, ``__graft_entry__.smoke()`` and ``bench.py``'s ``cpu_baseline``
/ ``--impl reference`` legs may import this package.  It imports nothing from
``paper_2402_00665_b200`` and shares no code with the CUDA path.

All functions take and return numpy arrays.  Codes are uint64 whatever ``bits`` is.
"""
from __future__ import annotations

import ctypes
import os
import subprocess
from ctypes import POINTER, c_float, c_int, c_int32, c_int64, c_uint32, c_uint64, c_void_p

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "bvh_oracle.cpp")
_LIB = os.path.join(_HERE, "libbvh_oracle.so")

# No -ffast-math, no -march: fp32 arithmetic must be one IEEE operation per statement.
CXXFLAGS = ["-O2", "-std=c++17", "-ffp-contract=off", "-fPIC", "-shared"]


def build(force: bool = False) -> str:
    """Compile the oracle shared library next to its source (g++)."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        tmp = _LIB + f".tmp{os.getpid()}"
        subprocess.check_call(["g++", *CXXFLAGS, _SRC, "-o", tmp])
        os.replace(tmp, _LIB)
    return _LIB


_lib = None


def _L():
    global _lib
    if _lib is None:
        lib = ctypes.CDLL(build())
        fp, i64, i32p, u32p, u64p = POINTER(c_float), c_int64, POINTER(c_int32), POINTER(c_uint32), POINTER(c_uint64)
        lib.oracle_scene_bounds.argtypes = [fp, i64, c_int, fp]
        lib.oracle_morton.argtypes = [fp, i64, c_int, fp, c_int, u64p]
        lib.oracle_sort.argtypes = [u64p, i64, u64p, u32p]
        lib.oracle_hierarchy.argtypes = [u64p, i64, i32p, i32p, i32p, i32p]
        lib.oracle_ropes.argtypes = [i32p, i32p, i64, i32p]
        lib.oracle_ropes_alg2.argtypes = [u64p, i32p, i32p, i64, i32p]
        lib.oracle_boxes.argtypes = [fp, c_int, u32p, i32p, i32p, i64, fp]
        lib.oracle_build.argtypes = [fp, i64, c_int, c_int, u64p, u32p, i32p, i32p, fp, fp, i32p]
        for name in ("oracle_query_spheres_tree", "oracle_query_boxes_tree", "oracle_query_rays_tree"):
            f = getattr(lib, name)
            f.argtypes = [fp, i32p, i32p, i64, fp, i64]
            f.restype = c_void_p
        for name in ("oracle_query_spheres_brute", "oracle_query_boxes_brute", "oracle_query_rays_brute"):
            f = getattr(lib, name)
            f.argtypes = [fp, i64, c_int, fp, i64]
            f.restype = c_void_p
        lib.oracle_result_nnz.argtypes = [c_void_p]
        lib.oracle_result_nnz.restype = c_int64
        lib.oracle_result_copy.argtypes = [c_void_p, POINTER(c_int64), i32p]
        lib.oracle_result_free.argtypes = [c_void_p]
        lib.oracle_walk_all.argtypes = [i32p, i32p, i64, i32p, i64]
        lib.oracle_walk_all.restype = c_int64
        for name in ("oracle_nearest_spheres_brute", "oracle_first_hit_rays_brute"):
            f = getattr(lib, name)
            f.argtypes = [fp, i64, c_int, fp, i64, i32p, fp]
            f.restype = None
        for name in ("oracle_nearest_spheres_tree", "oracle_first_hit_rays_tree"):
            f = getattr(lib, name)
            f.argtypes = [fp, i32p, i32p, i64, fp, i64, i32p, fp]
            f.restype = None
        lib.oracle_apetrei.argtypes = [u64p, i64, i32p, i32p, i32p]
        lib.oracle_apetrei.restype = None
        lib.oracle_ropes_from.argtypes = [i32p, i32p, i64, c_int32, i32p]
        lib.oracle_ropes_from.restype = None
        lib.oracle_boxes_from.argtypes = [fp, c_int, u32p, i32p, i32p, i64, c_int32, fp]
        lib.oracle_boxes_from.restype = None
        for name in ("oracle_scene_bounds", "oracle_morton", "oracle_sort", "oracle_hierarchy", "oracle_ropes",
                     "oracle_ropes_alg2", "oracle_boxes", "oracle_build", "oracle_result_copy", "oracle_result_free"):
            getattr(lib, name).restype = None
        _lib = lib
    return _lib


def _p(a: np.ndarray, ct):
    return a.ctypes.data_as(POINTER(ct))


def _prims(prim: np.ndarray):
    """Returns (contiguous float32 array, n, is_box) for an [n,3] point or [n,6] box array."""
    a = np.ascontiguousarray(prim, dtype=np.float32)
    assert a.ndim == 2 and a.shape[1] in (3, 6), a.shape
    return a, a.shape[0], int(a.shape[1] == 6)


# ---- D1 .. D7 --------------------------------------------------------------------------------------

def scene_bounds(prim) -> np.ndarray:
    a, n, is_box = _prims(prim)
    out = np.empty(6, np.float32)
    _L().oracle_scene_bounds(_p(a, c_float), n, is_box, _p(out, c_float))
    return out


def morton(prim, scene6, bits: int) -> np.ndarray:
    a, n, is_box = _prims(prim)
    s = np.ascontiguousarray(scene6, dtype=np.float32)
    codes = np.empty(n, np.uint64)
    _L().oracle_morton(_p(a, c_float), n, is_box, _p(s, c_float), int(bits), _p(codes, c_uint64))
    return codes


def sort_codes(codes):
    c = np.ascontiguousarray(codes, dtype=np.uint64)
    n = c.shape[0]
    sorted_ = np.empty(n, np.uint64)
    perm = np.empty(n, np.uint32)
    _L().oracle_sort(_p(c, c_uint64), n, _p(sorted_, c_uint64), _p(perm, c_uint32))
    return sorted_, perm


def hierarchy(sorted_codes):
    """Karras top-down tree over sorted codes. Returns left, right, first, last (each n-1, unified indices)."""
    c = np.ascontiguousarray(sorted_codes, dtype=np.uint64)
    n = c.shape[0]
    m = max(n - 1, 0)
    left, right, first, last = (np.empty(m, np.int32) for _ in range(4))
    if n >= 2:
        _L().oracle_hierarchy(_p(c, c_uint64), n, _p(left, c_int32), _p(right, c_int32), _p(first, c_int32),
                              _p(last, c_int32))
    return left, right, first, last


def ropes(left, right, n: int) -> np.ndarray:
    left = np.ascontiguousarray(left, np.int32)
    right = np.ascontiguousarray(right, np.int32)
    rope = np.empty(2 * n - 1, np.int32)
    _L().oracle_ropes(_p(left, c_int32), _p(right, c_int32), n, _p(rope, c_int32))
    return rope


def ropes_alg2(sorted_codes, first, last) -> np.ndarray:
    c = np.ascontiguousarray(sorted_codes, dtype=np.uint64)
    n = c.shape[0]
    first = np.ascontiguousarray(first, np.int32)
    last = np.ascontiguousarray(last, np.int32)
    rope = np.empty(2 * n - 1, np.int32)
    _L().oracle_ropes_alg2(_p(c, c_uint64), _p(first, c_int32), _p(last, c_int32), n, _p(rope, c_int32))
    return rope


def boxes(prim, perm, left, right) -> np.ndarray:
    a, n, is_box = _prims(prim)
    perm = np.ascontiguousarray(perm, np.uint32)
    left = np.ascontiguousarray(left, np.int32)
    right = np.ascontiguousarray(right, np.int32)
    aabb = np.empty((2 * n - 1, 6), np.float32)
    _L().oracle_boxes(_p(a, c_float), is_box, _p(perm, c_uint32), _p(left, c_int32), _p(right, c_int32), n,
                      _p(aabb, c_float))
    return aabb


class Bvh:
    """Result of :func:`build` -- the canonical arrays the boundary's ``bvh_export`` also produces."""

    __slots__ = ("n", "bits", "sorted_codes", "perm", "left_child", "rope", "aabb", "scene_bounds", "right_child")


def build_bvh(prim, bits: int) -> Bvh:
    a, n, is_box = _prims(prim)
    out = Bvh()
    out.n, out.bits = n, int(bits)
    m = max(2 * n - 1, 0)
    out.sorted_codes = np.empty(n, np.uint64)
    out.perm = np.empty(n, np.uint32)
    out.left_child = np.empty(m, np.int32)
    out.rope = np.empty(m, np.int32)
    out.aabb = np.empty((m, 6), np.float32)
    out.scene_bounds = np.zeros(6, np.float32)
    out.right_child = np.empty(max(n - 1, 0), np.int32)
    if n > 0:
        _L().oracle_build(_p(a, c_float), n, is_box, int(bits), _p(out.sorted_codes, c_uint64),
                          _p(out.perm, c_uint32), _p(out.left_child, c_int32), _p(out.rope, c_int32),
                          _p(out.aabb, c_float), _p(out.scene_bounds, c_float), _p(out.right_child, c_int32))
    return out


# ---- D8 --------------------------------------------------------------------------------------------

def _take(handle):
    lib = _L()
    nnz = lib.oracle_result_nnz(handle)
    return handle, nnz


def _finish(handle, q):
    lib = _L()
    nnz = lib.oracle_result_nnz(handle)
    offsets = np.empty(q + 1, np.int64)
    indices = np.empty(nnz, np.int32)
    lib.oracle_result_copy(handle, _p(offsets, c_int64), _p(indices, c_int32))
    lib.oracle_result_free(handle)
    return offsets, indices


def query_spheres_tree(bvh: Bvh, xyzr):
    """Stack traversal of the oracle tree. CSR (offsets int64[q+1], indices int32[nnz]) of original indices."""
    qa = np.ascontiguousarray(xyzr, np.float32)
    assert qa.ndim == 2 and qa.shape[1] == 4
    h = _L().oracle_query_spheres_tree(_p(bvh.aabb, c_float), _p(bvh.left_child, c_int32),
                                       _p(bvh.right_child, c_int32), bvh.n, _p(qa, c_float), qa.shape[0])
    return _finish(h, qa.shape[0])


def query_boxes_tree(bvh: Bvh, minmax):
    qa = np.ascontiguousarray(minmax, np.float32)
    assert qa.ndim == 2 and qa.shape[1] == 6
    h = _L().oracle_query_boxes_tree(_p(bvh.aabb, c_float), _p(bvh.left_child, c_int32),
                                     _p(bvh.right_child, c_int32), bvh.n, _p(qa, c_float), qa.shape[0])
    return _finish(h, qa.shape[0])


def query_spheres_brute(prim, xyzr):
    a, n, is_box = _prims(prim)
    qa = np.ascontiguousarray(xyzr, np.float32)
    h = _L().oracle_query_spheres_brute(_p(a, c_float), n, is_box, _p(qa, c_float), qa.shape[0])
    return _finish(h, qa.shape[0])


def query_boxes_brute(prim, minmax):
    a, n, is_box = _prims(prim)
    qa = np.ascontiguousarray(minmax, np.float32)
    h = _L().oracle_query_boxes_brute(_p(a, c_float), n, is_box, _p(qa, c_float), qa.shape[0])
    return _finish(h, qa.shape[0])


def query_rays_tree(bvh: Bvh, rays):
    """D9 (NEXT-1): rays [q,8] = {origin.xyz, direction.xyz, tmin, tmax}; stack traversal of the oracle tree."""
    qa = np.ascontiguousarray(rays, np.float32)
    assert qa.ndim == 2 and qa.shape[1] == 8
    h = _L().oracle_query_rays_tree(_p(bvh.aabb, c_float), _p(bvh.left_child, c_int32),
                                    _p(bvh.right_child, c_int32), bvh.n, _p(qa, c_float), qa.shape[0])
    return _finish(h, qa.shape[0])


def query_rays_brute(prim, rays):
    a, n, is_box = _prims(prim)
    qa = np.ascontiguousarray(rays, np.float32)
    assert qa.ndim == 2 and qa.shape[1] == 8
    h = _L().oracle_query_rays_brute(_p(a, c_float), n, is_box, _p(qa, c_float), qa.shape[0])
    return _finish(h, qa.shape[0])


def walk_all(left_child, rope, n: int) -> np.ndarray:
    """Algorithm 1 with an always-true predicate; returns the visit order (raises on a cycle)."""
    left_child = np.ascontiguousarray(left_child, np.int32)
    rope = np.ascontiguousarray(rope, np.int32)
    cap = 2 * n + 8
    order = np.empty(cap, np.int32)
    k = _L().oracle_walk_all(_p(left_child, c_int32), _p(rope, c_int32), n, _p(order, c_int32), cap)
    if k < 0:
        raise RuntimeError("stackless walk did not terminate within 2n+8 visits")
    return order[:k].copy()


# ---- D10 / D11: an operation at the leaf instead of a stored row ----------------------------------

def _reduce(fn_brute, fn_tree, queries, width, prim=None, bvh=None):
    qa = np.ascontiguousarray(queries, np.float32)
    assert qa.ndim == 2 and qa.shape[1] == width
    idx = np.empty(qa.shape[0], np.int32)
    key = np.empty(qa.shape[0], np.float32)
    if bvh is not None:
        fn_tree(_p(bvh.aabb, c_float), _p(bvh.left_child, c_int32), _p(bvh.right_child, c_int32), bvh.n, _p(qa, c_float),
                qa.shape[0], _p(idx, c_int32), _p(key, c_float))
    else:
        a, n, is_box = _prims(prim)
        fn_brute(_p(a, c_float), n, is_box, _p(qa, c_float), qa.shape[0], _p(idx, c_int32), _p(key, c_float))
    return idx, key


def nearest_spheres_brute(prim, xyzr):
    """D10: per sphere {x,y,z,r}, the primitive with the smallest D8 distance d2 <= r*r (ties: smallest index);
    returns (index or -1, d2 or +inf).  Tests every primitive."""
    return _reduce(_L().oracle_nearest_spheres_brute, None, xyzr, 4, prim=prim)


def nearest_spheres_tree(bvh: Bvh, xyzr):
    return _reduce(None, _L().oracle_nearest_spheres_tree, xyzr, 4, bvh=bvh)


def first_hit_rays_brute(prim, rays):
    """D11: per ray, the primitive whose box the ray enters first (smallest t_enter; ties: smallest index);
    returns (index or -1, t_enter or +inf).  Tests every primitive."""
    return _reduce(_L().oracle_first_hit_rays_brute, None, rays, 8, prim=prim)


def first_hit_rays_tree(bvh: Bvh, rays):
    return _reduce(None, _L().oracle_first_hit_rays_tree, rays, 8, bvh=bvh)


# ---- Algorithm 3: Apetrei's numbering (NEXT-2 a) ------------------------------------------------------------------

class ApetreiTree:
    """The hierarchy as the unmodified Algorithm 3 numbers it: internal node index = split position, root stored."""

    __slots__ = ("n", "root", "left", "right", "rope", "aabb")


def apetrei_tree(prim, bvh: Bvh) -> ApetreiTree:
    """Runs Algorithm 3 serially over bvh.sorted_codes, then skip-connections by their
    definition (a walk from the stored root) and boxes by post-order union."""
    a, n, is_box = _prims(prim)
    t = ApetreiTree()
    t.n = n
    m = max(n - 1, 0)
    t.left, t.right = np.empty(m, np.int32), np.empty(m, np.int32)
    root = np.zeros(1, np.int32)
    if n >= 2:
        _L().oracle_apetrei(_p(bvh.sorted_codes, c_uint64), n, _p(t.left, c_int32), _p(t.right, c_int32), _p(root, c_int32))
    t.root = int(root[0])
    t.rope = np.empty(max(2 * n - 1, 0), np.int32)
    t.aabb = np.empty((max(2 * n - 1, 0), 6), np.float32)
    if n >= 1:
        _L().oracle_ropes_from(_p(t.left, c_int32), _p(t.right, c_int32), n, t.root, _p(t.rope, c_int32))
        _L().oracle_boxes_from(_p(a, c_float), is_box, _p(bvh.perm, c_uint32), _p(t.left, c_int32), _p(t.right, c_int32),
                               n, t.root, _p(t.aabb, c_float))
    return t
