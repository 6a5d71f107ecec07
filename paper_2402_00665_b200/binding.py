"""Thin Python binding over the C ABI of ``libbvh_b200.so`` (include/bvh_b200.h).

Argument marshalling only: every function has the name and the argument list of its C entry point,
takes torch CUDA tensors (device memory) and passes their ``data_ptr()`` plus the current torch CUDA
stream.  No step of the path runs here.  There is NO CPU fallback: if the library is missing or
cannot be loaded, every call raises.

On top of the 1:1 functions, :class:`Bvh` and the ``query_*`` helpers chain the calls the way a user
would (sizes -> allocate with torch -> build; count -> scan -> read nnz -> allocate -> fill).
"""
from __future__ import annotations

import ctypes
import os
from ctypes import c_int, c_int64, c_size_t, c_void_p

import torch

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libbvh_b200.so")

BVH_OK = 0
ERRORS = {
    -1: "BVH_ERR_INVALID_ARGUMENT",
    -2: "BVH_ERR_MORTON_BITS",
    -3: "BVH_ERR_TOO_LARGE",
    -4: "BVH_ERR_SCRATCH",
    -5: "BVH_ERR_CUDA",
    -6: "BVH_ERR_STATIC_LIMIT",
}

# every symbol include/bvh_b200.h declares: (name, argtypes)
_P = c_void_p
SYMBOLS = {
    "bvh_version": [],
    "bvh_sizes": [c_int64, c_int, ctypes.POINTER(c_size_t), ctypes.POINTER(c_size_t)],
    "bvh_build_points": [_P, c_int64, c_int, _P, _P, c_size_t, _P],
    "bvh_build_boxes": [_P, c_int64, c_int, _P, _P, c_size_t, _P],
    "bvh_build_staged": [_P, c_int, c_int64, c_int, _P, _P, c_size_t, _P, ctypes.POINTER(c_void_p)],
    "bvh_query_order_sizes": [c_int64, ctypes.POINTER(c_size_t)],
    "bvh_query_order_spheres": [_P, c_int64, _P, c_int64, _P, _P, c_size_t, _P],
    "bvh_query_order_boxes": [_P, c_int64, _P, c_int64, _P, _P, c_size_t, _P],
    "bvh_query_spheres_count": [_P, c_int64, _P, c_int64, _P, _P, _P],
    "bvh_query_boxes_count": [_P, c_int64, _P, c_int64, _P, _P, _P],
    "bvh_scan_sizes": [c_int64, ctypes.POINTER(c_size_t)],
    "bvh_scan_counts": [_P, c_int64, _P, _P, c_size_t, _P],
    "bvh_scan_counts_static": [_P, c_int64, _P, _P],
    "bvh_query_spheres_fill": [_P, c_int64, _P, c_int64, _P, _P, _P, _P],
    "bvh_query_boxes_fill": [_P, c_int64, _P, c_int64, _P, _P, _P, _P],
    "bvh_query_spheres_nearest": [_P, c_int64, _P, c_int64, _P, _P, _P, _P],
    "bvh_query_rays_first_hit": [_P, c_int64, _P, c_int64, _P, _P, _P, _P],
    "bvh_query_any_hit": [_P, c_int64, _P, c_int, c_int64, _P, _P, _P],
    "bvh_query_collect": [_P, c_int64, _P, c_int, c_int64, _P, c_int64, _P, _P, _P],
    "bvh_rows_to_csr": [_P, c_int64, _P, _P, c_int64, _P, _P],
    "bvh_query_fill_overflow": [_P, c_int64, _P, c_int, c_int64, _P, c_int64, _P, _P, _P, _P],
    "bvh_query_csr_sizes": [c_int64, ctypes.POINTER(c_size_t)],
    "bvh_query_csr": [_P, c_int64, _P, c_int, c_int64, c_int64, _P, _P, _P, _P, _P, c_int64, _P, c_size_t, _P],
    "bvh_query_order_rays": [_P, c_int64, _P, c_int64, _P, _P, c_size_t, _P],
    "bvh_query_rays_count": [_P, c_int64, _P, c_int64, _P, _P, _P],
    "bvh_query_rays_fill": [_P, c_int64, _P, c_int64, _P, _P, _P, _P],
    "bvh_variant_sizes": [c_int64, c_int, c_int, ctypes.POINTER(c_size_t)],
    "bvh_build_variant": [_P, c_int, c_int64, c_int, _P, _P, c_size_t, c_int, _P, ctypes.POINTER(c_void_p)],
    "bvh_variant_export": [_P, _P, c_int64, c_int, c_int, _P, _P, _P, _P, _P, _P],
    "bvh_export": [_P, _P, c_int64, c_int, _P, _P, _P, _P, _P, _P, _P],
}


class BvhError(RuntimeError):
    pass


_lib = None


def load_library() -> ctypes.CDLL:
    """Load the C-ABI library (fails loudly if it has not been built: ``python -m paper_2402_00665_b200.build``)."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise BvhError(f"{LIB_PATH} is missing: build it with `python -m paper_2402_00665_b200.build` "
                           "(there is no CPU fallback)")
        lib = ctypes.CDLL(LIB_PATH)
        for name, argtypes in SYMBOLS.items():
            fn = getattr(lib, name)
            fn.argtypes = argtypes
            fn.restype = c_int
        _lib = lib
    return _lib


def _check(code: int, what: str) -> None:
    if code != BVH_OK:
        raise BvhError(f"{what} failed: {ERRORS.get(code, code)}")


def _ptr(t: torch.Tensor | None) -> int | None:
    if t is None:
        return None
    if not t.is_cuda:
        raise BvhError("the C ABI takes device memory: pass CUDA tensors (there is no CPU path)")
    if not t.is_contiguous():
        raise BvhError("tensors must be contiguous")
    return t.data_ptr()


def _stream() -> int:
    return torch.cuda.current_stream().cuda_stream


# ---- 1:1 with the C ABI -------------------------------------------------------------------------------

def bvh_version() -> int:
    return load_library().bvh_version()


def bvh_sizes(n: int, morton_bits: int) -> tuple[int, int]:
    nb, sb = c_size_t(), c_size_t()
    _check(load_library().bvh_sizes(n, morton_bits, ctypes.byref(nb), ctypes.byref(sb)), "bvh_sizes")
    return nb.value, sb.value


def bvh_build_points(xyz: torch.Tensor, n: int, morton_bits: int, nodes: torch.Tensor, scratch: torch.Tensor) -> None:
    _check(load_library().bvh_build_points(_ptr(xyz), n, morton_bits, _ptr(nodes), _ptr(scratch),
                                           scratch.numel() * scratch.element_size(), _stream()), "bvh_build_points")


def bvh_build_boxes(minmax: torch.Tensor, n: int, morton_bits: int, nodes: torch.Tensor, scratch: torch.Tensor) -> None:
    _check(load_library().bvh_build_boxes(_ptr(minmax), n, morton_bits, _ptr(nodes), _ptr(scratch),
                                          scratch.numel() * scratch.element_size(), _stream()), "bvh_build_boxes")


NUM_STAGE_EVENTS = 13
STAGE_NAMES = ["start", "init", "bounds", "morton"] + [f"sort_pass{p}" for p in range(8)] + ["hierarchy"]


def bvh_build_staged(prim: torch.Tensor, prim_is_box: int, n: int, morton_bits: int, nodes: torch.Tensor,
                     scratch: torch.Tensor, stage_events) -> None:
    """stage_events: sequence of NUM_STAGE_EVENTS entries, each a ``torch.cuda.Event(enable_timing=True)`` that has
    been recorded at least once (so that its cudaEvent_t exists) or None."""
    assert len(stage_events) == NUM_STAGE_EVENTS
    arr = (c_void_p * NUM_STAGE_EVENTS)(*[None if e is None else e.cuda_event for e in stage_events])
    _check(load_library().bvh_build_staged(_ptr(prim), int(prim_is_box), n, morton_bits, _ptr(nodes), _ptr(scratch),
                                           scratch.numel() * scratch.element_size(), _stream(), arr), "bvh_build_staged")


def bvh_query_order_sizes(q: int) -> int:
    sb = c_size_t()
    _check(load_library().bvh_query_order_sizes(q, ctypes.byref(sb)), "bvh_query_order_sizes")
    return sb.value


def bvh_query_order_spheres(nodes, n: int, xyzr, q: int, order, scratch) -> None:
    _check(load_library().bvh_query_order_spheres(_ptr(nodes), n, _ptr(xyzr), q, _ptr(order), _ptr(scratch),
                                                  scratch.numel() * scratch.element_size(), _stream()),
           "bvh_query_order_spheres")


def bvh_query_order_boxes(nodes, n: int, minmax, q: int, order, scratch) -> None:
    _check(load_library().bvh_query_order_boxes(_ptr(nodes), n, _ptr(minmax), q, _ptr(order), _ptr(scratch),
                                                scratch.numel() * scratch.element_size(), _stream()),
           "bvh_query_order_boxes")


def bvh_query_spheres_count(nodes, n: int, xyzr, q: int, order, counts) -> None:
    _check(load_library().bvh_query_spheres_count(_ptr(nodes), n, _ptr(xyzr), q, _ptr(order), _ptr(counts), _stream()),
           "bvh_query_spheres_count")


def bvh_query_boxes_count(nodes, n: int, minmax, q: int, order, counts) -> None:
    _check(load_library().bvh_query_boxes_count(_ptr(nodes), n, _ptr(minmax), q, _ptr(order), _ptr(counts), _stream()),
           "bvh_query_boxes_count")


def bvh_query_spheres_nearest(nodes, n: int, xyzr, q: int, order, index, d2) -> None:
    _check(load_library().bvh_query_spheres_nearest(_ptr(nodes), n, _ptr(xyzr), q, _ptr(order), _ptr(index), _ptr(d2),
                                                    _stream()), "bvh_query_spheres_nearest")


def bvh_query_rays_first_hit(nodes, n: int, rays, q: int, order, index, t) -> None:
    _check(load_library().bvh_query_rays_first_hit(_ptr(nodes), n, _ptr(rays), q, _ptr(order), _ptr(index), _ptr(t),
                                                   _stream()), "bvh_query_rays_first_hit")


def bvh_query_any_hit(nodes, n: int, queries, query_kind: int, q: int, order, hit) -> None:
    _check(load_library().bvh_query_any_hit(_ptr(nodes), n, _ptr(queries), query_kind, q, _ptr(order), _ptr(hit),
                                            _stream()), "bvh_query_any_hit")


def bvh_query_collect(nodes, n: int, queries, query_kind: int, q: int, order, cap: int, rows, counts) -> None:
    _check(load_library().bvh_query_collect(_ptr(nodes), n, _ptr(queries), query_kind, q, _ptr(order), cap, _ptr(rows),
                                            _ptr(counts), _stream()), "bvh_query_collect")


def bvh_rows_to_csr(rows, cap: int, counts, offsets, q: int, indices) -> None:
    _check(load_library().bvh_rows_to_csr(_ptr(rows), cap, _ptr(counts), _ptr(offsets), q, _ptr(indices), _stream()),
           "bvh_rows_to_csr")


def bvh_query_fill_overflow(nodes, n: int, queries, query_kind: int, q: int, order, cap: int, counts, offsets,
                            indices) -> None:
    _check(load_library().bvh_query_fill_overflow(_ptr(nodes), n, _ptr(queries), query_kind, q, _ptr(order), cap,
                                                  _ptr(counts), _ptr(offsets), _ptr(indices), _stream()),
           "bvh_query_fill_overflow")


def bvh_query_csr_sizes(q: int) -> int:
    b = c_size_t(0)
    _check(load_library().bvh_query_csr_sizes(q, ctypes.byref(b)), "bvh_query_csr_sizes")
    return int(b.value)


def bvh_query_csr(nodes, n: int, queries, query_kind: int, q: int, cap: int, rows, order, counts, offsets, indices,
                  indices_capacity: int, scratch) -> None:
    _check(load_library().bvh_query_csr(_ptr(nodes), n, _ptr(queries), query_kind, q, cap, _ptr(rows), _ptr(order),
                                        _ptr(counts), _ptr(offsets), _ptr(indices), indices_capacity, _ptr(scratch),
                                        0 if scratch is None else scratch.numel() * scratch.element_size(), _stream()),
           "bvh_query_csr")


def bvh_query_order_rays(nodes, n: int, rays, q: int, order, scratch) -> None:
    _check(load_library().bvh_query_order_rays(_ptr(nodes), n, _ptr(rays), q, _ptr(order), _ptr(scratch),
                                               scratch.numel() * scratch.element_size(), _stream()),
           "bvh_query_order_rays")


def bvh_query_rays_count(nodes, n: int, rays, q: int, order, counts) -> None:
    _check(load_library().bvh_query_rays_count(_ptr(nodes), n, _ptr(rays), q, _ptr(order), _ptr(counts), _stream()),
           "bvh_query_rays_count")


def bvh_query_rays_fill(nodes, n: int, rays, q: int, order, offsets, indices) -> None:
    _check(load_library().bvh_query_rays_fill(_ptr(nodes), n, _ptr(rays), q, _ptr(order), _ptr(offsets),
                                              _ptr(indices), _stream()), "bvh_query_rays_fill")


def bvh_variant_sizes(n: int, morton_bits: int, variant: int) -> int:
    sb = c_size_t()
    _check(load_library().bvh_variant_sizes(n, morton_bits, variant, ctypes.byref(sb)), "bvh_variant_sizes")
    return sb.value


def bvh_build_variant(prim, prim_is_box: int, n: int, morton_bits: int, nodes, scratch, variant: int) -> None:
    """NEXT-2 measurement variants: 1 = Karras top-down + Algorithm 2 + separate box pass (same `nodes` bytes as the
    product); 2 = unmodified Algorithm 3 (Apetrei numbering) + separate skip-connection pass (read with
    bvh_variant_export); 3 = Algorithm 4 as the paper writes it, one thread per leaf with a global `store` (same `nodes`
    bytes as the product)."""
    _check(load_library().bvh_build_variant(_ptr(prim), prim_is_box, n, morton_bits, _ptr(nodes), _ptr(scratch),
                                            scratch.numel() * scratch.element_size(), variant, _stream(), None),
           "bvh_build_variant")


def bvh_variant_export(nodes, scratch, n: int, morton_bits: int, variant: int, left=None, right=None, rope=None, aabb=None,
                       root=None) -> None:
    _check(load_library().bvh_variant_export(_ptr(nodes), _ptr(scratch), n, morton_bits, variant, _ptr(left), _ptr(right),
                                             _ptr(rope), _ptr(aabb), _ptr(root), _stream()), "bvh_variant_export")


def bvh_scan_sizes(q: int) -> int:
    sb = c_size_t()
    _check(load_library().bvh_scan_sizes(q, ctypes.byref(sb)), "bvh_scan_sizes")
    return sb.value


def bvh_scan_counts(counts, q: int, offsets, scratch) -> None:
    _check(load_library().bvh_scan_counts(_ptr(counts), q, _ptr(offsets), _ptr(scratch),
                                          scratch.numel() * scratch.element_size(), _stream()), "bvh_scan_counts")


SCAN_STATIC_MAX_Q = 8192 * 4096   # BVH_SCAN_STATIC_MAX_Q


def bvh_scan_counts_static(counts, q: int, offsets) -> None:
    """``bvh_scan_counts`` without a scratch argument, for code that may not allocate device memory when it runs
    (memory already committed to a pool, allocator calls forbidden by the host framework, no tolerance for the
    allocator's device-wide synchronisation).  The tile sums go to a 64 KB array inside the library, one per GPU and
    shared by all calls on it: at most ``SCAN_STATIC_MAX_Q`` counts (more raises ``BVH_ERR_STATIC_LIMIT``), and calls
    that may overlap on the GPU must be serialised by the caller.  Same offsets, bit for bit, as ``bvh_scan_counts``.
    Make the first call on each device at start-up (it resolves the array's address there)."""
    _check(load_library().bvh_scan_counts_static(_ptr(counts), q, _ptr(offsets), _stream()), "bvh_scan_counts_static")


def bvh_query_spheres_fill(nodes, n: int, xyzr, q: int, order, offsets, indices) -> None:
    _check(load_library().bvh_query_spheres_fill(_ptr(nodes), n, _ptr(xyzr), q, _ptr(order), _ptr(offsets),
                                                 _ptr(indices), _stream()), "bvh_query_spheres_fill")


def bvh_query_boxes_fill(nodes, n: int, minmax, q: int, order, offsets, indices) -> None:
    _check(load_library().bvh_query_boxes_fill(_ptr(nodes), n, _ptr(minmax), q, _ptr(order), _ptr(offsets),
                                               _ptr(indices), _stream()), "bvh_query_boxes_fill")


def bvh_export(nodes, scratch, n: int, morton_bits: int, sorted_codes=None, perm=None, left_child=None, rope=None,
               aabb=None, scene_bounds=None) -> None:
    _check(load_library().bvh_export(_ptr(nodes), _ptr(scratch), n, morton_bits, _ptr(sorted_codes), _ptr(perm),
                                     _ptr(left_child), _ptr(rope), _ptr(aabb), _ptr(scene_bounds), _stream()),
           "bvh_export")


# ---- the calls chained as a user would ------------------------------------------------------------------

class Bvh:
    """Device buffers of one hierarchy: ``nodes`` (the product) and ``scratch`` (kept for :meth:`export`)."""

    def __init__(self, n: int, morton_bits: int, device="cuda"):
        self.n = int(n)
        self.morton_bits = int(morton_bits)
        node_bytes, scratch_bytes = bvh_sizes(self.n, self.morton_bits)
        self.nodes = torch.empty(node_bytes, dtype=torch.uint8, device=device)
        self.scratch = torch.empty(scratch_bytes, dtype=torch.uint8, device=device)
        self.prim_kind = None

    def build(self, prims: torch.Tensor) -> "Bvh":
        """prims: float32 CUDA tensor [n,3] (points) or [n,6] (boxes).  Asynchronous on the current stream."""
        if prims.dtype != torch.float32 or prims.dim() != 2 or prims.shape[0] != self.n or prims.shape[1] not in (3, 6):
            raise BvhError(f"expected float32 [{self.n},3] or [{self.n},6], got {prims.dtype} {tuple(prims.shape)}")
        if prims.shape[1] == 3:
            bvh_build_points(prims, self.n, self.morton_bits, self.nodes, self.scratch)
        else:
            bvh_build_boxes(prims, self.n, self.morton_bits, self.nodes, self.scratch)
        self.prim_kind = "points" if prims.shape[1] == 3 else "boxes"
        return self

    def export(self) -> dict[str, torch.Tensor]:
        n, dev = self.n, self.nodes.device
        m = max(2 * n - 1, 0)
        out = {
            "sorted_codes": torch.zeros(n, dtype=torch.int32 if self.morton_bits == 30 else torch.int64, device=dev),
            "perm": torch.zeros(n, dtype=torch.int32, device=dev),
            "left_child": torch.zeros(m, dtype=torch.int32, device=dev),
            "rope": torch.zeros(m, dtype=torch.int32, device=dev),
            "aabb": torch.zeros((m, 6), dtype=torch.float32, device=dev),
            "scene_bounds": torch.zeros(6, dtype=torch.float32, device=dev),
        }
        bvh_export(self.nodes, self.scratch, n, self.morton_bits, **out)
        return out


class QueryWorkspace:
    """Reusable device buffers for ordered count-then-fill over up to ``q`` queries."""

    def __init__(self, q: int, device="cuda"):
        self.q = int(q)
        self.counts = torch.empty(max(self.q, 1), dtype=torch.int32, device=device)
        self.offsets = torch.empty(self.q + 1, dtype=torch.int64, device=device)
        self.scan_scratch = torch.empty(max(bvh_scan_sizes(self.q), 8), dtype=torch.uint8, device=device)
        self.order = torch.empty(max(self.q, 1), dtype=torch.int32, device=device)
        self.order_scratch = torch.empty(bvh_query_order_sizes(self.q), dtype=torch.uint8, device=device)


QUERY_KINDS = {4: 0, 6: 1, 8: 2}   # floats per query -> query_kind of the C ABI


def query(bvh: Bvh, queries: torch.Tensor, ws: QueryWorkspace | None = None, indices: torch.Tensor | None = None,
          ordered: bool = True, row_capacity: int | None = None, rows: torch.Tensor | None = None):
    """Range search.  queries: float32 CUDA [q,4] spheres {x,y,z,r}, [q,6] boxes {min,max} or [q,8] rays
    {origin, direction, tmin, tmax}.

    order (Morton schedule of the queries) -> count -> scan -> fill.  Returns (offsets int64[q+1], indices
    int32[nnz]) on the device.  Reads nnz back once (the path's only device->host sync) unless ``indices`` is
    passed in with enough room.

    ``row_capacity`` (a multiple of 8) selects the single-pass variant instead: order -> collect (one traversal
    into rows of that many entries + exact counts) -> scan -> rows_to_csr -> fill_overflow (only the rows that
    did not fit are traversed again).  Same result, byte for byte.  ``rows``: optional int32 buffer of
    q * row_capacity entries to reuse."""
    if queries.dtype != torch.float32 or queries.dim() != 2 or queries.shape[1] not in (4, 6, 8):
        raise BvhError(f"expected float32 [q,4], [q,6] or [q,8], got {queries.dtype} {tuple(queries.shape)}")
    q = int(queries.shape[0])
    if bvh.prim_kind is None:
        raise BvhError("query() on a Bvh that has not been built")
    ws = ws or QueryWorkspace(q, queries.device)
    if ws.q < q:
        raise BvhError(f"QueryWorkspace holds {ws.q} queries, {q} given")
    order_fn, count, fill = {
        4: (bvh_query_order_spheres, bvh_query_spheres_count, bvh_query_spheres_fill),
        6: (bvh_query_order_boxes, bvh_query_boxes_count, bvh_query_boxes_fill),
        8: (bvh_query_order_rays, bvh_query_rays_count, bvh_query_rays_fill),
    }[int(queries.shape[1])]
    order = None
    if ordered and q > 0:
        order_fn(bvh.nodes, bvh.n, queries, q, ws.order, ws.order_scratch)
        order = ws.order
    kind = QUERY_KINDS[int(queries.shape[1])]
    if row_capacity is not None:
        cap = int(row_capacity)
        if rows is None:
            rows = torch.empty(max(q, 1) * cap, dtype=torch.int32, device=queries.device)
        elif rows.numel() < q * cap:
            raise BvhError(f"rows holds {rows.numel()} entries, {q * cap} needed")
        bvh_query_collect(bvh.nodes, bvh.n, queries, kind, q, order, cap, rows, ws.counts)
    else:
        count(bvh.nodes, bvh.n, queries, q, order, ws.counts)
    bvh_scan_counts(ws.counts, q, ws.offsets, ws.scan_scratch)
    if indices is None:
        nnz = int(ws.offsets[q].item())
        indices = torch.empty(max(nnz, 1), dtype=torch.int32, device=queries.device)
    else:
        nnz = None   # the caller vouches for the size (reading offsets[q] back here would be the sync it avoids)
    if row_capacity is not None:
        bvh_rows_to_csr(rows, cap, ws.counts, ws.offsets, q, indices)
        bvh_query_fill_overflow(bvh.nodes, bvh.n, queries, kind, q, order, cap, ws.counts, ws.offsets, indices)
    else:
        fill(bvh.nodes, bvh.n, queries, q, order, ws.offsets, indices)
    offsets = ws.offsets[: q + 1]
    return offsets, (indices if nnz is None else indices[:nnz])


def query_csr(bvh: Bvh, queries: torch.Tensor, row_capacity: int, indices: torch.Tensor, ws: QueryWorkspace | None = None,
              rows: torch.Tensor | None = None):
    """The single-pass range search as ONE call of the C ABI (``bvh_query_csr``): nothing is read back, so the caller
    sizes ``indices`` beforehand (from the previous batch, say).  Returns (offsets int64[q+1], indices) on the device;
    ``offsets[q]`` is nnz: if it exceeds ``indices.numel()`` the rows that did not fit were skipped and the caller
    finishes with ``bvh_rows_to_csr`` + ``bvh_query_fill_overflow`` into a larger buffer."""
    if queries.dtype != torch.float32 or queries.dim() != 2 or queries.shape[1] not in (4, 6, 8):
        raise BvhError(f"expected float32 [q,4], [q,6] or [q,8], got {queries.dtype} {tuple(queries.shape)}")
    if bvh.prim_kind is None:
        raise BvhError("query_csr() on a Bvh that has not been built")
    q = int(queries.shape[0])
    cap = int(row_capacity)
    ws = ws or QueryWorkspace(q, queries.device)
    if ws.q < q:
        raise BvhError(f"QueryWorkspace holds {ws.q} queries, {q} given")
    if rows is None:
        rows = torch.empty(max(q, 1) * cap, dtype=torch.int32, device=queries.device)
    elif rows.numel() < q * cap:
        raise BvhError(f"rows holds {rows.numel()} entries, {q * cap} needed")
    bvh_query_csr(bvh.nodes, bvh.n, queries, QUERY_KINDS[int(queries.shape[1])], q, cap, rows, ws.order, ws.counts,
                  ws.offsets, indices, indices.numel(), ws.order_scratch)
    return ws.offsets[: q + 1], indices


class HostCsr:
    """Pinned host buffers that receive a CSR result: ``offsets`` int64[q + 1], ``indices`` int32[capacity]; ``nnz`` is
    set by :func:`query_to_host`."""

    def __init__(self, q: int, capacity: int):
        self.q = int(q)
        self.offsets = torch.empty(self.q + 1, dtype=torch.int64).pin_memory()
        self.indices = torch.empty(max(int(capacity), 1), dtype=torch.int32).pin_memory()
        self.nnz = 0


def query_to_host(bvh: Bvh, h_queries: torch.Tensor, out: HostCsr, row_capacity: int, chunks: int = 8, ordered: bool = True):
    """End-to-end range search from pinned host queries to a CSR in pinned host memory.

    The result (4 bytes per hit) is usually far larger than the queries, and its device->host copy far longer than the
    search; so the batch is searched in ``chunks`` contiguous blocks (single-pass path: order, collect, scan,
    rows_to_csr, fill_overflow on the current stream) and each block's rows are copied to the host on a second stream
    while the next block is searched.  Returns ``out`` with offsets[0..q] and indices[0..nnz) filled, synchronised."""
    if not (h_queries.is_pinned() and not h_queries.is_cuda):
        raise BvhError("query_to_host takes the queries in pinned host memory")
    q = int(h_queries.shape[0])
    if out.q != q:
        raise BvhError(f"HostCsr was made for {out.q} queries, {q} given")
    dev = bvh.nodes.device
    chunks = max(1, min(int(chunks), max(q, 1)))
    bounds = [(c * q // chunks, (c + 1) * q // chunks) for c in range(chunks)]
    qmax = max(hi - lo for lo, hi in bounds) if q > 0 else 0
    ws = QueryWorkspace(qmax, dev)
    cap = int(row_capacity)
    rows = torch.empty(max(qmax, 1) * cap, dtype=torch.int32, device=dev)
    main = torch.cuda.current_stream()
    copy = torch.cuda.Stream(device=dev)
    keep, base = [], 0
    for lo, hi in bounds:
        if hi == lo:
            continue
        dq = h_queries[lo:hi].to(dev, non_blocking=True)
        off, idx = query(bvh, dq, ws, ordered=ordered, row_capacity=cap, rows=rows)     # reads this block's nnz back
        nnz = int(idx.numel())
        if base + nnz > out.indices.numel():
            raise BvhError(f"HostCsr holds {out.indices.numel()} indices, more are needed")
        off_g = off[:-1] + base                                                           # global positions of the block's rows
        done = torch.cuda.Event()
        done.record(main)
        with torch.cuda.stream(copy):
            copy.wait_event(done)
            out.offsets[lo:hi].copy_(off_g, non_blocking=True)
            if nnz:
                out.indices[base: base + nnz].copy_(idx[:nnz], non_blocking=True)
        keep.append((off_g, idx, dq))                                                     # alive until the copies are done
        base += nnz
    copy.synchronize()
    main.synchronize()
    out.offsets[q] = base
    out.nnz = base
    return out


def reduce_query(bvh: Bvh, queries: torch.Tensor, op: str, ws: QueryWorkspace | None = None, ordered: bool = True):
    """"Perform an operation" at the leaves instead of storing rows.  op = "nearest" (spheres: index and
    squared distance of the nearest primitive within the radius), "first_hit" (rays: index and entry parameter of the
    first box the ray enters) or "any_hit" (any query kind: 0 / 1).  Returns device tensors."""
    q = int(queries.shape[0])
    if bvh.prim_kind is None:
        raise BvhError("reduce_query() on a Bvh that has not been built")
    if queries.dtype != torch.float32 or queries.dim() != 2 or int(queries.shape[1]) not in QUERY_KINDS:
        raise BvhError(f"expected float32 [q,4], [q,6] or [q,8], got {queries.dtype} {tuple(queries.shape)}")
    kind = QUERY_KINDS[int(queries.shape[1])]
    ws = ws or QueryWorkspace(q, queries.device)
    order = None
    if ordered and q > 0:
        (bvh_query_order_spheres, bvh_query_order_boxes, bvh_query_order_rays)[kind](bvh.nodes, bvh.n, queries, q, ws.order,
                                                                                   ws.order_scratch)
        order = ws.order
    index = torch.empty(max(q, 1), dtype=torch.int32, device=queries.device)
    if op == "any_hit":
        bvh_query_any_hit(bvh.nodes, bvh.n, queries, kind, q, order, index)
        return index[:q]
    key = torch.empty(max(q, 1), dtype=torch.float32, device=queries.device)
    if op == "nearest" and kind == 0:
        bvh_query_spheres_nearest(bvh.nodes, bvh.n, queries, q, order, index, key)
    elif op == "first_hit" and kind == 2:
        bvh_query_rays_first_hit(bvh.nodes, bvh.n, queries, q, order, index, key)
    else:
        raise BvhError(f"operation {op!r} is not defined for {tuple(queries.shape)} queries")
    return index[:q], key[:q]
