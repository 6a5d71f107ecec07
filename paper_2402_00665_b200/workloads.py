"""Seeded synthetic inputs for the five BASELINE.json configs (recipe: DESIGN.md "Input recipe").

This module holds NO arithmetic of the method (no bounds, Morton codes, sorting, trees or predicates):
it only draws primitives and queries.  It is the one module both the CUDA tests/bench and the oracle
tests use, so that both sides see the same bytes.  numpy only; nothing here touches the GPU.

Generator: counter-based.  Every random number is SplitMix64's output function applied to
``seed * 2**40 + stream * 2**32 + counter`` (seed < 2**24, stream < 256, counter < 2**32), so any
element can be drawn independently and the arrays do not depend on chunking.
  uniform24 = top 24 bits * 2**-24   (exact in fp32, in [0, 1))
  uniform53 = top 53 bits * 2**-53   (fp64)
  gaussian  = Box-Muller in fp64 from two uniform53 draws
All coordinates are cast to fp32 and then have +0.0f added, which turns -0.0 into +0.0 (reading G19).
The paper uses no dataset, so these shapes stand in for nothing; they come from BASELINE.json.
"""
from __future__ import annotations

from dataclasses import dataclass

import numpy as np

_M64 = np.uint64(0xFFFFFFFFFFFFFFFF)


def _splitmix64(x: np.ndarray) -> np.ndarray:
    with np.errstate(over="ignore"):
        z = x + np.uint64(0x9E3779B97F4A7C15)
        z = (z ^ (z >> np.uint64(30))) * np.uint64(0xBF58476D1CE4E5B9)
        z = (z ^ (z >> np.uint64(27))) * np.uint64(0x94D049BB133111EB)
        return z ^ (z >> np.uint64(31))


def _raw(seed: int, stream: int, counter: np.ndarray) -> np.ndarray:
    assert 0 <= seed < (1 << 24) and 0 <= stream < 256
    base = np.uint64((seed << 40) + (stream << 32))
    return _splitmix64(base + counter.astype(np.uint64))


def uniform24(seed: int, stream: int, counter: np.ndarray) -> np.ndarray:
    """fp32 uniform in [0,1): top 24 bits of the hash times 2**-24."""
    return (_raw(seed, stream, counter) >> np.uint64(40)).astype(np.float32) * np.float32(2.0 ** -24)


def uniform53(seed: int, stream: int, counter: np.ndarray) -> np.ndarray:
    return (_raw(seed, stream, counter) >> np.uint64(11)).astype(np.float64) * (2.0 ** -53)


def gaussian(seed: int, stream: int, counter: np.ndarray) -> np.ndarray:
    """fp64 standard normal (Box-Muller); uses streams ``stream`` and ``stream + 1``."""
    u1 = ((_raw(seed, stream, counter) >> np.uint64(11)).astype(np.float64) + 1.0) * (2.0 ** -53)  # (0,1]
    u2 = uniform53(seed, stream + 1, counter)
    return np.sqrt(-2.0 * np.log(u1)) * np.cos(2.0 * np.pi * u2)


def _f32(a: np.ndarray) -> np.ndarray:
    out = np.ascontiguousarray(a, dtype=np.float32)
    out += np.float32(0.0)  # -0.0 -> +0.0
    return out


def _chunks(n: int, step: int = 1 << 22):
    for s in range(0, n, step):
        yield s, min(n, s + step)


# ---- point clouds ------------------------------------------------------------------------------------

def uniform_cube(n: int, seed: int) -> np.ndarray:
    """n points uniform in [0,1)^3 (streams 0,1,2)."""
    out = np.empty((n, 3), np.float32)
    for s, e in _chunks(n):
        c = np.arange(s, e, dtype=np.uint64)
        for a in range(3):
            out[s:e, a] = uniform24(seed, a, c)
    return _f32(out)


def gaussian_mixture(n: int, seed: int, centre_seed: int, components: int = 100, sigma: float = 0.005) -> np.ndarray:
    """n samples of a ``components``-component isotropic Gaussian mixture clamped to [0,1]^3.

    Centres: uniform_cube(components, centre_seed) streams 0-2.  Sample i: component = floor(u * components)
    with u = uniform53 stream 3; offset = sigma * gaussian (streams 4-5, 6-7, 8-9), fp64; cast to fp32."""
    centres = uniform_cube(components, centre_seed).astype(np.float64)
    out = np.empty((n, 3), np.float32)
    for s, e in _chunks(n):
        c = np.arange(s, e, dtype=np.uint64)
        comp = np.minimum((uniform53(seed, 3, c) * components).astype(np.int64), components - 1)
        for a in range(3):
            x = centres[comp, a] + sigma * gaussian(seed, 4 + 2 * a, c)
            out[s:e, a] = np.clip(x, 0.0, 1.0).astype(np.float32)
    return _f32(out)


def sphere_surface(n: int, seed: int) -> np.ndarray:
    """n points on the unit sphere: normalised fp64 Gaussian triple (streams 0-1, 2-3, 4-5)."""
    out = np.empty((n, 3), np.float32)
    for s, e in _chunks(n):
        c = np.arange(s, e, dtype=np.uint64)
        g = np.stack([gaussian(seed, 2 * a, c) for a in range(3)], axis=1)
        norm = np.sqrt((g * g).sum(axis=1, keepdims=True))
        norm[norm == 0.0] = 1.0
        out[s:e] = (g / norm).astype(np.float32)
    return _f32(out)


def hollow_shell(n: int, seed: int) -> np.ndarray:
    """n points uniform in [0,1)^3 minus the open cube (0.1,0.9)^3, by counter-based rejection:
    attempt k of element i draws uniform24 with streams 3k, 3k+1, 3k+2 and counter i."""
    out = np.empty((n, 3), np.float32)
    for s, e in _chunks(n):
        todo = np.arange(s, e, dtype=np.uint64)
        k = 0
        while todo.size:
            assert 3 * k + 2 < 256, "rejection sampler ran out of streams"
            p = np.stack([uniform24(seed, 3 * k + a, todo) for a in range(3)], axis=1)
            inside = np.all((p > np.float32(0.1)) & (p < np.float32(0.9)), axis=1)
            ok = ~inside
            out[todo[ok].astype(np.int64)] = p[ok]
            todo = todo[inside]
            k += 1
    return _f32(out)


def boxes_around(centres: np.ndarray, half_edge: float) -> np.ndarray:
    """[n,6] fp32 boxes {c - h, c + h}, the subtraction and addition done in fp32."""
    h = np.float32(half_edge)
    c = centres.astype(np.float32)
    return _f32(np.concatenate([c - h, c + h], axis=1))


def spheres_at(centres: np.ndarray, radius: float) -> np.ndarray:
    """[q,4] fp32 {x, y, z, r}."""
    q = centres.shape[0]
    out = np.empty((q, 4), np.float32)
    out[:, :3] = centres
    out[:, 3] = np.float32(radius)
    return _f32(out)


def rays_at(origins: np.ndarray, directions: np.ndarray, tmin: float, tmax: float) -> np.ndarray:
    """[q,8] fp32 {origin.xyz, direction.xyz, tmin, tmax} (NEXT-1 ray queries: the segment o + t d, tmin <= t <= tmax)."""
    q = origins.shape[0]
    out = np.empty((q, 8), np.float32)
    out[:, :3] = origins
    out[:, 3:6] = directions
    out[:, 6] = np.float32(tmin)
    out[:, 7] = np.float32(tmax)
    return _f32(out)


# ---- the five configs ------------------------------------------------------------------------------

@dataclass
class Workload:
    name: str
    prims: np.ndarray          # [n,3] points or [n,6] boxes, fp32
    prim_kind: str             # "points" | "boxes"
    morton_bits: int           # 30 | 63
    queries: np.ndarray | None  # [q,4] spheres or [q,6] boxes, fp32
    query_kind: str | None     # "spheres" | "boxes"
    note: str = ""

    @property
    def n(self) -> int:
        return int(self.prims.shape[0])

    @property
    def q(self) -> int:
        return 0 if self.queries is None else int(self.queries.shape[0])


FULL_SIZES = {
    "C1": (4096, 4096),
    "C2": (1 << 20, 1 << 20),
    "C3": (10_000_000, 1_000_000),
    "C4": (4_000_000, 4_000_000),
    "C5": (1 << 24, 1 << 24),
}

C5_RADIUS_FULL = 0.00606  # 32 = (2**24 / 0.488) * (4/3) pi r^3


def make(name: str, n: int | None = None, q: int | None = None, radius: float | None = None,
         seed_offset: int = 0) -> Workload:
    """Build config ``name`` ("C1".."C5").  ``n``/``q`` override the full sizes (same distribution, same
    seeds, just fewer draws), ``radius`` overrides the query radius / half-edge scale; scaled-down cases
    are what the parity tests use.  q=0 gives a build-only workload.  ``seed_offset`` r adds 10000*r to every seed
    (independent replicas for the multi-GPU bench)."""
    so = 10000 * int(seed_offset)
    fn, fq = FULL_SIZES[name]
    n = fn if n is None else n
    q = fq if q is None else q
    if name == "C1":
        # 4096 fp32 points uniform in [0,1)^3 (seed 0) as degenerate AABBs, 30-bit; spheres on the points.
        pts = uniform_cube(n, seed=0 + so)
        r = 0.085 if radius is None else radius
        centres = pts[:q] if q <= n else uniform_cube(q, seed=0 + so)
        return Workload(name, boxes_around(pts, 0.0), "boxes", 30, spheres_at(centres, r) if q else None,
                        "spheres" if q else None, "uniform cube, degenerate boxes")
    if name == "C2":
        pts = uniform_cube(n, seed=2 + so)
        r = 0.0157 if radius is None else radius
        return Workload(name, pts, "points", 63, spheres_at(uniform_cube(q, seed=1002 + so), r) if q else None,
                        "spheres" if q else None, "uniform cube")
    if name == "C3":
        pts = gaussian_mixture(n, seed=3 + so, centre_seed=3 + so)
        r = 0.002 if radius is None else radius
        qs = spheres_at(gaussian_mixture(q, seed=1003 + so, centre_seed=3 + so), r) if q else None
        return Workload(name, pts, "points", 30, qs, "spheres" if q else None, "100-component mixture, sigma 0.005")
    if name == "C4":
        h = 5e-4 if radius is None else radius
        prims = boxes_around(sphere_surface(n, seed=4 + so), h)
        qs = boxes_around(sphere_surface(q, seed=1004 + so), 2.0 * h) if q else None
        return Workload(name, prims, "boxes", 63, qs, "boxes" if q else None, "boxes on the unit sphere surface")
    if name == "C5":
        pts = hollow_shell(n, seed=5 + so)
        r = C5_RADIUS_FULL if radius is None else radius
        qs = spheres_at(hollow_shell(q, seed=1005 + so), r) if q else None
        return Workload(name, pts, "points", 63, qs, "spheres" if q else None, "hollow cube shell")
    raise KeyError(name)


def previous_queries(name: str, q: int, radius: float | None = None, seed_offset: int = 0) -> np.ndarray:
    """ANOTHER batch of ``q`` queries of config ``name``: same scene, same distribution and radius, other seeds (the
    query seeds of :func:`make` + 500).  It stands for the batch a caller served before the one being measured -- what a
    row capacity "taken from the previous batch" can honestly be derived from."""
    so = 10000 * int(seed_offset)
    if name == "C1":
        return spheres_at(uniform_cube(q, seed=500 + so), 0.085 if radius is None else radius)
    if name == "C2":
        return spheres_at(uniform_cube(q, seed=1502 + so), 0.0157 if radius is None else radius)
    if name == "C3":
        return spheres_at(gaussian_mixture(q, seed=1503 + so, centre_seed=3 + so), 0.002 if radius is None else radius)
    if name == "C4":
        return boxes_around(sphere_surface(q, seed=1504 + so), 2.0 * (5e-4 if radius is None else radius))
    if name == "C5":
        return spheres_at(hollow_shell(q, seed=1505 + so), C5_RADIUS_FULL if radius is None else radius)
    raise KeyError(name)
