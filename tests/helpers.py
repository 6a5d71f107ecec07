"""Test-side helpers.  None of this is imported by the product or by the oracle.

``alg4_serial`` is a direct transliteration of the paper's Algorithm 4 (with the
readings G1, G2, G11, G14 of DESIGN.md) that runs the leaf "threads" one at a time in a given order;
a thread that arrives first at a parent stops (ATOMICCAS returned the invalid value), the second one
carries on.  It is an independent route to the hierarchy the oracle builds top-down.
"""
from __future__ import annotations

import numpy as np

INF = 1 << 200


def delta_star(codes, i: int, n: int) -> int:
    """XOR magnitude of adjacent augmented keys (code, position); +inf out of range (G1, G5)."""
    if i < 0 or i >= n - 1:
        return INF
    i = int(i)
    return ((int(codes[i]) << 32) | i) ^ ((int(codes[i + 1]) << 32) | (i + 1))


def alg4_serial(codes, order=None):
    """Returns (left_child[n-1], rope[2n-1]) in unified indices (I_k -> k, L_i -> n-1+i, sentinel -1)."""
    n = len(codes)
    lb = n - 1
    left = [None] * max(n - 1, 0)
    rope = [None] * (2 * n - 1)
    store = [-1] * max(n - 1, 0)
    d = lambda i: delta_star(codes, i, n)  # noqa: E731
    if order is None:
        order = range(n)
    for i in order:
        i = int(i)
        rl, rr = i, i
        dl, dr = d(i - 1), d(i)                       # L3-4
        if i == n - 1:                                # L5-6
            rope[lb + i] = -1
        else:                                         # L8
            rope[lb + i] = lb + i + 1 if dr < d(i + 1) else i + 1
        if n == 1:                                    # G11
            break
        while True:
            if dr < dl:                               # L10 left child of its parent
                p = rr                                # L11
                old, store[p] = store[p], (rl if store[p] == -1 else store[p])  # L12 ATOMICCAS
                if old == -1:
                    break                             # L13
                rr = old
                dr = d(rr)                            # L14
            else:                                     # right child of its parent
                p = rl - 1                            # L16
                old, store[p] = store[p], (rr if store[p] == -1 else store[p])  # L17
                if old == -1:
                    break                             # L18
                rl = old
                dl = d(rl - 1)                        # L19
            q = rr if dr < dl else rl                 # L20 Karras index
            left[q] = lb + p if rl == p else p        # L21 (reading G2: compares with p, child is L_p / I_p)
            if rr == n - 1:                           # L22-23
                rope[q] = -1
            else:
                r = rr + 1                            # L25
                rope[q] = lb + r if dr < d(r) else r  # L26
            if q == 0:                                # L28 until i = 0
                break
    return np.array(left, np.int32), np.array(rope, np.int32)


def csr_rows_sorted(offsets, indices):
    """CSR with each row sorted ascending (rows are sets: G13)."""
    offsets = np.asarray(offsets, np.int64)
    indices = np.asarray(indices)
    q = len(offsets) - 1
    if len(indices) == 0:
        return indices.copy()
    row = np.repeat(np.arange(q, dtype=np.int64), np.diff(offsets))
    order = np.lexsort((indices, row))
    return indices[order]
