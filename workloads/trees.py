"""Seeded random coalescent trees (inputs only).

Node numbering: tips 0..N-1, internal nodes N..2N-2 in order of creation going
backwards in time, so the root is 2N-2 (the library does not rely on this; tests
also feed relabelled trees).  PAPER.md:L64 "N-tipped F", 2N-1 nodes, bifurcating.
"""
from __future__ import annotations

import numpy as np


def coalescent(rng: np.random.Generator, tip_heights: np.ndarray, ne: float = 1.0):
    """Serially-sampled Kingman coalescent. `tip_heights` (N,) >= 0 are sampling heights (0 = most recent).
    Returns (parent int32 (2N-1,), height float64 (2N-1,))."""
    N = int(tip_heights.shape[0])
    order = np.argsort(tip_heights, kind="stable")
    parent = np.full(2 * N - 1, -1, dtype=np.int32)
    height = np.zeros(2 * N - 1, dtype=np.float64)
    height[:N] = tip_heights
    active = []
    nxt = 0            # next tip (in `order`) still to be sampled
    t = 0.0
    new = N
    while new < 2 * N - 1:
        k = len(active)
        if k < 2:
            tip = int(order[nxt]); nxt += 1
            t = max(t, float(tip_heights[tip]))
            active.append(tip)
            continue
        wait = rng.exponential(ne / (k * (k - 1) / 2.0))
        if nxt < N and t + wait > tip_heights[order[nxt]]:
            tip = int(order[nxt]); nxt += 1
            t = float(tip_heights[tip])
            active.append(tip)
            continue
        t = t + wait
        i, j = rng.choice(k, size=2, replace=False)
        a, b = active[i], active[j]
        for idx in sorted((int(i), int(j)), reverse=True):
            active.pop(idx)
        parent[a] = new
        parent[b] = new
        height[new] = t
        active.append(new)
        new += 1
    return parent, height


def stretch_above(height: np.ndarray, pivot: float, root_height: float) -> np.ndarray:
    """Map heights above `pivot` linearly so the maximum becomes `root_height` (monotone: order is kept)."""
    h = height.copy()
    top = h.max()
    if top <= pivot:
        raise ValueError("root is not above the pivot")
    above = h > pivot
    h[above] = pivot + (h[above] - pivot) * ((root_height - pivot) / (top - pivot))
    h[np.argmax(height)] = root_height
    return h


def relabel_internal(rng: np.random.Generator, parent: np.ndarray, height: np.ndarray):
    """Randomly permute the labels of the internal nodes (tips keep 0..N-1). For testing label-independence."""
    n = parent.shape[0]
    N = (n + 1) // 2
    perm = np.arange(n)
    perm[N:] = N + rng.permutation(n - N)      # old label -> new label
    new_parent = np.full(n, -1, dtype=np.int32)
    new_height = np.zeros(n, dtype=np.float64)
    for old in range(n):
        p = parent[old]
        new_parent[perm[old]] = -1 if p < 0 else perm[p]
        new_height[perm[old]] = height[old]
    return new_parent, new_height


def children_of(parent: np.ndarray):
    """(left, right) child arrays, -1 for tips; children ordered by label."""
    n = parent.shape[0]
    left = np.full(n, -1, dtype=np.int64)
    right = np.full(n, -1, dtype=np.int64)
    for c in range(n):
        p = parent[c]
        if p < 0:
            continue
        if left[p] < 0:
            left[p] = c
        else:
            right[p] = c
    return left, right
