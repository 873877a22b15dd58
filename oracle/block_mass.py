"""Block mass and block selectors -- TEST INFRASTRUCTURE, NOT THE PRODUCT.

PAPER.md:61-62 (Top-P: retain until the retained probability reaches the target; Top-K: a fixed budget), applied at
block level as in the paper's Table 1 / Fig. 3 comparison.  Plain definitions in fp64:

  mass[i, j] = sum over rows r of Q tile i and columns c of K tile j of softmax(scale * Q K^T)[r, c]
  Top-K: per row of tiles, retain the ceil(keep * T_c) tiles of largest mass
  Top-P: per row of tiles, retain tiles in order of decreasing mass until the retained share of the row's
         total mass reaches P (the tile that crosses P is retained)
Ties are broken by the lower tile index first.  Tile 0 is always retained (the kernel's MASK mode keeps it anyway).
"""
from __future__ import annotations

import math

import numpy as np


def block_mass(q: np.ndarray, k: np.ndarray, tile: int, scale: float | None = None) -> np.ndarray:
    """q, k: [N, D] float64 (widened bf16).  Returns [T, T] float64."""
    N, D = q.shape
    scale = 1.0 / math.sqrt(D) if scale is None else scale
    s = scale * (q @ k.T)
    p = np.exp(s - s.max(axis=1, keepdims=True))
    p /= p.sum(axis=1, keepdims=True)
    T = -(-N // tile)
    mass = np.zeros((T, T))
    for i in range(T):
        for j in range(T):
            mass[i, j] = p[i * tile:(i + 1) * tile, j * tile:(j + 1) * tile].sum()
    return mass


def _order(row: np.ndarray) -> np.ndarray:
    """Tile indices by decreasing mass, ties by increasing index."""
    return np.array(sorted(range(len(row)), key=lambda j: (-row[j], j)), dtype=np.int64)


def select_topk(mass: np.ndarray, keep: float) -> np.ndarray:
    """Returns the skip bitmap [T_r, T_c] (1 = skip)."""
    T_r, T_c = mass.shape
    n_keep = min(T_c, max(1, math.ceil(keep * T_c)))
    skip = np.ones((T_r, T_c), dtype=np.uint8)
    for i in range(T_r):
        skip[i, _order(mass[i])[:n_keep]] = 0
    skip[:, 0] = 0
    return skip


def select_topp(mass: np.ndarray, p: float) -> np.ndarray:
    T_r, T_c = mass.shape
    skip = np.ones((T_r, T_c), dtype=np.uint8)
    for i in range(T_r):
        total, acc = mass[i].sum(), 0.0
        for j in _order(mass[i]):
            if acc >= p * total:
                break
            skip[i, j] = 0
            acc += mass[i, j]
    skip[:, 0] = 0
    return skip
