"""Block mass and block selectors -- TEST INFRASTRUCTURE, NOT THE PRODUCT.

PAPER.md:61-62 (Top-P: retain until the retained probability reaches the target; Top-K: a fixed budget), applied at
block level as in the paper's Table 1 / Fig. 3 comparison.  Plain definitions in fp64:

  mass[i, j] = sum over rows r of Q tile i and columns c of K tile j of softmax(scale * Q K^T)[r, c]
  Top-K: per row of tiles, retain the ceil(keep * T_c) tiles of largest mass
  Top-P: per row of tiles, retain tiles in order of decreasing mass until the retained share of the row's
         total mass reaches P (the tile that crosses P is retained)
Ties are broken by the lower tile index first.  Tile 0 is always retained (the kernel's MASK mode keeps it anyway).

The "ideal" mask of PAPER.md section 3 (lines 105-109), at block level, under the variance bound of Eq. 3:
  sqmass[i, j] = sum over the same rows and columns of softmax(.)[r, c] ** 2
  P_j = mass[i, j] / rows_i,  q_j = sqmass[i, j] / rows_i   (block sums averaged over the valid rows of Q tile i: Eq. 3
        is written for one query row; a block mask takes one decision per row of TILES -- reading R14 of DESIGN.md)
  "Sort P_j in ascending order.  Initialize S = {}, K = {1..N}.  Sequentially move the smallest p_j from K to S, and
   dynamically update S_1 = sum_S p_j.  Calculate the current error variance metric in real time, and stop the
   computation when the condition represented by Eq. 3 is met":
  tiles j >= 1 are moved in order of increasing P_j (ties: lower index first) while, WITH the tile in S,
        sum_S q_j + (S_1 / (1 - S_1))^2 sum_K q_j <= Theta
  still holds; the first tile that would break it, and every larger one, stays in K.
Parity pins (tests/test_block_mass.py): uniform rows discard exactly min(T-1, floor(Theta N T / (1 + Theta N))) tiles
(closed form derived there), Theta = 0 discards nothing of positive mass, and the bound is checked by direct evaluation
of Eq. 3 on the returned set and on the set with one more tile.
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


def block_sqmass(q: np.ndarray, k: np.ndarray, tile: int, scale: float | None = None) -> np.ndarray:
    """Per-tile sum of squared dense probabilities.  q, k: [N, D] float64 (widened bf16).  Returns [T, T] float64."""
    N, D = q.shape
    scale = 1.0 / math.sqrt(D) if scale is None else scale
    s = scale * (q @ k.T)
    p = np.exp(s - s.max(axis=1, keepdims=True))
    p /= p.sum(axis=1, keepdims=True)
    p2 = p * p
    T = -(-N // tile)
    sq = np.zeros((T, T))
    for i in range(T):
        for j in range(T):
            sq[i, j] = p2[i * tile:(i + 1) * tile, j * tile:(j + 1) * tile].sum()
    return sq


def eq3_lhs(P: np.ndarray, q: np.ndarray, discarded) -> float:
    """Left side of Eq. 3 for one row: sum_S q_j + (S_1/(1-S_1))^2 sum_K q_j, S_1 = sum_S P_j."""
    d = np.zeros(len(P), dtype=bool)
    d[list(discarded)] = True
    s1 = P[d].sum()
    if not s1 < 1.0:
        return math.inf
    return q[d].sum() + (s1 / (1.0 - s1)) ** 2 * q[~d].sum()


def select_greedy(mass: np.ndarray, sqmass: np.ndarray, N: int, tile_q: int, theta: float) -> np.ndarray:
    """Returns the skip bitmap [T_r, T_c] (1 = skip) of the section-3 mask under Eq. 3 with tolerance `theta`."""
    T_r, T_c = mass.shape
    skip = np.zeros((T_r, T_c), dtype=np.uint8)
    for i in range(T_r):
        rows = min(tile_q, N - i * tile_q)
        P = mass[i].astype(np.float64) / rows
        q = sqmass[i].astype(np.float64) / rows
        ascending = sorted(range(1, T_c), key=lambda j: (mass[i, j], j))      # tile 0 is never a candidate
        S = []
        for j in ascending:
            if not eq3_lhs(P, q, S + [j]) <= theta:
                break
            S.append(j)
        skip[i, S] = 1
    return skip
