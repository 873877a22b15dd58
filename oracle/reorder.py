"""Token re-ordering oracle -- TEST INFRASTRUCTURE, NOT THE PRODUCT.

PAPER.md:139 (last sentence) and :25: tokens of the 1-D sequence are mapped back to their
[t, h, w] grid and regrouped into spatio-temporal blocks so that the tokens of one attention tile
are neighbours in time and space.  This is the plain definition, written with one Python loop per
token (slow, obviously correct): position p of the brick order holds the token with the p-th
smallest key (brick_t_index, brick_h_index, brick_w_index, t, h, w).  Bricks at the upper edges of
a grid whose sides are not multiples of the brick are simply smaller (no padding).

Pins (tests/test_reorder.py): it is a bijection; a brick that spans the whole grid, or one row of
it, gives the identity; on a grid whose sides are multiples of the brick it equals the closed form
reshape(T/bt, bt, H/bh, bh, W/bw, bw).transpose(0, 2, 4, 1, 3, 5); every full brick is contiguous.
"""
from __future__ import annotations

import numpy as np


def brick_permutation(grid, brick) -> np.ndarray:
    """perm[p] = original [t, h, w]-order index n of the token at position p of the brick order."""
    T, H, W = (int(x) for x in grid)
    bt, bh, bw = (int(x) for x in brick)
    keyed = []
    for t in range(T):
        for h in range(H):
            for w in range(W):
                n = (t * H + h) * W + w
                keyed.append(((t // bt, h // bh, w // bw, t, h, w), n))
    keyed.sort(key=lambda kv: kv[0])
    return np.array([n for _, n in keyed], dtype=np.int64)


def reorder(x: np.ndarray, perm: np.ndarray, inverse: bool = False) -> np.ndarray:
    """x: [..., N, D].  Forward: y[..., p, :] = x[..., perm[p], :].  Inverse: y[..., perm[p], :] = x[..., p, :]."""
    y = np.empty_like(x)
    N = x.shape[-2]
    for p in range(N):
        if inverse:
            y[..., int(perm[p]), :] = x[..., p, :]
        else:
            y[..., p, :] = x[..., int(perm[p]), :]
    return y
