"""Brute-force per-tile enumeration -- TEST INFRASTRUCTURE, NOT THE PRODUCT.

Second, independent formulation of the paper's rule for tiny inputs: the full
S matrix is materialised, and at every step j the cumulative energy LSE_i^(j-1) of Eq. 6 is
recomputed FROM SCRATCH as log(sum) over the explicit set of retained columns -- no running
state, no logaddexp.  The output is an explicit masked softmax over the retained columns (Eq. 1:
renormalised over the kept set).  Shares no code with dynsparse_oracle.c; used to pin it (P10).
"""
from __future__ import annotations

import math
from typing import Optional

import numpy as np

MODE_DENSE, MODE_FIXED, MODE_DYNAMIC = 0, 1, 2


def brute_force_head(q: np.ndarray, k: np.ndarray, v: np.ndarray, *, tile: int, lam: float, mode: int,
                     scale: Optional[float] = None, tile_k: Optional[int] = None):
    """q, k, v: float64 [N, D] (already widened from bf16).  Decision tiles are `tile` query rows by
    `tile_k` keys (default: square; the paper gives B_c only -- 128 for 14B, 32 for 5B).

    Returns dict(out [N, D], lse [N], skip [T_r, T_c] uint8, margin [T_r, T_c]).
    """
    N, D = q.shape
    if scale is None:
        scale = 1.0 / math.sqrt(D)
    width = tile if tile_k is None else tile_k
    T_r = -(-N // tile)
    T_c = -(-N // width)
    S = scale * (q @ k.T)                               # logits, S includes the scale
    out = np.zeros((N, D))
    lse = np.zeros(N)
    skip = np.zeros((T_r, T_c), dtype=np.uint8)
    margin = np.full((T_r, T_c), np.inf)
    for i in range(T_r):
        rows = range(i * tile, min(N, (i + 1) * tile))
        retained_cols = []                              # explicit set: columns of tiles k notin J_i
        for j in range(T_c):
            cols = list(range(j * width, min(N, (j + 1) * width)))
            if mode == MODE_DENSE or not retained_cols:
                keep = True                             # first tile: LSE^(0) = -inf, t = +inf
            else:
                t_max = -np.inf
                for r in rows:
                    mhat = max(S[r, c] for c in cols)
                    kept = S[r, retained_cols]
                    if mode == MODE_DYNAMIC:
                        ref = math.log(np.sum(np.exp(kept - kept.max()))) + kept.max()   # Eq. 6
                    else:
                        ref = kept.max()                # running max over retained tiles (BLASST)
                    t_max = max(t_max, mhat - ref)      # Eq. 5
                margin[i, j] = t_max - lam
                keep = not (t_max < lam)                # skip iff t < lambda for every row
            if keep:
                retained_cols.extend(cols)
            else:
                skip[i, j] = 1
        for r in rows:                                  # masked softmax over the retained columns
            s = S[r, retained_cols]
            m = s.max()
            e = np.exp(s - m)
            z = e.sum()
            out[r] = (e / z) @ v[retained_cols]
            lse[r] = m + math.log(z)
    return dict(out=out, lse=lse, skip=skip, margin=margin)
