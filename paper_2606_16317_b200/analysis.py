"""Mask comparison and row-level recall analysis (SURVEY.md 8(f) NEXT-4; PAPER.md:196-206 Fig. 3, :249-275 Appendix A.1).

Harness logic only, like calibrate.py: every number comes out of the C ABI (`sparse_attn_fwd` in its DENSE / FIXED /
DYNAMIC / MASK modes, `sparse_attn_block_stats`, the three selectors, `sparse_attn_recall_stats`,
`sparse_attn_output_error`, `sparse_attn_row_topk_curve`); this module sequences the calls and bisects each method's one
parameter.  torch provides device memory and the stream.

compare_masks: for one head, the block bitmaps of Top-K, Top-P, the section-3 greedy mask (Eq. 3), FIXED (BLASST) and
DYNAMIC (DynSparse), each with its parameter bisected to the same MEAN row recall ("under the same precision",
PAPER.md:206), with the sparsity, recall and output error each reaches.
topk_curves: the Appendix A.1 scatter -- excess kurtosis, and recall / MAE against K, of sampled rows.
"""
from __future__ import annotations

import math
from typing import Dict, Sequence

import numpy as np

from . import binding as sa
from .calibrate import bisect_lambda

METHODS = ("topk", "topp", "greedy_eq3", "fixed", "dynamic")


def _dev_bf16(torch, bits):
    return torch.from_numpy(np.ascontiguousarray(bits).view(np.int16)).cuda().view(torch.bfloat16)


def compare_masks(q_bits, k_bits, v_bits, target_recall: float = 0.95, iters: int = 16) -> Dict[str, dict]:
    """q/k/v bits: uint16 [1, 1, N, D] (one head).  Returns {method: {param, sparsity, recall_mean, recall_min,
    err_vs_dense_max_abs, err_vs_dense_mean_abs, mask}} with mask a uint8 [T, T] numpy array (1 = skipped)."""
    import torch

    B, H, N, D = q_bits.shape
    assert B == 1 and H == 1
    tile = 64 if D == 64 else 128
    T = -(-N // tile)
    st = torch.cuda.current_stream().cuda_stream
    q, k, v = (_dev_bf16(torch, x) for x in (q_bits, k_bits, v_bits))
    out_d, out = torch.empty_like(q), torch.empty_like(q)
    lse_d = torch.empty((1, 1, N), device="cuda", dtype=torch.float32)
    lse = torch.empty_like(lse_d)
    stats = torch.zeros((1, 1, 2), device="cuda", dtype=torch.int64)
    rs = torch.zeros(2, device="cuda", dtype=torch.float64)
    mass = torch.empty((1, 1, T, T), device="cuda", dtype=torch.float32)
    sq = torch.empty_like(mass)
    bitmap = torch.zeros((1, 1, T, T), device="cuda", dtype=torch.uint8)
    sa.sparse_attn_fwd(q, k, v, out_d, lse_d, 1, 1, N, D, sa.make_params(stream=st), sa.MODE_DENSE, stats)
    sa.sparse_attn_block_stats(q, k, lse_d, mass, sq, 1, 1, N, D, 0.0, st)

    def quality(param):
        sa.sparse_attn_recall_stats(lse, lse_d, N, rs, st)
        rmin, rsum = rs.tolist()
        sa.sparse_attn_output_error(out, out_d, N * D, rs, st)
        emax, esum = rs.tolist()
        executed, skipped = stats.reshape(2).tolist()
        return {"param": param, "sparsity": skipped / (executed + skipped), "recall_mean": rsum / N, "recall_min": rmin,
                "err_vs_dense_max_abs": emax, "err_vs_dense_mean_abs": esum / (N * D),
                "mask": bitmap.reshape(T, T).cpu().numpy().copy()}

    def run_mask(param):
        sa.sparse_attn_fwd(q, k, v, out, lse, 1, 1, N, D, sa.make_params(stream=st, skip_mask_in=bitmap), sa.MODE_MASK, stats)
        return quality(param)

    def run_loop(mode, lam):
        sa.sparse_attn_fwd(q, k, v, out, lse, 1, 1, N, D, sa.make_params(lam=lam, stream=st, skip_mask_out=bitmap), mode, stats)
        return quality(lam)

    # each method as f(x) with the recall non-increasing in x, so that one bisection ("largest x that still meets the
    # target") serves all of them: x = -kept fraction, -P, log10(Theta), lambda
    def topk(x):
        sa.sparse_attn_select_blocks(mass, bitmap, 1, 1, T, T, sa.SELECT_TOPK, -x, st)
        return run_mask(-x)

    def topp(x):
        sa.sparse_attn_select_blocks(mass, bitmap, 1, 1, T, T, sa.SELECT_TOPP, -x, st)
        return run_mask(-x)

    def greedy(x):
        sa.sparse_attn_select_blocks_greedy(mass, sq, bitmap, 1, 1, N, tile, T, 10.0 ** x, st)
        return run_mask(10.0 ** x)

    ranges = {"topk": (topk, -1.0, -1.0 / T), "topp": (topp, -1.0, -1e-3), "greedy_eq3": (greedy, -16.0, 0.0),
              "fixed": (lambda x: run_loop(sa.MODE_FIXED, x), -40.0, 0.0),
              "dynamic": (lambda x: run_loop(sa.MODE_DYNAMIC, x), -40.0, 0.0)}
    result = {}
    for name in METHODS:
        f, lo, hi = ranges[name]
        seen = {}

        def recall_at(x, f=f, seen=seen):
            seen[x] = f(x)
            return seen[x]["recall_mean"]

        x, _ = bisect_lambda(recall_at, target_recall, lo, hi, iters)
        result[name] = seen[x]
    return result


def mask_picture(mask: np.ndarray) -> list:
    """One string per row of tiles: '#' retained, '.' skipped (the rows of Fig. 3 as text)."""
    return ["".join("." if s else "#" for s in row) for row in mask]


def default_keep_grid(N: int) -> np.ndarray:
    """K values for the recall ablation: geometric from 1 up to N / 2 (24 steps), then every 1 % of N up to N."""
    geo = np.unique(np.round(np.geomspace(1, N / 2, 24)).astype(np.int64))
    lin = np.unique(np.round(np.linspace(0.5, 1.0, 51) * N).astype(np.int64))
    return np.unique(np.clip(np.concatenate([geo, lin]), 1, N)).astype(np.int32)


def topk_curves(q_bits, k_bits, v_bits, rows_per_head: int, seed: int, keep_counts: Sequence[int] = None):
    """q/k/v bits: uint16 [1, H, N, D].  Samples `rows_per_head` query rows per head (seeded) and returns
    (rows int32 [R, 2], keep int32 [n_K], kurtosis [R], recall [R, n_K], mae [R, n_K]) as numpy arrays."""
    import torch

    B, H, N, D = q_bits.shape
    assert B == 1
    rng = np.random.default_rng([seed, 78])
    rows = np.empty((H * rows_per_head, 2), dtype=np.int32)
    for h in range(H):
        rows[h * rows_per_head:(h + 1) * rows_per_head, 0] = h
        rows[h * rows_per_head:(h + 1) * rows_per_head, 1] = np.sort(rng.choice(N, size=rows_per_head, replace=False))
    keep = default_keep_grid(N) if keep_counts is None else np.ascontiguousarray(keep_counts, dtype=np.int32)
    q, k, v = (_dev_bf16(torch, x) for x in (q_bits, k_bits, v_bits))
    R, nK = rows.shape[0], keep.shape[0]
    kurt = torch.empty(R, device="cuda", dtype=torch.float64)
    recall = torch.empty((R, nK), device="cuda", dtype=torch.float64)
    mae = torch.empty((R, nK), device="cuda", dtype=torch.float64)
    sa.sparse_attn_row_topk_curve(q, k, v, 1, H, N, D, rows, keep, kurt, recall, mae, 0.0, torch.cuda.current_stream().cuda_stream)
    torch.cuda.synchronize()
    return rows, keep, kurt.cpu().numpy(), recall.cpu().numpy(), mae.cpu().numpy()
