"""Iso-recall calibration of the threshold lambda.

The paper compares methods at equal quality; on inputs where the worst-case map lambda = ln((1-R)/N)
skips nothing, the informative comparison is at equal ACHIEVED recall.  Recall costs nothing extra:
for every row r, recall_r = exp(lse_retained_r - lse_dense_r), the share of the softmax mass the
retained tiles hold.  This module bisects lambda until a statistic of recall (min or mean over rows)
meets a target.  Harness logic only: every attention call goes through `sparse_attn_fwd` and the recall
statistic through `sparse_attn_recall_stats`; torch provides device memory and the stream, no arithmetic.
"""
from __future__ import annotations

import math
from typing import Callable, Tuple


def bisect_lambda(recall_at: Callable[[float], float], target: float, lo: float = -30.0, hi: float = 0.0,
                  iters: int = 14) -> Tuple[float, float]:
    """Largest lambda in [lo, hi] (to the bisection resolution) whose recall statistic is >= target.

    `recall_at(lambda)` is non-increasing in lambda up to order effects (a larger threshold skips more).
    Returns (lambda, recall_at(lambda)).  If even `lo` misses the target, (lo, recall_at(lo)) is returned;
    if `hi` already meets it, (hi, recall_at(hi))."""
    r_hi = recall_at(hi)
    if r_hi >= target:
        return hi, r_hi
    r_lo = recall_at(lo)
    if r_lo < target:
        return lo, r_lo
    best, r_best = lo, r_lo
    for _ in range(iters):
        mid = 0.5 * (lo + hi)
        r = recall_at(mid)
        if r >= target:
            lo, best, r_best = mid, mid, r
        else:
            hi = mid
    return best, r_best


def calibrate_lambda(q, k, v, B, H, N, D, mode, target: float, statistic: str = "mean", lo: float = -30.0,
                     hi: float = 0.0, iters: int = 14, stream=None):
    """Bisects lambda for `mode` on device tensors q, k, v ([B, H, N, D] bf16) until `statistic` ("min" | "mean")
    of the per-row recall is >= target.  Returns dict(lambda, recall_min, recall_mean, sparsity, calls)."""
    import torch

    from . import binding as sa

    if statistic not in ("min", "mean"):
        raise ValueError("statistic must be 'min' or 'mean'")
    st = stream if stream is not None else torch.cuda.current_stream().cuda_stream
    out = torch.empty_like(q)
    lse_d = torch.empty((B, H, N), device=q.device, dtype=torch.float32)
    lse = torch.empty_like(lse_d)
    stats = torch.zeros((B, H, 2), device=q.device, dtype=torch.int64)
    rstats = torch.zeros(2, device=q.device, dtype=torch.float64)
    sa.sparse_attn_fwd(q, k, v, out, lse_d, B, H, N, D, sa.make_params(stream=st), sa.MODE_DENSE, stats)
    last = {}
    calls = [1]

    def recall_at(lam: float) -> float:
        upper = min(lam, 0.0) if mode == sa.MODE_FIXED else lam
        sa.sparse_attn_fwd(q, k, v, out, lse, B, H, N, D, sa.make_params(lam=upper, stream=st), mode, stats)
        calls[0] += 1
        sa.sparse_attn_recall_stats(lse, lse_d, B * H * N, rstats, st)
        rmin, rsum = rstats.tolist()                       # (.tolist() synchronises)
        executed, skipped = (sum(col) for col in zip(*stats.reshape(-1, 2).tolist()))
        last[lam] = {"lambda": lam, "recall_min": rmin, "recall_mean": rsum / (B * H * N),
                     "sparsity": skipped / max(executed + skipped, 1)}
        return last[lam]["recall_" + statistic]

    lam, _ = bisect_lambda(recall_at, target, lo, hi, iters)
    res = dict(last[lam])
    res["calls"] = calls[0]
    return res
