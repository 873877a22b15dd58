"""Row-level accuracy-vs-recall analysis of PAPER.md Appendix A.1 -- TEST INFRASTRUCTURE, NOT THE PRODUCT.

PAPER.md:253-257: "We sample random rows from the P matrix and apply Top-K with different K values to ablate the recall
rate.  Excess Kurtosis is used to measure the 'tailedness' of a data distribution."  Fig. 4 / Table 3
then relate the mean absolute error of the output to the recall, by excess-kurtosis bin.  Plain definitions, fp64, for
ONE query row with logits s_c = scale * <q, k_c> over all N keys:

  p            = softmax(s)                                                        (N values, sum 1)
  kurtosis     = m4 / m2^2 - 3,  m_n = mean_c (p_c - mean(p))^n                    (population excess kurtosis of the N values)
  Top-K        = the K keys of largest p (every key equal to the K-th largest value is retained: reading R15 of DESIGN.md)
  recall(K)    = sum_{c in Top-K} p_c                                              ("retained probability")
  O            = sum_c p_c v_c,     O'(K) = sum_{c in Top-K} p_c v_c / recall(K)   (Eq. 1: renormalised)
  MAE(K)       = mean_d |O_d - O'(K)_d|

Parity pins (tests/test_analysis.py): the kurtosis against scipy.stats.kurtosis and the Bernoulli closed form of a one-hot row
(N^2 / (N - 1) - 6), uniform rows (recall = K / N exactly), K = N (recall 1, MAE 0), Eq. 1's error
identity E = O' - O evaluated term by term on small rows, and brute force over explicit index sets.
"""
from __future__ import annotations

import math

import numpy as np

# Table 3's kurtosis bins: (lo, hi], first bin closed below at -inf, last open above
KURTOSIS_BINS = (-math.inf, 0.0, 1.0, 3.0, 10.0, 30.0, 100.0, 300.0, 1000.0, 3000.0, 10000.0, math.inf)


def excess_kurtosis(p: np.ndarray) -> float:
    """Population excess kurtosis of the values of p (a constant vector has none: returns nan)."""
    p = np.asarray(p, dtype=np.float64)
    d = p - p.mean()
    m2 = np.mean(d ** 2)
    m4 = np.mean(d ** 4)
    if m2 == 0.0:
        return math.nan
    return float(m4 / (m2 * m2) - 3.0)


def row_probabilities(q_row: np.ndarray, k: np.ndarray, scale: float | None = None) -> np.ndarray:
    """softmax(scale * k q) over all N keys.  q_row: [D], k: [N, D], fp64."""
    D = q_row.shape[0]
    scale = 1.0 / math.sqrt(D) if scale is None else scale
    s = scale * (k.astype(np.float64) @ q_row.astype(np.float64))
    e = np.exp(s - s.max())
    return e / e.sum()


def row_topk_curve(q_row: np.ndarray, k: np.ndarray, v: np.ndarray, keep_counts, scale: float | None = None):
    """Returns (kurtosis, recall[n_K], mae[n_K]) of one query row for every K in keep_counts (1 <= K <= N)."""
    p = row_probabilities(q_row, k, scale)
    v = v.astype(np.float64)
    N = p.shape[0]
    O = p @ v
    srt = np.sort(p)[::-1]
    recall, mae = [], []
    for K in keep_counts:
        K = int(K)
        assert 1 <= K <= N
        kept = p >= srt[K - 1]                     # every key equal to the K-th largest value is retained (R15)
        r = p[kept].sum()
        Oq = (p[kept] @ v[kept]) / r
        recall.append(r)
        mae.append(np.abs(O - Oq).mean())
    return excess_kurtosis(p), np.array(recall), np.array(mae)


def kurtosis_bin(kurt: float) -> int:
    """Index of Table 3's bin: bin b holds KURTOSIS_BINS[b] < kurt <= KURTOSIS_BINS[b + 1] (the last is open above)."""
    for b in range(len(KURTOSIS_BINS) - 1):
        if kurt <= KURTOSIS_BINS[b + 1]:
            return b
    return len(KURTOSIS_BINS) - 2


def table3(kurt: np.ndarray, recall: np.ndarray, mae: np.ndarray, recall_at=0.8, recall_tol=0.01, mae_at=0.05, mae_tol=0.005):
    """Table 3 from the scatter of (recall, MAE) points of all rows and all K: per kurtosis bin, mean and
    standard deviation of the MAE over the points with |recall - 0.8| <= 0.01, and mean and variance of the recall over the
    points with |MAE - 0.05| <= 0.005.  kurt: [R], recall, mae: [R, n_K].  Returns a list of dicts, one per bin."""
    bins = np.array([kurtosis_bin(x) for x in kurt])
    out = []
    for b in range(len(KURTOSIS_BINS) - 1):
        sel = bins == b
        rc, me = recall[sel].ravel(), mae[sel].ravel()
        a = me[np.abs(rc - recall_at) <= recall_tol]
        c = rc[np.abs(me - mae_at) <= mae_tol]
        out.append({"kurtosis_lo": KURTOSIS_BINS[b], "kurtosis_hi": KURTOSIS_BINS[b + 1], "rows": int(sel.sum()),
                    "mae_at_recall_n": int(a.size), "mae_at_recall_mean": float(a.mean()) if a.size else None,
                    "mae_at_recall_std": float(a.std()) if a.size else None,
                    "recall_at_mae_n": int(c.size), "recall_at_mae_mean": float(c.mean()) if c.size else None,
                    "recall_at_mae_var": float(c.var()) if c.size else None})
    return out
