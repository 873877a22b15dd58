"""Pins of oracle/analysis.py (Appendix A.1) and, on the GPU, parity of
sparse_attn_row_topk_curve with it."""
import itertools
import math

import numpy as np
import pytest
import scipy.stats

import oracle
from workloads import bf16_bits_to_f64, f32_to_bf16_bits


def _rows(seed, N, D, tau):
    rng = np.random.default_rng(seed)
    q = bf16_bits_to_f64(f32_to_bf16_bits((tau * rng.standard_normal(D)).astype(np.float32)))
    k = bf16_bits_to_f64(f32_to_bf16_bits(rng.standard_normal((N, D)).astype(np.float32)))
    v = bf16_bits_to_f64(f32_to_bf16_bits(rng.standard_normal((N, D)).astype(np.float32)))
    return q, k, v


def test_kurtosis_against_scipy_and_closed_forms():
    rng = np.random.default_rng(0)
    for n in (7, 100, 4097):
        x = rng.gamma(0.3, size=n)
        assert oracle.excess_kurtosis(x) == pytest.approx(scipy.stats.kurtosis(x, fisher=True, bias=True), rel=1e-12)
    # one-hot row of length N: a Bernoulli(1/N) sample, excess kurtosis 1/(pq) - 6 = N^2/(N-1) - 6
    for n in (2, 5, 214, 32760):
        onehot = np.zeros(n)
        onehot[n // 3] = 1.0
        assert oracle.excess_kurtosis(onehot) == pytest.approx(n * n / (n - 1.0) - 6.0, rel=1e-9)
    # two equal halves (a, b): every deviation has the same magnitude -> m4 = m2^2 -> excess kurtosis -2
    assert oracle.excess_kurtosis(np.array([0.1] * 8 + [0.025] * 8)) == pytest.approx(-2.0, abs=1e-12)
    assert math.isnan(oracle.excess_kurtosis(np.full(9, 1.0 / 9)))
    # invariance under scale and shift
    x = rng.random(1000)
    assert oracle.excess_kurtosis(3.0 * x + 2.0) == pytest.approx(oracle.excess_kurtosis(x), rel=1e-10)


def test_kurtosis_bins_are_table3s():
    assert len(oracle.KURTOSIS_BINS) - 1 == 11                               # eleven rows
    assert [oracle.kurtosis_bin(x) for x in (-1.2, 0.0, 0.5, 1.0, 2.0, 10.0, 10.1, 9999.0, 10000.0, 10001.0, 1e9)] == \
           [0, 0, 1, 1, 2, 3, 4, 9, 9, 10, 10]


def test_uniform_row_recall_is_k_over_n_and_full_k_is_exact():
    N, D = 96, 16
    rng = np.random.default_rng(1)
    v = rng.standard_normal((N, D))
    k = np.zeros((N, D))                                                      # all logits equal: p = 1/N
    q = rng.standard_normal(D)
    kurt, recall, mae = oracle.row_topk_curve(q, k, v, [1, 10, N])
    assert math.isnan(kurt)
    # every key ties with the K-th largest: all are retained (R15), so recall is 1 at every K
    assert np.allclose(recall, 1.0) and np.allclose(mae, 0.0, atol=1e-15)
    q, k, v = _rows(2, 300, 32, 2.0)
    _, recall, mae = oracle.row_topk_curve(q, k, v, [300])
    assert recall[0] == pytest.approx(1.0, abs=1e-14) and mae[0] < 1e-15


def test_curve_against_brute_force_index_sets():
    """Top-K as an explicit index set from a stable sort; recall, O' and the MAE recomputed from the definitions."""
    for seed, N, D, tau in ((3, 50, 8, 1.0), (4, 257, 64, 3.0), (5, 1000, 128, 0.5)):
        q, k, v = _rows(seed, N, D, tau)
        s = (k @ q) / math.sqrt(D)
        w = np.array([math.exp(x - s.max()) for x in s])
        p = w / w.sum()
        order = sorted(range(N), key=lambda c: -p[c])
        Ks = [1, 2, N // 7 + 1, N // 2, N - 1, N]
        kurt, recall, mae = oracle.row_topk_curve(q, k, v, Ks)
        assert kurt == pytest.approx(scipy.stats.kurtosis(p), rel=1e-10)
        O = sum(p[c] * v[c] for c in range(N))
        for K, r, e in zip(Ks, recall, mae):
            S = order[:K]
            rr = sum(p[c] for c in S)
            Oq = sum(p[c] * v[c] for c in S) / rr
            assert r == pytest.approx(rr, rel=1e-12)
            assert e == pytest.approx(float(np.mean(np.abs(O - Oq))), rel=1e-9, abs=1e-14)
            # Eq. 1: O' - O = (S1 / (1 - S1)) sum_kept p v - sum_discarded p v with S1 = 1 - recall
            if K < N:
                disc = order[K:]
                s1 = sum(p[c] for c in disc)
                E = (s1 / (1.0 - s1)) * sum(p[c] * v[c] for c in S) - sum(p[c] * v[c] for c in disc)
                assert np.allclose(Oq - O, E, rtol=1e-9, atol=1e-15)
        assert all(a <= b + 1e-15 for a, b in zip(recall, recall[1:]))       # recall grows with K


def test_table3_windows():
    kurt = np.array([-0.5, 50.0, 50.0])
    recall = np.array([[0.795, 0.9], [0.805, 0.3], [0.82, 0.31]])
    mae = np.array([[0.01, 0.001], [0.03, 0.051], [0.5, 0.046]])
    t = oracle.table3(kurt, recall, mae)
    assert t[0]["rows"] == 1 and t[0]["mae_at_recall_mean"] == pytest.approx(0.01) and t[0]["recall_at_mae_n"] == 0
    b = t[oracle.kurtosis_bin(50.0)]
    assert b["rows"] == 2 and b["mae_at_recall_n"] == 1 and b["mae_at_recall_mean"] == pytest.approx(0.03)
    assert b["recall_at_mae_n"] == 2 and b["recall_at_mae_mean"] == pytest.approx(0.305)
    assert b["recall_at_mae_var"] == pytest.approx(0.005 ** 2)
