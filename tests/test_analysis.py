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


# ------------------------------------------------------------------------------------------------ GPU parity
def _curve_case(q_bits, k_bits, v_bits, rows, keep):
    import torch

    import paper_2606_16317_b200 as sa
    B, H, N, D = q_bits.shape
    dev = [torch.from_numpy(np.ascontiguousarray(x).view(np.int16)).cuda().view(torch.bfloat16) for x in (q_bits, k_bits, v_bits)]
    R, nK = rows.shape[0], keep.shape[0]
    kurt = torch.full((R,), float("nan"), device="cuda", dtype=torch.float64)
    recall = torch.full((R, nK), float("nan"), device="cuda", dtype=torch.float64)
    mae = torch.full((R, nK), float("nan"), device="cuda", dtype=torch.float64)
    sa.sparse_attn_row_topk_curve(*dev, B, H, N, D, rows, keep, kurt, recall, mae)
    torch.cuda.synchronize()
    return kurt.cpu().numpy(), recall.cpu().numpy(), mae.cpu().numpy()


@pytest.mark.gpu
@pytest.mark.parametrize("D,N,H", [(128, 1000, 2), (64, 777, 1), (128, 4133, 1)])
def test_row_topk_curve_matches_the_oracle(D, N, H):
    rng = np.random.default_rng([11, D, N])
    base = rng.standard_normal((1, H, N, D)).astype(np.float32)
    taus = rng.uniform(0.3, 2.5, size=(1, H, 1, 1)).astype(np.float32)
    q_bits = f32_to_bf16_bits(taus * (0.6 * base + 0.4 * rng.standard_normal((1, H, N, D)).astype(np.float32)))
    k_bits = f32_to_bf16_bits(taus * (0.6 * base + 0.4 * rng.standard_normal((1, H, N, D)).astype(np.float32)))
    v_bits = f32_to_bf16_bits(rng.standard_normal((1, H, N, D)).astype(np.float32))
    rows = np.array([(h, r) for h in range(H) for r in sorted(rng.choice(N, size=12, replace=False))], dtype=np.int32)
    rows[0, 1], rows[-1, 1] = 0, N - 1
    keep = np.array([1, 2, 3, 17, N // 10, N // 3, N // 2, int(0.8 * N), N - 1, N], dtype=np.int32)
    kurt, recall, mae = _curve_case(q_bits, k_bits, v_bits, rows, keep)
    q64, k64, v64 = (bf16_bits_to_f64(x) for x in (q_bits, k_bits, v_bits))
    for i, (h, r) in enumerate(rows):
        okurt, orec, omae = oracle.row_topk_curve(q64[0, h, r], k64[0, h], v64[0, h], keep)
        assert kurt[i] == pytest.approx(okurt, rel=1e-3, abs=1e-3)
        # fp32 logits / exponentials against fp64: recall to 1e-5; the retained SET may differ from the oracle's only where
        # two probabilities agree to fp32 rounding, which moves O' by less than that probability
        assert np.abs(recall[i] - orec).max() < 2e-5, (i, recall[i], orec)
        assert np.all(np.abs(mae[i] - omae) <= 2e-5 + 2e-3 * omae), (i, mae[i], omae)
    assert np.all(recall[:, -1] > 1 - 1e-6) and np.all(mae[:, -1] < 1e-6)


@pytest.mark.gpu
def test_row_topk_curve_uniform_row_and_errors():
    import paper_2606_16317_b200 as sa
    N, D = 300, 128
    rng = np.random.default_rng(12)
    q_bits = f32_to_bf16_bits(rng.standard_normal((1, 1, N, D)).astype(np.float32))
    k_bits = np.zeros((1, 1, N, D), dtype=np.uint16)                          # all logits 0: p = 1 / N
    v_bits = f32_to_bf16_bits(rng.standard_normal((1, 1, N, D)).astype(np.float32))
    kurt, recall, mae = _curve_case(q_bits, k_bits, v_bits, np.array([[0, 5]], dtype=np.int32), np.array([1, 150, 300], dtype=np.int32))
    assert math.isnan(kurt[0]) and np.allclose(recall, 1.0) and np.all(mae < 1e-6)       # every key ties: all retained (R15)
    import torch
    x = torch.zeros((1, 1, N, D), device="cuda", dtype=torch.bfloat16)
    o = torch.zeros(8, device="cuda", dtype=torch.float64)
    for rows, keep in ((np.array([[0, N]], dtype=np.int32), np.array([1], dtype=np.int32)),
                       (np.array([[1, 0]], dtype=np.int32), np.array([1], dtype=np.int32)),
                       (np.array([[0, 0]], dtype=np.int32), np.array([0], dtype=np.int32)),
                       (np.array([[0, 0]], dtype=np.int32), np.array([N + 1], dtype=np.int32))):
        with pytest.raises(sa.SparseAttnError):
            sa.sparse_attn_row_topk_curve(x, x, x, 1, 1, N, D, rows, keep, o, o, o)


@pytest.mark.gpu
def test_mask_comparison_meets_the_target_and_fixed_depends_on_the_position_of_the_maximum():
    """compare_masks: every method reaches the target mean recall with its bisected parameter; its bitmaps are what the
    oracle's selectors / modes produce for that parameter; and the paper's Fig. 3 observation holds on the synthetic
    regimes (BLASST's mask depends on the POSITION of the maximum, "in the 4th column the maximum ... appears
    at the first token position, so the subsequent selection ratio drops significantly, while the 3rd column shows the
    opposite")."""
    from paper_2606_16317_b200 import analysis
    from workloads.scenarios import make_scenario
    res = {}
    for name in ("flat_max_first", "flat_max_last"):
        q, k, v = make_scenario(name, 5)
        res[name] = analysis.compare_masks(q, k, v, 0.9, iters=12)
        for m, r in res[name].items():
            assert r["recall_mean"] >= 0.9, (name, m, r["recall_mean"])
            assert r["mask"].shape == (32, 32) and not r["mask"][:, 0].any()
        # bitmaps against the oracle at the parameters the bisection found
        q64, k64, v64 = (bf16_bits_to_f64(x)[0, 0] for x in (q, k, v))
        mass, sq = oracle.block_mass(q64, k64, 128), oracle.block_sqmass(q64, k64, 128)
        r = res[name]["topk"]
        assert np.array_equal(r["mask"], oracle.select_topk(mass, r["param"]))
        for m, mode in (("fixed", oracle.MODE_FIXED), ("dynamic", oracle.MODE_DYNAMIC)):
            r = res[name][m]
            ref = oracle.run_head(*(x[0, 0] for x in (q, k, v)), tile=128, lam=r["param"], mode=mode)
            differ = ref.skip != r["mask"]
            assert not (differ & (np.abs(ref.margin) > 1e-3)).any()
            if not differ.any():
                assert r["sparsity"] == pytest.approx(ref.skipped / (ref.skipped + ref.executed))
    # At one FIXED threshold the running max is reached at once when the maximum comes first, and everything after it is
    # pruned; when it comes last nothing is.  DYNAMIC depends on the position much less (LSE accumulates mass from every tile).
    import paper_2606_16317_b200 as sa
    from parity_utils import run_gpu
    sp = {}
    for name in ("flat_max_first", "flat_max_last"):
        q, k, v = make_scenario(name, 5)
        for m, mode, lam in (("fixed", sa.MODE_FIXED, -1.0), ("dynamic", sa.MODE_DYNAMIC, -6.0)):
            st = run_gpu(q, k, v, mode=mode, lam=lam, tile=128).stats[0]
            sp[name, m] = st[1] / st.sum()
            ref = oracle.run_head(q[0, 0], k[0, 0], v[0, 0], tile=128, lam=lam, mode=getattr(oracle, "MODE_" + m.upper()))
            assert st[1] == ref.skipped
    gap_fixed = sp["flat_max_first", "fixed"] - sp["flat_max_last", "fixed"]
    gap_dyn = sp["flat_max_first", "dynamic"] - sp["flat_max_last", "dynamic"]
    assert gap_fixed > 0.5 and abs(gap_dyn) < gap_fixed


@pytest.mark.gpu
def test_recall_stats_reductions_and_nan_propagation():
    """sparse_attn_recall_stats: {min, sum} of e^(lse_retained - lse_dense) against NumPy, on more rows than one grid pass
    covers; a NaN row (a broken sparse run) must surface in the minimum instead of being dropped by fmin."""
    import torch

    import paper_2606_16317_b200 as sa
    rng = np.random.default_rng(13)
    n = 700_001
    dense = rng.normal(5.0, 2.0, size=n).astype(np.float32)
    kept = (dense + np.log(rng.uniform(0.2, 1.0, size=n))).astype(np.float32)
    rec = np.exp(kept.astype(np.float64) - dense.astype(np.float64))
    d_dense, d_kept = torch.from_numpy(dense).cuda(), torch.from_numpy(kept).cuda()
    out = torch.full((2,), -7.0, device="cuda", dtype=torch.float64)
    sa.sparse_attn_recall_stats(d_kept, d_dense, n, out)
    torch.cuda.synchronize()
    mn, sm = out.cpu().numpy()
    assert mn == rec.min() and sm == pytest.approx(rec.sum(), rel=1e-12)
    d_kept[123_456] = float("nan")
    sa.sparse_attn_recall_stats(d_kept, d_dense, n, out)
    torch.cuda.synchronize()
    mn, sm = out.cpu().numpy()
    assert math.isnan(mn) and math.isnan(sm)
    # the output-error reduction beside it
    a = torch.from_numpy(rng.standard_normal(100_000).astype(np.float32)).cuda().to(torch.bfloat16)
    b = torch.from_numpy(rng.standard_normal(100_000).astype(np.float32)).cuda().to(torch.bfloat16)
    sa.sparse_attn_output_error(a, b, a.numel(), out)
    torch.cuda.synchronize()
    diff = np.abs(a.float().cpu().numpy().astype(np.float64) - b.float().cpu().numpy().astype(np.float64))
    mx, sm = out.cpu().numpy()
    assert mx == diff.max() and sm == pytest.approx(diff.sum(), rel=1e-12)
