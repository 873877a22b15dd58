"""Pins of the CPU oracle against what the paper and the mathematics fix.

None of these tests touches the CUDA path.  Each pin is chosen so that a plausible mistake in
oracle/dynsparse_oracle.c (dropped scale, wrong sign, wrong reference statistic, state updated on
a skipped tile, transposed operand, non-strict inequality) fails at least one of them.
"""
import math
import os

import numpy as np
import pytest
import torch

import oracle
from oracle import MODE_DENSE, MODE_DYNAMIC, MODE_FIXED
from workloads import CONFIGS, bf16_bits_to_f64, f32_to_bf16_bits, make_head

GOLDEN = os.path.join(os.path.dirname(__file__), "golden", "paper_values.txt")


def _golden():
    vals = {}
    with open(GOLDEN) as f:
        for line in f:
            if line.startswith("#") or not line.strip():
                continue
            key, val, _cite = [s.strip() for s in line.split("|", 2)]
            vals[key] = float(val)
    return vals


def _rand_bits(rng, N, D, spread):
    """Random bf16 inputs whose logits have a few units of spread."""
    q = rng.standard_normal((N, D)).astype(np.float32) * spread
    k = rng.standard_normal((N, D)).astype(np.float32) * spread
    v = rng.standard_normal((N, D)).astype(np.float32)
    return f32_to_bf16_bits(q), f32_to_bf16_bits(k), f32_to_bf16_bits(v)


@pytest.fixture(scope="module")
def cfg0_head(seed):
    return make_head(CONFIGS["cfg0"], seed, 0)


# ---------------------------------------------------------------- P1: dense special case
@pytest.mark.parametrize("N,D,tile", [(1024, 64, 64), (200, 64, 64), (333, 128, 128), (64, 64, 64)])
def test_p1_dense_is_textbook_softmax(N, D, tile, seed):
    rng = np.random.default_rng([seed, N, D])
    qb, kb, vb = _rand_bits(rng, N, D, 1.5)
    q, k, v = (bf16_bits_to_f64(x) for x in (qb, kb, vb))
    scale = 1.0 / math.sqrt(D)
    o_ref, lse_ref, _ = oracle.dense_attention_textbook(q, k, v, scale)
    for mode, lam in [(MODE_DENSE, 0.0), (MODE_DYNAMIC, -math.inf), (MODE_FIXED, -math.inf)]:
        res = oracle.run_head(qb, kb, vb, tile=tile, lam=lam, mode=mode)
        o, lse = res.rows()
        assert res.skipped == 0
        np.testing.assert_allclose(o, o_ref, rtol=0, atol=1e-12)
        np.testing.assert_allclose(lse, lse_ref, rtol=0, atol=1e-12)
    # library routine: torch SDPA in fp64 on CPU
    tq, tk, tv = (torch.from_numpy(x)[None, None] for x in (q, k, v))
    o_t = torch.nn.functional.scaled_dot_product_attention(tq, tk, tv, scale=scale)[0, 0].numpy()
    np.testing.assert_allclose(o, o_t, rtol=0, atol=1e-12)


def test_p1_scale_override_is_honoured(seed):
    rng = np.random.default_rng([seed, 5])
    qb, kb, vb = _rand_bits(rng, 192, 64, 1.0)
    q, k, v = (bf16_bits_to_f64(x) for x in (qb, kb, vb))
    o_ref, lse_ref, _ = oracle.dense_attention_textbook(q, k, v, 0.37)
    o, lse = oracle.run_head(qb, kb, vb, tile=64, lam=0.0, mode=MODE_DENSE, scale=0.37).rows()
    np.testing.assert_allclose(o, o_ref, atol=1e-12)
    np.testing.assert_allclose(lse, lse_ref, atol=1e-12)


# ---------------------------------------------------------------- P2/P3/P4: recall guarantee and counts
@pytest.mark.parametrize("mode", [MODE_DYNAMIC, MODE_FIXED])
@pytest.mark.parametrize("lam", [-1.0, -2.0, -3.0, -4.0, -6.0])
def test_p2_p3_p4_recall_bound_on_cfg0(cfg0_head, mode, lam):
    qb, kb, vb = cfg0_head
    N, D, tile = 1024, 64, 64
    q, k = bf16_bits_to_f64(qb), bf16_bits_to_f64(kb)
    S = (q @ k.T) / math.sqrt(D)
    dense = oracle.run_head(qb, kb, vb, tile=tile, lam=0.0, mode=MODE_DENSE)
    res = oracle.run_head(qb, kb, vb, tile=tile, lam=lam, mode=mode)
    T = N // tile
    assert res.skip.shape == (T, T)
    assert not res.skip[:, 0].any()                                   # P4: tile 0 never skipped
    assert res.executed + res.skipped == T * T                        # P4
    _, L = res.rows()
    _, Ld = dense.rows()
    recall = np.exp(L - Ld)
    assert np.all(recall <= 1.0 + 1e-12)
    for i in range(T):
        rows = slice(i * tile, (i + 1) * tile)
        n_skipped_cols = 0
        for j in range(T):
            if res.skip[i, j]:
                n_skipped_cols += tile
                # P2: every logit of a skipped tile is below the final LSE + lambda
                assert np.all(S[rows, j * tile:(j + 1) * tile] < L[rows, None] + lam)
        # P3 (G4): lost share < (#skipped columns) e^lambda per row.
        # recall is measured against the dense normaliser, the bound against the retained one:
        # 1 - recall = lost/(kept+lost) <= lost/kept < n_skipped * e^lambda.
        assert np.all(1.0 - recall[rows] < n_skipped_cols * math.exp(lam) + 1e-15)


@pytest.mark.parametrize("mode", [MODE_DYNAMIC, MODE_FIXED])
@pytest.mark.parametrize("target", [0.90, 0.95, 0.99])
def test_p3_strict_map_meets_recall_target_on_every_row(seed, mode, target):
    # the strict map lambda = ln((1-R)/N) on an input where tiles really are skipped
    N, D, tile = 512, 64, 64
    rng = np.random.default_rng([seed, 77])
    q = rng.standard_normal((N, D)).astype(np.float32)
    k = rng.standard_normal((N, D)).astype(np.float32)
    k[:tile] = q[:tile] * 1.0                       # strong early keys so that later tiles fall below threshold
    q *= 6.0
    qb, kb = f32_to_bf16_bits(q), f32_to_bf16_bits(k * 3.0)
    vb = f32_to_bf16_bits(rng.standard_normal((N, D)).astype(np.float32))
    lam = oracle.lambda_from_recall(target, N)
    dense = oracle.run_head(qb, kb, vb, tile=tile, lam=0.0, mode=MODE_DENSE)
    res = oracle.run_head(qb, kb, vb, tile=tile, lam=lam, mode=mode)
    recall = np.exp(res.rows()[1] - dense.rows()[1])
    assert recall.min() > target


# ---------------------------------------------------------------- P5: Eq. 1 identity
@pytest.mark.parametrize("lam", [-2.0, -3.0])
def test_p5_eq1_error_decomposition(cfg0_head, lam):
    qb, kb, vb = cfg0_head
    N, D, tile = 1024, 64, 64
    q, k, v = (bf16_bits_to_f64(x) for x in (qb, kb, vb))
    o_dense, _, p = oracle.dense_attention_textbook(q, k, v, 1.0 / math.sqrt(D))
    res = oracle.run_head(qb, kb, vb, tile=tile, lam=lam, mode=MODE_DYNAMIC)
    assert res.skipped > 0
    o_sparse, _ = res.rows()
    discarded = np.repeat(np.repeat(res.skip.astype(bool), tile, axis=0), tile, axis=1)   # [N, N]
    pS = np.where(discarded, p, 0.0)
    pK = np.where(discarded, 0.0, p)
    S1 = pS.sum(axis=1, keepdims=True)
    # E = O - O' = sum_S p_j v_j - S1/(1-S1) sum_K p_j v_j   (Eq. 1)
    E = pS @ v - (S1 / (1.0 - S1)) * (pK @ v)
    np.testing.assert_allclose(o_dense - o_sparse, E, rtol=0, atol=1e-12)


# ---------------------------------------------------------------- P6: DYNAMIC skips a superset of FIXED
@pytest.mark.parametrize("lam", [-0.5, -1.0, -2.0, -3.0, -4.0, -6.0])
def test_p6_dynamic_superset_of_fixed(seed, lam):
    for name in ("cfg0", "cfg0_aligned"):
        qb, kb, vb = make_head(CONFIGS[name], seed, 1)
        dyn = oracle.run_head(qb, kb, vb, tile=64, lam=lam, mode=MODE_DYNAMIC)
        fix = oracle.run_head(qb, kb, vb, tile=64, lam=lam, mode=MODE_FIXED)
        assert np.all(dyn.skip >= fix.skip)
        assert dyn.sparsity >= fix.sparsity


# ---------------------------------------------------------------- P7: uniform closed form
@pytest.mark.parametrize("lam,kept", [(-6.0, 7), (-5.0, 3), (-7.5, 16)])
def test_p7_uniform_logits_closed_form(lam, kept):
    N, D, tile = 1024, 64, 64
    T = N // tile
    assert kept == min(T, int(math.floor(math.exp(-lam) / tile)) + 1)
    qb = np.zeros((N, D), dtype=np.uint16)                         # Q = 0: all logits equal
    rng = np.random.default_rng(3)
    kb = f32_to_bf16_bits(rng.standard_normal((N, D)).astype(np.float32))
    vb = f32_to_bf16_bits(rng.standard_normal((N, D)).astype(np.float32))
    dyn = oracle.run_head(qb, kb, vb, tile=tile, lam=lam, mode=MODE_DYNAMIC)
    expect = np.zeros((T, T), dtype=np.uint8)
    expect[:, kept:] = 1
    np.testing.assert_array_equal(dyn.skip, expect)
    fix = oracle.run_head(qb, kb, vb, tile=tile, lam=lam, mode=MODE_FIXED)
    assert fix.skipped == 0                                         # t = 0 is not < lambda
    # output: uniform average of V over the kept prefix; lse = ln(kept * tile)
    o, lse = dyn.rows()
    v = bf16_bits_to_f64(vb)
    np.testing.assert_allclose(o, np.broadcast_to(v[:kept * tile].mean(axis=0), o.shape), atol=1e-12)
    np.testing.assert_allclose(lse, math.log(kept * tile), atol=1e-12)


@pytest.mark.parametrize("lam", [-6.0, -5.0, -4.0, -8.0])
def test_p7_uniform_logits_rectangular_tiles(lam):
    """P7 with decision tiles of 128 rows x 32 keys ("block size 32"): with all logits
    equal, DYNAMIC keeps exactly floor(e^-lambda / 32) + 1 leading 32-key tiles.  A slip that takes T_c, the column
    offset or the tile width from tile_q instead of tile_k fails here."""
    N, D, tq, tk = 1024, 64, 128, 32
    T_r, T_c = N // tq, N // tk
    kept = min(T_c, int(math.floor(math.exp(-lam) / tk)) + 1)
    assert {-6.0: 13, -5.0: 5, -4.0: 2, -8.0: 32}[lam] == kept
    qb = np.zeros((N, D), dtype=np.uint16)
    rng = np.random.default_rng(5)
    kb = f32_to_bf16_bits(rng.standard_normal((N, D)).astype(np.float32))
    vb = f32_to_bf16_bits(rng.standard_normal((N, D)).astype(np.float32))
    dyn = oracle.run_head(qb, kb, vb, tile=tq, tile_k=tk, lam=lam, mode=MODE_DYNAMIC)
    assert dyn.skip.shape == (T_r, T_c)
    expect = np.zeros((T_r, T_c), dtype=np.uint8)
    expect[:, kept:] = 1
    np.testing.assert_array_equal(dyn.skip, expect)
    fix = oracle.run_head(qb, kb, vb, tile=tq, tile_k=tk, lam=lam, mode=MODE_FIXED)
    assert fix.skipped == 0
    o, lse = dyn.rows()
    v = bf16_bits_to_f64(vb)
    np.testing.assert_allclose(o, np.broadcast_to(v[:kept * tk].mean(axis=0), o.shape), atol=1e-12)
    np.testing.assert_allclose(lse, math.log(kept * tk), atol=1e-12)


def _winner_inputs(N, D, tile, winner_col, W):
    """Each row has logit W at column `winner_col` and 0 elsewhere (scale 1/sqrt(D))."""
    a = math.sqrt(W * math.sqrt(D))
    assert float(np.float32(a)) == a and bf16_bits_to_f64(f32_to_bf16_bits(np.float32([a])))[0] == a
    q = np.zeros((N, D), dtype=np.float32)
    k = np.zeros((N, D), dtype=np.float32)
    q[:, 0] = a
    k[winner_col, 0] = a
    rng = np.random.default_rng(4)
    v = rng.standard_normal((N, D)).astype(np.float32)
    return f32_to_bf16_bits(q), f32_to_bf16_bits(k), f32_to_bf16_bits(v)


# ---------------------------------------------------------------- P8: early winner
def test_p8_early_winner_skips_everything_after(seed):
    N, D, tile, lam, W = 1024, 64, 64, -6.0, 8.0
    T = N // tile
    qb, kb, vb = _winner_inputs(N, D, tile, winner_col=5, W=W)
    for mode in (MODE_DYNAMIC, MODE_FIXED):
        res = oracle.run_head(qb, kb, vb, tile=tile, lam=lam, mode=mode)
        expect = np.ones((T, T), dtype=np.uint8)
        expect[:, 0] = 0
        np.testing.assert_array_equal(res.skip, expect)
        assert res.sparsity == (T - 1) / T
        np.testing.assert_allclose(res.rows()[1], math.log(math.exp(W) + tile - 1), atol=1e-12)


# ---------------------------------------------------------------- P9: late winner (position dependence of BLASST)
def test_p9_late_winner():
    N, D, tile, lam, W = 1024, 64, 64, -6.0, 8.0
    T = N // tile
    qb, kb, vb = _winner_inputs(N, D, tile, winner_col=N - 3, W=W)
    fix = oracle.run_head(qb, kb, vb, tile=tile, lam=lam, mode=MODE_FIXED)
    assert fix.skipped == 0                                         # running max is 0 until the last tile
    dyn = oracle.run_head(qb, kb, vb, tile=tile, lam=lam, mode=MODE_DYNAMIC)
    kstar = int(math.floor(math.exp(-lam) / tile)) + 1              # 7 (P7)
    expect = np.zeros((T, T), dtype=np.uint8)
    expect[:, kstar:T - 1] = 1                                      # dilution tiles skipped, winner tile kept
    np.testing.assert_array_equal(dyn.skip, expect)
    np.testing.assert_allclose(dyn.rows()[1], math.log(kstar * tile + math.exp(W) + tile - 1), atol=1e-12)


@pytest.mark.parametrize("tq,tk", [(128, 32), (128, 64), (64, 16)])
def test_p8_p9_winner_rectangular_tiles(tq, tk):
    """P8 / P9 with tile_k != tile_q: the winner sits in the FIRST (col 5) or the LAST tile_k-wide decision tile."""
    N, D, lam, W = 1024, 64, -6.0, 8.0
    T_r, T_c = N // tq, N // tk
    kstar = int(math.floor(math.exp(-lam) / tk)) + 1
    # early winner: every decision tile after the first is skipped in both modes
    qb, kb, vb = _winner_inputs(N, D, tq, winner_col=5, W=W)
    for mode in (MODE_DYNAMIC, MODE_FIXED):
        res = oracle.run_head(qb, kb, vb, tile=tq, tile_k=tk, lam=lam, mode=mode)
        expect = np.ones((T_r, T_c), dtype=np.uint8)
        expect[:, 0] = 0
        np.testing.assert_array_equal(res.skip, expect)
        np.testing.assert_allclose(res.rows()[1], math.log(math.exp(W) + tk - 1), atol=1e-12)
    # late winner, in the last tile_k keys: FIXED skips nothing; DYNAMIC skips the dilution tiles, keeps the winner tile
    qb, kb, vb = _winner_inputs(N, D, tq, winner_col=N - 3, W=W)
    fix = oracle.run_head(qb, kb, vb, tile=tq, tile_k=tk, lam=lam, mode=MODE_FIXED)
    assert fix.skipped == 0
    dyn = oracle.run_head(qb, kb, vb, tile=tq, tile_k=tk, lam=lam, mode=MODE_DYNAMIC)
    expect = np.zeros((T_r, T_c), dtype=np.uint8)
    expect[:, kstar:T_c - 1] = 1
    np.testing.assert_array_equal(dyn.skip, expect)
    np.testing.assert_allclose(dyn.rows()[1], math.log(kstar * tk + math.exp(W) + tk - 1), atol=1e-12)


# ---------------------------------------------------------------- P10: brute force on tiny inputs
@pytest.mark.parametrize("N,D,tq,tk", [(330, 32, 128, 32), (200, 64, 128, 64), (150, 16, 64, 16), (257, 32, 128, 32)])
@pytest.mark.parametrize("mode", [MODE_DYNAMIC, MODE_FIXED])
def test_p10_brute_force_rectangular_tiles(N, D, tq, tk, mode, seed):
    """P10 with tile_k != tile_q (ragged N in both directions): the independent formulation takes its own tile_q /
    tile_k, so the streaming oracle's rectangular-tile regime (every 128 x 64 / 128 x 32 parity claim rests on it) is
    pinned like the square one."""
    rng = np.random.default_rng([seed, N, D, tq, tk, mode])
    qb, kb, vb = _rand_bits(rng, N, D, 1.8)
    q, k, v = (bf16_bits_to_f64(x) for x in (qb, kb, vb))
    T_r, T_c = -(-N // tq), -(-N // tk)
    probe = oracle.run_head(qb, kb, vb, tile=tq, tile_k=tk, lam=0.0, mode=mode, forced_skip=np.zeros((T_r, T_c), dtype=np.uint8))
    assert probe.skip.shape == (T_r, T_c)
    finite = probe.margin[np.isfinite(probe.margin)]
    n_skip_total = 0
    for lam in np.quantile(finite, [0.2, 0.5, 0.8]):
        lam = float(lam)
        res = oracle.run_head(qb, kb, vb, tile=tq, tile_k=tk, lam=lam, mode=mode)
        bf = oracle.brute_force_head(q, k, v, tile=tq, tile_k=tk, lam=lam, mode=mode)
        assert bf["skip"].shape == (T_r, T_c)
        safe = ~(np.abs(bf["margin"]) < 1e-9)
        np.testing.assert_array_equal(res.skip[safe], bf["skip"][safe])
        if np.array_equal(res.skip, bf["skip"]):
            o, lse = res.rows()
            np.testing.assert_allclose(o, bf["out"], rtol=0, atol=1e-11)
            np.testing.assert_allclose(lse, bf["lse"], rtol=0, atol=1e-11)
            fin = np.isfinite(bf["margin"])
            np.testing.assert_allclose(res.margin[fin], bf["margin"][fin], rtol=0, atol=1e-11)
        n_skip_total += res.skipped
    assert n_skip_total > 0


@pytest.mark.parametrize("N,D,tile", [(256, 64, 64), (200, 64, 64), (130, 32, 32), (384, 128, 128), (97, 16, 16)])
@pytest.mark.parametrize("mode", [MODE_DYNAMIC, MODE_FIXED])
def test_p10_brute_force_equals_streaming(N, D, tile, mode, seed):
    rng = np.random.default_rng([seed, N, D, tile, mode])
    qb, kb, vb = _rand_bits(rng, N, D, 1.8)
    q, k, v = (bf16_bits_to_f64(x) for x in (qb, kb, vb))
    # thresholds drawn near the typical margins of this input (so both outcomes occur)
    probe = oracle.run_head(qb, kb, vb, tile=tile, lam=0.0, mode=mode, forced_skip=np.zeros(
        (-(-N // tile), -(-N // tile)), dtype=np.uint8))
    finite = probe.margin[np.isfinite(probe.margin)]
    n_skip_total = 0
    for lam in np.quantile(finite, [0.2, 0.5, 0.8]) if finite.size else [-1.0]:
        lam = float(lam)
        res = oracle.run_head(qb, kb, vb, tile=tile, lam=lam, mode=mode)
        bf = oracle.brute_force_head(q, k, v, tile=tile, lam=lam, mode=mode)
        safe = ~(np.abs(bf["margin"]) < 1e-9)
        np.testing.assert_array_equal(res.skip[safe], bf["skip"][safe])
        if np.array_equal(res.skip, bf["skip"]):
            o, lse = res.rows()
            np.testing.assert_allclose(o, bf["out"], rtol=0, atol=1e-11)
            np.testing.assert_allclose(lse, bf["lse"], rtol=0, atol=1e-11)
            fin = np.isfinite(bf["margin"])
            np.testing.assert_allclose(res.margin[fin], bf["margin"][fin], rtol=0, atol=1e-11)
            assert np.array_equal(np.isfinite(res.margin), fin)
        n_skip_total += res.skipped
    assert n_skip_total > 0          # the skip path really ran


def test_p10_brute_force_on_cfg0(cfg0_head):
    qb, kb, vb = cfg0_head
    q, k, v = (bf16_bits_to_f64(x[:512]) for x in (qb, kb, vb))
    for mode in (MODE_DYNAMIC, MODE_FIXED):
        res = oracle.run_head(qb[:512], kb[:512], vb[:512], tile=64, lam=-2.0, mode=mode)
        bf = oracle.brute_force_head(q, k, v, tile=64, lam=-2.0, mode=mode)
        np.testing.assert_array_equal(res.skip, bf["skip"])
        np.testing.assert_allclose(res.rows()[0], bf["out"], atol=1e-11)


# ---------------------------------------------------------------- replay mode
def test_replay_reproduces_free_run_and_reports_margins(cfg0_head):
    qb, kb, vb = cfg0_head
    free = oracle.run_head(qb, kb, vb, tile=64, lam=-2.0, mode=MODE_DYNAMIC)
    rep = oracle.run_head(qb, kb, vb, tile=64, lam=-2.0, mode=MODE_DYNAMIC, forced_skip=free.skip)
    np.testing.assert_array_equal(rep.skip, free.skip)
    np.testing.assert_array_equal(rep.margin, free.margin)
    np.testing.assert_array_equal(rep.out, free.out)
    # forcing a different bitmap changes the state the later margins are evaluated from
    forced = free.skip.copy()
    forced[:, 1:] = 1
    rep2 = oracle.run_head(qb, kb, vb, tile=64, lam=-2.0, mode=MODE_DYNAMIC, forced_skip=forced)
    np.testing.assert_array_equal(rep2.skip, forced)
    # with only tile 0 kept the result is dense attention over the first 64 keys
    q, k, v = (bf16_bits_to_f64(x) for x in (qb, kb, vb))
    o_ref, lse_ref, _ = oracle.dense_attention_textbook(q, k[:64], v[:64], 1.0 / 8.0)
    np.testing.assert_allclose(rep2.rows()[0], o_ref, atol=1e-12)
    np.testing.assert_allclose(rep2.rows()[1], lse_ref, atol=1e-12)


def test_qtile_subset_matches_full_run(seed):
    qb, kb, vb = make_head(CONFIGS["cfg0"], seed, 1)
    qb, kb, vb = qb[:1000], kb[:1000], vb[:1000]                    # ragged: 1000 = 15*64 + 40
    full = oracle.run_head(qb, kb, vb, tile=64, lam=-2.0, mode=MODE_DYNAMIC)
    sub = oracle.run_head(qb, kb, vb, tile=64, lam=-2.0, mode=MODE_DYNAMIC, qtiles=[15, 0, 7])
    for t, i in enumerate([15, 0, 7]):
        np.testing.assert_array_equal(sub.skip[t], full.skip[i])
        np.testing.assert_array_equal(sub.out[t], full.out[i])
    assert np.all(full.out[15, 40:] == 0.0)                         # rows beyond N never written


# ---------------------------------------------------------------- P11: values the paper prints
def test_p11_paper_printed_values():
    g = _golden()
    from workloads import num_tiles
    assert num_tiles(27280, 128) == g["n_blk_27280_128"]
    lam = oracle.lambda_from_preal(g["p_real_transition"], 128, 75600)
    assert abs(lam - g["lambda_14b"]) < 0.03                        # ln(1.5) + ln(128/75600) = -5.976
    assert abs(oracle.lambda_from_preal(1.0, 128, 75600) - math.log(128 / 75600)) < 1e-15
    assert abs(oracle.lambda_from_recall(0.9, 1024) - (-9.2341)) < 1e-3
    # section 2.3 closed form (off-path sanity): std/delta = sqrt((N-K)/(N-1))/sqrt(K), N = 214 blocks
    for keep, key in ((0.80, "std_frac_keep80"), (0.95, "std_frac_keep95")):
        K = round(keep * 214)
        frac = math.sqrt((214 - K) / (214 - 1)) / math.sqrt(K)
        assert abs(frac - g[key]) < 6e-4
