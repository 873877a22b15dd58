"""Thresholds at the edge of what the ABI accepts (include/sparse_attn.h: lambda > 0 is allowed in DYNAMIC mode with the
default decision tiles; FIXED takes lambda <= 0, including 0 and -inf), against the oracle on the GPU.

With lambda > 0 the rule of Eq. 5 may skip a tile whose row maxima lie ABOVE the running log-sum-exp:
the skipped tile must leave m, l and O untouched (Eq. 6) even though its maximum exceeds the stabiliser the kernel holds,
and a later retained tile then raises the maximum by more than any tile before it.  P7 of SURVEY.md 8(c) (uniform logits)
has a closed form here too: only tile 0 of every row of tiles survives."""
import math

import numpy as np
import pytest

from oracle import MODE_DENSE, MODE_DYNAMIC, MODE_FIXED
from workloads import bf16_bits_to_f64, f32_to_bf16_bits

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def parity():
    import torch
    if not torch.cuda.is_available():
        pytest.fail("GPU tests need a CUDA device; there is no CPU fallback")
    import parity_utils
    return parity_utils


def _check(parity, qb, kb, vb, mode, lam, tile):
    H, N = qb.shape[1], qb.shape[2]
    gpu = parity.run_gpu(qb, kb, vb, mode=mode, lam=lam, tile=tile)
    parity.check_stats(gpu, N, tile)
    rep = parity.ParityReport()
    for h in range(H):
        parity.compare_head(gpu, h, qb[0, h], kb[0, h], vb[0, h], tile=tile, mode=mode, lam=lam, report=rep)
    assert rep.ok(), "\n".join(rep.failures[:10])
    plain = parity.run_gpu(qb, kb, vb, mode=mode, lam=lam, tile=tile, debug=False)      # the timed instantiation
    np.testing.assert_array_equal(plain.out, gpu.out)
    np.testing.assert_array_equal(plain.lse, gpu.lse)
    np.testing.assert_array_equal(plain.stats, gpu.stats)
    return gpu, rep


@pytest.mark.parametrize("D,N", [(128, 1000), (64, 777), (128, 2125)])
@pytest.mark.parametrize("lam", [0.0, 0.5, 2.0])
def test_dynamic_mode_with_non_negative_lambda_on_random_inputs(parity, D, N, lam):
    rng = np.random.default_rng([51, D, N])
    H = 2
    gains = np.array([1.0, 3.5], dtype=np.float32).reshape(1, H, 1, 1)       # a flat head and a peaked one
    q = rng.standard_normal((1, H, N, D), dtype=np.float32) * gains
    k = rng.standard_normal((1, H, N, D), dtype=np.float32)
    v = rng.standard_normal((1, H, N, D), dtype=np.float32)
    qb, kb, vb = (f32_to_bf16_bits(x) for x in (q, k, v))
    gpu, rep = _check(parity, qb, kb, vb, MODE_DYNAMIC, lam, 64 if D == 64 else 128)
    frac = gpu.stats[:, 1].sum() / gpu.stats.sum()
    assert frac > 0.3, frac                                                   # a non-negative threshold prunes hard
    print(f"[lambda={lam}] sparsity {frac:.3f}, out max-abs {rep.max_abs:.2e}, lse max-abs {rep.max_lse_abs:.2e}")


@pytest.mark.parametrize("D", [64, 128])
@pytest.mark.parametrize("lam", [0.0, 0.5, 2.0])
def test_p7_uniform_logits_with_non_negative_lambda_keeps_tile_0_only(parity, D, lam):
    """K = 0: every logit is 0, LSE after tile 0 is ln(B_c), so t = -ln(B_c) < 0 <= lambda for every later tile."""
    tile = 64 if D == 64 else 128
    N = 5 * tile + 17
    rng = np.random.default_rng([52, D])
    qb = f32_to_bf16_bits(rng.standard_normal((1, 1, N, D), dtype=np.float32))
    kb = np.zeros((1, 1, N, D), dtype=np.uint16)
    vb = f32_to_bf16_bits(rng.standard_normal((1, 1, N, D), dtype=np.float32))
    gpu, _ = _check(parity, qb, kb, vb, MODE_DYNAMIC, lam, tile)
    T = -(-N // tile)
    expect = np.ones((T, T), dtype=np.uint8)
    expect[:, 0] = 0
    np.testing.assert_array_equal(gpu.skip[0], expect)
    assert np.allclose(gpu.lse[0], math.log(tile), atol=1e-5)
    mean_v = bf16_bits_to_f64(vb[0, 0, :tile]).mean(axis=0)
    assert np.abs(gpu.out[0] - mean_v[None, :]).max() < 5e-3


@pytest.mark.parametrize("D", [64, 128])
def test_a_tile_above_the_running_lse_is_skipped_and_a_later_one_raises_the_maximum(parity, D):
    """Logits by construction (q = a e_0, k_c = b_c e_0): 0 everywhere except tile 3 (LSE + 1) and tile 5 (LSE + 9), with
    LSE = ln(B_c) from tile 0.  lambda = 2 skips tile 3 although its logits exceed every retained one, keeps tile 5;
    lambda = 0.5 keeps both (tile 5 then exceeds the LSE that includes tile 3 by about 3)."""
    tile = 64 if D == 64 else 128
    N = 7 * tile
    scale = 1.0 / math.sqrt(D)
    a = 8.0
    q = np.zeros((1, 1, N, D), dtype=np.float32)
    q[..., 0] = a
    k = np.zeros((1, 1, N, D), dtype=np.float32)
    lse0 = math.log(tile)
    k[0, 0, 3 * tile:4 * tile, 0] = (lse0 + 1.0) / (a * scale)
    k[0, 0, 5 * tile:6 * tile, 0] = (lse0 + 9.0) / (a * scale)
    rng = np.random.default_rng([53, D])
    v = rng.standard_normal((1, 1, N, D), dtype=np.float32)
    qb, kb, vb = (f32_to_bf16_bits(x) for x in (q, k, v))
    for lam, kept in ((2.0, [0, 5]), (0.5, [0, 3, 5])):
        gpu, _ = _check(parity, qb, kb, vb, MODE_DYNAMIC, lam, tile)
        expect = np.ones(7, dtype=np.uint8)
        expect[kept] = 0
        for i in range(7):
            np.testing.assert_array_equal(gpu.skip[0, i], expect, err_msg=f"lambda {lam}, Q tile {i}")


@pytest.mark.parametrize("D,N", [(128, 1000), (64, 500)])
def test_fixed_mode_at_lambda_zero_and_minus_infinity(parity, D, N):
    """FIXED: lambda = 0 skips exactly the tiles whose maximum lies strictly below the running maximum in
    every row; lambda = -inf skips nothing and must reproduce DENSE bit for bit."""
    rng = np.random.default_rng([54, D, N])
    q = rng.standard_normal((1, 2, N, D), dtype=np.float32) * 2.0
    k = rng.standard_normal((1, 2, N, D), dtype=np.float32)
    v = rng.standard_normal((1, 2, N, D), dtype=np.float32)
    qb, kb, vb = (f32_to_bf16_bits(x) for x in (q, k, v))
    tile = 64 if D == 64 else 128
    _check(parity, qb, kb, vb, MODE_FIXED, 0.0, tile)
    none, _ = _check(parity, qb, kb, vb, MODE_FIXED, -math.inf, tile)
    assert none.stats[:, 1].sum() == 0
    dense = parity.run_gpu(qb, kb, vb, mode=MODE_DENSE, tile=tile, debug=False)
    np.testing.assert_array_equal(none.out, dense.out)
    np.testing.assert_array_equal(none.lse, dense.lse)
