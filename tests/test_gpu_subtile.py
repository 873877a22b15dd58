"""GPU parity for decision tiles narrower than the MMA tile (block size 32):
128 x 64 and 128 x 32 decision tiles at D = 128, against the oracle run with tile_q = 128, tile_k = 64 / 32."""
import math

import numpy as np
import pytest

import oracle
from oracle import MODE_DYNAMIC, MODE_FIXED
from workloads import CONFIGS, f32_to_bf16_bits, make_qkv
from dataclasses import replace

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def parity():
    import torch
    if not torch.cuda.is_available():
        pytest.fail("GPU tests need a CUDA device; there is no CPU fallback")
    import parity_utils
    return parity_utils


def _small_cfg(aligned, grid=(4, 16, 16)):
    # config 0's grid and generator with D = 128 (the narrow decision tiles exist for D = 128 only)
    return replace(CONFIGS["cfg0"], name="cfg0_d128", D=128, tile=128, grid=grid, aligned=aligned)


@pytest.mark.parametrize("tile_k", [32, 64])
@pytest.mark.parametrize("aligned", [False, True])
def test_subtile_decisions_match_oracle(parity, seed, tile_k, aligned):
    cfg = _small_cfg(aligned)
    qb, kb, vb = make_qkv(cfg, seed)
    for mode in (MODE_FIXED, MODE_DYNAMIC):
        for lam in (-1.0, -2.0, -3.0, -4.0, -6.0):
            gpu = parity.run_gpu(qb, kb, vb, mode=mode, lam=lam, tile=128, tile_k=tile_k)
            parity.check_stats(gpu, cfg.N, 128, tile_k)
            rep = parity.ParityReport()
            for h in range(cfg.H):
                parity.compare_head(gpu, h, qb[0, h], kb[0, h], vb[0, h], tile=128, tile_k=tile_k, mode=mode, lam=lam,
                                    report=rep)
            # the timed (non-debug) build settles sub-tiles by a preliminary round, a certain-keep bound and lazy
            # statistics: its counts must equal the oracle's and its output must be within the same tolerance
            plain = parity.run_gpu(qb, kb, vb, mode=mode, lam=lam, tile=128, tile_k=tile_k, debug=False)
            for h in range(cfg.H):
                ref = oracle.run_head(qb[0, h], kb[0, h], vb[0, h], tile=128, tile_k=tile_k, lam=lam, mode=mode)
                assert (int(plain.stats[h, 0]), int(plain.stats[h, 1])) == (ref.executed, ref.skipped)
                err = np.abs(plain.out[h] - ref.rows()[0])
                assert err.max() < parity.OUT_MAX_ABS and err.mean() < parity.OUT_MEAN_ABS
                assert np.abs(plain.lse[h] - ref.rows()[1]).max() < parity.LSE_ABS
            print(f"[subtile] tile_k={tile_k} aligned={aligned} mode={mode} lam={lam}: sparsity "
                  f"{gpu.stats[:, 1].sum() / gpu.stats.sum():.3f} disagree={rep.disagreements} max-abs={rep.max_abs:.2e}")
            assert rep.ok(), "\n".join(rep.failures[:10])


@pytest.mark.parametrize("N,tile_k", [(1000, 32), (2125, 32), (193, 64), (129, 32), (97, 32), (33, 64), (4000, 64)])
def test_subtile_ragged_random_inputs(parity, seed, N, tile_k):
    rng = np.random.default_rng([seed, N, tile_k])
    B, H, D = 1, 2, 128
    q = rng.standard_normal((B, H, N, D), dtype=np.float32) * 1.3
    k = rng.standard_normal((B, H, N, D), dtype=np.float32) * 1.3
    k[:, :, : N // 3] *= 1.6                               # a heavier head of the sequence so that later tiles get skipped
    v = rng.standard_normal((B, H, N, D), dtype=np.float32)
    qb, kb, vb = (f32_to_bf16_bits(x) for x in (q, k, v))
    for mode, lam in ((MODE_DYNAMIC, -3.0), (MODE_DYNAMIC, -6.0), (MODE_FIXED, -2.0)):
        gpu = parity.run_gpu(qb, kb, vb, mode=mode, lam=lam, tile=128, tile_k=tile_k)
        parity.check_stats(gpu, N, 128, tile_k)
        rep = parity.ParityReport()
        for h in range(H):
            parity.compare_head(gpu, h, qb[0, h], kb[0, h], vb[0, h], tile=128, tile_k=tile_k, mode=mode, lam=lam, report=rep)
        assert rep.ok(), "\n".join(rep.failures[:10])


def test_subtile_at_bench_shape_sampled(parity, seed):
    """Config 1's shape (one head) in the launch configuration of the timed runs (no debug outputs for the stats run),
    oracle on sampled Q tiles: first, ragged last, two random."""
    cfg = CONFIGS["cfg1_aligned"]
    qb, kb, vb = make_qkv(cfg, seed, heads=[3])
    lam = math.log(1.5) + math.log(32 / cfg.N)              # Eq. 7 with B_c = 32
    plain = parity.run_gpu(qb, kb, vb, mode=MODE_DYNAMIC, lam=lam, tile=128, tile_k=32, debug=False)
    gpu = parity.run_gpu(qb, kb, vb, mode=MODE_DYNAMIC, lam=lam, tile=128, tile_k=32)
    # the debug and the plain build share the decision and statistics path: bit for bit the same
    np.testing.assert_array_equal(plain.stats, gpu.stats)
    np.testing.assert_array_equal(plain.out, gpu.out)
    np.testing.assert_array_equal(plain.lse, gpu.lse)
    parity.check_stats(gpu, cfg.N, 128, 32)
    rep = parity.ParityReport()
    parity.compare_head(gpu, 0, qb[0, 0], kb[0, 0], vb[0, 0], tile=128, tile_k=32, mode=MODE_DYNAMIC, lam=lam,
                        qtiles=[0, 255, 77, 190], report=rep)
    print(f"[subtile] cfg1_aligned head 3: sparsity {gpu.stats[:, 1].sum() / gpu.stats.sum():.3f}")
    assert rep.ok(), "\n".join(rep.failures[:10])


def test_subtile_rejected_where_unsupported():
    import torch
    import paper_2606_16317_b200 as sa
    q = torch.zeros((1, 1, 256, 64), device="cuda", dtype=torch.bfloat16)
    out = torch.empty_like(q)
    with pytest.raises(sa.SparseAttnError) as e:           # D = 64 has 64 x 64 decision tiles only
        sa.sparse_attn_fwd(q, q, q, out, None, 1, 1, 256, 64, sa.make_params(lam=-3.0, tile_q=64, tile_k=32),
                           sa.MODE_DYNAMIC, None)
    assert e.value.status == -4
    q = torch.zeros((1, 1, 256, 128), device="cuda", dtype=torch.bfloat16)
    out = torch.empty_like(q)
    with pytest.raises(sa.SparseAttnError) as e:           # DENSE mode takes no decisions
        sa.sparse_attn_fwd(q, q, q, out, None, 1, 1, 256, 128, sa.make_params(tile_q=128, tile_k=32), sa.MODE_DENSE, None)
    assert e.value.status == -4


@pytest.mark.parametrize("tile_k", [32, 64])
@pytest.mark.parametrize("mode", [MODE_DYNAMIC, MODE_FIXED])
def test_subtile_decisions_that_depend_on_earlier_subtiles(parity, tile_k, mode):
    """Inputs built so that, inside ONE 128-key MMA tile, the fate of a sub-tile depends on which earlier sub-tiles were
    retained (Eq. 6 is sequential): every key of a sub-tile carries the same logit level, levels drawn so that most
    sub-tiles pass the test against the statistics before the MMA tile and are then decided by the levels ahead of them
    (the hypothesis bits of the kernel's second vote round).  Rows fall into four groups with shifted levels, one group per
    warp, so the all-rows vote crosses warps.  Decisions, counts and outputs against the oracle."""
    rng = np.random.default_rng([7, tile_k, mode])
    D, N, S = 128, 1024 + 77, tile_k
    n_sub = -(-N // S)
    e0 = np.zeros(D, dtype=np.float32)
    e0[0] = 1.0
    worked = 0
    for trial in range(6):
        level = rng.uniform(0.0, 6.0, size=n_sub).astype(np.float32)          # logit level of every sub-tile
        level[:: 128 // S] += rng.uniform(0.0, 3.0, size=len(level[:: 128 // S])).astype(np.float32)   # a strong first sub-tile
        shift = np.repeat(rng.uniform(0.6, 1.0, size=4), 32)                      # four row groups (one per warp of a Q tile)
        q = np.zeros((N, D), dtype=np.float32)
        q[:, 0] = math.sqrt(D) * np.tile(shift, -(-N // 128))[:N]                 # logit(r, c) = shift_r * level_c (+ noise)
        k = np.zeros((N, D), dtype=np.float32)
        k[:, 0] = np.repeat(level, S)[:N]
        k[:, 1:] = 0.02 * rng.standard_normal((N, D - 1)).astype(np.float32)
        q[:, 1:] = 0.02 * rng.standard_normal((N, D - 1)).astype(np.float32)
        v = rng.standard_normal((N, D)).astype(np.float32)
        qb, kb, vb = (f32_to_bf16_bits(x)[None, None] for x in (q, k, v))
        for lam in (-1.0, -2.5):
            gpu = parity.run_gpu(qb, kb, vb, mode=mode, lam=lam, tile=128, tile_k=tile_k)
            parity.check_stats(gpu, N, 128, tile_k)
            rep = parity.compare_head(gpu, 0, qb[0, 0], kb[0, 0], vb[0, 0], tile=128, tile_k=tile_k, mode=mode, lam=lam)
            assert rep.ok(), "\n".join(rep.failures[:10])
            plain = parity.run_gpu(qb, kb, vb, mode=mode, lam=lam, tile=128, tile_k=tile_k, debug=False)
            np.testing.assert_array_equal(plain.stats, gpu.stats)
            np.testing.assert_array_equal(plain.out, gpu.out)
            np.testing.assert_array_equal(plain.lse, gpu.lse)
            # the case is only interesting if sub-tiles are skipped INSIDE retained MMA tiles
            sk = gpu.skip[0].reshape(gpu.skip.shape[1], -1)
            per_mma = sk[:, : (sk.shape[1] // (128 // S)) * (128 // S)].reshape(sk.shape[0], -1, 128 // S)
            worked += int(((per_mma.sum(-1) > 0) & (per_mma.sum(-1) < 128 // S)).sum())
    assert worked > 20, worked


def test_subtile_logits_that_leave_the_fp32_range_inside_one_mma_tile(parity):
    """Random-walk Q / K with logits of several hundred nats: rows whose logits rise by more than 126 log2 units above their
    running LSE inside ONE 128-key MMA tile.  Sums relative to the tile's row max underflow there; the kernel's references
    for such rows come from per-sub-tile log-sums instead.  Decisions and margins against the oracle (a soak run found the
    case as margins off by 0.4 - 3.8 nats before that branch existed)."""
    N, D, H, gain, lam = 1423, 128, 3, 2.9630839477090753, -5.9537085225695545
    rng = np.random.default_rng(793270137)
    q = rng.standard_normal((1, H, N, D), dtype=np.float32) * gain
    k = rng.standard_normal((1, H, N, D), dtype=np.float32)
    base = np.cumsum(rng.standard_normal((1, H, N, D), dtype=np.float32), axis=2) / 8.0
    q = (base + 0.3 * q) * gain
    k = base + 0.3 * k
    v = rng.standard_normal((1, H, N, D), dtype=np.float32)
    qb, kb, vb = (f32_to_bf16_bits(x) for x in (q, k, v))
    for tile_k in (32, 64):
        gpu = parity.run_gpu(qb, kb, vb, mode=MODE_DYNAMIC, lam=lam, tile=128, tile_k=tile_k)
        parity.check_stats(gpu, N, 128, tile_k)
        rep = parity.ParityReport()
        for h in range(H):
            parity.compare_head(gpu, h, qb[0, h], kb[0, h], vb[0, h], tile=128, tile_k=tile_k, mode=MODE_DYNAMIC, lam=lam,
                                report=rep)
        assert rep.ok(), "\n".join(rep.failures[:10])
        assert rep.max_margin_abs < 1e-3
