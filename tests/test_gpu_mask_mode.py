"""MASK mode (first part): the kernel driven by a precomputed block bitmap, against the oracle's
replay of the same bitmap (oracle/dynsparse_oracle.c `forced_skip`)."""
import math

import numpy as np
import pytest
import torch

import oracle
import paper_2606_16317_b200 as sa
from workloads import CONFIGS, bf16_bits_to_f64, f32_to_bf16_bits, make_qkv

pytestmark = pytest.mark.gpu


def _run_mask(qb, kb, vb, bitmap, tile, lam=-3.0):
    B, H, N, D = qb.shape
    q, k, v = (torch.from_numpy(np.ascontiguousarray(x).view(np.int16)).cuda().view(torch.bfloat16) for x in (qb, kb, vb))
    out = torch.full_like(q, float("nan"))
    lse = torch.full((B, H, N), float("nan"), device="cuda", dtype=torch.float32)
    stats = torch.full((B, H, 2), -1, device="cuda", dtype=torch.int64)
    T = -(-N // tile)
    dmask = torch.from_numpy(np.ascontiguousarray(bitmap, dtype=np.uint8)).cuda()
    echo = torch.full((B, H, T, T), 255, device="cuda", dtype=torch.uint8)
    margin = torch.full((B, H, T, T), float("nan"), device="cuda", dtype=torch.float32)
    p = sa.make_params(lam=lam, skip_mask_in=dmask, skip_mask_out=echo, margin_out=margin)
    sa.sparse_attn_fwd(q, k, v, out, lse, B, H, N, D, p, sa.MODE_MASK, stats)
    torch.cuda.synchronize()
    o = bf16_bits_to_f64(out.view(torch.int16).cpu().numpy().view(np.uint16))
    return o, lse.cpu().numpy(), stats.cpu().numpy(), echo.cpu().numpy(), margin.cpu().numpy()


@pytest.mark.parametrize("N,D", [(1024, 64), (1000, 128), (2125, 128), (193, 64), (64, 64)])
def test_mask_mode_matches_oracle_replay(seed, N, D):
    rng = np.random.default_rng([seed, N, D])
    B, H = 1, 2
    tile = 64 if D == 64 else 128
    T = -(-N // tile)
    qb, kb, vb = (f32_to_bf16_bits(rng.standard_normal((B, H, N, D), dtype=np.float32)) for _ in range(3))
    for density in (0.0, 0.3, 0.8, 1.0):
        bitmap = (rng.random((B, H, T, T)) < density).astype(np.uint8)
        want = bitmap.copy()
        want[..., 0] = 0                                       # tile 0 is retained whatever its byte says
        lam = -3.0
        o, lse, stats, echo, margin = _run_mask(qb, kb, vb, bitmap, tile, lam)
        assert np.array_equal(echo, want)
        for h in range(H):
            assert (int(stats[0, h, 0]), int(stats[0, h, 1])) == (int((want[0, h] == 0).sum()), int(want[0, h].sum()))
            ref = oracle.run_head(qb[0, h], kb[0, h], vb[0, h], tile=tile, lam=lam, mode=oracle.MODE_DYNAMIC,
                                  forced_skip=want[0, h])
            ro, rl = ref.rows()
            assert np.abs(o[0, h] - ro).max() < 2e-2 and np.abs(o[0, h] - ro).mean() < 2e-3
            assert np.abs(lse[0, h] - rl).max() < 2e-3
            fin = np.isfinite(ref.margin)
            assert np.array_equal(np.isfinite(margin[0, h]), fin)
            if fin.any():
                assert np.abs(margin[0, h][fin] - ref.margin[fin]).max() < 1e-3


def test_mask_mode_reproduces_dynamic_mode_bit_for_bit(seed):
    """Feeding DYNAMIC mode's own decisions back as a mask gives the same bits: same tiles, same arithmetic."""
    cfg = CONFIGS["cfg0_aligned"]
    qb, kb, vb = make_qkv(cfg, seed)
    q, k, v = (torch.from_numpy(x.view(np.int16)).cuda().view(torch.bfloat16) for x in (qb, kb, vb))
    B, H, N, D = cfg.B, cfg.H, cfg.N, cfg.D
    T = N // cfg.tile
    out1, out2 = torch.empty_like(q), torch.empty_like(q)
    lse1 = torch.empty((B, H, N), device="cuda", dtype=torch.float32)
    lse2 = torch.empty_like(lse1)
    st1 = torch.zeros((B, H, 2), device="cuda", dtype=torch.int64)
    st2 = torch.zeros_like(st1)
    mask = torch.zeros((B, H, T, T), device="cuda", dtype=torch.uint8)
    sa.sparse_attn_fwd(q, k, v, out1, lse1, B, H, N, D, sa.make_params(lam=-2.0, skip_mask_out=mask), sa.MODE_DYNAMIC, st1)
    sa.sparse_attn_fwd(q, k, v, out2, lse2, B, H, N, D, sa.make_params(lam=-2.0, skip_mask_in=mask), sa.MODE_MASK, st2)
    torch.cuda.synchronize()
    assert int(st1[..., 1].sum()) > 0
    assert torch.equal(st1, st2) and torch.equal(out1.view(torch.int16), out2.view(torch.int16)) and torch.equal(lse1, lse2)


def test_mask_mode_through_the_host_buffer_entry(seed):
    """sparse_attn_fwd_host copies the bitmap to the device itself: same result as the device entry."""
    rng = np.random.default_rng([seed, 77])
    B, H, N, D, tile = 1, 2, 700, 128, 128
    T = -(-N // tile)
    qb, kb, vb = (f32_to_bf16_bits(rng.standard_normal((B, H, N, D), dtype=np.float32)) for _ in range(3))
    bitmap = (rng.random((B, H, T, T)) < 0.5).astype(np.uint8)
    o_dev, lse_dev, st_dev, _, _ = _run_mask(qb, kb, vb, bitmap, tile)
    out = np.zeros((B, H, N, D), dtype=np.uint16)
    lse = np.zeros((B, H, N), dtype=np.float32)
    stats = np.zeros((B, H, 2), dtype=np.int64)
    p = sa.make_params(lam=-3.0, skip_mask_in=bitmap)
    sa.sparse_attn_fwd_host(qb, kb, vb, out, lse, B, H, N, D, p, sa.MODE_MASK, stats)
    assert np.array_equal(stats, st_dev)
    assert np.array_equal(bf16_bits_to_f64(out), o_dev) and np.array_equal(lse, lse_dev)
