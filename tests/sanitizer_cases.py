#!/usr/bin/env python
"""Small invocations of every kernel instantiation for compute-sanitizer:

    compute-sanitizer --tool memcheck|racecheck|synccheck python tests/sanitizer_cases.py

Config 0 (D = 64 kernels) in all modes, a ragged D = 128 case with 128x128 / 128x64 / 128x32 decision tiles with and
without the parity outputs, MASK mode, block stats, the selectors, token re-ordering and the quality reductions.  Results
are checked for finiteness and count consistency only (parity is tests/test_gpu_*.py's job); the summaries kept under
profiles/ are the sanitizer's own.
"""
import math
import os
import sys

import numpy as np
import torch

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)
import paper_2606_16317_b200 as sa  # noqa: E402
from workloads import CONFIGS, f32_to_bf16_bits, make_qkv  # noqa: E402


def dev(bits):
    return torch.from_numpy(np.ascontiguousarray(bits).view(np.int16)).cuda().view(torch.bfloat16)


def run(q, k, v, mode, lam, tile, tile_k=0, debug=False, mask_in=None):
    B, H, N, D = q.shape
    out = torch.empty_like(q)
    lse = torch.empty((B, H, N), device="cuda", dtype=torch.float32)
    stats = torch.zeros((B, H, 2), device="cuda", dtype=torch.int64)
    T, Tc = -(-N // tile), -(-N // (tile_k or tile))
    mask = torch.zeros((B, H, T, Tc), device="cuda", dtype=torch.uint8) if debug else None
    margin = torch.zeros((B, H, T, Tc), device="cuda", dtype=torch.float32) if debug else None
    p = sa.make_params(lam=lam, tile_q=tile if tile_k else 0, tile_k=tile_k, skip_mask_out=mask, margin_out=margin,
                       skip_mask_in=mask_in)
    sa.sparse_attn_fwd(q, k, v, out, lse, B, H, N, D, p, mode, stats)
    torch.cuda.synchronize()
    assert torch.isfinite(out.float()).all() and torch.isfinite(lse).all()
    assert int(stats.sum()) == B * H * T * Tc
    return out, lse, stats, mask


def main():
    torch.cuda.set_device(0)
    n = 0
    cfg = CONFIGS["cfg0_aligned"]
    q, k, v = (dev(x) for x in make_qkv(cfg, 20261104))
    for mode, lam in ((sa.MODE_DENSE, -math.inf), (sa.MODE_FIXED, -3.0), (sa.MODE_DYNAMIC, -3.0), (sa.MODE_DYNAMIC, -6.0)):
        for debug in (False, True):
            run(q, k, v, mode, lam, cfg.tile, debug=debug)
            n += 1
    rng = np.random.default_rng(7)
    N, D = 700, 128                                       # ragged: 5 full tiles + 60 rows
    base = rng.standard_normal((1, 1, N, D)).astype(np.float32)
    q2 = dev(f32_to_bf16_bits(base * 1.5 + 0.3 * rng.standard_normal((1, 1, N, D)).astype(np.float32)))
    k2 = dev(f32_to_bf16_bits(base * 1.5 + 0.3 * rng.standard_normal((1, 1, N, D)).astype(np.float32)))
    v2 = dev(f32_to_bf16_bits(rng.standard_normal((1, 1, N, D)).astype(np.float32)))
    skipped = 0
    for tile_k in (0, 64, 32):
        for mode, lam in ((sa.MODE_DENSE, -math.inf), (sa.MODE_FIXED, -4.0), (sa.MODE_DYNAMIC, -4.0), (sa.MODE_DYNAMIC, -1.0)):
            if mode == sa.MODE_DENSE and tile_k:
                continue
            for debug in (False, True):
                _, _, st, mask = run(q2, k2, v2, mode, lam, 128, tile_k=tile_k, debug=debug)
                skipped += int(st[..., 1].sum())
                n += 1
    assert skipped > 0
    _, lse_d, _, _ = run(q2, k2, v2, sa.MODE_DENSE, -math.inf, 128)
    _, lse_s, _, mask = run(q2, k2, v2, sa.MODE_DYNAMIC, -2.0, 128, debug=True)
    run(q2, k2, v2, sa.MODE_MASK, 0.0, 128, mask_in=mask)
    T = -(-N // 128)
    mass = torch.empty((1, 1, T, T), device="cuda", dtype=torch.float32)
    sq = torch.empty_like(mass)
    bitmap = torch.empty((1, 1, T, T), device="cuda", dtype=torch.uint8)
    sa.sparse_attn_block_stats(q2, k2, lse_d, mass, sq, 1, 1, N, D)
    sa.sparse_attn_block_mass(q2, k2, lse_d, mass, 1, 1, N, D)
    sa.sparse_attn_select_blocks(mass, bitmap, 1, 1, T, T, sa.SELECT_TOPK, 0.5)
    sa.sparse_attn_select_blocks(mass, bitmap, 1, 1, T, T, sa.SELECT_TOPP, 0.9)
    sa.sparse_attn_select_blocks_greedy(mass, sq, bitmap, 1, 1, N, 128, T, 1e-3)
    rs = torch.zeros(2, device="cuda", dtype=torch.float64)
    sa.sparse_attn_recall_stats(lse_s, lse_d, N, rs)
    sa.sparse_attn_output_error(q2, k2, N * D, rs)
    perm = np.empty(cfg.N, dtype=np.int32)
    sa.sparse_attn_brick_permutation(*cfg.grid, 2, 4, 8, perm)
    dst = torch.empty_like(q)
    sa.sparse_attn_reorder_tokens(q, dst, cfg.B, cfg.H, cfg.N, cfg.D, torch.from_numpy(perm).cuda(), 0)
    torch.cuda.synchronize()
    assert torch.isfinite(mass).all() and torch.isfinite(sq).all()
    print(f"sanitizer_cases: {n + 12} launches OK")


if __name__ == "__main__":
    main()
