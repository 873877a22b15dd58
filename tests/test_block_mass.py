"""Block mass of the dense probabilities (first half of the offline selectors).
CPU: pins of the oracle.  GPU: sparse_attn_block_mass against the oracle."""
import numpy as np
import pytest
import torch

import oracle
import paper_2606_16317_b200 as sa
from workloads import CONFIGS, bf16_bits_to_f64, f32_to_bf16_bits, make_qkv


def test_oracle_block_mass_rows_sum_to_tile_rows_and_match_textbook():
    rng = np.random.default_rng(5)
    N, D, tile = 200, 16, 64
    q, k = rng.standard_normal((N, D)), rng.standard_normal((N, D))
    m = oracle.block_mass(q, k, tile)
    rows = np.array([64, 64, 64, 8])
    assert np.allclose(m.sum(axis=1), rows, atol=1e-9)          # probabilities of each row sum to one
    # one tile against the probabilities of torch's softmax (library routine)
    p = torch.softmax(torch.from_numpy(q @ k.T / 4.0), dim=1).numpy()
    assert abs(m[1, 2] - p[64:128, 128:192].sum()) < 1e-9
    # uniform logits: mass proportional to the tile's share of the keys
    mu = oracle.block_mass(np.zeros((N, D)), k, tile)
    assert np.allclose(mu[0], 64 * np.array([64, 64, 64, 8]) / 200)


def test_oracle_selectors_closed_forms():
    mass = np.array([[5.0, 1.0, 3.0, 1.0], [0.1, 0.1, 0.1, 9.7]])
    assert oracle.select_topk(mass, 0.5).tolist() == [[0, 1, 0, 1], [0, 1, 1, 0]]   # tile 0 always kept; ties -> low index
    assert oracle.select_topp(mass, 0.8).tolist() == [[0, 1, 0, 1], [0, 1, 1, 0]]   # 5 + 3 = 8 of 10; 9.7 of 10 (+ tile 0)
    assert oracle.select_topp(mass, 1.0).sum() == 0 and oracle.select_topk(mass, 1.0).sum() == 0


@pytest.mark.gpu
@pytest.mark.parametrize("name,N", [("cfg0_aligned", None), ("d128", 1000), ("d128", 193), ("d64", 700)])
def test_gpu_block_mass_matches_oracle(seed, name, N):
    if name == "cfg0_aligned":
        cfg = CONFIGS[name]
        qb, kb, vb = make_qkv(cfg, seed)
        B, H, N, D, tile = cfg.B, cfg.H, cfg.N, cfg.D, cfg.tile
    else:
        D, tile = (128, 128) if name == "d128" else (64, 64)
        B, H = 1, 2
        rng = np.random.default_rng([seed, N, D])
        qb, kb, vb = (f32_to_bf16_bits(rng.standard_normal((B, H, N, D), dtype=np.float32) * 1.2) for _ in range(3))
    q, k, v = (torch.from_numpy(np.ascontiguousarray(x).view(np.int16)).cuda().view(torch.bfloat16) for x in (qb, kb, vb))
    out = torch.empty_like(q)
    lse = torch.empty((B, H, N), device="cuda", dtype=torch.float32)
    sa.sparse_attn_fwd(q, k, v, out, lse, B, H, N, D, sa.make_params(), sa.MODE_DENSE, None)
    T = -(-N // tile)
    mass = torch.full((B, H, T, T), float("nan"), device="cuda", dtype=torch.float32)
    sa.sparse_attn_block_mass(q, k, lse, mass, B, H, N, D)
    torch.cuda.synchronize()
    got = mass.cpu().numpy().astype(np.float64)
    for h in range(H):
        ref = oracle.block_mass(bf16_bits_to_f64(qb[0, h]), bf16_bits_to_f64(kb[0, h]), tile)
        assert np.abs(got[0, h] - ref).max() < 1e-3 * tile + 1e-3 * np.abs(ref).max()
        assert np.allclose(got[0, h].sum(axis=1), ref.sum(axis=1), rtol=1e-3)
