"""Block mass of the dense probabilities (first half of the offline selectors).
CPU: pins of the oracle.  GPU: sparse_attn_block_mass against the oracle."""
import math

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


def test_oracle_sqmass_and_eq3_against_definitions():
    rng = np.random.default_rng(6)
    N, D, tile = 200, 16, 64
    q, k = rng.standard_normal((N, D)), rng.standard_normal((N, D))
    p = torch.softmax(torch.from_numpy(q @ k.T / 4.0), dim=1).numpy()       # library softmax
    sq = oracle.block_sqmass(q, k, tile)
    assert abs(sq[2, 1] - (p[128:192, 64:128] ** 2).sum()) < 1e-12
    assert np.allclose(sq.sum(axis=1), [(p[i * 64:(i + 1) * 64] ** 2).sum() for i in range(4)], atol=1e-12)
    # Eq. 3 typed out for one row of 4 tokens, S = {1, 3}: sum_S p^2 + (S1/(1-S1))^2 sum_K p^2
    P = np.array([0.5, 0.1, 0.3, 0.1])
    assert abs(oracle.eq3_lhs(P, P ** 2, [1, 3]) - (0.02 + (0.2 / 0.8) ** 2 * (0.25 + 0.09))) < 1e-15
    assert oracle.eq3_lhs(P, P ** 2, []) == 0.0


@pytest.mark.parametrize("T,tile", [(16, 64), (32, 128), (9, 64)])
@pytest.mark.parametrize("theta_n", [0.0, 0.05, 0.3, 1.0, 5.0, 1e6])
def test_oracle_greedy_uniform_closed_form(T, tile, theta_n):
    """Uniform attention (every p = 1/N): discarding n of the T tiles gives S1 = n/T, sum_S q = n B_c / N^2 and
    sum_K q = (T - n) B_c / N^2, so Eq. 3's left side is (B_c / N^2) (n + n^2 / (T - n)) = n / ((T - n) N); it grows
    with n, and the largest n with n / ((T - n) N) <= Theta is floor(Theta N T / (1 + Theta N)), capped at T - 1 because
    tile 0 is never a candidate.  (Theta is given here as theta_n = Theta * N.)"""
    N = T * tile
    theta = theta_n / N
    mass = np.full((T, T), tile * tile / N)               # rows * (tile / N)
    sq = np.full((T, T), tile * tile / N ** 2)
    skip = oracle.select_greedy(mass, sq, N, tile, theta)
    n_expect = min(T - 1, int(math.floor(theta_n * T / (1.0 + theta_n) + 1e-9)))
    assert np.all(skip.sum(axis=1) == n_expect), (skip.sum(axis=1), n_expect)
    assert not skip[:, 0].any()
    if n_expect:                                          # ties: lower index first
        assert np.all(skip[:, 1:1 + n_expect] == 1)


def test_oracle_greedy_respects_eq3_and_is_maximal(seed):
    cfg = CONFIGS["cfg0_aligned"]
    qb, kb, _ = make_qkv(cfg, seed, heads=[0])
    q, k = bf16_bits_to_f64(qb[0, 0]), bf16_bits_to_f64(kb[0, 0])
    mass, sq = oracle.block_mass(q, k, cfg.tile), oracle.block_sqmass(q, k, cfg.tile)
    n_disc = []
    for theta in (0.0, 1e-5, 1e-4, 1e-3, 1e-2):
        skip = oracle.select_greedy(mass, sq, cfg.N, cfg.tile, theta)
        n_disc.append(int(skip.sum()))
        for i in range(mass.shape[0]):
            P, qq = mass[i] / cfg.tile, sq[i] / cfg.tile
            S = list(np.nonzero(skip[i])[0])
            assert oracle.eq3_lhs(P, qq, S) <= theta                   # the returned set satisfies Eq. 3 ...
            rest = [j for j in range(1, mass.shape[1]) if not skip[i, j]]
            if rest:                                                    # ... and the next-smallest tile would break it
                nxt = min(rest, key=lambda j: (mass[i, j], j))
                assert oracle.eq3_lhs(P, qq, S + [nxt]) > theta
            if S and rest:                                              # discarded tiles are the smallest ones
                assert mass[i, S].max() <= mass[i, rest].min()
    assert n_disc == sorted(n_disc) and n_disc[0] == 0 and n_disc[-1] > 0   # a larger tolerance discards more


@pytest.mark.gpu
def test_gpu_block_stats_and_greedy_selector(seed):
    """sparse_attn_block_stats' second output against the fp64 definition; sparse_attn_select_blocks_greedy against the
    oracle's selection on the same (GPU) masses; the bitmap then drives MASK mode and equals the oracle's replay."""
    for name, N in (("cfg0_aligned", None), ("d128", 1000)):
        if name == "cfg0_aligned":
            cfg = CONFIGS[name]
            qb, kb, vb = make_qkv(cfg, seed)
            B, H, N, D, tile = cfg.B, cfg.H, cfg.N, cfg.D, cfg.tile
        else:
            D, tile, B, H = 128, 128, 1, 2
            rng = np.random.default_rng([seed, N, D, 9])
            qb, kb = (f32_to_bf16_bits(rng.standard_normal((B, H, N, D), dtype=np.float32) * 1.6) for _ in range(2))
            vb = f32_to_bf16_bits(rng.standard_normal((B, H, N, D), dtype=np.float32))     # V ~ N(0,1) as in the configs
        q, k, v = (torch.from_numpy(np.ascontiguousarray(x).view(np.int16)).cuda().view(torch.bfloat16) for x in (qb, kb, vb))
        out = torch.empty_like(q)
        lse = torch.empty((B, H, N), device="cuda", dtype=torch.float32)
        sa.sparse_attn_fwd(q, k, v, out, lse, B, H, N, D, sa.make_params(), sa.MODE_DENSE, None)
        T = -(-N // tile)
        mass = torch.full((B, H, T, T), float("nan"), device="cuda", dtype=torch.float32)
        sq = torch.full((B, H, T, T), float("nan"), device="cuda", dtype=torch.float32)
        sa.sparse_attn_block_stats(q, k, lse, mass, sq, B, H, N, D)
        torch.cuda.synchronize()
        m64, s64 = mass.cpu().numpy().astype(np.float64), sq.cpu().numpy().astype(np.float64)
        for h in range(H):
            qh, kh = bf16_bits_to_f64(qb[0, h]), bf16_bits_to_f64(kb[0, h])
            ref_m, ref_s = oracle.block_mass(qh, kh, tile), oracle.block_sqmass(qh, kh, tile)
            assert np.abs(m64[0, h] - ref_m).max() < 1e-3 * tile + 1e-3 * np.abs(ref_m).max()
            assert np.abs(s64[0, h] - ref_s).max() < 2e-3 * np.abs(ref_s).max() + 1e-9
        total = 0
        for theta in (1e-6, 1e-4, 1e-3, 3e-2):
            bitmap = torch.full((B, H, T, T), 255, device="cuda", dtype=torch.uint8)
            sa.sparse_attn_select_blocks_greedy(mass, sq, bitmap, B, H, N, tile, T, theta)
            torch.cuda.synchronize()
            got = bitmap.cpu().numpy()
            for h in range(H):
                assert np.array_equal(got[0, h], oracle.select_greedy(m64[0, h], s64[0, h], N, tile, theta)), (name, theta, h)
            total += int(got.sum())
            stats = torch.zeros((B, H, 2), device="cuda", dtype=torch.int64)
            sa.sparse_attn_fwd(q, k, v, out, None, B, H, N, D, sa.make_params(skip_mask_in=bitmap), sa.MODE_MASK, stats)
            torch.cuda.synchronize()
            o = bf16_bits_to_f64(out.view(torch.int16).cpu().numpy().view(np.uint16))
            for h in range(H):
                assert int(stats[0, h, 1]) == int(got[0, h].sum())
                ref = oracle.run_head(qb[0, h], kb[0, h], vb[0, h], tile=tile, lam=0.0, mode=oracle.MODE_DYNAMIC,
                                      forced_skip=got[0, h])
                assert np.abs(o[0, h] - ref.rows()[0]).max() < 2e-2
        assert total > 0


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


def test_select_blocks_validates_on_host():
    a = np.zeros(1024, dtype=np.float32)
    b = np.zeros(1024, dtype=np.uint8)
    cases = [((None, b, 1, 1, 4, 4, 0, 0.5), -1), ((a, None, 1, 1, 4, 4, 0, 0.5), -1), ((a, b, 1, 1, 0, 4, 0, 0.5), -2),
             ((a, b, 1, 1, 4, 5000, 0, 0.5), -2), ((a, b, 1, 1, 4, 4, 2, 0.5), -5), ((a, b, 1, 1, 4, 4, 0, 0.0), -6),
             ((a, b, 1, 1, 4, 4, 1, 1.5), -6)]
    for args, status in cases:
        with pytest.raises(sa.SparseAttnError) as e:
            sa.sparse_attn_select_blocks(*args)
        assert e.value.status == status, args
    q = np.zeros(4096, dtype=np.uint16)
    with pytest.raises(sa.SparseAttnError) as e:
        sa.sparse_attn_block_mass(q, q, None, a, 1, 1, 16, 64)
    assert e.value.status == -1
    with pytest.raises(sa.SparseAttnError) as e:
        sa.sparse_attn_block_mass(q, q, a, a, 1, 1, 16, 96)
    assert e.value.status == -3
    for args, status in [((None, a, b, 1, 1, 256, 64, 4, 0.1), -1), ((a, a, b, 1, 1, 256, 96, 4, 0.1), -4),
                         ((a, a, b, 1, 1, 256, 64, 0, 0.1), -2), ((a, a, b, 1, 1, 256, 64, 4, -1.0), -6),
                         ((a, a, b, 1, 1, 256, 64, 4, float("nan")), -6)]:
        with pytest.raises(sa.SparseAttnError) as e:
            sa.sparse_attn_select_blocks_greedy(*args)
        assert e.value.status == status, args


@pytest.mark.gpu
def test_gpu_selectors_match_oracle_and_drive_mask_mode(seed):
    """Top-K / Top-P bitmaps from the GPU equal the oracle's selection on the same mass values; the bitmap then drives
    MASK mode, whose output equals the oracle's replay of it, and Top-P's bitmap retains at least P of every row of
    tiles' mass."""
    cfg = CONFIGS["cfg0_aligned"]
    qb, kb, vb = make_qkv(cfg, seed)
    B, H, N, D, tile = cfg.B, cfg.H, cfg.N, cfg.D, cfg.tile
    T = N // tile
    q, k, v = (torch.from_numpy(x.view(np.int16)).cuda().view(torch.bfloat16) for x in (qb, kb, vb))
    out = torch.empty_like(q)
    lse = torch.empty((B, H, N), device="cuda", dtype=torch.float32)
    sa.sparse_attn_fwd(q, k, v, out, lse, B, H, N, D, sa.make_params(), sa.MODE_DENSE, None)
    mass = torch.empty((B, H, T, T), device="cuda", dtype=torch.float32)
    sa.sparse_attn_block_mass(q, k, lse, mass, B, H, N, D)
    torch.cuda.synchronize()
    m64 = mass.cpu().numpy().astype(np.float64)
    for kind, param, sel in ((sa.SELECT_TOPK, 0.25, oracle.select_topk), (sa.SELECT_TOPK, 0.6, oracle.select_topk),
                             (sa.SELECT_TOPP, 0.9, oracle.select_topp), (sa.SELECT_TOPP, 0.99, oracle.select_topp)):
        bitmap = torch.full((B, H, T, T), 255, device="cuda", dtype=torch.uint8)
        sa.sparse_attn_select_blocks(mass, bitmap, B, H, T, T, kind, param)
        torch.cuda.synchronize()
        got = bitmap.cpu().numpy()
        for h in range(H):
            assert np.array_equal(got[0, h], sel(m64[0, h], param)), (kind, param, h)
            if kind == sa.SELECT_TOPP:
                kept = (m64[0, h] * (got[0, h] == 0)).sum(axis=1)
                assert np.all(kept >= param * m64[0, h].sum(axis=1) * (1 - 1e-12))
        stats = torch.zeros((B, H, 2), device="cuda", dtype=torch.int64)
        lse_m = torch.empty_like(lse)
        sa.sparse_attn_fwd(q, k, v, out, lse_m, B, H, N, D, sa.make_params(lam=-3.0, skip_mask_in=bitmap), sa.MODE_MASK, stats)
        torch.cuda.synchronize()
        o = bf16_bits_to_f64(out.view(torch.int16).cpu().numpy().view(np.uint16))
        for h in range(H):
            assert int(stats[0, h, 1]) == int(got[0, h].sum())
            ref = oracle.run_head(qb[0, h], kb[0, h], vb[0, h], tile=tile, lam=-3.0, mode=oracle.MODE_DYNAMIC,
                                  forced_skip=got[0, h])
            assert np.abs(o[0, h] - ref.rows()[0]).max() < 2e-2
        if kind == sa.SELECT_TOPP:                          # row recall >= share of the row's own tile masses kept: sanity
            rec = torch.exp(lse_m - lse)
            assert float(rec.mean()) > param - 0.05


@pytest.mark.gpu
def test_gpu_selectors_at_the_documented_maximum_row_length(seed):
    """T_c = 4096 is the largest row of tiles the selectors accept; the greedy kernel then needs exactly 48 KB of shared
    memory (it used to need 4 bytes more than the default limit and failed to launch).  Random mass rows, one Q tile per
    head, against the oracle's selections."""
    import torch
    T_c, tile = 4096, 128
    N = tile                                                                    # T_r = 1 row of tiles per head
    rng = np.random.default_rng([seed, 4096])
    H = 3
    p = rng.dirichlet(np.full(T_c, 0.3), size=(1, H, 1)).astype(np.float32)     # P_j of a row, sums to 1
    mass = (p * tile).astype(np.float32)                                        # block sums over 128 rows
    sq = (p ** 2 * tile * rng.uniform(0.5, 1.5, size=p.shape)).astype(np.float32)
    dm, ds = torch.from_numpy(mass).cuda(), torch.from_numpy(sq).cuda()
    bitmap = torch.full((1, H, 1, T_c), 255, device="cuda", dtype=torch.uint8)
    for theta in (1e-7, 1e-5):
        sa.sparse_attn_select_blocks_greedy(dm, ds, bitmap, 1, H, N, tile, T_c, theta)
        torch.cuda.synchronize()
        got = bitmap.cpu().numpy()
        for h in range(H):
            ref = oracle.select_greedy(mass[0, h].astype(np.float64), sq[0, h].astype(np.float64), N, tile, theta)
            assert np.array_equal(got[0, h], ref), (theta, h, int(got[0, h].sum()), int(ref.sum()))
        assert 0 < got.sum() < H * T_c
    for kind, param in ((sa.SELECT_TOPK, 0.25), (sa.SELECT_TOPP, 0.9)):
        sa.sparse_attn_select_blocks(dm, bitmap, 1, H, 1, T_c, kind, param)
        torch.cuda.synchronize()
        got = bitmap.cpu().numpy()
        for h in range(H):
            ref = (oracle.select_topk if kind == sa.SELECT_TOPK else oracle.select_topp)(mass[0, h].astype(np.float64), param)
            assert np.array_equal(got[0, h], ref), (kind, h)
