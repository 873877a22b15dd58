"""Spatio-temporal token re-ordering.

CPU (-m "not gpu"): the oracle against what the definition fixes (pins), the C host function
sparse_attn_brick_permutation against the oracle, and the error paths of both entry points.
GPU (-m gpu): sparse_attn_reorder_tokens bit-exact against the oracle's row-by-row loop, the
round trip, and the equivariance of the attention call under the permutation."""
import math

import numpy as np
import pytest
import torch

import oracle
import paper_2606_16317_b200 as sa
from paper_2606_16317_b200 import build
from workloads import CONFIGS, bf16_bits_to_f64, make_qkv

GRIDS = [((4, 16, 16), (2, 8, 8)), ((21, 30, 52), (2, 8, 8)), ((21, 30, 52), (4, 4, 8)), ((5, 7, 9), (2, 3, 4)),
         ((3, 5, 7), (8, 8, 8)), ((1, 1, 40), (1, 1, 16)), ((21, 45, 80), (1, 8, 16))]


@pytest.fixture(scope="module", autouse=True)
def built():
    build.build()


def c_perm(grid, brick):
    out = np.full(grid[0] * grid[1] * grid[2], -1, dtype=np.int32)
    sa.sparse_attn_brick_permutation(*grid, *brick, out)
    return out


# ------------------------------------------------------------------ oracle pins
@pytest.mark.parametrize("grid,brick", GRIDS[:6])
def test_oracle_perm_is_a_bijection(grid, brick):
    p = oracle.brick_permutation(grid, brick)
    assert sorted(p.tolist()) == list(range(grid[0] * grid[1] * grid[2]))


@pytest.mark.parametrize("grid", [(4, 6, 8), (3, 5, 7)])
def test_oracle_perm_identity_cases(grid):
    T, H, W = grid
    N = T * H * W
    for brick in ((T, H, W), (1, 1, W), (1, H, W), (T + 3, H + 1, W + 2)):
        assert np.array_equal(oracle.brick_permutation(grid, brick), np.arange(N)), brick


def test_oracle_perm_closed_form_on_divisible_grid():
    grid, brick = (4, 16, 24), (2, 8, 8)
    T, H, W = grid
    bt, bh, bw = brick
    idx = np.arange(T * H * W).reshape(T // bt, bt, H // bh, bh, W // bw, bw).transpose(0, 2, 4, 1, 3, 5).reshape(-1)
    assert np.array_equal(oracle.brick_permutation(grid, brick), idx)


def test_oracle_bricks_are_contiguous_and_local():
    grid, brick = (21, 30, 52), (2, 8, 8)
    p = oracle.brick_permutation(grid, brick)
    T, H, W = grid
    t, h, w = p // (H * W), (p // W) % H, p % W
    first = p[:128]                                     # the first full brick: one 128-token attention tile
    assert len(set((first // (H * W)).tolist())) == 2 and np.ptp((first // W) % H) == 7 and np.ptp(first % W) == 7
    # brick coordinates never decrease along the new order in lexicographic (t, h, w) brick order
    key = ((t // 2) * 100 + (h // 8)) * 100 + (w // 8)
    assert np.all(np.diff(key) >= 0)


def test_oracle_reorder_round_trip_and_definition():
    rng = np.random.default_rng(3)
    x = rng.integers(0, 65536, size=(2, 3, 60, 8)).astype(np.uint16)
    p = oracle.brick_permutation((3, 4, 5), (2, 2, 2))
    y = oracle.reorder(x, p)
    assert np.array_equal(y, x[:, :, p])                # gather definition, by fancy indexing (library routine)
    assert np.array_equal(oracle.reorder(y, p, inverse=True), x)
    inv = np.argsort(p)
    assert np.array_equal(oracle.reorder(x, p, inverse=True), x[:, :, inv])


# ------------------------------------------------------------------ C host function against the oracle
@pytest.mark.parametrize("grid,brick", GRIDS)
def test_c_permutation_equals_oracle(grid, brick):
    if grid == (21, 45, 80):                            # 75600 tokens: the Python-loop oracle is slow but fine once
        pass
    assert np.array_equal(c_perm(grid, brick).astype(np.int64), oracle.brick_permutation(grid, brick))


def test_permutation_error_paths():
    out = np.zeros(8, dtype=np.int32)
    for args, status in (((0, 2, 2, 1, 1, 1), -2), ((2, 2, 2, 0, 1, 1), -2), ((1 << 12, 1 << 12, 2, 1, 1, 1), -2)):
        with pytest.raises(sa.SparseAttnError) as e:
            sa.sparse_attn_brick_permutation(*args, out)
        assert e.value.status == status
    with pytest.raises(sa.SparseAttnError) as e:
        sa.sparse_attn_brick_permutation(2, 2, 2, 1, 1, 1, None)
    assert e.value.status == -1


def test_reorder_validates_before_touching_a_device():
    a = np.zeros(4096 + 64, dtype=np.uint8)
    base = a.ctypes.data + ((-a.ctypes.data) % 64)
    perm = np.zeros(4, dtype=np.int32)
    cases = [((None, base, 1, 1, 4, 64, perm, 0), -1), ((base, base + 1024, 1, 1, 4, 64, None, 0), -1),
             ((base, base + 1024, 0, 1, 4, 64, perm, 0), -2), ((base, base + 1024, 1, 1, 4, 96, perm, 0), -3),
             ((base + 2, base + 1024, 1, 1, 4, 64, perm, 0), -7), ((base, base + 256, 1, 1, 4, 64, perm, 0), -6)]
    for args, status in cases:
        with pytest.raises(sa.SparseAttnError) as e:
            sa.sparse_attn_reorder_tokens(*args)
        assert e.value.status == status, args
    if not torch.cuda.is_available():                   # no CPU fallback
        with pytest.raises(sa.SparseAttnError) as e:
            sa.sparse_attn_reorder_tokens(base, base + 2048, 1, 1, 4, 64, perm, 0)
        assert e.value.status == -8


# ------------------------------------------------------------------ GPU parity (through the C ABI)
def _dev(bits):
    return torch.from_numpy(np.ascontiguousarray(bits).view(np.int16)).cuda()


@pytest.mark.gpu
@pytest.mark.parametrize("B,H,grid,brick,D", [(1, 2, (4, 16, 16), (2, 8, 8), 64), (2, 3, (5, 7, 9), (2, 3, 4), 128),
                                              (1, 1, (1, 1, 1), (1, 1, 1), 64), (1, 2, (3, 5, 7), (8, 8, 8), 128),
                                              (1, 5, (7, 13, 11), (2, 4, 4), 128)])
def test_gpu_reorder_bit_exact(B, H, grid, brick, D):
    N = grid[0] * grid[1] * grid[2]
    rng = np.random.default_rng([7, N, D])
    x = rng.integers(0, 65536, size=(B, H, N, D)).astype(np.uint16)
    perm = c_perm(grid, brick)
    dperm = torch.from_numpy(perm).cuda()
    src = _dev(x)
    for inverse in (0, 1):
        dst = torch.full_like(src, -1)
        sa.sparse_attn_reorder_tokens(src, dst, B, H, N, D, dperm, inverse, torch.cuda.current_stream().cuda_stream)
        torch.cuda.synchronize()
        got = dst.cpu().numpy().view(np.uint16)
        assert np.array_equal(got, oracle.reorder(x, perm.astype(np.int64), inverse=bool(inverse)))
    # round trip
    mid, back = torch.empty_like(src), torch.empty_like(src)
    sa.sparse_attn_reorder_tokens(src, mid, B, H, N, D, dperm, 0)
    sa.sparse_attn_reorder_tokens(mid, back, B, H, N, D, dperm, 1)
    torch.cuda.synchronize()
    assert torch.equal(back, src)


@pytest.mark.gpu
def test_gpu_reorder_full_size_sampled(seed):
    """Config 1's shape in the launch configuration bench.py times; rows sampled against the definition."""
    cfg = CONFIGS["cfg1"]
    H = 4
    rng = np.random.default_rng(seed)
    x = rng.integers(0, 65536, size=(1, H, cfg.N, cfg.D), dtype=np.uint16)
    perm = c_perm(cfg.grid, (4, 4, 8))
    assert np.array_equal(np.sort(perm), np.arange(cfg.N))
    dperm = torch.from_numpy(perm).cuda()
    src, dst = _dev(x), torch.empty(x.shape, dtype=torch.int16, device="cuda")
    sa.sparse_attn_reorder_tokens(src, dst, 1, H, cfg.N, cfg.D, dperm, 0)
    torch.cuda.synchronize()
    got = dst.cpu().numpy().view(np.uint16)
    for p in [0, 1, 127, 128, cfg.N - 1] + rng.integers(0, cfg.N, 200).tolist():
        for h in range(H):
            assert np.array_equal(got[0, h, p], x[0, h, perm[p]])
    assert np.array_equal(np.sort(got[0, 0].astype(np.int64).sum(axis=1)), np.sort(x[0, 0].astype(np.int64).sum(axis=1)))


@pytest.mark.gpu
def test_gpu_attention_is_equivariant_under_reordering(seed):
    """DENSE attention on re-ordered q, k, v, scattered back, equals the un-permuted call up to summation order;
    DYNAMIC mode on the re-ordered inputs matches the oracle run on the same re-ordered inputs."""
    cfg = CONFIGS["cfg0"]
    qb, kb, vb = make_qkv(cfg, seed)
    perm = c_perm(cfg.grid, (2, 4, 8))
    dperm = torch.from_numpy(perm).cuda()
    B, H, N, D = cfg.B, cfg.H, cfg.N, cfg.D
    q, k, v = (_dev(x).view(torch.bfloat16) for x in (qb, kb, vb))
    qp, kp, vp = (torch.empty_like(q) for _ in range(3))
    for s, d in ((q, qp), (k, kp), (v, vp)):
        sa.sparse_attn_reorder_tokens(s, d, B, H, N, D, dperm, 0)
    out, outp, outb = (torch.empty_like(q) for _ in range(3))
    lse = torch.empty((B, H, N), device="cuda", dtype=torch.float32)
    stats = torch.zeros((B, H, 2), device="cuda", dtype=torch.int64)
    p = sa.make_params()
    sa.sparse_attn_fwd(q, k, v, out, lse, B, H, N, D, p, sa.MODE_DENSE, stats)
    sa.sparse_attn_fwd(qp, kp, vp, outp, lse, B, H, N, D, p, sa.MODE_DENSE, stats)
    sa.sparse_attn_reorder_tokens(outp, outb, B, H, N, D, dperm, 1)
    torch.cuda.synchronize()
    d = (out.float() - outb.float()).abs()
    assert d.max().item() < 2e-2 and d.mean().item() < 2e-3
    # sparse mode on the re-ordered inputs against the oracle on the oracle's own re-ordering
    lam = -2.0
    mask = torch.zeros((B, H, N // cfg.tile, N // cfg.tile), device="cuda", dtype=torch.uint8)
    p = sa.make_params(lam=lam, skip_mask_out=mask)
    sa.sparse_attn_fwd(qp, kp, vp, outp, lse, B, H, N, D, p, sa.MODE_DYNAMIC, stats)
    torch.cuda.synchronize()
    o = bf16_bits_to_f64(outp.view(torch.int16).cpu().numpy().view(np.uint16))
    operm = oracle.brick_permutation(cfg.grid, (2, 4, 8))
    for h in range(H):
        ref = oracle.run_head(oracle.reorder(qb[0, h], operm), oracle.reorder(kb[0, h], operm),
                              oracle.reorder(vb[0, h], operm), tile=cfg.tile, lam=lam, mode=oracle.MODE_DYNAMIC)
        assert np.array_equal(ref.skip, mask[0, h].cpu().numpy())
        assert np.abs(o[0, h] - ref.rows()[0]).max() < 2e-2
        assert int(stats[0, h, 1]) == ref.skipped
