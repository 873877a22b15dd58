"""`sparse_attn_fwd_host` against the device entry `sparse_attn_fwd`, bit for bit, in the shapes the chunked pipeline
actually meets: more heads than chunks (20), so that chunks hold several heads, and head counts that do not divide evenly
(B*H = 21, 24, 41, 45), with every optional buffer set (lse, stats, skip_mask_out, margin_out, skip_mask_in), from pinned
and from pageable host memory.  The per-chunk pointer offsets of all nine buffers are what is under test; the arithmetic
is the device entry's, which tests/test_gpu_parity.py checks against the oracle."""
import numpy as np
import pytest
from workloads import f32_to_bf16_bits

pytestmark = pytest.mark.gpu


def _inputs(B, H, N, D, seed):
    rng = np.random.default_rng([41, seed, B, H, N, D])
    # per-head temperatures: flat heads skip a lot at lambda = -3, peaked heads little -> stats differ from head to head
    tau = rng.uniform(0.4, 3.0, size=(B, H, 1, 1)).astype(np.float32)
    base = rng.standard_normal((B, H, N, D)).astype(np.float32)
    q = f32_to_bf16_bits(tau * (0.5 * base + 0.5 * rng.standard_normal((B, H, N, D)).astype(np.float32)))
    k = f32_to_bf16_bits(tau * (0.5 * base + 0.5 * rng.standard_normal((B, H, N, D)).astype(np.float32)))
    v = f32_to_bf16_bits(rng.standard_normal((B, H, N, D)).astype(np.float32))
    return q, k, v


def _host_buffers(arrays, pinned):
    """numpy views of pinned torch tensors, or plain (pageable) numpy arrays."""
    import torch
    if not pinned:
        return [np.ascontiguousarray(a).copy() for a in arrays], None
    keep = []
    out = []
    for a in arrays:
        t = torch.from_numpy(np.ascontiguousarray(a).view(np.int16 if a.dtype == np.uint16 else a.dtype)).pin_memory()
        keep.append(t)
        out.append(t.numpy().view(a.dtype))
    return out, keep


@pytest.mark.parametrize("B,H,N,D,pinned", [(1, 41, 300, 128, True), (2, 21, 300, 128, False), (1, 24, 257, 128, True),
                                            (3, 15, 200, 64, True), (1, 40, 129, 128, False)])
def test_host_entry_equals_device_entry_with_many_heads_per_chunk(B, H, N, D, pinned, seed):
    import torch

    import paper_2606_16317_b200 as sa
    import parity_utils
    tile = 64 if D == 64 else 128
    T = -(-N // tile)
    q, k, v = _inputs(B, H, N, D, seed)
    lam = -3.0
    dev = parity_utils.run_gpu(q, k, v, mode=sa.MODE_DYNAMIC, lam=lam, tile=tile)
    frac = dev.stats[:, 1].sum() / dev.stats.sum()
    assert 0.05 < frac < 0.95 and len({tuple(s) for s in dev.stats}) >= 3, "the workload must mix decisions across heads"

    def host_call(mode, mask_in=None):
        bufs = [q, k, v,
                np.full((B, H, N, D), 0x7fc0, dtype=np.uint16),                  # out: bf16 NaN
                np.full((B, H, N), np.nan, dtype=np.float32),                     # lse
                np.full((B, H, 2), -1, dtype=np.int64),                           # stats
                np.full((B, H, T, T), 255, dtype=np.uint8),                       # skip_mask_out
                np.full((B, H, T, T), np.nan, dtype=np.float32)]                  # margin_out
        if mask_in is not None:
            bufs.append(mask_in)
        (hq, hk, hv, hout, hlse, hstats, hmask, hmargin, *rest), keep = _host_buffers(bufs, pinned)
        p = sa.make_params(lam=lam, skip_mask_out=hmask, margin_out=hmargin, skip_mask_in=rest[0] if rest else None)
        sa.sparse_attn_fwd_host(hq, hk, hv, hout, hlse, B, H, N, D, p, mode, hstats)
        del keep
        return hout, hlse, hstats, hmask, hmargin

    hout, hlse, hstats, hmask, hmargin = host_call(sa.MODE_DYNAMIC)
    dev_bits = f32_to_bf16_bits(dev.out.astype(np.float32)).reshape(B, H, N, D)   # (bf16 -> f64 -> bf16 is exact)
    np.testing.assert_array_equal(hout, dev_bits)
    np.testing.assert_array_equal(hlse.reshape(B * H, N), dev.lse)
    np.testing.assert_array_equal(hstats.reshape(B * H, 2), dev.stats)
    np.testing.assert_array_equal(hmask.reshape(B * H, T, T), dev.skip)
    np.testing.assert_array_equal(hmargin.reshape(B * H, T, T), dev.margin)

    # MASK mode: a random bitmap (tile 0 of every row is retained whatever its byte says) through both entries
    rng = np.random.default_rng([42, seed, B, H])
    bitmap = (rng.random((B, H, T, T)) < 0.4).astype(np.uint8)
    mq, mk, mv = (parity_utils.to_dev_bf16(np.ascontiguousarray(x)) for x in (q, k, v))
    dout = torch.full((B, H, N, D), float("nan"), device="cuda", dtype=torch.bfloat16)
    dlse = torch.full((B, H, N), float("nan"), device="cuda", dtype=torch.float32)
    dstats = torch.full((B, H, 2), -1, device="cuda", dtype=torch.int64)
    dmask = torch.full((B, H, T, T), 255, device="cuda", dtype=torch.uint8)
    dmargin = torch.full((B, H, T, T), float("nan"), device="cuda", dtype=torch.float32)
    p = sa.make_params(lam=lam, skip_mask_out=dmask, margin_out=dmargin, skip_mask_in=torch.from_numpy(bitmap).cuda(),
                       stream=torch.cuda.current_stream().cuda_stream)
    sa.sparse_attn_fwd(mq, mk, mv, dout, dlse, B, H, N, D, p, sa.MODE_MASK, dstats)
    torch.cuda.synchronize()
    hout, hlse, hstats, hmask, hmargin = host_call(sa.MODE_MASK, bitmap)
    np.testing.assert_array_equal(hout.view(np.int16), dout.view(torch.int16).cpu().numpy())
    np.testing.assert_array_equal(hlse, dlse.cpu().numpy())
    np.testing.assert_array_equal(hstats, dstats.cpu().numpy())
    np.testing.assert_array_equal(hmask, dmask.cpu().numpy())
    np.testing.assert_array_equal(hmargin, dmargin.cpu().numpy())
    expect = bitmap.copy()
    expect[..., 0] = 0
    np.testing.assert_array_equal(hmask, expect)


def test_host_entry_scratch_lives_in_the_library_pool_and_can_be_released(seed):
    """The device copies come from a pool of the library's own: they stay there after the call (so the next call does not
    pay for them again) and sparse_attn_release_scratch hands them back to the driver."""
    import torch

    import paper_2606_16317_b200 as sa
    B, H, N, D = 1, 41, 1000, 128                                              # 4 tensors x 10.5 MB of scratch
    q, k, v = _inputs(B, H, N, D, seed)
    out = np.zeros_like(q)

    def call():
        sa.sparse_attn_fwd_host(q, k, v, out, None, B, H, N, D, sa.make_params(lam=-3.0), sa.MODE_DYNAMIC, None)
        torch.cuda.synchronize()

    call()                                                                     # loads the kernels, creates the pool
    first = out.copy()
    sa.sparse_attn_release_scratch()
    free0, _ = torch.cuda.mem_get_info()
    call()
    free1, _ = torch.cuda.mem_get_info()
    assert free0 - free1 >= 30 << 20, (free0, free1)                           # the scratch is retained ...
    sa.sparse_attn_release_scratch()
    free2, _ = torch.cuda.mem_get_info()
    assert free2 >= free0 - (2 << 20), (free0, free2)                          # ... until it is released
    call()                                                                     # and the entry works again afterwards
    np.testing.assert_array_equal(out, first)
    sa.sparse_attn_release_scratch()
