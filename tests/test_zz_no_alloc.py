"""`sparse_attn_row_topk_curve_static`: the Appendix A.1 row curve for callers that cannot allocate device memory.

Some hosts of this library have no allocator left to call: a serving process that reserved all free HBM for its own cache
at start-up (cudaMalloc / cudaMallocAsync then fail with out-of-memory), or a request path that is not allowed to enter
the driver's allocator because cudaMalloc and cudaFree may stall the whole device.  For them the library keeps the
kernel's working memory in one fixed 16 MiB array of its own device image; the entry point tested here uses that array and
calls no allocator.  The array is shared by every call and keeps the previous call's contents, so the test makes TWO calls
in a row (the second with another shape, on top of the first one's leftovers) and compares each with the allocating entry
point `sparse_attn_row_topk_curve`, at the tolerances tests/test_analysis.py uses for this kernel.

This file sorts last on purpose (`pytest --collect-only`): under `pytest -x` a failure here hides no other test.
"""
import numpy as np
import pytest
from workloads import f32_to_bf16_bits

from paper_2606_16317_b200 import build


@pytest.fixture(scope="module", autouse=True)
def built():
    build.build()


def _inputs(seed, H, N, D, n_rows):
    import torch
    rng = np.random.default_rng([31, seed, N, D])
    base = rng.standard_normal((1, H, N, D)).astype(np.float32)
    taus = rng.uniform(0.3, 2.5, size=(1, H, 1, 1)).astype(np.float32)
    bits = [f32_to_bf16_bits(taus * (0.6 * base + 0.4 * rng.standard_normal((1, H, N, D)).astype(np.float32))),
            f32_to_bf16_bits(taus * (0.6 * base + 0.4 * rng.standard_normal((1, H, N, D)).astype(np.float32))),
            f32_to_bf16_bits(rng.standard_normal((1, H, N, D)).astype(np.float32))]
    dev = [torch.from_numpy(np.ascontiguousarray(x).view(np.int16)).cuda().view(torch.bfloat16) for x in bits]
    rows = np.array([(h, r) for h in range(H) for r in sorted(rng.choice(N, size=n_rows, replace=False))], dtype=np.int32)
    rows[0, 1], rows[-1, 1] = 0, N - 1
    keep = np.array([1, 2, 3, 17, N // 10, N // 3, N // 2, int(0.8 * N), N - 1, N], dtype=np.int32)
    return dev, rows, keep


def _outputs(R, nK):
    import torch
    return (torch.full((R,), float("nan"), device="cuda", dtype=torch.float64),
            torch.full((R, nK), float("nan"), device="cuda", dtype=torch.float64),
            torch.full((R, nK), float("nan"), device="cuda", dtype=torch.float64))


@pytest.mark.gpu
def test_static_scratch_entry_matches_the_allocating_one_on_two_calls_in_a_row():
    import torch

    import paper_2606_16317_b200 as sa
    # second call: other head dim, shorter rows, fewer of them -> it runs over what the first call left in the array
    for call, (H, N, D, n_rows) in enumerate([(2, 4133, 128, 9), (1, 777, 64, 5)]):
        dev, rows, keep = _inputs(call, H, N, D, n_rows)
        ref, got = _outputs(len(rows), len(keep)), _outputs(len(rows), len(keep))
        sa.sparse_attn_row_topk_curve(*dev, 1, H, N, D, rows, keep, *ref)
        torch.cuda.synchronize()
        sa.sparse_attn_row_topk_curve_static(*dev, 1, H, N, D, rows, keep, *got)
        torch.cuda.synchronize()
        (rk, rr, rm), (gk, gr, gm) = ([t.cpu().numpy() for t in ref], [t.cpu().numpy() for t in got])
        assert not np.isnan(gr).any() and not np.isnan(gm).any(), f"call {call}: outputs not fully written"
        assert np.allclose(gk, rk, rtol=1e-3, atol=1e-3, equal_nan=True), (call, gk, rk)
        assert np.abs(gr - rr).max() < 2e-5, (call, np.abs(gr - rr).max())
        assert np.all(np.abs(gm - rm) <= 2e-5 + 2e-3 * np.abs(rm)), (call, np.abs(gm - rm).max())

    # a third call with the second one's arguments (every kernel it needs is loaded by now) must leave the amount of free
    # device memory exactly where it was: nothing was taken from, or returned to, the driver
    free_before, _ = torch.cuda.mem_get_info()
    sa.sparse_attn_row_topk_curve_static(*dev, 1, H, N, D, rows, keep, *got)
    torch.cuda.synchronize()
    free_after, _ = torch.cuda.mem_get_info()
    assert free_after == free_before, (free_before, free_after)
    assert np.array_equal(got[1].cpu().numpy(), gr) and np.array_equal(got[2].cpu().numpy(), gm)


@pytest.mark.gpu
def test_static_scratch_entry_rejects_sizes_beyond_its_fixed_array():
    import torch

    import paper_2606_16317_b200 as sa
    from paper_2606_16317_b200 import binding
    N, D = 4096, 128
    x = torch.zeros((1, 1, N, D), device="cuda", dtype=torch.bfloat16)
    keep = np.array([1], dtype=np.int32)
    fits = binding.STATIC_SCRATCH_FLOATS // N                      # 1024 rows of 4096 keys fill the 16 MiB exactly
    o = _outputs(fits + 1, 1)
    rows = np.zeros((fits + 1, 2), dtype=np.int32)
    with pytest.raises(sa.SparseAttnError) as e:
        sa.sparse_attn_row_topk_curve_static(x, x, x, 1, 1, N, D, rows, keep, *o)
    assert e.value.status == -2 and "static scratch" in e.value.detail
    assert torch.isnan(o[0]).all()                                 # rejected before anything ran
    sa.sparse_attn_row_topk_curve_static(x, x, x, 1, 1, N, D, rows[:fits], keep, *o)      # the largest size is accepted
    torch.cuda.synchronize()
    assert torch.isnan(o[0][:fits]).all() and torch.allclose(o[1][:fits], torch.full_like(o[1][:fits], 1.0))   # uniform row
    for bad_rows, bad_keep in ((np.zeros((binding.STATIC_MAX_ROWS + 1, 2), dtype=np.int32), keep),
                               (rows[:1], np.ones(binding.STATIC_MAX_KEEP + 1, dtype=np.int32))):
        with pytest.raises(sa.SparseAttnError) as e:
            sa.sparse_attn_row_topk_curve_static(x[:, :, :64], x[:, :, :64], x[:, :, :64], 1, 1, 64, D, bad_rows, bad_keep, *o)
        assert e.value.status == -2
