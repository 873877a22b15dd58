"""Property tests on random small shapes (tier 6): hypothesis draws N (ragged), D, mode,
lambda, the decision tile and a logit scale; the CUDA path (through the C ABI) must match the oracle on every draw."""
import math

import numpy as np
import pytest
from hypothesis import HealthCheck, given, settings, strategies as st

from oracle import MODE_DENSE, MODE_DYNAMIC, MODE_FIXED
from workloads import f32_to_bf16_bits

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def parity():
    import torch
    if not torch.cuda.is_available():
        pytest.fail("GPU tests need a CUDA device; there is no CPU fallback")
    import parity_utils
    return parity_utils


@settings(max_examples=40, deadline=None, suppress_health_check=[HealthCheck.function_scoped_fixture], derandomize=True)
@given(N=st.integers(1, 700), D=st.sampled_from([64, 128]), mode=st.sampled_from([MODE_DENSE, MODE_FIXED, MODE_DYNAMIC]),
       lam=st.floats(-8.0, 2.0), sub=st.sampled_from([0, 32, 64]), gain=st.floats(0.3, 3.0), H=st.integers(1, 3),
       seed=st.integers(0, 2 ** 20), head_heavy=st.booleans())
def test_random_shapes_match_oracle(parity, N, D, mode, lam, sub, gain, H, seed, head_heavy):
    rng = np.random.default_rng(seed)
    q = rng.standard_normal((1, H, N, D), dtype=np.float32) * gain
    k = rng.standard_normal((1, H, N, D), dtype=np.float32)
    if head_heavy:
        k[:, :, : max(1, N // 4)] *= 2.0                 # early winners: later tiles get skipped
    v = rng.standard_normal((1, H, N, D), dtype=np.float32)
    qb, kb, vb = (f32_to_bf16_bits(x) for x in (q, k, v))
    tile = 64 if D == 64 else 128
    tile_k = sub if (D == 128 and mode != MODE_DENSE) else 0
    if mode == MODE_FIXED or tile_k:
        lam = min(lam, 0.0)                              # the ABI takes lambda > 0 in DYNAMIC mode with default tiles only
    gpu = parity.run_gpu(qb, kb, vb, mode=mode, lam=lam if mode != MODE_DENSE else -math.inf, tile=tile, tile_k=tile_k)
    parity.check_stats(gpu, N, tile, tile_k or None)
    rep = parity.ParityReport()
    for h in range(H):
        parity.compare_head(gpu, h, qb[0, h], kb[0, h], vb[0, h], tile=tile, tile_k=tile_k or None, mode=mode,
                            lam=lam if mode != MODE_DENSE else -math.inf, report=rep)
    assert rep.ok(), "\n".join(rep.failures[:10])
