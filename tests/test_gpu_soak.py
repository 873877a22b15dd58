"""A bounded, seeded soak over input families far outside the contract workloads (tolerances), in
place of an untracked script: 60 draws of shape, mode, threshold, decision tile and logit range -- Gaussian inputs with
gains up to 6, random-walk logits that sweep +-1500 nats along the keys, and near one-hot rows on values with |v| > 4.
Everywhere: decisions equal to the oracle's wherever |g| exceeds the margin tolerance, lse within 2e-3, margins within
that tolerance -- 1e-3 + 1e-6 max|S|: BASELINE.json's 1e-3 on logits of the contract's size, plus the fp32 resolution of
S itself where logits reach hundreds of nats (ulp(1500) = 1.2e-4, a margin is a difference of such numbers).  For the output
the 2e-2 of BASELINE.json is a statement about the contract workloads (|o| << 1, |v| <= 4.5); here the scale-free bound
of parity_utils.scale_free_out_tol is asserted (2^-8 (|o| + max|v|) + 1e-3: the two bf16 roundings of the path), and,
on the draws whose values stay inside the contract's range (|v| <= 4.5), the 2e-2 as well."""
import math

import numpy as np
import pytest

from oracle import MODE_DENSE, MODE_DYNAMIC, MODE_FIXED
from workloads import bf16_bits_to_f64, f32_to_bf16_bits

pytestmark = pytest.mark.gpu

N_DRAWS = 60


def _draw(i):
    rng = np.random.default_rng([61, i])
    family = ("gauss", "walk", "onehot")[i % 3]
    D = int(rng.choice([64, 128]))
    N = int(rng.integers(1, 900))
    H = int(rng.integers(1, 3))
    mode = int(rng.choice([MODE_DENSE, MODE_FIXED, MODE_DYNAMIC]))
    tile_k = int(rng.choice([0, 32, 64])) if (D == 128 and mode != MODE_DENSE) else 0
    lam = -math.inf if mode == MODE_DENSE else float(rng.uniform(-10.0, 0.0))
    if mode == MODE_DYNAMIC and tile_k == 0 and rng.random() < 0.3:
        lam = float(rng.uniform(0.0, 2.0))
    vgain = 1.0
    if family == "gauss":
        q = rng.standard_normal((1, H, N, D), dtype=np.float32) * float(rng.uniform(0.3, 6.0))
        k = rng.standard_normal((1, H, N, D), dtype=np.float32)
    elif family == "walk":
        # logits = scale * a * walk_c along the keys: a random walk whose range is stretched to +-span nats
        span = float(rng.choice([20.0, 200.0, 1500.0]))
        walk = np.cumsum(rng.standard_normal((1, H, N)), axis=-1)
        walk = walk / max(1e-9, np.abs(walk).max()) * 256.0
        a = span * math.sqrt(D) / 256.0
        q = rng.standard_normal((1, H, N, D), dtype=np.float32) * 0.05
        q[..., 0] = a * rng.choice([-1.0, 1.0], size=(1, H, N))
        k = rng.standard_normal((1, H, N, D), dtype=np.float32) * 0.05
        k[..., 0] = walk
    else:
        q = rng.standard_normal((1, H, N, D), dtype=np.float32) * float(rng.uniform(8.0, 20.0))
        k = rng.standard_normal((1, H, N, D), dtype=np.float32)
        vgain = 3.0
    v = rng.standard_normal((1, H, N, D), dtype=np.float32) * vgain
    return family, D, N, H, mode, tile_k, lam, tuple(f32_to_bf16_bits(x) for x in (q, k, v))


@pytest.mark.parametrize("block", range(6))
def test_soak_block(block):
    import torch
    if not torch.cuda.is_available():
        pytest.fail("GPU tests need a CUDA device; there is no CPU fallback")
    import parity_utils as parity
    worst = {"out_over_contract": 0.0, "lse": 0.0, "margin": 0.0}
    for i in range(block * (N_DRAWS // 6), (block + 1) * (N_DRAWS // 6)):
        family, D, N, H, mode, tile_k, lam, (qb, kb, vb) = _draw(i)
        tile = 64 if D == 64 else 128
        gpu = parity.run_gpu(qb, kb, vb, mode=mode, lam=lam, tile=tile, tile_k=tile_k)
        parity.check_stats(gpu, N, tile, tile_k or None)
        rep = parity.ParityReport()
        for h in range(H):
            v64 = bf16_bits_to_f64(vb[0, h])
            smax = float(np.abs(bf16_bits_to_f64(qb[0, h]) @ bf16_bits_to_f64(kb[0, h]).T).max()) / math.sqrt(D)
            mtol = parity.MARGIN_TOL + 1e-6 * smax
            in_contract_range = np.abs(v64).max() <= 4.5
            parity.compare_head(gpu, h, qb[0, h], kb[0, h], vb[0, h], tile=tile, tile_k=tile_k or None, mode=mode, lam=lam,
                                report=rep, out_tol=parity.scale_free_out_tol(v64), margin_tol=mtol)
            if in_contract_range:
                before = len(rep.failures)
                r2 = parity.compare_head(gpu, h, qb[0, h], kb[0, h], vb[0, h], tile=tile, tile_k=tile_k or None, mode=mode, lam=lam,
                                         margin_tol=mtol)
                rep.failures.extend(f for f in r2.failures if "out " in f)
                worst["out_over_contract"] = max(worst["out_over_contract"], r2.max_abs)
                assert len(rep.failures) >= before
        worst["lse"] = max(worst["lse"], rep.max_lse_abs)
        worst["margin"] = max(worst["margin"], rep.max_margin_abs)
        assert rep.ok(), f"draw {i} ({family}, D={D}, N={N}, H={H}, mode={mode}, tile_k={tile_k}, lam={lam:.3f}):\n" + "\n".join(rep.failures[:10])
        plain = parity.run_gpu(qb, kb, vb, mode=mode, lam=lam, tile=tile, tile_k=tile_k, debug=False)
        assert np.array_equal(plain.out, gpu.out) and np.array_equal(plain.stats, gpu.stats), f"draw {i}: plain != debug build"
    print(f"[soak block {block}] worst out max-abs on |v| <= 4.5 draws {worst['out_over_contract']:.2e}, "
          f"lse {worst['lse']:.2e}, margin {worst['margin']:.2e}")
