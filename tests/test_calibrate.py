"""Iso-recall calibration: bisection logic on the CPU, the GPU loop against the oracle."""
import math

import numpy as np
import pytest
import torch

from paper_2606_16317_b200.calibrate import bisect_lambda


def test_bisection_finds_the_largest_lambda_meeting_the_target():
    f = lambda lam: 1.0 / (1.0 + math.exp(lam + 7.0))       # smooth, decreasing; f(lam) = 0.9 at lam = -7 - ln 9
    lam, r = bisect_lambda(f, 0.9, -30.0, 0.0, iters=30)
    assert abs(lam - (-7.0 - math.log(9.0))) < 1e-6 and r >= 0.9
    steps = lambda lam: 1.0 if lam < -5 else (0.8 if lam < -2 else 0.1)   # plateaus, as tile decisions produce
    lam, r = bisect_lambda(steps, 0.75, -30.0, 0.0, iters=30)
    assert -2.0 - 1e-6 < lam < -2.0 and r == 0.8
    assert bisect_lambda(steps, 0.05, -30.0, 0.0) == (0.0, 0.1)          # hi already meets the target
    assert bisect_lambda(lambda lam: 0.5, 0.9, -30.0, 0.0) == (-30.0, 0.5)   # unreachable: lo is returned


@pytest.mark.gpu
@pytest.mark.parametrize("mode_name,target,stat", [("dynamic", 0.95, "mean"), ("fixed", 0.99, "min"), ("dynamic", 0.9, "min")])
def test_gpu_calibration_meets_target_and_agrees_with_oracle(seed, mode_name, target, stat):
    import oracle
    import paper_2606_16317_b200 as sa
    from paper_2606_16317_b200.calibrate import calibrate_lambda
    from workloads import CONFIGS, make_qkv

    cfg = CONFIGS["cfg0_aligned"]
    qb, kb, vb = make_qkv(cfg, seed)
    q, k, v = (torch.from_numpy(x.view(np.int16)).cuda().view(torch.bfloat16) for x in (qb, kb, vb))
    mode = {"fixed": sa.MODE_FIXED, "dynamic": sa.MODE_DYNAMIC}[mode_name]
    res = calibrate_lambda(q, k, v, cfg.B, cfg.H, cfg.N, cfg.D, mode, target, statistic=stat, iters=12)
    assert res["recall_" + stat] >= target
    assert res["sparsity"] > 0.0                          # this workload has tiles to skip at these targets
    # the oracle at the calibrated lambda measures the same recall and the same sparsity
    omode = {"fixed": oracle.MODE_FIXED, "dynamic": oracle.MODE_DYNAMIC}[mode_name]
    rec, skipped, total = [], 0, 0
    for h in range(cfg.H):
        dense = oracle.run_head(qb[0, h], kb[0, h], vb[0, h], tile=cfg.tile, lam=-math.inf, mode=oracle.MODE_DENSE)
        sp = oracle.run_head(qb[0, h], kb[0, h], vb[0, h], tile=cfg.tile, lam=np.float32(res["lambda"]), mode=omode)
        rec.append(np.exp(sp.rows()[1] - dense.rows()[1]))
        skipped += sp.skipped
        total += sp.skipped + sp.executed
    rec = np.concatenate(rec)
    o_stat = rec.min() if stat == "min" else rec.mean()
    assert abs(o_stat - res["recall_" + stat]) < 2e-3
    assert abs(skipped / total - res["sparsity"]) < 0.02   # near-margin tiles may differ (R13)
