"""GPU parity tests: the CUDA path (through the C ABI) against the CPU oracle, element by element.

Run with `-m gpu` on a B200.  Tolerances are BASELINE.json's (tests/parity_utils.py).
"""
import math

import numpy as np
import pytest

import oracle
from oracle import MODE_DENSE, MODE_DYNAMIC, MODE_FIXED
from workloads import CONFIGS, bf16_bits_to_f64, f32_to_bf16_bits, make_head, make_qkv

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def parity():
    import torch
    if not torch.cuda.is_available():
        pytest.fail("GPU tests need a CUDA device; there is no CPU fallback")
    import parity_utils
    return parity_utils


def _assert_ok(rep, what):
    print(f"[parity] {what}: tiles={rep.tiles_checked} decisions={rep.decisions_checked} "
          f"disagree={rep.disagreements} near-margin-first={rep.near_margin_disagreements} "
          f"diverged_qtiles={rep.diverged_qtiles} out max-abs={rep.max_abs:.3e} mean-abs={rep.mean_abs:.3e} "
          f"lse max-abs={rep.max_lse_abs:.3e} margin max-abs={rep.max_margin_abs:.3e}")
    assert rep.ok(), "\n".join(rep.failures[:10])


# ------------------------------------------------------------------ config 0 in full (and its aligned variant)
CFG0_LAMBDAS = [oracle.lambda_from_recall(r, 1024) for r in (0.90, 0.95, 0.99)] + [-1.0, -2.0, -3.0, -4.0, -6.0]


@pytest.mark.parametrize("name", ["cfg0", "cfg0_aligned"])
def test_cfg0_full_all_modes(parity, seed, name):
    cfg = CONFIGS[name]
    q, k, v = make_qkv(cfg, seed)
    settings = [(MODE_DENSE, -math.inf)] + [(m, lam) for m in (MODE_FIXED, MODE_DYNAMIC) for lam in CFG0_LAMBDAS]
    total_skipped = 0
    for mode, lam in settings:
        gpu = parity.run_gpu(q, k, v, mode=mode, lam=lam, tile=cfg.tile)
        parity.check_stats(gpu, cfg.N, cfg.tile)
        rep = parity.ParityReport()
        for h in range(cfg.H):
            parity.compare_head(gpu, h, q[0, h], k[0, h], v[0, h], tile=cfg.tile, mode=mode, lam=lam, report=rep)
        _assert_ok(rep, f"{name} mode={mode} lambda={lam:.3f} sparsity={gpu.stats[:, 1].sum() / gpu.stats.sum():.3f}")
        if mode == MODE_DENSE:
            assert gpu.stats[:, 1].sum() == 0
        total_skipped += int(gpu.stats[:, 1].sum())
    assert total_skipped > 0       # the skip path really ran


# ------------------------------------------------------------------ ragged shapes, several tiles, both head dims
@pytest.mark.parametrize("B,H,N,D", [(1, 2, 1000, 64), (2, 1, 1000, 128), (1, 1, 40, 64), (1, 1, 129, 128),
                                     (1, 1, 1, 128), (1, 3, 2125, 128), (1, 1, 64, 64), (1, 1, 193, 64)])
def test_ragged_random_inputs(parity, seed, B, H, N, D):
    tile = 64 if D == 64 else 128
    rng = np.random.default_rng([seed, B, H, N, D])
    q = f32_to_bf16_bits(rng.standard_normal((B, H, N, D)).astype(np.float32) * 1.8)
    k = f32_to_bf16_bits(rng.standard_normal((B, H, N, D)).astype(np.float32) * 1.8)
    v = f32_to_bf16_bits(rng.standard_normal((B, H, N, D)).astype(np.float32))
    for mode, lam in [(MODE_DENSE, 0.0), (MODE_DYNAMIC, -2.0), (MODE_DYNAMIC, -4.0), (MODE_FIXED, -1.0),
                      (MODE_FIXED, -3.0), (MODE_DYNAMIC, -math.inf)]:
        gpu = parity.run_gpu(q, k, v, mode=mode, lam=lam, tile=tile)
        parity.check_stats(gpu, N, tile)
        rep = parity.ParityReport()
        for b in range(B):
            for h in range(H):
                parity.compare_head(gpu, b * H + h, q[b, h], k[b, h], v[b, h], tile=tile, mode=mode, lam=lam,
                                    report=rep)
        _assert_ok(rep, f"ragged B{B} H{H} N{N} D{D} mode={mode} lambda={lam}")


def test_softmax_scale_override(parity, seed):
    rng = np.random.default_rng([seed, 31])
    q, k, v = (f32_to_bf16_bits(rng.standard_normal((1, 1, 300, 128)).astype(np.float32)) for _ in range(3))
    gpu = parity.run_gpu(q, k, v, mode=MODE_DYNAMIC, lam=-3.0, tile=128, scale=0.2)
    rep = parity.compare_head(gpu, 0, q[0, 0], k[0, 0], v[0, 0], tile=128, mode=MODE_DYNAMIC, lam=-3.0, scale=0.2)
    _assert_ok(rep, "scale override")


# ------------------------------------------------------------------ closed forms, decisions bit-exact
def _uniform_inputs(N, D, seed):
    rng = np.random.default_rng(seed)
    q = np.zeros((1, 1, N, D), dtype=np.uint16)
    k = f32_to_bf16_bits(rng.standard_normal((1, 1, N, D)).astype(np.float32))
    v = f32_to_bf16_bits(rng.standard_normal((1, 1, N, D)).astype(np.float32))
    return q, k, v


@pytest.mark.parametrize("D,tile,N,lam", [(64, 64, 1024, -6.0), (64, 64, 1024, -5.0), (64, 64, 1024, -7.5),
                                          (128, 128, 2048, -6.0), (128, 128, 2000, -7.0)])
def test_uniform_closed_form_on_gpu(parity, D, tile, N, lam):
    """P7 on the GPU: all logits equal -> DYNAMIC keeps exactly k* leading tiles, FIXED skips nothing."""
    T = -(-N // tile)
    kept = min(T, int(math.floor(math.exp(-lam) / tile)) + 1)
    q, k, v = _uniform_inputs(N, D, 3)
    gpu = parity.run_gpu(q, k, v, mode=MODE_DYNAMIC, lam=lam, tile=tile)
    expect = np.zeros((T, T), dtype=np.uint8)
    expect[:, kept:] = 1
    np.testing.assert_array_equal(gpu.skip[0], expect)
    assert gpu.stats[0].tolist() == [T * kept, T * (T - kept)]
    vv = bf16_bits_to_f64(v[0, 0])
    np.testing.assert_allclose(gpu.out[0], np.broadcast_to(vv[:min(N, kept * tile)].mean(axis=0), (N, D)),
                               atol=parity.OUT_MAX_ABS)
    np.testing.assert_allclose(gpu.lse[0], math.log(min(N, kept * tile)), atol=parity.LSE_ABS)
    fix = parity.run_gpu(q, k, v, mode=MODE_FIXED, lam=lam, tile=tile)
    assert fix.stats[0].tolist() == [T * T, 0]


@pytest.mark.parametrize("winner_last", [False, True])
def test_winner_closed_forms_on_gpu(parity, winner_last):
    """P8 / P9 on the GPU (D = 128, 128 x 128 tiles)."""
    N, D, tile, lam, W = 2048, 128, 128, -6.0, 8.0
    T = N // tile
    a = math.sqrt(W * math.sqrt(D))
    a = float(bf16_bits_to_f64(f32_to_bf16_bits(np.float32([a])))[0])
    Wb = a * a / math.sqrt(D)
    qf = np.zeros((1, 1, N, D), dtype=np.float32)
    kf = np.zeros((1, 1, N, D), dtype=np.float32)
    qf[..., 0] = a
    kf[0, 0, N - 3 if winner_last else 5, 0] = a
    v = f32_to_bf16_bits(np.random.default_rng(4).standard_normal((1, 1, N, D)).astype(np.float32))
    q, k = f32_to_bf16_bits(qf), f32_to_bf16_bits(kf)
    dyn = parity.run_gpu(q, k, v, mode=MODE_DYNAMIC, lam=lam, tile=tile)
    fix = parity.run_gpu(q, k, v, mode=MODE_FIXED, lam=lam, tile=tile)
    expect = np.zeros((T, T), dtype=np.uint8)
    if winner_last:
        kstar = int(math.floor(math.exp(-lam) / tile)) + 1
        expect[:, kstar:T - 1] = 1
        np.testing.assert_array_equal(dyn.skip[0], expect)
        assert fix.stats[0, 1] == 0
        np.testing.assert_allclose(dyn.lse[0], math.log(kstar * tile + math.exp(Wb) + tile - 1), atol=parity.LSE_ABS)
    else:
        expect[:, 1:] = 1
        np.testing.assert_array_equal(dyn.skip[0], expect)
        np.testing.assert_array_equal(fix.skip[0], expect)
        np.testing.assert_allclose(dyn.lse[0], math.log(math.exp(Wb) + tile - 1), atol=parity.LSE_ABS)


# ------------------------------------------------------------------ full-size configs, oracle on sampled Q tiles
def _sample_qtiles(T, rng, n_random):
    return sorted(set([0, T - 1] + [int(x) for x in rng.choice(np.arange(1, T - 1), size=n_random, replace=False)]))


def _assert_plain_build_equals_debug_build(parity, q, k, v, dbg, *, mode, lam, tile):
    """The instantiation bench.py times (no parity outputs: kDebug = false) against the oracle-checked debug run of the
    same call: equal tile counts, bit-equal out and lse.  The debug build synchronises the vote with named barriers, the
    plain build with the dec mbarrier and the speculative re-issue path; decisions and arithmetic order are the same."""
    plain = parity.run_gpu(q, k, v, mode=mode, lam=lam, tile=tile, debug=False)
    np.testing.assert_array_equal(plain.stats, dbg.stats)
    np.testing.assert_array_equal(plain.out, dbg.out)
    np.testing.assert_array_equal(plain.lse, dbg.lse)


@pytest.mark.parametrize("name,lam_dyn,lam_fix", [("cfg1", -3.0, -1.0), ("cfg1_aligned", -6.0, -6.0)])
def test_cfg1_full_size_sampled_tiles(parity, seed, name, lam_dyn, lam_fix):
    """Config 1 (B=1, H=24, N=32760, D=128) at full size.  The debug build (skip_mask_out / margin_out set) is checked
    against the oracle on the first, the last (ragged) and random Q tiles of 3 heads, all 256 K tiles; the plain build
    -- the launch configuration bench.py times -- must then reproduce the debug run bit for bit."""
    cfg = CONFIGS[name]
    q, k, v = make_qkv(cfg, seed)
    rng = np.random.default_rng([seed, 1234])
    heads = [0, 11, 23]
    for mode, lam in [(MODE_DENSE, -math.inf), (MODE_DYNAMIC, lam_dyn), (MODE_FIXED, lam_fix),
                      (MODE_DYNAMIC, oracle.lambda_from_preal(1.5, cfg.tile, cfg.N))]:
        gpu = parity.run_gpu(q, k, v, mode=mode, lam=lam, tile=cfg.tile)
        parity.check_stats(gpu, cfg.N, cfg.tile)
        rep = parity.ParityReport()
        for h in heads:
            qt = _sample_qtiles(256, rng, 2)
            parity.compare_head(gpu, h, q[0, h], k[0, h], v[0, h], tile=cfg.tile, mode=mode, lam=lam, qtiles=qt,
                                report=rep)
        _assert_ok(rep, f"{name} mode={mode} lambda={lam} sparsity={gpu.stats[:, 1].sum() / gpu.stats.sum():.4f}")
        _assert_plain_build_equals_debug_build(parity, q, k, v, gpu, mode=mode, lam=lam, tile=cfg.tile)


def test_cfg2_contract_generator_extreme_heads(parity, seed):
    """Config 2's generator (per-head temperature tau_h in [1, 2.5], field sigma_h in [1, 6]): the heads with the
    smallest and the largest tau_h (logits up to tau^2 sqrt(D) = 11 and 71: different exponent ranges), sampled Q tiles."""
    from workloads.generator import head_params
    cfg = CONFIGS["cfg2"]
    taus = [head_params(cfg, seed, h)[0] for h in range(cfg.H)]
    heads = [int(np.argmin(taus)), int(np.argmax(taus))]
    q, k, v = make_qkv(cfg, seed, heads=heads)
    rng = np.random.default_rng([seed, 222])
    T = -(-cfg.N // cfg.tile)
    for mode, lam in [(MODE_DENSE, -math.inf), (MODE_DYNAMIC, oracle.lambda_from_preal(1.5, cfg.tile, cfg.N)),
                      (MODE_DYNAMIC, -3.0), (MODE_FIXED, -2.0)]:
        gpu = parity.run_gpu(q, k, v, mode=mode, lam=lam, tile=cfg.tile)
        parity.check_stats(gpu, cfg.N, cfg.tile)
        rep = parity.ParityReport()
        for i in range(2):
            parity.compare_head(gpu, i, q[0, i], k[0, i], v[0, i], tile=cfg.tile, mode=mode, lam=lam,
                                qtiles=_sample_qtiles(T, rng, 2), report=rep)
        _assert_ok(rep, f"cfg2 heads {heads} (tau {taus[heads[0]]:.2f}, {taus[heads[1]]:.2f}) mode={mode} lambda={lam:.3f} "
                        f"sparsity={gpu.stats[:, 1].sum() / gpu.stats.sum():.4f}")
        _assert_plain_build_equals_debug_build(parity, q, k, v, gpu, mode=mode, lam=lam, tile=cfg.tile)


def test_cfg3_contract_generator_sampled_tiles(parity, seed):
    """Config 3 as BASELINE.json states it (N = 75600: 591 tiles, 80-row ragged tail; per-head tau / sigma), three heads,
    first / ragged-last / four random Q tiles, DYNAMIC at the paper's lambda = -6 and -8 and at the
    strict map of recall 0.9, FIXED at -6."""
    cfg = CONFIGS["cfg3"]
    heads = [0, 19, 39]
    q, k, v = make_qkv(cfg, seed, heads=heads)
    rng = np.random.default_rng([seed, 333])
    T = -(-cfg.N // cfg.tile)
    assert T == 591 and cfg.N - 590 * 128 == 80
    for mode, lam in [(MODE_DYNAMIC, -6.0), (MODE_DYNAMIC, -8.0), (MODE_DYNAMIC, oracle.lambda_from_recall(0.9, cfg.N)),
                      (MODE_FIXED, -6.0)]:
        gpu = parity.run_gpu(q, k, v, mode=mode, lam=lam, tile=cfg.tile)
        parity.check_stats(gpu, cfg.N, cfg.tile)
        rep = parity.ParityReport()
        for i in range(len(heads)):
            parity.compare_head(gpu, i, q[0, i], k[0, i], v[0, i], tile=cfg.tile, mode=mode, lam=lam,
                                qtiles=_sample_qtiles(T, rng, 4), report=rep)
        _assert_ok(rep, f"cfg3 heads {heads} mode={mode} lambda={lam:.3f} sparsity={gpu.stats[:, 1].sum() / gpu.stats.sum():.4f}")
        _assert_plain_build_equals_debug_build(parity, q, k, v, gpu, mode=mode, lam=lam, tile=cfg.tile)


@pytest.mark.parametrize("noise_a", [0.1, 0.9])
def test_cfg4_drift_generator_sampled_tiles(parity, seed, noise_a):
    """Config 4 (drift sweep at the 720p shape): X = (1 - a) field + a noise at the two ends of the sweep."""
    cfg = CONFIGS["cfg4"]
    heads = [5, 30]
    q, k, v = make_qkv(cfg, seed, heads=heads, noise_a=noise_a)
    rng = np.random.default_rng([seed, 444, int(noise_a * 10)])
    T = -(-cfg.N // cfg.tile)
    lam = oracle.lambda_from_preal(1.5, cfg.tile, cfg.N)
    for mode in (MODE_DYNAMIC, MODE_FIXED):
        gpu = parity.run_gpu(q, k, v, mode=mode, lam=lam, tile=cfg.tile)
        parity.check_stats(gpu, cfg.N, cfg.tile)
        rep = parity.ParityReport()
        for i in range(len(heads)):
            parity.compare_head(gpu, i, q[0, i], k[0, i], v[0, i], tile=cfg.tile, mode=mode, lam=lam,
                                qtiles=_sample_qtiles(T, rng, 2), report=rep)
        _assert_ok(rep, f"cfg4 a={noise_a} mode={mode} lambda={lam:.3f} sparsity={gpu.stats[:, 1].sum() / gpu.stats.sum():.4f}")
        _assert_plain_build_equals_debug_build(parity, q, k, v, gpu, mode=mode, lam=lam, tile=cfg.tile)


def test_cfg3_shape_sampled_tiles(parity, seed):
    """Config 3's N = 75600 on 2 heads of the supplementary aligned variant (where most tiles are skipped: long skip runs,
    the speculative Q K^T path)."""
    cfg = CONFIGS["cfg3_aligned"]
    q, k, v = make_qkv(cfg, seed, heads=[3, 17])
    rng = np.random.default_rng([seed, 4321])
    for mode, lam in [(MODE_DYNAMIC, -6.0), (MODE_FIXED, -6.0)]:
        gpu = parity.run_gpu(q, k, v, mode=mode, lam=lam, tile=cfg.tile)
        parity.check_stats(gpu, cfg.N, cfg.tile)
        rep = parity.ParityReport()
        for h in range(2):
            qt = [0, 590] + [int(x) for x in rng.choice(np.arange(1, 590), size=1)]
            parity.compare_head(gpu, h, q[0, h], k[0, h], v[0, h], tile=cfg.tile, mode=mode, lam=lam, qtiles=qt,
                                report=rep)
        _assert_ok(rep, f"cfg3_aligned mode={mode} lambda={lam} sparsity={gpu.stats[:, 1].sum() / gpu.stats.sum():.4f}")
        _assert_plain_build_equals_debug_build(parity, q, k, v, gpu, mode=mode, lam=lam, tile=cfg.tile)


# ------------------------------------------------------------------ invariants that hold at any size
def test_dynamic_superset_of_fixed_and_recall_on_gpu(parity, seed):
    """P6 and P3 evaluated from GPU outputs alone on full config-1-shaped heads (aligned variant)."""
    cfg = CONFIGS["cfg1_aligned"]
    q, k, v = make_qkv(cfg, seed, heads=[2, 9])
    lam = -8.0
    dense = parity.run_gpu(q, k, v, mode=MODE_DENSE, tile=cfg.tile, debug=False)
    dyn = parity.run_gpu(q, k, v, mode=MODE_DYNAMIC, lam=lam, tile=cfg.tile)
    fix = parity.run_gpu(q, k, v, mode=MODE_FIXED, lam=lam, tile=cfg.tile)
    # P6 holds exactly in exact arithmetic; on the GPU allow disagreement only at near-margin tiles
    viol = (fix.skip == 1) & (dyn.skip == 0)
    assert np.all(np.abs(dyn.margin[viol]) <= parity.MARGIN_TOL)
    assert dyn.stats[:, 1].sum() >= fix.stats[:, 1].sum() - viol.sum()
    for res in (dyn, fix):
        recall = np.exp(res.lse.astype(np.float64) - dense.lse.astype(np.float64))
        skipped_cols = np.repeat(res.skip.sum(axis=2) * cfg.tile, cfg.tile, axis=1)[:, :cfg.N]
        assert np.all(1.0 - recall < skipped_cols * math.exp(lam) + 5e-3)   # P3 (+ fp32 lse rounding)


def test_host_buffer_entry_point(parity, seed):
    import paper_2606_16317_b200 as sa
    cfg = CONFIGS["cfg0"]
    q, k, v = make_qkv(cfg, seed)
    out = np.zeros_like(q)
    lse = np.zeros((1, cfg.H, cfg.N), dtype=np.float32)
    stats = np.zeros((1, cfg.H, 2), dtype=np.int64)
    p = sa.make_params(lam=-2.0)
    sa.sparse_attn_fwd_host(q, k, v, out, lse, 1, cfg.H, cfg.N, cfg.D, p, MODE_DYNAMIC, stats)
    dev = parity.run_gpu(q, k, v, mode=MODE_DYNAMIC, lam=-2.0, tile=cfg.tile)
    np.testing.assert_array_equal(bf16_bits_to_f64(out).reshape(cfg.H, cfg.N, cfg.D), dev.out)
    np.testing.assert_array_equal(stats.reshape(cfg.H, 2), dev.stats)


# ------------------------------------------------------------------ in place of compute-sanitizer (profiles/sanitizer_r02.md)
def test_sanitizer_cases_run_clean():
    """Every kernel instantiation on small cases (the script written for compute-sanitizer, which this pool does not
    allow): finite outputs, consistent counts, no CUDA error."""
    import importlib.util
    import os
    spec = importlib.util.spec_from_file_location("sanitizer_cases", os.path.join(os.path.dirname(__file__), "sanitizer_cases.py"))
    mod = importlib.util.module_from_spec(spec)
    spec.loader.exec_module(mod)
    mod.main()


@pytest.mark.parametrize("tile_k", [0, 32])
def test_repeated_launches_are_bit_identical(parity, seed, tile_k):
    """The timed build on a workload with mixed skip / keep decisions (speculative Q K^T, re-issue after a mis-speculated
    skip, on-demand V, vote ring), 20 launches: a race between the softmax warps, the issuers and the V producer would
    show up as a run that differs from the others.  The first run is the one the oracle checks."""
    import torch
    cfg = CONFIGS["cfg1_aligned"]
    heads = [0, 7]
    q, k, v = make_qkv(cfg, seed, heads=heads)
    lam = oracle.lambda_from_preal(1.5, tile_k or cfg.tile, cfg.N)
    first = parity.run_gpu(q, k, v, mode=MODE_DYNAMIC, lam=lam, tile=cfg.tile, tile_k=tile_k, debug=False)
    assert 0.2 < first.stats[:, 1].sum() / first.stats.sum() < 0.95
    T = 256
    for i, h in enumerate(heads):
        ref = oracle.run_head(q[0, i], k[0, i], v[0, i], tile=cfg.tile, tile_k=tile_k or cfg.tile, lam=lam, mode=MODE_DYNAMIC,
                              qtiles=[0, 100, T - 1])
        o_ref, lse_ref = ref.rows()
        rows = np.concatenate([np.arange(t * 128, min((t + 1) * 128, cfg.N)) for t in (0, 100, T - 1)])
        if np.all(np.abs(ref.margin) > parity.MARGIN_TOL):
            assert np.abs(first.out[i][rows] - o_ref).max() < parity.OUT_MAX_ABS
            assert np.abs(first.lse[i][rows] - lse_ref).max() < parity.LSE_ABS
    for _ in range(19):
        again = parity.run_gpu(q, k, v, mode=MODE_DYNAMIC, lam=lam, tile=cfg.tile, tile_k=tile_k, debug=False)
        np.testing.assert_array_equal(again.stats, first.stats)
        np.testing.assert_array_equal(again.out, first.out)
        np.testing.assert_array_equal(again.lse, first.lse)
    torch.cuda.synchronize()


def test_cycle_counters_of_the_debug_instantiation(parity, seed):
    """params->cycles_out (measurement support of bench.py): {sum of per-CTA clock64 cycles, CTAs of the launch}; the
    buffer is overwritten on every call, selecting the debug instantiation changes no result, and the host-buffer entry
    refuses it."""
    import torch

    import paper_2606_16317_b200 as sa
    for name in ("cfg0",):
        cfg = CONFIGS[name]
        q, k, v = make_qkv(cfg, seed)
        dq, dk, dv = (parity.to_dev_bf16(np.ascontiguousarray(x)) for x in (q, k, v))
        out = torch.empty_like(dq)
        ref = torch.empty_like(dq)
        cyc = torch.full((2,), 12345, device="cuda", dtype=torch.int64)
        ctas_per_head = (-(-cfg.N // 128) + 1) // 2                       # two 128-row MMA tiles per CTA
        for mode, lam in ((MODE_DENSE, -math.inf), (MODE_DYNAMIC, -3.0)):
            sa.sparse_attn_fwd(dq, dk, dv, ref, None, cfg.B, cfg.H, cfg.N, cfg.D, sa.make_params(lam=lam), mode, None)
            for _ in range(2):
                sa.sparse_attn_fwd(dq, dk, dv, out, None, cfg.B, cfg.H, cfg.N, cfg.D, sa.make_params(lam=lam, cycles_out=cyc), mode, None)
                torch.cuda.synchronize()
                cycles, ctas = cyc.tolist()
                assert ctas == cfg.B * cfg.H * ctas_per_head
                assert 1000 * ctas < cycles < 10 ** 9 * ctas
            assert torch.equal(out.view(torch.int16), ref.view(torch.int16))
    with pytest.raises(sa.SparseAttnError) as e:
        sa.sparse_attn_fwd_host(q, k, v, np.zeros_like(q), None, cfg.B, cfg.H, cfg.N, cfg.D, sa.make_params(lam=-3.0, cycles_out=cyc),
                                MODE_DYNAMIC, None)
    assert e.value.status == -6
