#!/usr/bin/env python
"""bench.py -- times the tile-skipping attention forward on synthetic Wan-2.2-shaped inputs.

One "step" = one sparse_attn_fwd call (the whole hot path) over one batch of
BASELINE.json config 3 (B=1, H=40, N=75600, D=128, 128x128 tiles: the Wan2.2-14B 720p shape the paper quotes its
threshold for) in DYNAMIC mode at the paper's Eq. 7 threshold (P_real = 1.5 -> lambda = -5.98, the paper's "-6",
PAPER.md:139).  The same kernel's DENSE and FIXED modes are timed beside it, on the contract generator, on the
supplementary aligned variant and on the contract data re-ordered into bricks.

  python bench.py [--gpus N] [--steps K] [--warmup W] [--impl reference] [--config cfgX]
  python bench.py --report cfg2|cfg3|cfg4|masks|kurtosis     (the sweeps BASELINE.json configs[2..4] ask for; JSON)

Prints ONE JSON line on rank 0.  N > 1 (under torchrun): every rank runs its own batch (heads are independent
units: no data-path collective, weak scaling), stats are all-gathered.
"""
from __future__ import annotations

import argparse
import json
import math
import os
import re
import subprocess
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

from workloads import CONFIGS, make_qkv  # noqa: E402

METRIC = "attention ms & effective TFLOP/s vs dense mode at Wan-2.2 shapes; sparsity %; % tensor peak"
UNIT = "TFLOP/s (dense-equivalent attention FLOP / time)"       # the same string in both arms
DEFAULT_CONFIG = "cfg3"
P_REAL = 1.5            # Eq. 7 "transition region" constant
FALLBACK_TFLOPS = 1590.0
BRICK = (4, 4, 8)       # token re-ordering brick (t, h, w): 128 tokens = one attention tile
ROUNDS = ("r03", "r02")          # tracked ncu summaries, newest first


# ---------------------------------------------------------------------------------------------- peaks, names, profiles
def measured_peaks():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(path):
        with open(path) as f:
            p = json.load(f)
        return float(p["bf16_tflops"]), float(p.get("bf16_tflops_sustained", p["bf16_tflops"])), "measured"
    return FALLBACK_TFLOPS, 1400.0, "fallback"


def measured_hbm():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(path):
        with open(path) as f:
            return float(json.load(f)["hbm_gbs"])
    return 6650.0                                           # fallback stated in B200_PROFILING.md


def eq7_lambda(cfg, tile_k=None, p_real=P_REAL):
    return math.log(p_real) + math.log((tile_k or cfg.tile) / cfg.N)        # Eq. 7


def workload_name(cfg):
    kind = "supplementary aligned variant of " if cfg.aligned else ""
    gen = (f"per-head tau~U[1,2.5] sigma~U[1,6] a={cfg.noise_a}" if cfg.per_head
           else f"sigma={cfg.sigma} a={cfg.noise_a} tau={cfg.tau}")
    return (f"{kind}BASELINE.json configs[{cfg.config_id}] ({cfg.name}): B={cfg.B} H={cfg.H} N={cfg.N} (grid {cfg.grid}) "
            f"D={cfg.D}, {cfg.tile}x{cfg.tile} tiles, generator {gen}")


def _ncu_summary(config, mode):
    """The newest tracked ncu summary of this config and mode (profiles/ncu_<mode>_<config>_<round>.md, written from one
    `ncu --set full` capture): ({metric: value in base units}, relative path) or ({}, None)."""
    scale = {"byte": 1.0, "Kbyte": 1e3, "Mbyte": 1e6, "Gbyte": 1e9, "Tbyte": 1e12, "cycle": 1.0, "ms": 1e-3, "%": 1.0}
    for rnd in ROUNDS:
        path = os.path.join(ROOT, "profiles", f"ncu_{mode}_{config}_{rnd}.md")
        if not os.path.exists(path):
            continue
        vals = {}
        with open(path) as f:
            for line in f:
                m = re.match(r"\|\s*([\w.]+)\s*\|\s*([0-9.,]+)\s*\|\s*([\w%]*)\s*\|", line)
                if m and m.group(3) in scale:
                    vals[m.group(1)] = float(m.group(2).replace(",", "")) * scale[m.group(3)]
        return vals, os.path.relpath(path, ROOT)
    return {}, None


def ncu_traffic(config, mode):
    """dram__bytes_read.sum + dram__bytes_write.sum of one launch, from the tracked ncu summary; None if there is none."""
    vals, path = _ncu_summary(config, mode)
    total = vals.get("dram__bytes_read.sum", 0.0) + vals.get("dram__bytes_write.sum", 0.0)
    return (total or None), path


def dense_flop(BH, N, D):
    return 4.0 * BH * N * N * D


def executed_flop(BH, N, D, stats):
    """QK^T for every tile + P V for executed tiles; ragged tiles counted as full
    in the P V term (error < 1/T_c)."""
    qk = 2.0 * BH * N * N * D
    frac_exec = float(stats[..., 0].sum()) / float(stats.sum())   # executed / all decision tiles (any tile_k)
    return qk + 2.0 * BH * N * N * D * frac_exec


def host_workers():
    try:
        return max(1, min(16, len(os.sched_getaffinity(0))))
    except AttributeError:
        return max(1, min(16, os.cpu_count() or 1))


class ClockSampler:
    """Samples nvidia-smi clocks / throttle reasons while the timed region runs."""
    QUERY = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
             "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
             "clocks_event_reasons.sw_power_cap")

    def __init__(self, index=0):
        self.samples, self._stop, self.index = [], threading.Event(), index
        self.active = threading.Event()         # set only while a timed region runs: idle gaps are not sampled
        self._t = threading.Thread(target=self._run, daemon=True)

    def _run(self):
        while not self._stop.is_set():
            if not self.active.is_set():
                self._stop.wait(0.005)
                continue
            try:
                out = subprocess.run(["nvidia-smi", f"--query-gpu={self.QUERY}", "--format=csv,noheader,nounits",
                                      "-i", str(self.index)], capture_output=True, text=True, timeout=5).stdout
                if self.active.is_set():         # the region was still running when nvidia-smi returned
                    self.samples.append([s.strip() for s in out.strip().split(",")])
            except Exception:
                pass
            self._stop.wait(0.02)

    def __enter__(self):
        self._t.start()
        return self

    def __exit__(self, *a):
        self._stop.set()
        self._t.join(timeout=6)

    def summary(self):
        sm = [float(s[0]) for s in self.samples if len(s) >= 7 and s[0].replace(".", "").isdigit()]
        reasons = set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for s in self.samples:
            if len(s) >= 7:
                for n, val in zip(names, s[3:7]):
                    if val.lower().startswith("active"):
                        reasons.add(n)
        mx = [float(s[1]) for s in self.samples if len(s) >= 7 and s[1].replace(".", "").isdigit()]
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "reasons": sorted(reasons), "samples": len(self.samples)}


# ---------------------------------------------------------------------------------------------- oracle arm
def oracle_sample_time(cfg, seed, lam, mode, head=0, reps=1):
    """Time the oracle, as it stands, on a bounded sample: 4 x (host threads) evenly spaced Q tiles of one head (first
    and ragged last included), all K tiles -- about 6 s of work per repetition at config 3 on 16 cores."""
    import oracle
    q, k, v = make_qkv(cfg, seed, heads=[head])
    cores = oracle.max_threads()
    T = -(-cfg.N // cfg.tile)
    qt = sorted(set(int(x) for x in np.linspace(0, T - 1, min(T, 4 * cores)).round()))
    times = []
    for _ in range(reps):
        t0 = time.perf_counter()
        oracle.run_head(q[0, 0], k[0, 0], v[0, 0], tile=cfg.tile, lam=lam, mode=mode, qtiles=qt)
        times.append(time.perf_counter() - t0)
    rows = sum(min(cfg.tile, cfg.N - i * cfg.tile) for i in qt)
    flop = 4.0 * rows * cfg.N * cfg.D                    # dense-equivalent FLOP of the sampled Q tiles
    return {"seconds": times, "flop": flop, "cores": cores, "n_qtiles": len(qt),
            "sample": f"{len(qt)} of {T} Q tiles (evenly spaced, incl. first and ragged last) of head {head}, "
                      f"all {T} K tiles, mode {mode}, lambda {lam:.3f}"}


def run_reference(args, cfg, lam):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    res = oracle_sample_time(cfg, args.seed, lam, 2, reps=args.warmup + args.steps)
    secs = res["seconds"][args.warmup:]
    mean_s = float(np.mean(secs))
    val = res["flop"] / mean_s / 1e12
    line = {
        "impl": "reference", "metric": METRIC, "value": val, "unit": UNIT,
        "n_gpus": args.gpus, "steps": args.steps, "warmup": args.warmup, "ms_per_step": mean_s * 1e3,
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": workload_name(cfg), "mode": "dynamic", "lambda": lam, "step": res["sample"]},
        "cpu_baseline": {"value": val, "unit": UNIT, "cores": res["cores"], "kind": "oracle", "sample": res["sample"]},
        "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line), flush=True)


# ---------------------------------------------------------------------------------------------- GPU arm helpers
class Gpu:
    """Device buffers of one workload plus the timing / quality helpers (every value through the C ABI)."""

    def __init__(self, sa, torch, cfg, qb, kb, vb, barrier=lambda: None):
        self.sa, self.torch, self.cfg, self.barrier = sa, torch, cfg, barrier
        self.B, self.H, self.N, self.D = qb.shape

        def to_dev(bits):
            return torch.from_numpy(np.ascontiguousarray(bits).view(np.int16)).cuda().view(torch.bfloat16)

        self.q, self.k, self.v = to_dev(qb), to_dev(kb), to_dev(vb)
        self.out = torch.empty_like(self.q)
        self.lse = torch.empty((self.B, self.H, self.N), device="cuda", dtype=torch.float32)
        self.stats = torch.zeros((self.B, self.H, 2), device="cuda", dtype=torch.int64)
        self.out_dense = self.lse_dense = None
        self._rs = torch.zeros(2, device="cuda", dtype=torch.float64)
        self.stream = torch.cuda.current_stream()

    def call(self, mode, lam=-math.inf, tile_k=0, mask_in=None, skip_mask_out=None):
        p = self.sa.make_params(lam=lam, stream=self.stream.cuda_stream, tile_q=self.cfg.tile if tile_k else 0,
                                tile_k=tile_k, skip_mask_in=mask_in, skip_mask_out=skip_mask_out)
        self.sa.sparse_attn_fwd(self.q, self.k, self.v, self.out, self.lse, self.B, self.H, self.N, self.D, p, mode, self.stats)

    def preheat(self, seconds):
        """Untimed DENSE calls: after the idle seconds of input generation the first timed mode would otherwise run at
        burst clocks and the later ones under the power cap, which biases every ratio between modes by a few percent."""
        t0 = time.perf_counter()
        while time.perf_counter() - t0 < seconds:
            for _ in range(4):
                self.call(self.sa.MODE_DENSE)
            self.torch.cuda.synchronize()

    def time(self, mode, lam, steps, warmup, tile_k=0, mask_in=None, sampler=None):
        """Returns (total_ms over `steps` calls, per-call ms list, stats [B,H,2])."""
        torch = self.torch
        for _ in range(warmup):
            self.call(mode, lam, tile_k, mask_in)
        evs = [torch.cuda.Event(enable_timing=True) for _ in range(steps + 1)]
        self.barrier()
        torch.cuda.synchronize()
        if sampler is not None:
            sampler.active.set()
        evs[0].record(self.stream)
        for i in range(steps):
            self.call(mode, lam, tile_k, mask_in)
            evs[i + 1].record(self.stream)
        torch.cuda.synchronize()
        if sampler is not None:
            sampler.active.clear()
        self.barrier()
        per = [evs[i].elapsed_time(evs[i + 1]) for i in range(steps)]
        return evs[0].elapsed_time(evs[-1]), per, self.stats.cpu().numpy().copy()

    def effective_clock(self, mode, lam):
        """The SM clock a launch actually runs at, from the kernel's own counters: the debug instantiation sums clock64()
        cycles over its CTAs (params->cycles_out); with one CTA resident per SM and whole waves, sum / (SMs * time) is the
        clock.  Called right after a timed loop (chip hot), outside every timed region."""
        torch = self.torch
        n_sm = torch.cuda.get_device_properties(torch.cuda.current_device()).multi_processor_count
        cyc = torch.zeros(2, device="cuda", dtype=torch.int64)
        p = self.sa.make_params(lam=lam, stream=self.stream.cuda_stream, cycles_out=cyc)
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        for i in range(3):                                    # two to settle, the third is measured
            if i == 2:
                e0.record(self.stream)
            self.sa.sparse_attn_fwd(self.q, self.k, self.v, self.out, self.lse, self.B, self.H, self.N, self.D, p, mode, self.stats)
        e1.record(self.stream)
        torch.cuda.synchronize()
        ms = e0.elapsed_time(e1)
        cycles, ctas = (int(x) for x in cyc.tolist())
        return {"cta_cycles_sum": cycles, "ctas": ctas, "waves": ctas / n_sm, "debug_launch_ms": ms,
                "sm_mhz_effective": cycles / (n_sm * ms * 1e3)}

    def keep_dense(self):
        self.out_dense, self.lse_dense = self.out.clone(), self.lse.clone()

    def quality(self, heads=None):
        """Achieved recall per row = exp(lse_retained - lse_dense) and error against the dense output,
        reduced on the device by sparse_attn_recall_stats / sparse_attn_output_error."""
        if self.lse_dense is None:
            return {}
        sa, st = self.sa, self.stream.cuda_stream
        lse, lse_d, out, out_d = self.lse, self.lse_dense, self.out, self.out_dense
        if heads is not None:
            h0, h1 = heads
            lse, lse_d, out, out_d = lse[:, h0:h1], lse_d[:, h0:h1], out[:, h0:h1], out_d[:, h0:h1]
            assert self.B == 1
        n_rows, n_el = lse.numel(), out.numel()
        sa.sparse_attn_recall_stats(lse, lse_d, n_rows, self._rs, st)
        rmin, rsum = self._rs.tolist()
        sa.sparse_attn_output_error(out, out_d, n_el, self._rs, st)
        emax, esum = self._rs.tolist()
        return {"recall_min": rmin, "recall_mean": rsum / n_rows, "err_vs_dense_max_abs": emax,
                "err_vs_dense_mean_abs": esum / n_el}


def mode_entry(g, BH_total, ms, per, st_all, st_local):
    cfg = g.cfg
    ex = executed_flop(BH_total, cfg.N, cfg.D, st_all)
    return {"ms": ms, "ms_min": float(np.min(per)), "ms_median": float(np.median(per)),
            "sparsity": float(st_all[..., 1].sum() / st_all.sum()),
            "effective_tflops": dense_flop(BH_total, cfg.N, cfg.D) / (ms * 1e-3) / 1e12,
            "executed_tflops": ex / (ms * 1e-3) / 1e12,
            "kernel_ms_avg_rank0": float(np.mean(per)),
            "executed_flop_per_launch_rank0": executed_flop(g.B * g.H, cfg.N, cfg.D, st_local)}


def pair_stats(mask):
    """Diagnostic of the two-Q-tiles-per-CTA design: the two slots of a CTA stream the same K / V tiles in
    lock-step, so a K tile costs the CTA less only when BOTH of its Q tiles skip it.  mask: uint8 [B, H, T_r, T_c], 1 = skip
    (DYNAMIC mode's own decisions).  Returns the fraction of (CTA, K tile) pairs skipped by both / by exactly one slot and the
    speed-up bound 1 / (1 - joint / 2) of the lock-step pair (the MMA-bound model of a single Q tile is 1 / (1 - s / 2))."""
    m = mask.reshape(-1, mask.shape[-2], mask.shape[-1]).astype(bool)
    T_r = m.shape[1]
    even, odd = m[:, 0:T_r - (T_r % 2):2], m[:, 1::2]
    joint, one = float((even & odd).sum()), float((even ^ odd).sum())
    pairs = float(even.size)
    if T_r % 2:                                             # the last CTA of a head holds one Q tile
        joint += float(m[:, -1].sum())
        pairs += float(m[:, -1].size)
    return {"both_slots_skip": joint / pairs, "one_slot_skips": one / pairs, "lockstep_model": 1.0 / (1.0 - joint / pairs / 2.0)}


def time_reorder(sa, torch, cfg, brick, qkv, scratch_out, steps, warmup):
    """Re-orders q, k, v into brick order with sparse_attn_reorder_tokens and times the four passes a call needs
    (three gathers before the attention, one scatter of `out` after it)."""
    perm = np.empty(cfg.N, dtype=np.int32)
    sa.sparse_attn_brick_permutation(*cfg.grid, *brick, perm)
    dperm = torch.from_numpy(perm).cuda()
    stream = torch.cuda.current_stream()
    dst = [torch.empty_like(t) for t in qkv]
    back = torch.empty_like(scratch_out)

    def four_passes():
        for s_, d_ in zip(qkv, dst):
            sa.sparse_attn_reorder_tokens(s_, d_, cfg.B, cfg.H, cfg.N, cfg.D, dperm, 0, stream.cuda_stream)
        sa.sparse_attn_reorder_tokens(dst[0], back, cfg.B, cfg.H, cfg.N, cfg.D, dperm, 1, stream.cuda_stream)

    for _ in range(max(warmup, 1)):
        four_passes()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    torch.cuda.synchronize()
    e0.record(stream)
    for _ in range(steps):
        four_passes()
    e1.record(stream)
    torch.cuda.synchronize()
    assert torch.equal(back, qkv[0]), "gather followed by scatter must give the input back"
    ms = e0.elapsed_time(e1) / steps
    nbytes = 4 * 2 * qkv[0].numel() * 2                     # 4 passes, each reads and writes the tensor once
    hbm = measured_hbm()
    info = {"brick": list(brick), "ms_4_passes": ms, "bytes_4_passes": nbytes, "achieved_gbs": nbytes / (ms * 1e-3) / 1e9,
            "hbm_peak_gbs": hbm, "frac_of_hbm_peak": nbytes / (ms * 1e-3) / 1e9 / hbm,
            "note": "3 gathers (q, k, v) + 1 scatter (out) per attention call; %.0f MB read + %.0f MB written, larger than L2"
                    % (nbytes / 2e6, nbytes / 2e6)}
    del back
    return info, tuple(dst)


def timed_call(torch, fn, n, warm=2):
    stream = torch.cuda.current_stream()
    for _ in range(warm):
        fn()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    torch.cuda.synchronize()
    e0.record(stream)
    for _ in range(n):
        fn()
    e1.record(stream)
    torch.cuda.synchronize()
    return e0.elapsed_time(e1) / n


def selector_comparison(g, dyn, steps, warmup, theta_grid=(1e-7, 1e-6, 1e-5, 1e-4)):
    """the block-mask comparison methods of PAPER.md:61-62 and the section-3 "ideal" mask
     through the same kernel.  Block sums of p and p^2 of the dense probabilities -> Top-K at DYNAMIC
    mode's tile budget, Top-P at DYNAMIC mode's mean recall, the greedy mask under Eq. 3 over a Theta grid -> MASK mode."""
    sa, torch, cfg = g.sa, g.torch, g.cfg
    st = g.stream.cuda_stream
    T = -(-cfg.N // cfg.tile)
    mass = torch.empty((g.B, g.H, T, T), device="cuda", dtype=torch.float32)
    sq = torch.empty_like(mass)
    bitmap = torch.empty((g.B, g.H, T, T), device="cuda", dtype=torch.uint8)
    n = max(3, steps // 4)
    ms_mass = timed_call(torch, lambda: sa.sparse_attn_block_mass(g.q, g.k, g.lse_dense, mass, g.B, g.H, g.N, g.D, 0.0, st), n)
    ms_stats = timed_call(torch, lambda: sa.sparse_attn_block_stats(g.q, g.k, g.lse_dense, mass, sq, g.B, g.H, g.N, g.D, 0.0, st), n)
    qk_flop = 2.0 * g.B * g.H * g.N * g.N * g.D
    res = {"block_mass_ms": ms_mass, "block_mass_tflops": qk_flop / (ms_mass * 1e-3) / 1e12,
           "block_stats_ms": ms_stats, "block_stats_tflops": qk_flop / (ms_stats * 1e-3) / 1e12,
           "note": "mass and selection are a pre-pass the in-loop rule does not need (PAPER.md:109, :133)"}
    jobs = [("topk_at_dynamic_budget", lambda: sa.sparse_attn_select_blocks(mass, bitmap, g.B, g.H, T, T, sa.SELECT_TOPK,
                                                                            max(1.0 - dyn["sparsity"], 1.0 / T), st),
             max(1.0 - dyn["sparsity"], 1.0 / T), ms_mass),
            ("topp_at_dynamic_recall", lambda: sa.sparse_attn_select_blocks(mass, bitmap, g.B, g.H, T, T, sa.SELECT_TOPP,
                                                                            min(max(dyn["recall_mean"], 0.01), 1.0), st),
             min(max(dyn["recall_mean"], 0.01), 1.0), ms_mass)]
    for theta in theta_grid:
        jobs.append((f"greedy_eq3_theta_{theta:g}",
                     (lambda th: lambda: sa.sparse_attn_select_blocks_greedy(mass, sq, bitmap, g.B, g.H, g.N, cfg.tile, T, th, st))(theta),
                     theta, ms_stats))
    for name, select, param, ms_pre in jobs:
        ms_sel = timed_call(torch, select, 3, warm=1)
        total, per, stt = g.time(sa.MODE_MASK, -math.inf, max(3, steps // 2), min(warmup, 2), mask_in=bitmap)
        ms_att = total / max(3, steps // 2)
        res[name] = {"param": param, "select_ms": ms_sel, "attention_ms": ms_att,
                     "sparsity": float(stt[..., 1].sum() / stt.sum()), **g.quality(),
                     "ms_incl_prepass": ms_att + ms_pre + ms_sel}
    return res


# ---------------------------------------------------------------------------------------------- reports (configs 2-4, masks)
def sweep_point(g, mode, lam, steps, warmup, dense_ms, tile_k=0):
    total, per, st = g.time(mode, lam, steps, warmup, tile_k=tile_k)
    ms = total / steps
    s = float(st[..., 1].sum() / st.sum())
    return {"lambda": lam, "ms": ms, "sparsity": s, "speedup_vs_dense": dense_ms / ms, "mma_bound_model": 1.0 / (1.0 - s / 2.0),
            **g.quality()}


def report_cfg2(args, sa, torch):
    """BASELINE.json configs[2]: per-head sparsity against (tau_h, sigma_h)."""
    from workloads.generator import head_params
    cfg = CONFIGS["cfg2"]
    qb, kb, vb = make_qkv(cfg, args.seed, workers=host_workers())
    g = Gpu(sa, torch, cfg, qb, kb, vb)
    lam = eq7_lambda(cfg)
    g.preheat(args.preheat)
    total, per, _ = g.time(sa.MODE_DENSE, -math.inf, args.steps, args.warmup)
    dense_ms = total / args.steps
    g.keep_dense()
    out = {"report": "cfg2", "workload": workload_name(cfg), "lambda": lam, "lambda_rule": f"Eq. 7, P_real={P_REAL}",
           "dense_ms": dense_ms, "dense_tflops": dense_flop(cfg.H, cfg.N, cfg.D) / (dense_ms * 1e-3) / 1e12, "heads": []}
    per_mode = {}
    for mname, mode in (("fixed", sa.MODE_FIXED), ("dynamic", sa.MODE_DYNAMIC)):
        out[mname] = sweep_point(g, mode, lam, args.steps, args.warmup, dense_ms)
        st = g.stats.cpu().numpy()[0]
        per_mode[mname] = [{"sparsity": float(st[h, 1] / st[h].sum()), **{k_: v_ for k_, v_ in g.quality((h, h + 1)).items()
                                                                          if k_.startswith("recall")}} for h in range(cfg.H)]
    taus, sigmas = zip(*(head_params(cfg, args.seed, h) for h in range(cfg.H)))
    for h in range(cfg.H):
        out["heads"].append({"head": h, "tau": taus[h], "sigma": sigmas[h],
                             "fixed": per_mode["fixed"][h], "dynamic": per_mode["dynamic"][h]})
    sp = np.array([e["sparsity"] for e in per_mode["dynamic"]])
    out["dynamic_sparsity_corr_with_tau"] = float(np.corrcoef(sp, np.array(taus))[0, 1])
    out["dynamic_sparsity_corr_with_sigma"] = float(np.corrcoef(sp, np.array(sigmas))[0, 1])
    return out


def report_cfg3(args, sa, torch):
    """BASELINE.json configs[3]: recall-target sweep 0.85-0.99 (strict map, and the calibrated map of
    SURVEY.md NEXT-3), the paper's lambda grid {-6,-8,-9,-11} and Eq. 7 with P_real in {0.5,1,1.5,3}
    (PAPER.md:137-139): sparsity vs speed-up, DYNAMIC against FIXED, on the contract generator and the aligned variant."""
    from paper_2606_16317_b200.calibrate import calibrate_lambda
    out = {"report": "cfg3", "variants": {}}
    targets = (0.85, 0.90, 0.95, 0.97, 0.99)
    for name in ("cfg3", "cfg3_aligned"):
        cfg = CONFIGS[name]
        qb, kb, vb = make_qkv(cfg, args.seed, workers=host_workers())
        g = Gpu(sa, torch, cfg, qb, kb, vb)
        del qb, kb, vb
        g.preheat(args.preheat)
        total, per, _ = g.time(sa.MODE_DENSE, -math.inf, args.steps, args.warmup)
        dense_ms = total / args.steps
        g.keep_dense()
        v = {"workload": workload_name(cfg), "dense_ms": dense_ms,
             "dense_tflops": dense_flop(cfg.H, cfg.N, cfg.D) / (dense_ms * 1e-3) / 1e12, "sweeps": []}
        modes = (("fixed", sa.MODE_FIXED), ("dynamic", sa.MODE_DYNAMIC))
        for R in targets:
            lam = math.log((1.0 - R) / cfg.N)
            v["sweeps"].append({"rule": "strict map lambda = ln((1-R)/N)", "recall_target": R,
                                **{m: sweep_point(g, mode, lam, args.steps, args.warmup, dense_ms) for m, mode in modes}})
        for R in targets:
            e = {"rule": "calibrated: largest lambda with MEAN row recall >= R (bisection, 12 iterations)", "recall_target": R}
            for m, mode in modes:
                cal = calibrate_lambda(g.q, g.k, g.v, cfg.B, cfg.H, cfg.N, cfg.D, mode, R, statistic="mean", iters=12)
                e[m] = sweep_point(g, mode, cal["lambda"], args.steps, args.warmup, dense_ms)
            v["sweeps"].append(e)
        for lam in (-6.0, -8.0, -9.0, -11.0):
            v["sweeps"].append({"rule": "paper lambda grid (Table 2)", "lambda": lam,
                                **{m: sweep_point(g, mode, lam, args.steps, args.warmup, dense_ms) for m, mode in modes}})
        for pr in (0.5, 1.0, 1.5, 3.0):
            lam = eq7_lambda(cfg, p_real=pr)
            v["sweeps"].append({"rule": "Eq. 7", "p_real": pr,
                                **{m: sweep_point(g, mode, lam, args.steps, args.warmup, dense_ms) for m, mode in modes}})
        out["variants"][name] = v
        del g
        torch.cuda.empty_cache()
    return out


def report_cfg4(args, sa, torch):
    """BASELINE.json configs[4]: denoising-step drift sweep at the 720p shape, all 40 heads: X = (1-a) field + a noise."""
    from paper_2606_16317_b200.calibrate import calibrate_lambda
    cfg = CONFIGS["cfg4"]
    lam = eq7_lambda(cfg)
    out = {"report": "cfg4", "workload": workload_name(cfg), "lambda": lam, "lambda_rule": f"Eq. 7, P_real={P_REAL}", "sweep": []}
    for a in (0.1, 0.3, 0.5, 0.7, 0.9):
        qb, kb, vb = make_qkv(cfg, args.seed, noise_a=a, workers=host_workers())
        g = Gpu(sa, torch, cfg, qb, kb, vb)
        del qb, kb, vb
        g.preheat(args.preheat)
        total, per, _ = g.time(sa.MODE_DENSE, -math.inf, args.steps, args.warmup)
        dense_ms = total / args.steps
        g.keep_dense()
        row = {"noise_a": a, "dense_ms": dense_ms}
        for m, mode in (("fixed", sa.MODE_FIXED), ("dynamic", sa.MODE_DYNAMIC)):
            row[m] = sweep_point(g, mode, lam, args.steps, args.warmup, dense_ms)
            cal = calibrate_lambda(g.q, g.k, g.v, cfg.B, cfg.H, cfg.N, cfg.D, mode, 0.95, statistic="mean", iters=10)
            row[m + "_at_mean_recall_0.95"] = sweep_point(g, mode, cal["lambda"], args.steps, args.warmup, dense_ms)
        out["sweep"].append(row)
        del g
        torch.cuda.empty_cache()
    return out


def report_masks(args, sa, torch):
    """SURVEY.md 8(f) NEXT-4 / PAPER.md:196-206 (Fig. 3): block masks of Top-K, Top-P, the section-3 greedy mask, FIXED
    (BLASST) and DYNAMIC (DynSparse) on synthetic P-matrix regimes, every method's parameter bisected to the same mean row
    recall; the bitmaps as text ('#' retained, '.' skipped)."""
    from paper_2606_16317_b200 import analysis
    from workloads.scenarios import SCENARIOS, make_scenario, scenario_notes
    notes = scenario_notes()
    out = {"report": "masks", "shape": "one head, N=4096, D=128, 128x128 tiles (32x32 bitmaps)", "targets": {}}
    for target in (0.90, 0.95, 0.99):
        per = {}
        for name in SCENARIOS:
            q, k, v = make_scenario(name, args.seed)
            res = analysis.compare_masks(q, k, v, target)
            per[name] = {"note": notes[name],
                         "methods": {m: {**{k_: v_ for k_, v_ in r.items() if k_ != "mask"},
                                         **({"mask": analysis.mask_picture(r["mask"])} if target == 0.95 else {})}
                                     for m, r in res.items()}}
        mean_sp = {m: float(np.mean([per[n]["methods"][m]["sparsity"] for n in SCENARIOS])) for m in analysis.METHODS}
        out["targets"]["mean_recall_%.2f" % target] = {"scenarios": per, "mean_sparsity_over_scenarios": mean_sp}
    return out


# Table 3's kurtosis bins, (lo, hi]
KURT_EDGES = (-math.inf, 0.0, 1.0, 3.0, 10.0, 30.0, 100.0, 300.0, 1000.0, 3000.0, 10000.0, math.inf)


def report_kurtosis(args, sa, torch):
    """SURVEY.md 8(f) NEXT-4 / PAPER.md:249-275 (Appendix A.1, Fig. 4, Table 3): sampled rows of P from flat to peaked heads,
    Top-K over a grid of K, MAE against recall by excess-kurtosis bin: MAE at recall 0.8 +- 0.01 and recall at MAE 0.05 +- 0.005."""
    from paper_2606_16317_b200 import analysis
    from workloads.scenarios import kurtosis_heads
    q, k, v, params = kurtosis_heads(args.seed)
    t0 = time.perf_counter()
    rows, keep, kurt, recall, mae = analysis.topk_curves(q, k, v, rows_per_head=128, seed=args.seed)
    secs = time.perf_counter() - t0
    edges = np.array(KURT_EDGES[1:-1])
    bins = np.searchsorted(edges, kurt, side="left")          # bin b: edges[b-1] < kurt <= edges[b]
    table = []
    for b in range(len(KURT_EDGES) - 1):
        sel = bins == b
        rc, me = recall[sel].ravel(), mae[sel].ravel()
        a = me[np.abs(rc - 0.8) <= 0.01]
        c = rc[np.abs(me - 0.05) <= 0.005]
        table.append({"kurtosis_range": [KURT_EDGES[b], KURT_EDGES[b + 1]], "rows": int(sel.sum()),
                      "mae_at_recall_0.8": {"n": int(a.size), "mean": float(a.mean()) if a.size else None,
                                            "std": float(a.std()) if a.size else None},
                      "recall_at_mae_0.05": {"n": int(c.size), "mean": float(c.mean()) if c.size else None,
                                             "var": float(c.var()) if c.size else None}})
    heads = [{"head": h, "tau": params[h][0], "aligned": params[h][1],
              "kurtosis_median": float(np.median(kurt[rows[:, 0] == h]))} for h in range(len(params))]
    return {"report": "kurtosis", "shape": f"{len(params)} heads, N={q.shape[2]}, D={q.shape[3]}, 128 sampled rows per head",
            "n_keep_values": int(keep.size), "seconds_row_topk_curve": secs, "heads": heads, "table3": table,
            "note": "synthetic rows stand in for Wan 2.2-5B's (PAPER.md:253): the trend, not the numbers, is comparable"}


def run_report(args):
    import torch
    import paper_2606_16317_b200 as sa
    if not torch.cuda.is_available():
        raise RuntimeError("bench.py needs a CUDA device (B200); there is no CPU fallback")
    torch.cuda.set_device(0)
    fn = {"cfg2": report_cfg2, "cfg3": report_cfg3, "cfg4": report_cfg4, "masks": report_masks, "kurtosis": report_kurtosis}
    print(json.dumps(fn[args.report](args, sa, torch)), flush=True)


# ---------------------------------------------------------------------------------------------- main
def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=5)
    ap.add_argument("--impl", default="b200", choices=["b200", "reference"])
    ap.add_argument("--seed", type=int, default=20261104)
    ap.add_argument("--config", default=DEFAULT_CONFIG)
    ap.add_argument("--no-aligned", action="store_true", help="skip the supplementary aligned / re-ordered workloads")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--preheat", type=float, default=1.5, help="seconds of untimed DENSE calls before each workload's timed modes")
    ap.add_argument("--modes", default="dense,fixed,dynamic", help="subset of modes to time (profiling runs)")
    ap.add_argument("--scaling", default="weak", choices=["weak", "strong"],
                    help="N > 1: weak = every rank its own full batch (default, the driver's contract); strong = ONE batch, its heads "
                         "sharded over the ranks (SURVEY.md 8(e)), each rank generating only its own heads")
    ap.add_argument("--report", default=None, choices=["cfg2", "cfg3", "cfg4", "masks", "kurtosis"],
                    help="run one of the sweeps BASELINE.json configs[2..4] / SURVEY.md NEXT-4 ask for and print it as JSON")
    args = ap.parse_args()
    args.warmup = max(args.warmup, 0)

    cfg = CONFIGS[args.config]
    lam = eq7_lambda(cfg)
    if args.impl == "reference":
        run_reference(args, cfg, lam)
        return
    if args.report:
        run_report(args)
        return

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    workers = max(1, host_workers() // max(1, min(world, 8)))
    cfg_full = cfg
    strong = args.scaling == "strong" and world > 1
    if strong:
        # strong scaling: ONE batch of cfg.H heads, rank r owns the contiguous range shard_heads(H, world, r) and draws
        # only those heads (same seed on every rank: head h has the bits it has in the single-GPU run)
        import dataclasses
        from paper_2606_16317_b200.sharding import shard_heads
        if world > cfg.H:
            raise SystemExit(f"--scaling strong needs at most {cfg.H} ranks (one head per rank)")
        h0, h1 = shard_heads(cfg.H, world, rank)
        host_data = {args.config: make_qkv(cfg, args.seed, heads=range(h0, h1), workers=workers)}
        cfg = dataclasses.replace(cfg, H=h1 - h0)            # the local problem: everything below sees its own heads only
        args.no_aligned = True
    else:
        # inputs first (spawned workers): weak scaling, every rank draws its own batch (different seed), same shape
        host_data = {args.config: make_qkv(cfg, args.seed + 1000 * rank, workers=workers)}
    aligned_name = args.config + "_aligned"
    if not args.no_aligned and aligned_name in CONFIGS:
        host_data[aligned_name] = make_qkv(CONFIGS[aligned_name], args.seed + 1000 * rank, workers=workers)

    import torch
    import paper_2606_16317_b200 as sa   # raises if the CUDA extension is missing: no fallback

    if not torch.cuda.is_available():
        raise RuntimeError("bench.py needs a CUDA device (B200); there is no CPU fallback")
    torch.cuda.set_device(local_rank)
    dist = None
    if world > 1:
        import torch.distributed as dist_mod
        dist = dist_mod
        dist.init_process_group("nccl", device_id=torch.device("cuda", local_rank))

    def barrier():
        if dist is not None:
            dist.barrier()

    tb, ts, peak_kind = measured_peaks()
    BH = cfg.B * cfg.H                                       # heads of THIS rank
    BH_total = cfg_full.B * cfg_full.H if strong else BH * world
    results = {}
    # (result key, generator config, brick of the token re-ordering or None)
    variants = [(args.config, args.config, None)]
    if not args.no_aligned:
        if aligned_name in host_data:
            variants.append((aligned_name, aligned_name, None))
        # SURVEY.md 8(f) NEXT-1 / PAPER.md:139: the contract workload with its tokens re-ordered into bricks
        variants.append((args.config + "_brick%dx%dx%d" % BRICK, args.config, BRICK))
    reorder_info = selectors = head_total_ms = None
    sampler = ClockSampler(local_rank)
    sampler.__enter__()                     # clocks / throttle reasons are sampled inside every timed region below
    headline_launches = 0
    want = args.modes.split(",")
    for vi, (name, gen_name, brick) in enumerate(variants):
        vcfg = cfg if gen_name == args.config else CONFIGS[gen_name]
        g = Gpu(sa, torch, vcfg, *host_data[gen_name], barrier=barrier)
        if brick is not None:
            reorder_info, (g.q, g.k, g.v) = time_reorder(sa, torch, vcfg, brick, (g.q, g.k, g.v), g.out, args.steps, args.warmup)
        g.preheat(args.preheat)
        res = {}
        lam32 = eq7_lambda(cfg, tile_k=32)                    # Eq. 7 with B_c = 32
        for mname, mode, mlam, mtk in (("dense", sa.MODE_DENSE, -math.inf, 0), ("fixed", sa.MODE_FIXED, lam, 0),
                                       ("dynamic", sa.MODE_DYNAMIC, lam, 0), ("dynamic_bc32", sa.MODE_DYNAMIC, lam32, 32),
                                       ("mask_replay", sa.MODE_MASK, lam, 0)):
            mmask = None
            if mname == "mask_replay":
                # MASK mode fed DYNAMIC mode's own decisions: same tiles, decisions read instead of taken in the loop
                if args.no_aligned or "dynamic" not in res or vi != 1:
                    continue
                T_dec = -(-cfg.N // cfg.tile)
                mmask = torch.zeros((cfg.B, cfg.H, T_dec, T_dec), device="cuda", dtype=torch.uint8)
                g.call(sa.MODE_DYNAMIC, lam, skip_mask_out=mmask)
                torch.cuda.synchronize()
            elif mname.split("_")[0] not in want or (mtk and (args.no_aligned or cfg.D != 128)):
                continue
            headline = (vi == 0 and mname == "dynamic")
            l0 = sa.launch_count()
            total, per, st = g.time(mode, mlam, args.steps, args.warmup, tile_k=mtk, mask_in=mmask, sampler=sampler)
            if headline:
                headline_launches = sa.launch_count() - l0 - args.warmup
                head_total_ms = total
            if dist is not None:
                t = torch.tensor([total], device="cuda")
                dist.all_reduce(t, op=dist.ReduceOp.MAX)
                total = float(t.item())
                from paper_2606_16317_b200.sharding import gather_stats
                # weak: every rank owns cfg.H heads of the (world * H)-head job; strong: its shard of the H heads (sizes may
                # differ by one) -- assemble the per-head counts in rank order
                st_all = gather_stats(torch.from_numpy(st).cuda(), BH_total // cfg.B).cpu().numpy()[None]
            else:
                st_all = st[None]
            res[mname] = mode_entry(g, BH_total, total / args.steps, per, st_all, st[None])
            if vi == 0 and mname in ("dense", "dynamic"):
                res[mname]["clock"] = g.effective_clock(mode, mlam)
            if mname == "dense":
                g.keep_dense()
            else:
                res[mname].update(g.quality())
            if mname == "dynamic_bc32":
                res[mname]["lambda"] = lam32
                res[mname]["decision_tile"] = "128x32"
            if mname != "dense" and "dense" in res:
                res[mname]["speedup_vs_dense"] = res["dense"]["ms"] / res[mname]["ms"]
                res[mname]["mma_bound_model"] = 1.0 / (1.0 - res[mname]["sparsity"] / 2.0)
            if mname == "dynamic" and brick is None:
                # which skips the pair of Q tiles of a CTA can turn into time (outside the timed region; debug build)
                T_dec = -(-vcfg.N // vcfg.tile)
                dmask = torch.zeros((vcfg.B, vcfg.H, T_dec, T_dec), device="cuda", dtype=torch.uint8)
                g.call(sa.MODE_DYNAMIC, mlam, skip_mask_out=dmask)
                torch.cuda.synchronize()
                res[mname]["cta_pair"] = pair_stats(dmask.cpu().numpy())
                del dmask
        if vi == 1 and brick is None and "dynamic" in res and "dense" in res:
            selectors = selector_comparison(g, res["dynamic"], args.steps, args.warmup)
        if brick is not None and reorder_info is not None:
            for mname in ("fixed", "dynamic", "dynamic_bc32"):
                if mname in res and "dense" in results.get(variants[0][0], {}):
                    # whole re-ordered pipeline (3 gathers + attention + 1 scatter) against the plain DENSE call
                    res[mname]["ms_with_reorder"] = res[mname]["ms"] + reorder_info["ms_4_passes"]
                    res[mname]["speedup_vs_plain_dense_incl_reorder"] = (
                        results[variants[0][0]]["dense"]["ms"] / res[mname]["ms_with_reorder"])
        results[name] = res
        del g
        torch.cuda.empty_cache()

    sampler.__exit__()
    clocks = sampler.summary()
    for mname in ("dense", "dynamic"):                       # the clock the kernels' own cycle counters imply, beside the sampled one
        eff = results.get(variants[0][0], {}).get(mname, {}).get("clock")
        if eff:
            clocks["sm_mhz_effective_" + mname] = eff["sm_mhz_effective"]
    if selectors is not None and clocks.get("sm_mhz"):
        # the block-sum pre-pass has one ex2 per logit and no P V to hide it behind: its roofline is the MUFU pipe
        # (16 ex2 / clk / SM, 148 SMs), i.e. 2 D FLOP of Q K^T per ex2; clock = the median sampled in the
        # timed loops of this run
        # The bound is stated in CYCLES, not through a clock: N^2 B H exponentials / (16 per clock per SM x 148 SMs) against the
        # kernel's own sm__cycles_elapsed from the tracked ncu capture of the same shape.  (Round 2 converted with the
        # clock nvidia-smi sampled; this kernel draws less power than the forward kernels and runs well above that clock, so
        # that fraction came out near or above 1.)  implied_sm_mhz = those cycles over the time measured in this run.
        vals, src = _ncu_summary(args.config, "mass")
        min_cycles = float(cfg.N) * cfg.N * BH / (16.0 * 148)
        entry = {"bound": "alu", "pipe": "MUFU ex2, 16 / clk / SM", "unit": "SM cycles per launch", "peak": min_cycles,
                 "achieved_tflops_of_qk": selectors["block_mass_tflops"], "sm_mhz_sampled": clocks["sm_mhz"]}
        if vals.get("sm__cycles_elapsed.avg"):
            cyc = vals["sm__cycles_elapsed.avg"]
            entry.update({"achieved": cyc, "frac": min_cycles / cyc, "cycles_source": src,
                          "pipe_xu_active_pct": vals.get("sm__inst_executed_pipe_xu.avg.pct_of_peak_sustained_active"),
                          "implied_sm_mhz": cyc / (selectors["block_mass_ms"] * 1e3)})
        else:
            entry.update({"achieved": None, "frac": None, "note": "no tracked ncu summary of the block-sum kernel for this config"})
        selectors["block_mass_roofline"] = entry

    # ------------------------------------------------------------------ end-to-end through the host-buffer C entry point
    qb, kb, vb = host_data[args.config]
    hq, hk, hv = (torch.from_numpy(x.view(np.int16)).pin_memory() for x in (qb, kb, vb))
    hout = torch.empty_like(hq).pin_memory()
    hlse = torch.empty((cfg.B, cfg.H, cfg.N), dtype=torch.float32).pin_memory()
    hstats = torch.zeros((cfg.B, cfg.H, 2), dtype=torch.int64).pin_memory()
    p = sa.make_params(lam=lam, stream=torch.cuda.current_stream().cuda_stream)
    e2e_steps = max(3, min(args.steps, 5))
    sa.sparse_attn_fwd_host(hq, hk, hv, hout, hlse, cfg.B, cfg.H, cfg.N, cfg.D, p, sa.MODE_DYNAMIC, hstats)
    barrier()
    torch.cuda.synchronize()
    t0 = time.perf_counter()
    for _ in range(e2e_steps):
        sa.sparse_attn_fwd_host(hq, hk, hv, hout, hlse, cfg.B, cfg.H, cfg.N, cfg.D, p, sa.MODE_DYNAMIC, hstats)
    torch.cuda.synchronize()
    e2e_s = (time.perf_counter() - t0) / e2e_steps
    if dist is not None:
        t = torch.tensor([e2e_s], device="cuda")
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        e2e_s = float(t.item())
    barrier()
    h2d = 3 * hq.numel() * 2
    d2h = hout.numel() * 2 + hlse.numel() * 4 + hstats.numel() * 8
    # the timed host-buffer call must have produced what the device entry produces on the same inputs, bit for bit
    # (20 head chunks over four streams against one launch); checked outside the timed region
    sa.sparse_attn_release_scratch()
    dq, dk, dv = (x.cuda().view(torch.bfloat16) for x in (hq, hk, hv))
    dout = torch.empty_like(dq)
    dlse = torch.empty((cfg.B, cfg.H, cfg.N), dtype=torch.float32, device="cuda")
    dstats = torch.zeros((cfg.B, cfg.H, 2), dtype=torch.int64, device="cuda")
    sa.sparse_attn_fwd(dq, dk, dv, dout, dlse, cfg.B, cfg.H, cfg.N, cfg.D, p, sa.MODE_DYNAMIC, dstats)
    torch.cuda.synchronize()
    e2e_equal = (torch.equal(dout.view(torch.int16).cpu(), hout) and torch.equal(dlse.cpu(), hlse)
                 and torch.equal(dstats.cpu(), hstats))
    if not e2e_equal:
        raise RuntimeError("sparse_attn_fwd_host and sparse_attn_fwd disagree on the bench workload")
    del dq, dk, dv, dout, dlse, dstats

    if rank != 0:
        if dist is not None:
            dist.destroy_process_group()
        return

    # ------------------------------------------------------------------ CPU baseline: the oracle as it stands
    cpu_baseline = None
    if not args.no_cpu_baseline and world == 1:
        r = oracle_sample_time(cfg, args.seed, lam, 2)
        cpu_baseline = {"value": r["flop"] / r["seconds"][0] / 1e12, "unit": UNIT,
                        "cores": r["cores"], "kind": "oracle", "sample": r["sample"], "seconds": r["seconds"][0],
                        "extrapolated_full_config_seconds": r["seconds"][0] * dense_flop(BH, cfg.N, cfg.D) / r["flop"]}

    if set(want) != {"dense", "fixed", "dynamic"}:      # profiling run: raw numbers only
        print(json.dumps({"partial": True, "modes": results, "lambda": lam}), flush=True)
        return
    main_res = results[args.config]["dynamic"]
    dense_res = results[args.config]["dense"]
    # Roofline of the dominant (only) kernel IN THE HEADLINE LAUNCH (DYNAMIC mode): executed FLOP of that launch (Q K^T for
    # every tile + P V for the executed ones, from stats_out) / its own CUDA-event time; the same kernel's DENSE launch beside it.
    ach_dyn = main_res["executed_flop_per_launch_rank0"] / (main_res["kernel_ms_avg_rank0"] * 1e-3) / 1e12
    ach_dense = dense_res["executed_flop_per_launch_rank0"] / (dense_res["kernel_ms_avg_rank0"] * 1e-3) / 1e12
    traffic, traffic_src = ncu_traffic(args.config, "dynamic")
    alg_bytes = 4 * BH * cfg.N * cfg.D * 2 + BH * cfg.N * 4
    line = {
        "metric": METRIC,
        "value": main_res["effective_tflops"],
        "unit": UNIT,
        "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
        "ms_per_step": head_total_ms / args.steps if world == 1 else main_res["ms"],
        "higher_is_better": True, "scaling": "strong" if strong else "weak", "vs_baseline": None, "dtype": "bf16", "data": "synthetic",
        "config": {"workload": workload_name(cfg_full), "mode": "dynamic", "lambda": lam,
                   "lambda_rule": f"Eq. 7, P_real={P_REAL}",
                   "l2": "q+k+v+out = %.0f MB per step > 126 MB L2, no flush" % (4 * BH * cfg.N * cfg.D * 2 / 1e6),
                   "preheat_s": args.preheat,
                   "parallelism": (f"one batch, its {cfg_full.H} heads sharded over {world} ranks, no data-path collective" if strong
                                   else f"heads sharded, {world} rank(s) with one batch each, no data-path collective")},
        "sparsity_pct": 100.0 * main_res["sparsity"],
        "speedup_vs_dense": main_res["speedup_vs_dense"],
        "pct_tensor_peak_executed": {"dense": 100.0 * ach_dense / tb, "dynamic": 100.0 * ach_dyn / tb,
                                     "of": f"{tb} TFLOP/s ({peak_kind} burst)"},
        "modes": results,
        "roofline": {"bound": "tensor", "achieved": ach_dyn, "peak": tb, "unit": "TFLOP/s", "frac": ach_dyn / tb,
                     "traffic": traffic, "traffic_source": traffic_src, "algorithmic_bytes": alg_bytes,
                     "kernel": "sparse_attn_fwd_kernel<128,128,1,3,2,true,false,1>, DYNAMIC mode (the headline launch)",
                     "peak_kind": f"{peak_kind} bf16 burst; sustained {ts}", "frac_sustained": ach_dyn / ts,
                     "flop_per_launch": main_res["executed_flop_per_launch_rank0"],
                     "launch_ms": main_res["kernel_ms_avg_rank0"],
                     "frac_dense": ach_dense / tb, "frac_dense_sustained": ach_dense / ts,
                     "dense_flop_per_launch": dense_res["executed_flop_per_launch_rank0"],
                     "dense_launch_ms": dense_res["kernel_ms_avg_rank0"]},
        "cpu_baseline": cpu_baseline,
        "e2e": {"value": dense_flop(BH_total, cfg.N, cfg.D) / e2e_s / 1e12, "unit": UNIT,
                "ms_per_step": e2e_s * 1e3, "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": d2h,
                "path": "sparse_attn_fwd_host: pinned host buffers, H2D + kernel + D2H pipelined over head chunks",
                "equals_device_entry": bool(e2e_equal)},
        "token_reordering": reorder_info,
        "block_selectors_on_aligned_workload": selectors,
        "gpu_launches": headline_launches,
        "clocks": clocks,
    }
    print(json.dumps(line), flush=True)
    if dist is not None:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
