"""Shared GPU-vs-oracle comparison (SURVEY.md section 8(c) "free-running comparison" and "replay").

Tolerances are BASELINE.json's: output max-abs 2e-2 and mean-abs 2e-3 against the oracle's sparse
output; skip decisions agree on every tile whose margin to the threshold exceeds 1e-3 logit units.
"""
from __future__ import annotations

import math
from dataclasses import dataclass, field
from typing import List, Optional, Sequence

import numpy as np
import torch

import oracle
import paper_2606_16317_b200 as sa
from workloads import bf16_bits_to_f64

OUT_MAX_ABS = 2e-2
OUT_MEAN_ABS = 2e-3
LSE_ABS = 2e-3          # fp32 running sum of ex2.approx values; derivation in DESIGN.md section 6
MARGIN_TOL = 1e-3       # decisions must agree where |g_ij| exceeds this (BASELINE.json north_star)


@dataclass
class GpuResult:
    out: np.ndarray       # [BH, N, D] float64 (widened bf16)
    lse: np.ndarray       # [BH, N] float32
    stats: np.ndarray     # [BH, 2] int64
    skip: np.ndarray      # [BH, T_r, T_c] uint8
    margin: np.ndarray    # [BH, T_r, T_c] float32


def to_dev_bf16(bits: np.ndarray) -> torch.Tensor:
    return torch.from_numpy(bits.view(np.int16)).cuda().view(torch.bfloat16)


def run_gpu(q_bits: np.ndarray, k_bits: np.ndarray, v_bits: np.ndarray, *, mode: int, lam: float = -math.inf,
            tile: int, debug: bool = True, scale: float = 0.0, tile_k: int = 0) -> GpuResult:
    """q/k/v bits: uint16 [B, H, N, D].  Calls the C ABI through the binding on cuda:0."""
    B, H, N, D = q_bits.shape
    q, k, v = (to_dev_bf16(np.ascontiguousarray(x)) for x in (q_bits, k_bits, v_bits))
    out = torch.full((B, H, N, D), float("nan"), device="cuda", dtype=torch.bfloat16)
    lse = torch.full((B, H, N), float("nan"), device="cuda", dtype=torch.float32)
    stats = torch.full((B, H, 2), -1, device="cuda", dtype=torch.int64)
    T = -(-N // tile)
    Tc = -(-N // (tile_k or tile))                     # decision tiles along the keys (tile_k < tile: SURVEY.md NEXT-2)
    mask = torch.full((B, H, T, Tc), 255, device="cuda", dtype=torch.uint8) if debug else None
    margin = torch.full((B, H, T, Tc), float("nan"), device="cuda", dtype=torch.float32) if debug else None
    p = sa.make_params(lam=lam, softmax_scale=scale, stream=torch.cuda.current_stream().cuda_stream,
                       skip_mask_out=mask, margin_out=margin, tile_q=tile if tile_k else 0, tile_k=tile_k)
    sa.sparse_attn_fwd(q, k, v, out, lse, B, H, N, D, p, mode, stats)
    torch.cuda.synchronize()
    out64 = bf16_bits_to_f64(out.view(torch.int16).cpu().numpy().view(np.uint16)).reshape(B * H, N, D)
    return GpuResult(out64, lse.cpu().numpy().reshape(B * H, N), stats.cpu().numpy().reshape(B * H, 2),
                     mask.cpu().numpy().reshape(B * H, T, Tc) if debug else None,
                     margin.cpu().numpy().reshape(B * H, T, Tc) if debug else None)


def scale_free_out_tol(v64: np.ndarray):
    """Output allowance that holds for ANY input scale: the kernel rounds P to bf16 before P V
    (relative 2^-8 per probability, so at most 2^-8 max_c |v_cd| in column d after the division by the unrounded row
    sum) and rounds the output to bf16 (2^-8 |o|); 1e-3 covers the fp32 accumulation, ex2.approx and the FMA-pipe
    polynomial.  On the contract workloads (|o| << 1, |v| <= 4.5) this is the 2e-2 of BASELINE.json."""
    vmax = np.abs(v64).max(axis=0)                             # [D]
    mean_tol = OUT_MEAN_ABS * max(1.0, float(vmax.max()) / 4.0)
    return (lambda o_ref: 2.0 ** -8 * (np.abs(o_ref) + vmax[None, :]) + 1e-3), mean_tol


@dataclass
class ParityReport:
    tiles_checked: int = 0
    decisions_checked: int = 0
    disagreements: int = 0              # free-running disagreements (all of them)
    near_margin_disagreements: int = 0  # of which |g| <= MARGIN_TOL at the point of first divergence
    diverged_qtiles: int = 0
    max_abs: float = 0.0
    mean_abs_sum: float = 0.0
    mean_abs_n: int = 0
    max_lse_abs: float = 0.0
    max_margin_abs: float = 0.0
    failures: List[str] = field(default_factory=list)

    @property
    def mean_abs(self) -> float:
        return self.mean_abs_sum / max(1, self.mean_abs_n)

    def ok(self) -> bool:
        return not self.failures


def compare_head(gpu: GpuResult, bh: int, q_bits, k_bits, v_bits, *, tile: int, mode: int, lam: float,
                 qtiles: Optional[Sequence[int]] = None, report: Optional[ParityReport] = None,
                 scale: Optional[float] = None, tile_k: Optional[int] = None, out_tol=None,
                 margin_tol: float = MARGIN_TOL) -> ParityReport:
    """Compare one head of a GPU run with the oracle on the given decision tiles (all if None).

    out_tol: None = BASELINE.json's output bounds (OUT_MAX_ABS / OUT_MEAN_ABS, which hold on the contract workloads);
    otherwise `scale_free_out_tol(v)`: (per-column max-abs allowance function of o_ref, mean-abs allowance) for inputs
    whose values leave the contract's range.
    margin_tol: the decision / margin tolerance; BASELINE.json's 1e-3 logit units by default, which presumes logits of the
    contract's size -- S is an fp32 number, so a margin between logits of +-1500 nats carries a few ulp(1500) = 1e-4
    each; tests that draw such inputs pass 1e-3 + 1e-6 max|S|."""
    rep = report if report is not None else ParityReport()
    N, D = q_bits.shape
    T = -(-N // tile)
    qt = list(range(T)) if qtiles is None else list(qtiles)
    free = oracle.run_head(q_bits, k_bits, v_bits, tile=tile, lam=lam, mode=mode, qtiles=qt, scale=scale, tile_k=tile_k)
    gskip = gpu.skip[bh][qt]                                   # [n, T]
    diverged = [t for t in range(len(qt)) if not np.array_equal(gskip[t], free.skip[t])]
    replay = None
    if diverged:
        replay = oracle.run_head(q_bits, k_bits, v_bits, tile=tile, lam=lam, mode=mode,
                                 qtiles=[qt[t] for t in diverged], forced_skip=gskip[diverged], scale=scale,
                                 tile_k=tile_k)
    for t, i in enumerate(qt):
        rows = min(tile, N - i * tile)
        r0 = i * tile
        rep.tiles_checked += 1
        rep.decisions_checked += gskip.shape[1]
        if t in diverged:
            d = diverged.index(t)
            rep.diverged_qtiles += 1
            dis = np.nonzero(gskip[t] != free.skip[t])[0]
            rep.disagreements += len(dis)
            first = int(dis[0])
            g_first = free.margin[t, first]                    # same state on both sides up to `first`
            if abs(g_first) <= margin_tol:
                rep.near_margin_disagreements += 1
            else:
                rep.failures.append(f"head {bh} qtile {i}: first disagreement at j={first} has margin {g_first:.3e}")
            # replay: the GPU's decision must equal (g < 0) wherever |g| > tol, g evaluated from the GPU's kept set
            g = replay.margin[d]
            must = np.abs(g) > margin_tol
            bad = must & ((g < 0) != (gskip[t] != 0))
            if bad.any():
                j = int(np.nonzero(bad)[0][0])
                rep.failures.append(f"head {bh} qtile {i}: replay mismatch at j={j}, g={g[j]:.3e}, gpu_skip={gskip[t, j]}")
            o_ref, l_ref, g_ref = replay.out[d, :rows], replay.lse[d, :rows], g
        else:
            o_ref, l_ref, g_ref = free.out[t, :rows], free.lse[t, :rows], free.margin[t]
        o_gpu = gpu.out[bh, r0:r0 + rows]
        l_gpu = gpu.lse[bh, r0:r0 + rows].astype(np.float64)
        if not np.all(np.isfinite(o_gpu)) or not np.all(np.isfinite(l_gpu)):
            rep.failures.append(f"head {bh} qtile {i}: non-finite GPU output")
            continue
        err = np.abs(o_gpu - o_ref)
        rep.max_abs = max(rep.max_abs, float(err.max()))
        rep.mean_abs_sum += float(err.sum())
        rep.mean_abs_n += err.size
        rep.max_lse_abs = max(rep.max_lse_abs, float(np.abs(l_gpu - l_ref).max()))
        if out_tol is None:
            if err.max() > OUT_MAX_ABS:
                rep.failures.append(f"head {bh} qtile {i}: out max-abs {err.max():.3e} > {OUT_MAX_ABS}")
            if err.mean() > OUT_MEAN_ABS:
                rep.failures.append(f"head {bh} qtile {i}: out mean-abs {err.mean():.3e} > {OUT_MEAN_ABS}")
        else:
            elem_tol, mean_tol = out_tol
            over = err - elem_tol(o_ref)
            if over.max() > 0:
                r, c = np.unravel_index(int(over.argmax()), over.shape)
                rep.failures.append(f"head {bh} qtile {i}: out err {err[r, c]:.3e} at |o| = {abs(o_ref[r, c]):.3f} exceeds the "
                                    f"scale-free bound {elem_tol(o_ref)[r, c]:.3e}")
            if err.mean() > mean_tol:
                rep.failures.append(f"head {bh} qtile {i}: out mean-abs {err.mean():.3e} > {mean_tol:.3e}")
        if np.abs(l_gpu - l_ref).max() > LSE_ABS:
            rep.failures.append(f"head {bh} qtile {i}: lse abs err {np.abs(l_gpu - l_ref).max():.3e} > {LSE_ABS}")
        # margins the GPU evaluated (debug output) against the oracle's, same kept set
        gm = gpu.margin[bh, i].astype(np.float64)
        fin = np.isfinite(g_ref)
        if not np.array_equal(np.isfinite(gm), fin):
            rep.failures.append(f"head {bh} qtile {i}: margin finiteness pattern differs")
        elif fin.any():
            merr = float(np.abs(gm[fin] - g_ref[fin]).max())
            rep.max_margin_abs = max(rep.max_margin_abs, merr)
            if merr > margin_tol:
                rep.failures.append(f"head {bh} qtile {i}: margin abs err {merr:.3e} > {margin_tol}")
    return rep


def check_stats(gpu: GpuResult, N: int, tile: int, tile_k: Optional[int] = None) -> None:
    """stats_out = {executed, skipped} per head must equal the bitmap's counts; executed + skipped = T_r T_c."""
    T = -(-N // tile)
    for bh in range(gpu.stats.shape[0]):
        skipped = int(gpu.skip[bh].sum())
        assert gpu.skip[bh].max() <= 1
        assert gpu.stats[bh, 1] == skipped, (bh, gpu.stats[bh], skipped)
        assert gpu.stats[bh, 0] + gpu.stats[bh, 1] == T * -(-N // (tile_k or tile))
        assert not gpu.skip[bh][:, 0].any()          # tile 0 never skipped
