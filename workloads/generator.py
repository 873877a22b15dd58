"""Seeded Q/K/V generator for the Wan-2.2-shaped configs of BASELINE.json.

Recipe (BASELINE.json `configs`; readings recorded in DESIGN.md §4):

1. tokens live on a 3-D latent grid (t, h, w), token index n = (t_i*h + h_i)*w + w_i;
2. for Q and K, per head and per channel: white N(0,1) noise on the grid convolved with an
   isotropic 3-D Gaussian of `sigma` cells (boundary `wrap`, kernel truncated at 4 sigma),
   then standardised to zero mean / unit variance per (head, channel);
3. X = (1 - a) * field + a * N(0,1) iid noise  (a = 0.3 unless swept);
4. every token row is normalised to unit L2 norm and scaled by sqrt(D) * tau (tau = 1.5);
5. V ~ N(0,1) iid; Q, K, V are rounded once to bf16 (round-to-nearest-even) and those
   bits are what both the oracle and the GPU consume.

`aligned=True` is the supplementary (non-contract) workload of SURVEY.md §8(d): K's smooth
field is the same draw as Q's (noise independent), which gives the diagonal-local,
tile-coherent attention of a real video DiT.

Everything is drawn head by head from `numpy.random.default_rng([seed, config_id, head, k])`
substreams, so any single head can be regenerated without generating the others.
"""
from __future__ import annotations

from dataclasses import dataclass, replace
from typing import Dict, Optional, Tuple

import numpy as np
from scipy import ndimage


@dataclass(frozen=True)
class WorkloadConfig:
    name: str
    config_id: int
    B: int
    H: int
    D: int
    grid: Tuple[int, int, int]          # (t, h, w)
    tile: int                           # square decision tile B_r = B_c
    sigma: float                        # smooth-field sigma in cells (per-head draw if per_head)
    tau: float = 1.5                    # temperature: rows scaled to sqrt(D) * tau
    noise_a: float = 0.3                # X = (1-a) field + a noise
    per_head: bool = False              # configs 2-4: tau_h ~ U[1, 2.5], sigma_h ~ U[1, 6]
    aligned: bool = False               # supplementary workload: K field = Q field

    @property
    def N(self) -> int:
        t, h, w = self.grid
        return t * h * w


CONFIGS: Dict[str, WorkloadConfig] = {
    # BASELINE.json configs[0..4]
    "cfg0": WorkloadConfig("cfg0", 0, 1, 2, 64, (4, 16, 16), 64, 2.0),
    "cfg1": WorkloadConfig("cfg1", 1, 1, 24, 128, (21, 30, 52), 128, 3.0),
    "cfg2": WorkloadConfig("cfg2", 2, 1, 40, 128, (21, 30, 52), 128, 3.0, per_head=True),
    "cfg3": WorkloadConfig("cfg3", 3, 1, 40, 128, (21, 45, 80), 128, 3.0, per_head=True),
    "cfg4": WorkloadConfig("cfg4", 4, 1, 40, 128, (21, 45, 80), 128, 3.0, per_head=True),
}
# supplementary (labelled non-contract) aligned variants
for _k in ("cfg0", "cfg1", "cfg3"):
    CONFIGS[_k + "_aligned"] = replace(CONFIGS[_k], name=_k + "_aligned", aligned=True)


def num_tiles(N: int, tile: int) -> int:
    return (N + tile - 1) // tile


def f32_to_bf16_bits(x: np.ndarray) -> np.ndarray:
    """Round float32 to bf16 (round-to-nearest-even); returns the uint16 bit patterns."""
    x = np.ascontiguousarray(x, dtype=np.float32)
    u = x.view(np.uint32)
    rounding_bias = ((u >> 16) & 1) + np.uint32(0x7FFF)
    return ((u + rounding_bias) >> 16).astype(np.uint16)


def bf16_bits_to_f64(bits: np.ndarray) -> np.ndarray:
    """Widen bf16 bit patterns exactly to float64."""
    u = bits.astype(np.uint32) << 16
    return u.view(np.float32).astype(np.float64)


def _head_params(cfg: WorkloadConfig, seed: int, head: int) -> Tuple[float, float]:
    if not cfg.per_head:
        return cfg.tau, cfg.sigma
    r = np.random.default_rng([seed, cfg.config_id, head, 99])
    tau = float(r.uniform(1.0, 2.5))
    sigma = float(r.uniform(1.0, 6.0))
    return tau, sigma


def _smooth_field(rng: np.random.Generator, cfg: WorkloadConfig, sigma: float) -> np.ndarray:
    t, h, w = cfg.grid
    white = rng.standard_normal((cfg.D, t, h, w), dtype=np.float32)
    f = ndimage.gaussian_filter(white, sigma=(0, sigma, sigma, sigma), mode="wrap", truncate=4.0)
    f = f.reshape(cfg.D, -1)
    f -= f.mean(axis=1, keepdims=True)
    f /= f.std(axis=1, keepdims=True)
    return f.T  # [N, D]


def _mix_and_scale(field: np.ndarray, rng: np.random.Generator, cfg: WorkloadConfig,
                   tau: float, a: float) -> np.ndarray:
    x = (1.0 - a) * field + a * rng.standard_normal(field.shape, dtype=np.float32)
    x /= np.linalg.norm(x, axis=1, keepdims=True)
    x *= np.float32(np.sqrt(cfg.D) * tau)
    return x


def make_head(cfg: WorkloadConfig, seed: int, head: int, noise_a: Optional[float] = None):
    """Returns (q, k, v) bf16 bit patterns, each uint16 [N, D], for one (batch 0, head)."""
    a = cfg.noise_a if noise_a is None else noise_a
    tau, sigma = _head_params(cfg, seed, head)
    rq = np.random.default_rng([seed, cfg.config_id, head, 0])
    rk = np.random.default_rng([seed, cfg.config_id, head, 1])
    rv = np.random.default_rng([seed, cfg.config_id, head, 2])
    fq = _smooth_field(rq, cfg, sigma)
    fk = fq if cfg.aligned else _smooth_field(rk, cfg, sigma)
    q = _mix_and_scale(fq, rq, cfg, tau, a)
    k = _mix_and_scale(fk, rk, cfg, tau, a)
    v = rv.standard_normal((cfg.N, cfg.D), dtype=np.float32)
    return f32_to_bf16_bits(q), f32_to_bf16_bits(k), f32_to_bf16_bits(v)


def _make_head_job(args):
    return make_head(*args)


def make_qkv(cfg: WorkloadConfig, seed: int, heads=None, noise_a: Optional[float] = None, workers: int = 0):
    """Returns (q, k, v) uint16 arrays [B, len(heads), N, D]; B is 1 in every contract config.

    workers > 1 draws the heads in that many spawned processes (every head has its own substreams, so the bits do not
    depend on the worker count); `spawn`, not `fork`: the caller may already hold a CUDA context."""
    heads = list(range(cfg.H)) if heads is None else list(heads)
    q = np.empty((cfg.B, len(heads), cfg.N, cfg.D), dtype=np.uint16)
    k = np.empty_like(q)
    v = np.empty_like(q)
    jobs = [(cfg, seed + 7919 * b, h, noise_a) for b in range(cfg.B) for h in heads]
    if workers > 1 and len(jobs) > 1:
        import multiprocessing as mp
        with mp.get_context("spawn").Pool(min(workers, len(jobs))) as pool:
            results = pool.map(_make_head_job, jobs, chunksize=1)
    else:
        results = [make_head(*j) for j in jobs]
    for n, (hq, hk, hv) in enumerate(results):
        b, i = divmod(n, len(heads))
        q[b, i], k[b, i], v[b, i] = hq, hk, hv
    return q, k, v


def head_params(cfg: WorkloadConfig, seed: int, head: int) -> Tuple[float, float]:
    """(tau_h, sigma_h) actually used for `head` (for per-head sparsity reports)."""
    return _head_params(cfg, seed, head)
