"""Seeded single-head inputs whose attention matrix P has a prescribed structure -- input generation only.

The paper's Fig. 3 compares block masks "under different P matrix distributions": columns where
"all activation values are similar" (including one where "the maximum value in each row of the P matrix appears at the
first token position" and one where it is the opposite), columns where "some elements have larger activation values"
with "the maximum value in each row ... on the diagonal", and columns with few extreme values.  Its P matrices come
from Wan 2.2 and are not available; the scenarios below construct Q and K whose logits have those structures.  The
Appendix A.1 analysis needs rows of P from flat to very peaked: `kurtosis_heads`.

No attention arithmetic lives here: only Q, K, V bits.  logit(r, c) = <q_r, k_c> / sqrt(D).
"""
from __future__ import annotations

from dataclasses import replace
from typing import Dict, List, Tuple

import numpy as np

from .generator import CONFIGS, WorkloadConfig, _mix_and_scale, _smooth_field, f32_to_bf16_bits, make_head

SCENARIO_D = 128
SCENARIO_TILE = 128
SCENARIO_GRID = (4, 32, 32)            # N = 4096 tokens = 32 tiles of 128
SCENARIOS: Tuple[str, ...] = ("flat", "flat_max_first", "flat_max_last", "diagonal", "diagonal_sharp",
                              "sparse_columns", "sparse_blocks")


def _pack(q, k, v):
    return tuple(f32_to_bf16_bits(x.astype(np.float32))[None, None] for x in (q, k, v))


def make_scenario(name: str, seed: int):
    """Returns (q, k, v) bf16 bit patterns [1, 1, N, D] (N = 4096, D = 128) for one of SCENARIOS."""
    if name not in SCENARIOS:
        raise KeyError(name)
    t, h, w = SCENARIO_GRID
    N, D = t * h * w, SCENARIO_D
    rng = np.random.default_rng([seed, 77, SCENARIOS.index(name)])
    v = rng.standard_normal((N, D))
    root = np.sqrt(np.sqrt(D))                                # a bonus b in logit units: q += sqrt(b) D^(1/4) u, k likewise
    u = rng.standard_normal(D)
    u /= np.linalg.norm(u)
    if name.startswith("flat") or name.startswith("sparse"):
        q = 0.6 * rng.standard_normal((N, D))                 # logits ~ N(0, 0.36^2): every activation similar
        k = 0.6 * rng.standard_normal((N, D))
        if name in ("flat_max_first", "flat_max_last"):
            # every query carries the direction u; the keys of one tile carry it too: +2 logit units there
            q += np.sqrt(2.0) * root * u
            sl = slice(0, SCENARIO_TILE) if name == "flat_max_first" else slice(N - SCENARIO_TILE, N)
            k[sl] += np.sqrt(2.0) * root * u
        elif name == "sparse_columns":
            # a few heavy-hitter keys every query attends to: +7 logit units on 24 random keys
            q += np.sqrt(7.0) * root * u
            k[rng.choice(N, size=24, replace=False)] += np.sqrt(7.0) * root * u
        elif name == "sparse_blocks":
            # 16 clusters: a query tile and a key tile of the same cluster share a direction: +6 logit units
            dirs = np.linalg.qr(rng.standard_normal((D, 16)))[0].T
            cq = rng.integers(0, 16, size=N // SCENARIO_TILE)
            ck = rng.integers(0, 16, size=N // SCENARIO_TILE)
            for i in range(N // SCENARIO_TILE):
                q[i * SCENARIO_TILE:(i + 1) * SCENARIO_TILE] += np.sqrt(6.0) * root * dirs[cq[i]]
                k[i * SCENARIO_TILE:(i + 1) * SCENARIO_TILE] += np.sqrt(6.0) * root * dirs[ck[i]]
        return _pack(q, k, v)
    # diagonal: K's smooth field is Q's (the aligned generator of DESIGN.md section 4), maxima on the diagonal
    cfg = WorkloadConfig("scenario_" + name, 70, 1, 1, D, SCENARIO_GRID, SCENARIO_TILE, sigma=2.0,
                         tau=1.5 if name == "diagonal" else 2.2, aligned=True)
    f = _smooth_field(rng, cfg, cfg.sigma)
    q = _mix_and_scale(f, rng, cfg, cfg.tau, cfg.noise_a)
    k = _mix_and_scale(f, rng, cfg, cfg.tau, cfg.noise_a)
    return _pack(q, k, v)


# Appendix A.1: heads of the 480p shape (N = 32760) from flat to very peaked rows: (tau, aligned)
KURTOSIS_HEADS: Tuple[Tuple[float, bool], ...] = ((0.35, False), (0.5, False), (0.75, False), (1.0, False),
                                                  (1.25, False), (1.5, False), (2.0, False), (2.5, False),
                                                  (1.0, True), (1.5, True), (2.0, True), (3.0, True))


def kurtosis_heads(seed: int, grid=None, heads=None):
    """Returns (q, k, v) bf16 bit patterns [1, H, N, D] with head i drawn at KURTOSIS_HEADS[i] = (tau, aligned) on config
    1's grid (sigma = 3, a = 0.3), and the list of (tau, aligned) used."""
    base = CONFIGS["cfg1"]
    if grid is not None:
        base = replace(base, grid=tuple(grid))
    params = list(KURTOSIS_HEADS if heads is None else heads)
    out: List[np.ndarray] = [np.empty((1, len(params), base.N, base.D), dtype=np.uint16) for _ in range(3)]
    for i, (tau, aligned) in enumerate(params):
        cfg = replace(base, name="kurtosis_head", config_id=71, H=1, tau=tau, aligned=aligned)
        hq, hk, hv = make_head(cfg, seed, i)
        out[0][0, i], out[1][0, i], out[2][0, i] = hq, hk, hv
    return out[0], out[1], out[2], params


def scenario_notes() -> Dict[str, str]:
    return {
        "flat": "iid Gaussian Q, K at low temperature: every activation similar (Fig. 3, first group)",
        "flat_max_first": "flat, plus +2 logit units on the keys of the FIRST tile: every row's maximum is at the first positions",
        "flat_max_last": "flat, plus +2 logit units on the keys of the LAST tile (the opposite case)",
        "diagonal": "K's smooth field = Q's (tau 1.5): larger activations around the diagonal (Fig. 3, second group)",
        "diagonal_sharp": "as diagonal at tau 2.2",
        "sparse_columns": "flat, plus +7 logit units on 24 heavy-hitter keys: few extreme values (Fig. 3, last group)",
        "sparse_blocks": "flat, plus +6 logit units where the query tile and the key tile share one of 16 clusters",
    }
