"""Multi-GPU host logic: heads are the independent units of the path.

Each (b, h) needs its own Q and the whole K, V of its head and nothing else, so ranks take disjoint
head ranges and run `sparse_attn_fwd` on them with NO collective in the data path.  Only the per-head
`stats_out` slices are assembled afterwards (all-gather of [B, H_local, 2] int64).  K-dimension
(ring / context-parallel) sharding is deliberately not offered: the decisions are order dependent
(R4), a rank visiting K tiles in another order would change them.
"""
from __future__ import annotations

from typing import List, Tuple

import torch
import torch.distributed as dist


def shard_heads(H: int, world_size: int, rank: int) -> Tuple[int, int]:
    """Contiguous head range [h0, h1) of `rank`; the first H % world_size ranks get one extra head."""
    if not (0 <= rank < world_size):
        raise ValueError("rank out of range")
    base, extra = divmod(H, world_size)
    h0 = rank * base + min(rank, extra)
    return h0, h0 + base + (1 if rank < extra else 0)


def gather_stats(local_stats: torch.Tensor, H: int, group=None) -> torch.Tensor:
    """Assemble the full [B, H, 2] stats from every rank's [B, H_local, 2] slice (heads in rank order).

    Works with any backend (nccl on GPUs, gloo on CPU); ranks may own different numbers of heads.
    """
    world = dist.get_world_size(group)
    B = local_stats.shape[0]
    h_max = -(-H // world)
    padded = torch.zeros((B, h_max, 2), dtype=local_stats.dtype, device=local_stats.device)
    padded[:, : local_stats.shape[1]] = local_stats
    parts: List[torch.Tensor] = [torch.empty_like(padded) for _ in range(world)]
    dist.all_gather(parts, padded, group=group)
    out = []
    for r, p in enumerate(parts):
        h0, h1 = shard_heads(H, world, r)
        out.append(p[:, : h1 - h0])
    return torch.cat(out, dim=1)
