"""gloo tests (world size 2 and 3) of the multi-GPU host logic: heads sharded, stats all-gathered -- the code path of
`bench.py --gpus N` in both its weak (every rank a full batch) and strong (`--scaling strong`: one batch, uneven shards) forms."""
import os
import socket

import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from paper_2606_16317_b200.sharding import gather_stats, shard_heads


def test_shard_heads_partitions_exactly():
    for H in (1, 2, 24, 40, 41):
        for world in (1, 2, 3, 8):
            ranges = [shard_heads(H, world, r) for r in range(world)]
            assert ranges[0][0] == 0 and ranges[-1][1] == H
            for (a0, a1), (b0, b1) in zip(ranges, ranges[1:]):
                assert a1 == b0 and a0 <= a1
            sizes = [b - a for a, b in ranges]
            assert max(sizes) - min(sizes) <= 1
    with pytest.raises(ValueError):
        shard_heads(4, 2, 2)


def _worker(rank, world, port, H, ret):
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    h0, h1 = shard_heads(H, world, rank)
    # what each rank's sparse_attn_fwd would have written for its own heads: {executed, skipped} per head
    local = torch.stack([torch.tensor([1000 + h, 7 * h], dtype=torch.int64) for h in range(h0, h1)])[None]
    full = gather_stats(local, H)
    ret[rank] = full.clone()
    dist.barrier()
    dist.destroy_process_group()


def _run(world, H):
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    port = s.getsockname()[1]
    s.close()
    mgr = mp.Manager()
    ret = mgr.dict()
    mp.spawn(_worker, args=(world, port, H, ret), nprocs=world, join=True)
    expect = torch.stack([torch.tensor([1000 + h, 7 * h], dtype=torch.int64) for h in range(H)])[None]
    for r in range(world):
        assert torch.equal(ret[r], expect)


@pytest.mark.parametrize("H", [24, 5])
def test_gather_stats_world_size_2_gloo(H):
    _run(2, H)


def test_gather_stats_uneven_strong_scaling_split_40_heads_over_3_ranks():
    """Config 3's 40 heads over 3 ranks (14 + 13 + 13): the split `bench.py --scaling strong` makes."""
    assert [shard_heads(40, 3, r) for r in range(3)] == [(0, 14), (14, 27), (27, 40)]
    _run(3, 40)
