"""N > 1 host logic: shard a seek batch over ranks, decode each slice
independently, all-gather. Runs with the gloo backend and world_size 2 on CPU; the per-rank decode is
the oracle's isolated decoder here (the CUDA path needs a GPU), the sharding code is the product's."""
import os
import socket

import numpy as np
import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

import oracle
from paper_2606_24531_b200 import sharding
from paper_2606_24531_b200 import workloads as W

B = 16384


def test_shard_bounds_cover_every_item_once():
    for n in (0, 1, 2, 7, 64, 100003):
        for world in (1, 2, 3, 8):
            spans = [sharding.shard_bounds(n, r, world) for r in range(world)]
            assert spans[0][0] == 0 and spans[-1][1] == n
            assert all(spans[i][1] == spans[i + 1][0] for i in range(world - 1))
            sizes = [hi - lo for lo, hi in spans]
            assert max(sizes) - min(sizes) <= 1
    with pytest.raises(ValueError):
        sharding.shard_bounds(4, 2, 2)


def _worker(rank, world, port, container, ids, want):
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        mine = sharding.shard_ids(ids, rank, world)
        local = np.zeros(len(mine) * B, np.uint8)
        with oracle.Isolated(container) as iso:
            for i, b in enumerate(mine):
                blk = iso.decode(int(b))
                local[i * B:i * B + blk.size] = blk
        got = sharding.gather_packed(torch.from_numpy(local), len(ids)).numpy()
        assert np.array_equal(got, want), f"rank {rank}: gathered blocks differ"
    finally:
        dist.destroy_process_group()


def test_sharded_seek_batch_world2_gloo():
    cfg = W.CONFIGS["markov_1m"]
    data = cfg.data(12 * B + 123)
    c = oracle.encode(data, offset_width=cfg.offset_width, min_match=8, max_depth=8, window=2, batch=2)
    full = oracle.decode_all(c)
    nb = (data.size + B - 1) // B
    ids = W.seek_ids(nb, 9, W.SEED_BASE + 0x77)                   # odd count: uneven slices
    want = np.zeros(len(ids) * B, np.uint8)
    for i, b in enumerate(ids):
        blk = full[int(b) * B:(int(b) + 1) * B]
        want[i * B:i * B + blk.size] = blk
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        port = s.getsockname()[1]
    mp.spawn(_worker, args=(2, port, c, ids, want), nprocs=2, join=True)
