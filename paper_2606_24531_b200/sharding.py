"""Host-side sharding for more than one GPU ("replicas only").

``decode_all`` of one container does not shard without an exchange (a match may read any earlier
output byte). What shards with no data-path collective is a batch of isolated decodes: every rank
holds a replica of the container, takes a contiguous slice of the id list, decodes it with
``aceapex_decode_blocks`` and — only if the caller wants the blocks in one place — the slices are
concatenated with one all-gather. This module holds that bookkeeping and no codec arithmetic.
"""
from __future__ import annotations

import numpy as np

B = 16384


def shard_bounds(n: int, rank: int, world: int) -> tuple[int, int]:
    """Contiguous, balanced slice [lo, hi) of n items for `rank` of `world` (sizes differ by at most 1)."""
    if world < 1 or not 0 <= rank < world or n < 0:
        raise ValueError("bad shard arguments")
    q, r = divmod(n, world)
    lo = rank * q + min(rank, r)
    return lo, lo + q + (1 if rank < r else 0)


def shard_ids(ids, rank: int, world: int) -> np.ndarray:
    ids = np.ascontiguousarray(np.asarray(ids, dtype=np.uint64))
    lo, hi = shard_bounds(len(ids), rank, world)
    return ids[lo:hi]


def gather_packed(local, n_total: int, group=None):
    """All-gather the packed blocks of every rank's slice (a torch uint8 tensor of len(slice) * 16384
    bytes on any device the process group supports) into one tensor of n_total * 16384 bytes, in id order."""
    import torch
    import torch.distributed as dist
    world = dist.get_world_size(group)
    sizes = [(hi - lo) * B for lo, hi in (shard_bounds(n_total, r, world) for r in range(world))]
    width = max(sizes) if sizes else 0                               # all_gather wants equal sizes: pad, then trim
    padded = torch.zeros(width, dtype=torch.uint8, device=local.device)
    padded[: local.numel()] = local.reshape(-1)
    parts = [torch.empty(width, dtype=torch.uint8, device=local.device) for _ in range(world)]
    dist.all_gather(parts, padded, group=group)
    return torch.cat([p[:n] for p, n in zip(parts, sizes)])
