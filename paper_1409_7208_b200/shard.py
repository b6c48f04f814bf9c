"""Sharding of the path by ranges of l=8 partitions (SURVEY.md §8(e) variant (i), §8(f) rank 4): every rank
holds the packed reads, plans the same contiguous ranges from the same partition histogram and counts only its own
range; the per-rank outputs, concatenated in rank order, are the output of sdbg_count_edges. The only exchange is an
all-gather of the per-rank edge counts (offsets into the concatenation). Host logic only: the work is done by
sdbg_bucket_hist / sdbg_plan_shards / sdbg_count_edges_range of the C library."""
from __future__ import annotations

import numpy as np

from . import binding as sd


def shard_bounds(ctx: sd.Context, reads: sd.Reads, k: int, world: int) -> np.ndarray:
    """Partition bounds of `world` shards, balanced by raw records; identical on every rank (same reads, same k)."""
    import torch
    hist = torch.zeros(sd.SDBG_NUM_BUCKETS, dtype=torch.int64, device=f"cuda:{ctx.device}")
    sd.sdbg_bucket_hist(ctx, reads, k, hist)
    return sd.sdbg_plan_shards(hist.cpu().numpy().view(np.uint64), world)


def gather_counts(n_local: int, device="cpu"):
    """All-gather of the per-rank edge counts -> (counts of all ranks, offset of this rank, total). Without a process
    group: one rank."""
    import torch
    import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size() == 1:
        return [int(n_local)], 0, int(n_local)
    world, rank = dist.get_world_size(), dist.get_rank()
    mine = torch.tensor([int(n_local)], dtype=torch.int64, device=device)
    allc = [torch.zeros(1, dtype=torch.int64, device=device) for _ in range(world)]
    dist.all_gather(allc, mine)
    counts = [int(c.item()) for c in allc]
    return counts, sum(counts[:rank]), sum(counts)


def count_edges_sharded(ctx: sd.Context, reads: sd.Reads, n: int, k: int, d: int, out: sd.Edges, rank: int, world: int,
                        stats: sd.Stats | None = None, bounds: np.ndarray | None = None):
    """This rank's share of sdbg_count_edges: returns (edges of this rank, partition bounds). out holds the edges of
    partitions [bounds[rank], bounds[rank + 1]) in order."""
    if bounds is None:
        bounds = shard_bounds(ctx, reads, k, world)
    n_local = sd.sdbg_count_edges_range(ctx, reads, n, k, d, int(bounds[rank]), int(bounds[rank + 1]), out, stats)
    return n_local, bounds
