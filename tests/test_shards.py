"""Host logic of the sharded path without a GPU: the shard planner, and two gloo ranks that
plan from the same histogram, take their slice and all-gather the counts (the only exchange of the sharded path)."""
import os
import socket
import sys

import numpy as np
import pytest
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _plan(hist, n):
    import paper_1409_7208_b200 as sd
    return sd.sdbg_plan_shards(np.asarray(hist, dtype=np.uint64), n)


def test_plan_shards_is_contiguous_balanced_and_deterministic():
    rng = np.random.default_rng(7)
    for trial in range(20):
        hist = rng.integers(0, 1000, size=65536).astype(np.uint64)
        if trial % 3 == 0:
            hist[rng.integers(0, 65536, size=60000)] = 0          # mostly empty partitions
        if trial % 4 == 0:
            hist[rng.integers(0, 65536)] = 50_000_000             # one dominant partition
        total = int(hist.sum())
        cum = np.concatenate([[0], np.cumsum(hist)])
        for n in (1, 2, 3, 8, 64):
            b = _plan(hist, n)
            assert b[0] == 0 and b[-1] == 65536 and np.all(np.diff(b.astype(np.int64)) >= 0)
            assert np.array_equal(b, _plan(hist, n))
            for i in range(1, n):
                # shard i starts at the first partition where the running sum would exceed i/n of the records
                assert cum[b[i]] <= total * i // n
                assert b[i] == 65536 or cum[b[i] + 1] > total * i // n
            # no shard exceeds its fair share by more than one partition
            sizes = np.diff(cum[b])
            assert sizes.max() <= total // n + int(hist.max()) + 1


def test_plan_shards_edge_cases():
    import paper_1409_7208_b200 as sd
    z = np.zeros(65536, dtype=np.uint64)
    b = _plan(z, 4)
    assert b[0] == 0 and b[-1] == 65536
    one = z.copy(); one[12345] = 10
    b = _plan(one, 4)
    sizes = [int(one[b[i]:b[i + 1]].sum()) for i in range(4)]
    assert sum(sizes) == 10 and max(sizes) == 10
    with pytest.raises(sd.SdbgError):
        _plan(z, 0)


def _worker(rank, world, port, out):
    sys.path.insert(0, ROOT)
    import paper_1409_7208_b200 as sd
    from paper_1409_7208_b200.shard import gather_counts
    from oracle import run_oracle
    from workloads import ReadGenerator, get_config
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    w = get_config(1, scale=0.02)
    bases, offs = ReadGenerator(w).host()
    full = run_oracle((bases, offs), w.k, w.d)            # every rank holds the same reads (replicated)
    part = (full.distinct_keys[:, 0] >> np.uint64(48)).astype(np.int64)
    hist = np.bincount(part, weights=full.distinct_cnt.astype(np.float64), minlength=65536).astype(np.uint64)
    bounds = sd.sdbg_plan_shards(hist, world)
    spart = (full.keys[:, 0] >> np.uint64(48)).astype(np.int64)
    mine = np.nonzero((spart >= bounds[rank]) & (spart < bounds[rank + 1]))[0]     # what sdbg_count_edges_range yields
    counts, offset, total = gather_counts(len(mine))
    dist.barrier()
    out[rank] = dict(bounds=bounds.tolist(), counts=counts, offset=offset, total=total, first=int(mine[0]) if len(mine) else -1,
                     n=len(mine), n_solid=int(full.n_solid), raw=int(hist[bounds[rank]:bounds[rank + 1]].sum()), n_raw=int(full.n_raw))
    dist.destroy_process_group()


def test_two_gloo_ranks_plan_alike_and_concatenate():
    s = socket.socket(); s.bind(("127.0.0.1", 0)); port = s.getsockname()[1]; s.close()
    with mp.Manager() as m:
        out = m.dict()
        mp.spawn(_worker, args=(2, port, out), nprocs=2, join=True)
        r0, r1 = out[0], out[1]
    assert r0["bounds"] == r1["bounds"] and r0["counts"] == r1["counts"] == [r0["n"], r1["n"]]
    assert r0["offset"] == 0 and r1["offset"] == r0["n"] and r0["total"] == r1["total"] == r0["n_solid"]
    assert r0["first"] == 0 and r1["first"] == r0["n"]            # rank 1's slice starts where rank 0's ends: concatenation = full list
    assert r0["raw"] + r1["raw"] == r0["n_raw"]
    assert abs(r0["raw"] - r1["raw"]) < 0.2 * r0["n_raw"]           # balanced by raw records
