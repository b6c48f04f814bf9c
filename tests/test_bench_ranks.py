"""The N>1 host logic of bench.py ("replicas only") on CPU: two gloo ranks, max-over-ranks timing,
whole-job value, per-rank seeds. The path has no data-path collective to test: it does not shard."""
import os
import socket
import sys

import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _worker(rank, world, port, out):
    sys.path.insert(0, ROOT)
    import bench
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    ms = bench.max_over_ranks([10.0 + 5.0 * rank, 30.0 - 7.0 * rank])       # rank 1 is slower in the first, faster in the second
    dist.barrier()
    out[rank] = (ms, bench.rank_seed(140972082, rank))
    dist.destroy_process_group()


def test_two_gloo_ranks_take_the_max_and_sum_the_records():
    sys.path.insert(0, ROOT)
    import bench
    s = socket.socket(); s.bind(("127.0.0.1", 0)); port = s.getsockname()[1]; s.close()
    with mp.Manager() as m:
        out = m.dict()
        mp.spawn(_worker, args=(2, port, out), nprocs=2, join=True)
        (ms0, seed0), (ms1, seed1) = out[0], out[1]
    assert ms0 == ms1 == [15.0, 30.0]                   # both ranks agree on the max over ranks
    assert seed0 != seed1                               # independent replicas
    # 2 ranks x 1000 records x 4 steps in 15 ms (the slowest rank)
    assert bench.whole_job_value(1000, 2, 4, ms0[0]) == 2 * 1000 * 4 / 15e-3
    assert bench.max_over_ranks([1.5]) == [1.5]         # no process group: identity
