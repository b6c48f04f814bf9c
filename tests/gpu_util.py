"""Helpers of the -m gpu parity tests: run the CUDA path through the C ABI binding and compare with the oracle."""
from __future__ import annotations

import numpy as np

import paper_1409_7208_b200 as sd


def to_arrays(reads):
    """list[str] -> (uint8 bases, uint64 offsets)"""
    offs = np.zeros(len(reads) + 1, dtype=np.uint64)
    for i, r in enumerate(reads):
        offs[i + 1] = offs[i] + np.uint64(len(r))
    return np.frombuffer("".join(reads).encode(), dtype=np.uint8).copy(), offs


class GpuResult:
    pass


def run_gpu(reads, k, d, workspace_bytes=None, host_input=False, cap=None, checksums=True, bucket_hist=False,
            n_calls=1, ctx=None):
    """reads: list[str] or (bases uint8, offsets uint64) numpy pair or (torch cuda bases, torch cuda offsets)."""
    import torch
    if isinstance(reads, list):
        bases, offs = to_arrays(reads)
    else:
        bases, offs = reads
    n = len(offs) - 1
    if isinstance(bases, np.ndarray):
        nb = int(offs[-1] - offs[0])
        if not host_input:
            bases_t = torch.from_numpy(bases).cuda() if bases.size else torch.zeros(1, dtype=torch.uint8, device="cuda")
            offs_t = torch.from_numpy(offs.view(np.int64)).cuda()
        else:
            bases_t, offs_t = (bases if bases.size else np.zeros(1, np.uint8)), offs
    else:
        bases_t, offs_t = bases, offs
        nb = int((offs[-1] - offs[0]).item())
    W = sd.sdbg_key_words(k)
    N_ub = 2 * nb
    own_ctx = ctx is None
    if ctx is None:
        ws = workspace_bytes if workspace_bytes is not None else sd.sdbg_full_workspace(nb, k) + max(nb, 1 << 20)
        ctx = sd.Context(ws)
    rd = sd.Reads(nb, n_calls)
    if n_calls == 1:
        sd.sdbg_pack_reads(ctx, bases_t, offs_t, n, rd)
    else:   # split the reads over several appending calls
        cuts = [n * i // n_calls for i in range(n_calls + 1)]
        for a, b in zip(cuts, cuts[1:]):
            sd.sdbg_pack_reads(ctx, bases_t, offs_t[a:b + 1], b - a, rd)
    cap = max(N_ub // max(d, 1), 16) if cap is None else cap
    ed = sd.Edges(cap, k)
    st = sd.Stats(want_checksums=checksums, want_bucket_hist=bucket_hist)
    res = GpuResult()
    res.ctx, res.reads, res.edges, res.stats = ctx, rd, ed, st
    sd.sdbg_count_edges(ctx, rd, rd.n_reads, k, d, ed, st)
    g = sd.Graph(ed.n)
    sd.sdbg_build(ctx, ed, sd.SDBG_SORTED, g)
    torch.cuda.synchronize()
    res.graph = g
    res.n = ed.n
    res.keys = ed.keys_np()
    res.mult = ed.mult_np()
    res.W = g.W_np()
    res.last_bits = g.last_bits_np()
    res.gmult = g.mult_np()
    res.W_words = W
    return res


def assert_matches_oracle(res, orc, check_stats=True):
    """Bit-exact comparison of every output array with the oracle result (integer work: no tolerance)."""
    assert res.n == orc.n_solid, (res.n, orc.n_solid)
    assert np.array_equal(res.keys, orc.keys), "keys differ"
    assert np.array_equal(res.mult, orc.mult), "mult differs"
    assert np.array_equal(res.gmult, orc.mult), "graph mult differs"
    assert np.array_equal(res.W, orc.Wbyte), "W differs"
    assert np.array_equal(res.last_bits, orc.last_bits), "last differs"
    if check_stats:
        s = res.stats
        assert s.n_raw == orc.n_seen and s.n_distinct == orc.n_distinct and s.n_solid == orc.n_solid
        assert s.sum_solid_mult == orc.sum_solid_mult
