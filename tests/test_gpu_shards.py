"""-m gpu: the sharded path (sdbg_bucket_hist, sdbg_plan_shards, sdbg_count_edges_range) on ONE
GPU: the shards of a plan are counted one after the other (they do not wait on one another) and their outputs,
concatenated in shard order, must equal the unsharded output bit for bit — edges, multiplicities, and for k >= 9 the
arrays of sdbg_build over each shard; statistics and checksums must add up."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu


def _setup(cfg, k=None, scale=None):
    import torch
    import paper_1409_7208_b200 as sd
    from workloads import ReadGenerator, get_config
    from dataclasses import replace
    w = get_config(cfg, scale=scale) if scale else get_config(cfg)
    if k:
        w = replace(w, k=k)
    bases_d, offs_d = ReadGenerator(w).device()
    ctx = sd.Context(sd.sdbg_workspace_for_records(w.n_raw_edges, w.k))
    reads = sd.Reads(w.n_bases)
    sd.sdbg_pack_reads(ctx, bases_d, offs_d, w.n_reads, reads)
    return w, ctx, reads


def _bits(t, n):
    import torch
    return ((t[:(n + 63) // 64].unsqueeze(1) >> torch.arange(64, device=t.device)) & 1).reshape(-1)[:n]


def _check(w, ctx, reads, n_shards, workspace_ctx=None, min_ranges=1):
    import torch
    import paper_1409_7208_b200 as sd
    from paper_1409_7208_b200.shard import count_edges_sharded, shard_bounds
    N = w.n_raw_edges
    full = sd.Edges(N // w.d, w.k)
    st = sd.Stats(want_checksums=True, want_bucket_hist=True)
    sd.sdbg_count_edges(ctx, reads, w.n_reads, w.k, w.d, full, st)
    S = full.n
    g_full = sd.Graph(S)
    sd.sdbg_build(ctx, full, sd.SDBG_SORTED, g_full)
    torch.cuda.synchronize()
    bounds = shard_bounds(ctx, reads, w.k, n_shards)
    hist = st.bucket_hist.cpu().numpy().view(np.uint64)
    assert np.array_equal(bounds, sd.sdbg_plan_shards(hist, n_shards))       # sdbg_bucket_hist = the histogram of the full run
    cctx = workspace_ctx or ctx
    off = 0
    tot = dict(n_raw=0, n_distinct=0, sum_solid_mult=0, csum_raw=0, csum_distinct=0)
    raws = []
    for r in range(n_shards):
        part = sd.Edges(S, w.k)
        ps = sd.Stats(want_checksums=True)
        n_r, b2 = count_edges_sharded(cctx, reads, w.n_reads, w.k, w.d, part, r, n_shards, ps, bounds)
        assert np.array_equal(b2, bounds)
        assert ps.n_raw == int(hist[bounds[r]:bounds[r + 1]].sum()) and ps.n_solid == n_r
        assert ps.csum_raw == ps.csum_distinct and (ps.n_ranges >= min_ranges or ps.n_raw == 0)
        raws.append(ps.n_raw)
        W = full.w
        assert torch.equal(part.keys[:n_r * W], full.keys[off * W:(off + n_r) * W]), f"shard {r}: keys differ"
        assert torch.equal(part.mult[:n_r], full.mult[off:off + n_r]), f"shard {r}: mult differs"
        if n_r:
            kp = (part.keys[:n_r * W:W] >> 48) & 0xffff
            assert int(kp.min()) >= bounds[r] and int(kp.max()) < bounds[r + 1]
        if w.k >= 9 and n_r:
            g = sd.Graph(n_r)
            sd.sdbg_build(cctx, part, sd.SDBG_SORTED, g)
            torch.cuda.synchronize()
            assert torch.equal(g.W[:n_r], g_full.W[off:off + n_r]), f"shard {r}: W differs"
            assert torch.equal(_bits(g.last_bits, n_r), _bits(g_full.last_bits, S)[off:off + n_r]), f"shard {r}: last differs"
        if w.d >= 2 and full.w == 1 and w.k >= 15 and ps.n_raw >= 4096:
            # the launch configuration of bench.py --shard: no checksums asked for, so the shard takes the default path
            # (top passes for the record density of its range, then the table count) and must give the same edges
            part2 = sd.Edges(S, w.k)
            cctx.get_timing()
            n2, _ = count_edges_sharded(cctx, reads, w.n_reads, w.k, w.d, part2, r, n_shards, None, bounds)
            assert cctx.get_timing().launches["table"] >= 1, "the shard did not take the table-count path"
            assert n2 == n_r and torch.equal(part2.keys[:n_r], part.keys[:n_r]) and torch.equal(part2.mult[:n_r], part.mult[:n_r])
            del part2
        for f in ("n_raw", "n_distinct", "sum_solid_mult"):
            tot[f] += getattr(ps, f)
        for f in ("csum_raw", "csum_distinct"):
            tot[f] = (tot[f] + getattr(ps, f)) % 2 ** 64
        off += n_r
    assert off == S
    assert tot["n_raw"] == st.n_raw == N and tot["n_distinct"] == st.n_distinct and tot["sum_solid_mult"] == st.sum_solid_mult
    assert tot["csum_raw"] == st.csum_raw and tot["csum_distinct"] == st.csum_distinct
    if n_shards > 1 and N > 100000:
        assert max(raws) - min(raws) <= 0.1 * N / n_shards + int(hist.max())
    return S, bounds


@pytest.mark.parametrize("k", [5, 9, 21, 31, 40, 99])
def test_shards_concatenate_to_the_unsharded_output(k):
    w, ctx, reads = _setup(1, k=k, scale=0.3)
    for n in (1, 2, 3, 8):
        _check(w, ctx, reads, n)


def test_more_shards_than_partitions_with_records_and_a_blockwise_shard():
    import paper_1409_7208_b200 as sd
    w, ctx, reads = _setup(1, k=3, scale=0.05)            # 4^4 = 256 distinct edges in 256 partitions at most
    _check(w, ctx, reads, 64)
    # a shard that itself needs block-wise passes: workspace for a fifth of the records, two shards
    w, ctx, reads = _setup(1, k=21)
    small = sd.Context(max(sd.sdbg_workspace_for_records(w.n_raw_edges // 5, w.k), sd.sdbg_min_workspace()))
    _check(w, ctx, reads, 2, workspace_ctx=small, min_ranges=2)


def test_config2_full_size_in_eight_shards():
    w, ctx, reads = _setup(2)
    S, bounds = _check(w, ctx, reads, 8)
    assert S > 10_000_000


def test_bad_range_is_rejected():
    import paper_1409_7208_b200 as sd
    w, ctx, reads = _setup(1, scale=0.05)
    out = sd.Edges(1000, w.k)
    for lo, hi in ((5, 4), (0, 65537)):
        with pytest.raises(sd.SdbgError) as ei:
            sd.sdbg_count_edges_range(ctx, reads, w.n_reads, w.k, w.d, lo, hi, out)
        assert ei.value.name == "SDBG_E_INVAL"
    assert sd.sdbg_count_edges_range(ctx, reads, w.n_reads, w.k, w.d, 7, 7, out) == 0     # empty range
