"""-m gpu: sdbg_mercy_edges (mercy-kmers of PAPER.md:35) against Oracle.mercy(): the same multiset of records, and the
graph rebuilt from solid + mercy records (sdbg_build on unsorted input) against the oracle's merge of the two."""
import random

import numpy as np
import pytest

from oracle import Oracle
from oracle.sdbg_oracle import reads_to_arrays
from tests.helpers import rc

pytestmark = pytest.mark.gpu


def _sorted_rows(a):
    a = np.ascontiguousarray(a)
    return a[np.lexsort(a.T[::-1])] if len(a) else a


def _run(reads, k, d):
    import torch
    import paper_1409_7208_b200 as sd
    bases, offs = reads if isinstance(reads, tuple) else reads_to_arrays(list(reads))
    bases = np.array(bases, dtype=np.uint8)
    o = Oracle(k, d)
    o.add_reads(bases, offs)
    res = o.finish()
    want = o.mercy(bases, offs)
    o.close()
    nb = int(offs[-1])
    ctx = sd.Context(sd.sdbg_full_workspace(max(nb, 1), k) + (1 << 24))
    rd = sd.Reads(nb)
    sd.sdbg_pack_reads(ctx, torch.from_numpy(bases).cuda(), torch.from_numpy(offs.view(np.int64)).cuda(), len(offs) - 1, rd)
    ed = sd.Edges(max(res.n_solid, 1), k)
    sd.sdbg_count_edges(ctx, rd, rd.n_reads, k, d, ed, None)
    n_want = len(want["keys"])
    me = sd.Edges(max(n_want, 1), k)
    unstable_before = sd.sdbg_unstable_radix_launches()
    n = sd.sdbg_mercy_edges(ctx, rd, ed, me)
    assert sd.sdbg_unstable_radix_launches() == unstable_before, "sdbg_mercy_edges launched the unstable radix pass"
    assert n == n_want
    got = me.keys_np()
    assert np.array_equal(_sorted_rows(got), _sorted_rows(want["keys"])), "mercy records differ"
    assert np.all(me.mult_np() == 1)
    return ctx, rd, ed, me, res, want


def test_bridged_gap_closed_form():
    rng = random.Random(3)
    g = "".join(rng.choice("ACGT") for _ in range(120))
    ctx, rd, ed, me, res, want = _run([g[0:50]] * 3 + [g[70:120]] * 3 + [g[30:90]], 11, 2)
    assert me.n == 62
    ctx, rd, ed, me, res, want = _run([g[0:50]] * 3 + [g[70:120]] * 3 + [g[30:90]] * 2, 11, 2)
    assert me.n == 0


@pytest.mark.parametrize("k", [3, 8, 11, 21, 31, 32, 40, 63, 64, 70, 99, 127])
def test_random_low_coverage_reads(k):
    """Reads cut from a few sources at low coverage: gaps bridged by single reads occur; every key width."""
    rng = random.Random(900 + k)
    total = 0
    for trial in range(3):
        src = ["".join(rng.choice("ACGT") for _ in range(rng.randint(3 * k + 10, 3 * k + 200))) for _ in range(3)]
        reads = []
        for _ in range(40):
            s = rng.choice(src)
            a = rng.randint(0, len(s) - k - 1); b = rng.randint(a, len(s))
            reads.append(s[a:b] if rng.random() < 0.6 else rc(s[a:b]))
        ctx, rd, ed, me, res, want = _run(reads, k, 2)
        total += me.n
    assert total > 0 or k < 8


def test_synthetic_workload_and_rebuild():
    """Config-1-like reads at low coverage (many gaps), several pack calls; then the graph over solid + mercy records:
    sdbg_build on the unsorted union == the oracle's sort/merge of the same union."""
    import torch
    import paper_1409_7208_b200 as sd
    from dataclasses import replace
    from workloads import ReadGenerator, get_config
    k = 21
    cfg = replace(get_config(1, scale=0.2), n_reads=1800)              # ~9x coverage of a 20 kbp genome: d=2 leaves gaps
    bases, offs = ReadGenerator(cfg).host()
    ctx, rd, ed, me, res, want = _run((bases, offs), k, 2)
    assert me.n > 100
    # capacity one short -> needed count
    small = sd.Edges(me.n - 1, k)
    with pytest.raises(sd.SdbgError) as ei:
        sd.sdbg_mercy_edges(ctx, rd, ed, small)
    assert ei.value.name == "SDBG_E_CAPACITY" and small.n == me.n
    # union -> sdbg_build (unsorted): equal keys merged, mult summed
    S, M, w = ed.n, me.n, ed.w
    allk = sd.Edges(S + M, k)
    allk.keys[: S * w] = ed.keys[: S * w]; allk.keys[S * w:(S + M) * w] = me.keys[: M * w]
    allk.mult[:S] = ed.mult[:S]; allk.mult[S:S + M] = me.mult[:M]
    allk.c.n = S + M
    g = sd.Graph(S + M)
    sd.sdbg_build(ctx, allk, 0, g)
    torch.cuda.synchronize()
    # oracle side: counts of the union, by plain dict
    cnt = {}
    for row, m in zip(res.keys, res.mult):
        cnt[tuple(int(x) for x in row)] = int(m)
    for row in want["keys"]:
        t = tuple(int(x) for x in row)
        cnt[t] = cnt.get(t, 0) + 1
    keys_sorted = sorted(cnt)
    assert allk.n == len(keys_sorted)
    assert [tuple(int(x) for x in r) for r in allk.keys_np()] == keys_sorted
    assert list(allk.mult_np()) == [cnt[t] for t in keys_sorted]
