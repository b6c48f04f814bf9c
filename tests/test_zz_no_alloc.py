"""-m gpu: sdbg_index_build_static (include/sdbg.h) — the traversal index built with the library's static
device scratch, for callers that cannot allocate — against sdbg_index_build on the same graphs: every cell word, every
select sample, the ones counts and rank_H(F[c]) bit for bit, and the same forward / backward images, on two calls in a
row (the second on another graph, so whatever the first left in the shared scratch must not leak), then the first graph
again. The entry point is refused beyond its stated maximum. Collected last on purpose (the name): a failure here hides
no other test under pytest -x. Needs no state from other tests."""
import random

import numpy as np
import pytest

pytestmark = pytest.mark.gpu


def _reads(seed, glen, n, rlen):
    from tests.helpers import rc
    rng = random.Random(seed)
    genome = "".join(rng.choice("ACGT") for _ in range(glen))
    out = []
    for _ in range(n):
        a = rng.randint(0, glen - rlen)
        x = genome[a:a + rlen]
        out.append(x if rng.random() < 0.5 else rc(x))
    return out


def _full_graph(reads, k, d):
    """sdbg_pack_reads -> sdbg_count_edges -> sdbg_build_full through the ordinary ctx path."""
    import torch
    import paper_1409_7208_b200 as sd
    bases = np.frombuffer("".join(reads).encode(), dtype=np.uint8).copy()
    offs = np.zeros(len(reads) + 1, dtype=np.uint64)
    offs[1:] = np.cumsum([len(r) for r in reads])
    ctx = sd.Context(sd.sdbg_full_workspace(len(bases), k) + (64 << 20))
    pr = sd.Reads(len(bases))
    sd.sdbg_pack_reads(ctx, torch.from_numpy(bases).cuda(), torch.from_numpy(offs.astype(np.int64)).cuda(), len(reads), pr)
    n_raw = 2 * sum(max(0, len(r) - k) for r in reads)
    edges = sd.Edges(max(n_raw, 1), k)
    sd.sdbg_count_edges(ctx, pr, len(reads), k, d, edges, sd.Stats())
    fg = sd.FullGraph(2 * edges.n + 8, edges.n + 8, k)
    sd.sdbg_build_full(ctx, edges, fg)
    torch.cuda.synchronize()
    return ctx, fg, (pr, edges)


def _index_words(ix, m):
    """cells and select samples of the block (the part both entry points define), as numpy."""
    import paper_1409_7208_b200 as sd
    n = sd.lib().sdbg_index_static_bytes(m) // 8
    cells = ix.cells[:n].cpu().numpy()
    n_cells = m // 448 + 1
    body = cells[:5 * n_cells * 8].copy()
    samples = cells[5 * n_cells * 8:].view(np.uint32)
    per = (len(samples)) // 5
    used = [samples[c * per: c * per + (ix.ones[c] + 511) // 512].copy() for c in range(5)]
    return body, used


def _compare(ctx, fg, stream=None):
    import torch
    import paper_1409_7208_b200 as sd
    m = fg.m
    want = sd.Index(m)
    sd.sdbg_index_build(ctx, fg, want)
    got = sd.Index(m)
    got.cells.fill_(-1)                                   # the static path must write everything it defines
    torch.cuda.synchronize()                              # (the fill runs on torch's stream, the build may not)
    sd.sdbg_index_build_static(fg, got, stream)
    assert got.m == want.m == m and got.ones == want.ones and got.HF == want.HF
    assert [int(x) for x in got.c.F] == [int(x) for x in want.c.F] and got.c.n_cells == want.c.n_cells
    wb, ws = _index_words(want, m)
    gb, gs = _index_words(got, m)
    assert np.array_equal(wb, gb), "cells differ"
    for c in range(5):
        assert np.array_equal(ws[c], gs[c]), f"select samples of vector {c} differ"
    q = torch.arange(m + 2, dtype=torch.int64, device="cuda")
    outs = []
    for ix in (want, got):
        f = torch.empty(m + 2, dtype=torch.int64, device="cuda")
        b = torch.empty(m + 2, dtype=torch.int64, device="cuda")
        sd.sdbg_forward(ctx, ix, q, m + 2, f)
        sd.sdbg_backward(ctx, ix, q, m + 2, b)
        torch.cuda.synchronize()
        outs.append((f.cpu().numpy(), b.cpu().numpy()))
    assert np.array_equal(outs[0][0], outs[1][0]) and np.array_equal(outs[0][1], outs[1][1])
    return m


def test_static_index_build_matches_the_ctx_path_on_calls_in_a_row():
    import torch
    ctx_a, fg_a, keep_a = _full_graph(_reads(11, 60000, 6000, 100), 21, 2)     # ~ 10^5 edges: hundreds of cells, several blocks
    ctx_b, fg_b, keep_b = _full_graph(_reads(12, 3000, 400, 80), 31, 2)        # a few thousand edges
    m_a = _compare(ctx_a, fg_a)
    m_b = _compare(ctx_b, fg_b)                                                # second call in a row, smaller graph
    assert m_a > 64 * 448 * 3 and 0 < m_b < m_a
    assert _compare(ctx_a, fg_a, torch.cuda.Stream()) == m_a                   # third: the first graph again, own stream


def test_static_index_build_refuses_what_does_not_fit():
    import paper_1409_7208_b200 as sd
    L = sd.lib()
    cap = L.sdbg_index_static_max_edges()
    assert cap == 1 << 28
    ctx, fg, keep = _full_graph(_reads(13, 2000, 200, 60), 15, 2)
    ix = sd.Index(fg.m)
    m_true = fg.c.m
    fg.c.m = cap + 1                                      # beyond the static scratch: refused before anything runs
    with pytest.raises(sd.SdbgError) as ei:
        sd.sdbg_index_build_static(fg, ix)
    assert ei.value.name == "SDBG_E_CAPACITY" and "at most" in str(ei.value)
    fg.c.m = m_true
    small = sd.Index(fg.m)
    small.c.bytes = L.sdbg_index_static_bytes(fg.m) - 8   # the caller's block too small
    with pytest.raises(sd.SdbgError) as ei:
        sd.sdbg_index_build_static(fg, small)
    assert ei.value.name == "SDBG_E_CAPACITY"
    sd.sdbg_index_build_static(fg, ix)                    # and it still works afterwards
    assert ix.m == m_true
