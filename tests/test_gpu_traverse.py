"""-m gpu: sdbg_index_build / sdbg_forward / sdbg_backward (traversal by rank/select; SURVEY.md §8(f)
rank 3; readings A24-A26) against oracle/sdbg_traverse.py (node strings only), for every edge, bit for bit; zin_bits
and F of sdbg_build_full against the same oracle."""
import random

import numpy as np
import pytest

from oracle.sdbg_traverse import navigation
from tests.helpers import de_bruijn, rc
from tests.test_gpu_full_graph import _run

pytestmark = pytest.mark.gpu


def _check(reads, k, d):
    import torch
    import paper_1409_7208_b200 as sd
    fg, want, ctx, ed = _run(reads, k, d)
    nav = navigation(want, k)
    m = want["m"]
    assert np.array_equal(fg.zin_bits_np(), nav["zin_bits"]), "zin bits differ"
    assert fg.F == nav["F"], (fg.F, nav["F"])
    ix = sd.Index(m)
    sd.sdbg_index_build(ctx, fg, ix)
    W = want["W"]
    ones = [int(((W == c + 1)).sum()) for c in range(4)] + [int(want["last"].sum()) - int(nav["zin"].sum())]
    assert ix.m == m and ix.ones == ones
    q = torch.arange(m + 3, dtype=torch.int64, device="cuda")          # three indices past the end
    out_f = torch.empty(m + 3, dtype=torch.int64, device="cuda")
    out_b = torch.empty(m + 3, dtype=torch.int64, device="cuda")
    sd.sdbg_forward(ctx, ix, q, m + 3, out_f)
    sd.sdbg_backward(ctx, ix, q, m + 3, out_b)
    torch.cuda.synchronize()
    f, b = out_f.cpu().numpy(), out_b.cpu().numpy()
    assert np.array_equal(f[:m], nav["forward"]), "forward differs"
    assert np.array_equal(b[:m], nav["backward"]), "backward differs"
    assert np.all(f[m:] == -2) and np.all(b[m:] == -2)
    # queries in random order with repeats give the same answers
    if m:
        rng = np.random.default_rng(k)
        idx = rng.integers(0, m, size=min(4 * m, 20000))
        qi = torch.from_numpy(idx).cuda()
        o = torch.empty(len(idx), dtype=torch.int64, device="cuda")
        sd.sdbg_forward(ctx, ix, qi, len(idx), o)
        torch.cuda.synchronize()
        assert np.array_equal(o.cpu().numpy(), nav["forward"][idx])
    return fg, want, nav, ix, ctx


def test_simple_path_complete_graph_and_empty_graph():
    r = "ACGGATTCAGCA"
    fg, want, nav, ix, _ = _check([r, r], 4, 2)
    assert int(nav["zin"].sum()) == 2 and int((nav["backward"] == -1).sum()) >= 2
    for k in (3, 4, 5):                                   # m = 4^(k+1): no dummies, F splits the edges in four
        fg, want, nav, ix, _ = _check([de_bruijn("ACGT", k + 1)], k, 2)
        assert fg.F == [0, want["m"] // 4, want["m"] // 2, 3 * want["m"] // 4, want["m"]]
    _check(["ACG"], 5, 2)                                  # no window at all: m = 0, every query is out of range


@pytest.mark.parametrize("k", [2, 3, 5, 16, 21, 31, 32, 33, 63, 64, 65, 99, 127])
def test_ragged_reads_all_key_widths(k):
    rng = random.Random(2000 + k)
    src = ["".join(rng.choice("ACGT") for _ in range(rng.randint(k + 1, k + 120))) for _ in range(4)]
    reads = []
    for _ in range(80):
        s = rng.choice(src)
        a = rng.randint(0, len(s)); b = rng.randint(a, len(s))
        x = s[a:b] if rng.random() < 0.6 else rc(s[a:b])
        if x and rng.random() < 0.2:
            q = rng.randrange(len(x)); x = x[:q] + rng.choice("ACGT") + x[q + 1:]
        reads.append(x)
    for d in (1, 2):
        _check(reads, k, d)


@pytest.mark.parametrize("k", [5, 8, 21, 31, 40])
def test_synthetic_medium_spans_many_cells_and_samples(k):
    """Hundreds of 448-edge cells and several select samples per vector; k = 5 and 8 give dense graphs with many minus
    edges and long runs of one base (the select samples then lie many cells apart for some vectors)."""
    from workloads import ReadGenerator, get_config
    cfg = get_config(1, scale=0.08)
    bases, offs = ReadGenerator(cfg).host()
    fg, want, nav, ix, _ = _check((bases, offs), k, 2 if k > 8 else 1)
    assert want["m"] > 448 * (4 if k == 5 else 20)
    if k <= 8:
        assert int((want["W"] > 4).sum()) > 0


def test_argument_errors():
    import torch
    import paper_1409_7208_b200 as sd
    r = "ACGGATTCAGCA"
    fg, want, nav, ix, ctx = _check([r, r], 4, 2)
    small = sd.Index(want["m"])
    small.c.bytes = 64
    with pytest.raises(sd.SdbgError) as ei:
        sd.sdbg_index_build(ctx, fg, small)
    assert ei.value.name == "SDBG_E_CAPACITY"
    fg.c.zin_bits = None
    with pytest.raises(sd.SdbgError) as ei:
        sd.sdbg_index_build(ctx, fg, sd.Index(want["m"]))
    assert ei.value.name == "SDBG_E_INVAL"


def test_config1_at_full_size_every_edge():
    """BASELINE config 1 (30,000 reads of 100 bp, k = 21): about 0.7 M edges, 1,500 cells, hundreds of select samples."""
    from workloads import ReadGenerator, get_config
    cfg = get_config(1)
    bases, offs = ReadGenerator(cfg).host()
    fg, want, nav, ix, _ = _check((bases, offs), cfg.k, 1)
    assert want["m"] > 448 * 1000


def test_edge_count_a_multiple_of_the_cell_size():
    """m = 448 j exactly: rank at position m reads the extra (empty) cell behind the last full one."""
    from oracle import Oracle
    from oracle.sdbg_oracle import reads_to_arrays
    k, found = 5, None
    for seed in range(4000):
        rng = random.Random(seed)
        n_src = rng.randint(1, 3)
        src = ["".join(rng.choice("ACGT") for _ in range(rng.randint(150, 400))) for _ in range(n_src)]
        o = Oracle(k, 1)
        o.add_reads(*reads_to_arrays(src))
        res = o.finish(want_distinct=False)
        # m = solid edges + nodes without outgoing edge; computed here from the strings, cheaply
        S = res.solid_strings()
        src_nodes = {e[:k] for e in S}
        m = len(S) + len({e[1:] for e in S} - src_nodes)
        o.close()
        if m >= 448 and m % 448 == 0:
            found = src
            break
    assert found is not None, "no seed gave m = 448 j"
    fg, want, nav, ix, _ = _check(found, k, 1)
    assert want["m"] % 448 == 0


def test_two_letter_reads_leave_two_classes_empty():
    """Reads over {A, T} only (closed under reverse complement): no node ends with C or G, so F[1] = F[2] = F[3] and the
    vectors B_C, B_G have no one at all."""
    rng = random.Random(11)
    reads = ["".join(rng.choice("AT") for _ in range(rng.randint(20, 90))) for _ in range(40)]
    for k in (3, 7, 12):
        fg, want, nav, ix, _ = _check(reads, k, 1)
        assert fg.F[1] == fg.F[2] == fg.F[3] and ix.ones[1] == 0 and ix.ones[2] == 0 and ix.ones[0] > 0 and ix.ones[3] > 0
