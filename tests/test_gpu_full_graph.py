"""-m gpu: sdbg_build_full (the lossless extras of PAPER.md:31: '$' edges, zero-indegree vector, validity bits) against
Oracle.full_graph(), bit for bit."""
import random

import numpy as np
import pytest

from oracle import Oracle
from oracle.sdbg_oracle import reads_to_arrays
from tests.helpers import de_bruijn, rc

pytestmark = pytest.mark.gpu


def _run(reads, k, d, workspace_extra=0):
    import torch
    import paper_1409_7208_b200 as sd
    bases, offs = reads if isinstance(reads, tuple) else reads_to_arrays(list(reads))
    o = Oracle(k, d)
    o.add_reads(bases, offs)
    res = o.finish()
    want = o.full_graph()
    o.close()
    nb = int(offs[-1])
    ctx = sd.Context(sd.sdbg_full_workspace(max(nb, 1), k) + (1 << 22) + workspace_extra)
    rd = sd.Reads(nb)
    b = torch.from_numpy(np.array(bases, dtype=np.uint8)).cuda() if len(bases) else torch.zeros(1, dtype=torch.uint8, device="cuda")
    sd.sdbg_pack_reads(ctx, b, torch.from_numpy(offs.view(np.int64)).cuda(), len(offs) - 1, rd)
    ed = sd.Edges(max(res.n_solid, 1), k)
    sd.sdbg_count_edges(ctx, rd, rd.n_reads, k, d, ed, None)
    assert ed.n == res.n_solid
    fg = sd.FullGraph(want["m"], want["t"], k)
    unstable_before = sd.sdbg_unstable_radix_launches()
    sd.sdbg_build_full(ctx, ed, fg)
    # its single radix pass refines an existing order: it must be the stable kernel (include/sdbg.h, kernels.cuh RadixArgs)
    assert sd.sdbg_unstable_radix_launches() == unstable_before, "sdbg_build_full launched the unstable radix pass"
    assert (fg.m, fg.t, fg.n_zero_out) == (want["m"], want["t"], want["n_zero_out"])
    assert np.array_equal(fg.W_np(), want["W"]), "W differs"
    assert np.array_equal(fg.mult_np(), want["mult"]), "mult differs"
    assert np.array_equal(fg.last_bits_np(), want["last_bits"]), "last differs"
    assert np.array_equal(fg.valid_bits_np(), want["valid_bits"]), "validity bits differ"
    assert np.array_equal(fg.aux_bits_np(), want["aux_bits"]), "auxiliary vector differs"
    return fg, want, ctx, ed


def test_simple_path_and_complete_graph():
    r = "ACGGATTCAGCA"
    fg, want, _, _ = _run([r, r], 4, 2)
    assert fg.t == 2 and fg.n_zero_out == 2
    fg, _, _, _ = _run([de_bruijn("ACGT", 4)], 3, 2)
    assert fg.t == 0 and fg.n_zero_out == 0


@pytest.mark.parametrize("k", [2, 3, 5, 15, 16, 21, 31, 32, 33, 47, 63, 64, 65, 95, 96, 99, 127])
def test_ragged_reads_all_key_widths(k):
    rng = random.Random(1000 + k)
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
        _run(reads, k, d)


@pytest.mark.parametrize("k", [21, 31, 40, 99])
def test_synthetic_medium(k):
    from workloads import ReadGenerator, get_config
    cfg = get_config(1, scale=0.08) if k < 99 else get_config(2, scale=0.002)
    bases, offs = ReadGenerator(cfg).host()
    fg, want, _, _ = _run((bases, offs), k, 2)
    assert fg.t == fg.n_zero_out > 0           # strand symmetry; coverage gaps and read ends leave open nodes


def test_capacity_and_argument_errors():
    import paper_1409_7208_b200 as sd
    r = "ACGGATTCAGCA"
    fg, want, ctx, ed = _run([r, r], 4, 2)
    small = sd.FullGraph(want["m"] - 1, want["t"], 4)
    with pytest.raises(sd.SdbgError) as ei:
        sd.sdbg_build_full(ctx, ed, small)
    assert ei.value.name == "SDBG_E_CAPACITY" and small.m == want["m"] and small.t == want["t"]
    small = sd.FullGraph(want["m"], want["t"] - 1, 4)
    with pytest.raises(sd.SdbgError) as ei:
        sd.sdbg_build_full(ctx, ed, small)
    assert ei.value.name == "SDBG_E_CAPACITY"
    ed1 = sd.Edges(4, 1)
    with pytest.raises(sd.SdbgError) as ei:
        sd.sdbg_build_full(ctx, ed1, sd.FullGraph(4, 4, 1))
    assert ei.value.name == "SDBG_E_UNSUPPORTED"
