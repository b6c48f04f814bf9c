"""-m gpu: the CUDA path (through the C ABI binding) against the CPU oracle, element by element, bit-exact."""
import random

import numpy as np
import pytest

from oracle import run_oracle
from tests.gpu_util import assert_matches_oracle, run_gpu, to_arrays
from tests.helpers import de_bruijn, key_mix_np, rc

pytestmark = pytest.mark.gpu

T0_READS = ["ACGTTGCA", "CGTTGCAT", "TTGCATGA"]
ALL_K = [1, 2, 3, 5, 8, 9, 12, 15, 16, 21, 30, 31, 32, 33, 47, 62, 63, 64, 65, 95, 96, 99, 126, 127]


def _ragged_reads(rng, k, n_src=4, n_reads=60):
    """Reads cut from a few source strings (so counts >= 2 and branching occur), some reverse-complemented, some with
    a substitution, some shorter than k+1 or empty, some lower case."""
    src = ["".join(rng.choice("ACGT") for _ in range(rng.randint(k + 1, k + 90))) for _ in range(n_src)]
    reads = []
    for i in range(n_reads):
        b = rng.choice(src)
        a = rng.randint(0, len(b))
        e = rng.randint(a, len(b))
        x = b[a:e]
        if rng.random() < 0.4:
            x = rc(x)
        if x and rng.random() < 0.3:
            p = rng.randrange(len(x))
            x = x[:p] + rng.choice("ACGT") + x[p + 1:]
        if i % 5 == 0:
            x = x.lower()
        reads.append(x)
    return reads


def test_T0_handworked():
    res = run_gpu(T0_READS, 3, 2)
    orc = run_oracle(T0_READS, 3, 2)
    assert_matches_oracle(res, orc)
    assert res.n == 11 and int(res.last_bits[0]) == 0x7FD and list(res.W) == [2, 1, 4, 3, 1, 4, 2, 6, 3, 4, 3]


@pytest.mark.parametrize("k", ALL_K)
def test_ragged_tiny_all_k(k):
    rng = random.Random(4242 + k)
    for trial in range(3):
        reads = _ragged_reads(rng, k)
        for d in (1, 2, 3):
            assert_matches_oracle(run_gpu(reads, k, d), run_oracle(reads, k, d))


@pytest.mark.parametrize("k", [1, 2, 3, 4, 5, 6])
def test_complete_de_bruijn(k):
    s = de_bruijn("ACGT", k + 1)
    res = run_gpu([s], k, 2)
    S = 4 ** (k + 1)
    assert res.n == S and np.all(res.mult == 2)
    assert list(res.W & 3) == [1, 2, 3, 0] * (S // 4)            # bytes 1..4 (+4): A,C,G,T repeating
    assert_matches_oracle(res, run_oracle([s], k, 2))


@pytest.mark.parametrize("k,d", [(21, 2), (31, 2), (31, 1), (32, 2), (63, 2), (99, 2), (127, 2), (11, 3)])
def test_synthetic_medium(k, d):
    """A few hundred thousand records: many radix tiles and a ragged last tile, for every key width."""
    from workloads import ReadGenerator, get_config
    cfg = get_config(1, scale=0.08) if k < 99 else get_config(2, scale=0.002)     # 150 bp reads for the long keys
    bases, offs = ReadGenerator(cfg).host()
    res = run_gpu((bases, offs), k, d)
    orc = run_oracle((bases, offs), k, d)
    assert orc.n_solid > 100
    assert_matches_oracle(res, orc)
    # P4: the order-independent checksums agree and equal the definition evaluated on the oracle's output
    want = int((key_mix_np(orc.distinct_keys) * orc.distinct_cnt.astype(np.uint64)).sum(dtype=np.uint64))
    assert res.stats.csum_raw == res.stats.csum_distinct == want


@pytest.mark.parametrize("k", [8, 12, 16, 27, 32, 33, 47, 48, 63, 64, 65, 80, 95, 96, 97, 127])
@pytest.mark.parametrize("d", [2, 3])
def test_default_path_every_key_shape(k, d):
    """The default path (no checksums: top passes + table count) at a few hundred thousand records for the key shapes
    where something changes: the last word just begun (k = 32, 64, 96), just filled (31 is covered elsewhere; 63, 95, 127),
    one past (33, 65, 97), keys whose top passes are all there is of a word (k = 8: 18 bits), and both d. The number of
    table launches says that the path ran; the result and the statistics are the oracle's."""
    from workloads import ReadGenerator, get_config
    cfg = get_config(1, scale=0.1) if k < 80 else get_config(2, scale=0.003)      # 150 bp reads for the long keys
    bases, offs = ReadGenerator(cfg).host()
    orc = run_oracle((bases, offs), k, d)
    res = run_gpu((bases, offs), k, d, checksums=False)
    assert_matches_oracle(res, orc, check_stats=True)
    tim = res.ctx.get_timing()
    P = (2 * (k + 1) + 7) // 8
    assert tim.launches["table"] == 1 and tim.launches["radix"] < P, (k, d, tim.launches)


def test_config1_full_and_host_input():
    from workloads import ReadGenerator, get_config
    w = get_config(1)
    bases, offs = ReadGenerator(w).host()
    orc = run_oracle((bases, offs), w.k, w.d)
    res = run_gpu((bases, offs), w.k, w.d, bucket_hist=True)
    assert res.stats.n_raw == w.n_raw_edges and res.stats.n_ranges == 1
    assert_matches_oracle(res, orc)
    # bucket histogram (A11) against the oracle's raw records
    o1 = run_oracle((bases, offs), w.k, 1)
    want = np.bincount((o1.distinct_keys[:, 0] >> np.uint64(48)).astype(np.int64), weights=o1.distinct_cnt, minlength=65536)
    assert np.array_equal(res.stats.bucket_hist.cpu().numpy(), want.astype(np.int64))
    # the same through HOST buffers (H2D staged by the library), packed by 3 appending calls
    res2 = run_gpu((bases, offs), w.k, w.d, host_input=True, n_calls=3)
    assert_matches_oracle(res2, orc)


@pytest.mark.parametrize("k", [21, 40, 99])
def test_P8_plan_independence_blockwise(k):
    """Forcing a tiny workspace (many block-wise ranges of l=8 partitions) gives identical output."""
    import paper_1409_7208_b200 as sd
    from workloads import ReadGenerator, get_config
    cfg = get_config(1, scale=0.3) if k < 99 else get_config(2, scale=0.004)      # 150 bp reads for the long keys
    bases, offs = ReadGenerator(cfg).host()
    orc = run_oracle((bases, offs), k, 2)
    res = run_gpu((bases, offs), k, 2, workspace_bytes=sd.sdbg_min_workspace())
    assert res.stats.n_ranges >= 3, res.stats.n_ranges
    assert_matches_oracle(res, orc)
    # without checksums one-word keys take the default path INSIDE every block-wise range: the most significant passes
    # for the record density of the range, then the table count (launch accounting: table launches, and fewer radix
    # launches than ranges x passes; a last range of a few records alone may go the plain way)
    res2 = run_gpu((bases, offs), k, 2, workspace_bytes=sd.sdbg_min_workspace(), checksums=False)
    assert_matches_oracle(res2, orc)
    tim = res2.ctx.get_timing()
    P = (2 * (k + 1) + 7) // 8
    if k <= 31:
        assert tim.launches["table"] >= res2.stats.n_ranges - 1 and tim.launches["radix"] < res2.stats.n_ranges * P, tim.launches
    else:   # keys of several words take it too where a range holds enough records (short ranges go the plain way)
        assert tim.launches["table"] <= res2.stats.n_ranges


def test_edge_cases():
    import paper_1409_7208_b200 as sd
    # n = 0
    res = run_gpu([], 5, 2)
    assert res.n == 0 and res.stats.n_raw == 0
    # all reads shorter than k+1 / empty
    res = run_gpu(["ACG", "", "AC", "ACGTA"], 5, 1)
    assert res.n == 0 and res.stats.n_raw == 0
    # a read of length exactly k+1
    assert_matches_oracle(run_gpu(["ACGTAC"], 5, 1), run_oracle(["ACGTAC"], 5, 1))
    # d above every count
    assert run_gpu(["ACGTAC", "ACGTAC"], 5, 5).n == 0
    # palindromes double (A5)
    res = run_gpu(["ACGT"] * 5, 3, 2)
    assert res.n == 1 and list(res.mult) == [10]
    # lower case == upper case
    a, b = run_gpu([r.lower() for r in T0_READS], 3, 2), run_gpu(T0_READS, 3, 2)
    assert np.array_equal(a.keys, b.keys) and np.array_equal(a.mult, b.mult)
    # bad base
    with pytest.raises(sd.SdbgError) as ei:
        run_gpu(["ACGTACGT", "ACGNACGT"], 3, 1)
    assert ei.value.name == "SDBG_E_BADBASE" and "index 11" in str(ei.value)
    with pytest.raises(sd.SdbgError) as ei:
        run_gpu(["ACGTACGT", "ACGNACGT"], 3, 1, host_input=True)
    assert ei.value.name == "SDBG_E_BADBASE"
    # capacity one short -> SDBG_E_CAPACITY and out->n = needed
    with pytest.raises(sd.SdbgError) as ei:
        run_gpu(T0_READS, 3, 2, cap=10)
    assert ei.value.name == "SDBG_E_CAPACITY"
    # bad k / d
    for k, d, name in ((0, 2, "SDBG_E_UNSUPPORTED"), (128, 2, "SDBG_E_UNSUPPORTED"), (5, 0, "SDBG_E_INVAL")):
        with pytest.raises(sd.SdbgError) as ei:
            run_gpu(T0_READS, k, d)
        assert ei.value.name == name


def test_capacity_reports_needed_count():
    import paper_1409_7208_b200 as sd
    bases, offs = to_arrays(T0_READS)
    import torch
    ctx = sd.Context(sd.sdbg_min_workspace())
    rd = sd.Reads(len(bases))
    sd.sdbg_pack_reads(ctx, torch.from_numpy(bases).cuda(), torch.from_numpy(offs.view(np.int64)).cuda(), 3, rd)
    ed = sd.Edges(10, 3)
    with pytest.raises(sd.SdbgError):
        sd.sdbg_count_edges(ctx, rd, 3, 3, 2, ed)
    assert ed.n == 11


@pytest.mark.parametrize("k", [5, 31, 33, 99])
def test_build_unsorted_equals_count(k):
    """sdbg_build over raw records with mult 1 (unsorted, with repeats) == sdbg_count_edges at d=1 (one semantics)."""
    import torch
    import paper_1409_7208_b200 as sd
    rng = random.Random(99 + k)
    reads = _ragged_reads(rng, k, n_reads=80)
    orc = run_oracle(reads, k, 1)
    # raw records = the oracle's distinct keys repeated by their counts, shuffled
    keys = np.repeat(orc.distinct_keys, orc.distinct_cnt.astype(np.int64), axis=0)
    perm = np.random.default_rng(k).permutation(len(keys))
    keys = np.ascontiguousarray(keys[perm])
    n, w = len(keys), orc.w
    ctx = sd.Context(sd.sdbg_min_workspace() + 64 * n * w)
    ed = sd.Edges(n, k)
    ed.keys[: n * w] = torch.from_numpy(keys.reshape(-1).view(np.int64)).cuda()
    ed.mult[:n] = 1
    ed.c.n = n
    g = sd.Graph(n)
    sd.sdbg_build(ctx, ed, 0, g)
    torch.cuda.synchronize()
    assert ed.n == orc.n_distinct == g.n
    assert np.array_equal(ed.keys_np(), orc.distinct_keys)
    assert np.array_equal(ed.mult_np(), orc.distinct_cnt)
    assert np.array_equal(g.W_np(), orc.Wbyte) and np.array_equal(g.last_bits_np(), orc.last_bits)


@pytest.mark.parametrize("k", [21, 99])
def test_build_unsorted_many_chunks_and_long_runs(k):
    """sdbg_build on unsorted input whose runs of equal keys cross rounds (32), chunks (1,024) and blocks (8,192):
    raw records of a synthetic workload (every distinct key repeated by its count) plus one key repeated 20,000
    times with large multiplicities (saturating sum, reading A9)."""
    import torch
    import paper_1409_7208_b200 as sd
    from workloads import ReadGenerator, get_config
    cfg = get_config(1, scale=0.05) if k < 99 else get_config(2, scale=0.001)
    bases, offs = ReadGenerator(cfg).host()
    orc = run_oracle((bases, offs), k, 1)
    w = orc.w
    keys = np.repeat(orc.distinct_keys, orc.distinct_cnt.astype(np.int64), axis=0)
    mult = np.ones(len(keys), dtype=np.uint32)
    big = orc.distinct_keys[len(orc.distinct_keys) // 2]
    keys = np.concatenate([keys, np.repeat(big[None, :], 20000, axis=0)])
    mult = np.concatenate([mult, np.full(20000, 300000, dtype=np.uint32)])          # 20,000 x 300,000 > 2^32
    perm = np.random.default_rng(7 + k).permutation(len(keys))
    keys, mult = np.ascontiguousarray(keys[perm]), np.ascontiguousarray(mult[perm])
    n = len(keys)
    ctx = sd.Context(sd.sdbg_min_workspace() + 64 * n * w)
    ed = sd.Edges(n, k)
    ed.keys[: n * w] = torch.from_numpy(keys.reshape(-1).view(np.int64)).cuda()
    ed.mult[:n] = torch.from_numpy(mult.view(np.int32)).cuda()
    ed.c.n = n
    g = sd.Graph(n)
    sd.sdbg_build(ctx, ed, 0, g)
    torch.cuda.synchronize()
    want = orc.distinct_cnt.astype(np.uint64)
    want[len(orc.distinct_keys) // 2] += np.uint64(20000) * np.uint64(300000)
    want = np.minimum(want, np.uint64(2 ** 32 - 1)).astype(np.uint32)
    assert ed.n == orc.n_distinct == g.n
    assert np.array_equal(ed.keys_np(), orc.distinct_keys)
    assert np.array_equal(ed.mult_np(), want) and np.array_equal(g.mult_np(), want)
    assert np.array_equal(g.W_np(), orc.Wbyte) and np.array_equal(g.last_bits_np(), orc.last_bits)


def test_degenerate_long_runs_poly_A():
    """Thousands of identical reads of one letter: every record of a strand is the same key, so one run spans every
    chunk and block of the count sweeps (32-ary run-start search), every radix tile holds one digit value per pass,
    and the multiplicity is the whole record count. Mixed with ordinary reads so that other keys surround the runs."""
    from workloads import ReadGenerator, get_config
    k = 31
    bases, offs = ReadGenerator(get_config(1, scale=0.02)).host()
    extra = ["A" * 150] * 3500 + ["T" * 150] * 500 + ["ACGT" * 40] * 300
    eb, eo = to_arrays(extra)
    bases2 = np.concatenate([bases, eb])
    offs2 = np.concatenate([offs, eo[1:] + offs[-1]])
    orc = run_oracle((bases2, offs2), k, 2)
    assert int(orc.mult.max()) >= 4000 * (150 - k)          # poly-A forward + poly-T reverse strand
    import paper_1409_7208_b200 as sd
    assert_matches_oracle(run_gpu((bases2, offs2), k, 2), orc)
    # block-wise: the poly-A partition alone holds 476,000 records; a workspace for 520,000 forces more than one range
    res = run_gpu((bases2, offs2), k, 2, workspace_bytes=sd.sdbg_workspace_for_records(520000, k))
    assert res.stats.n_ranges >= 2
    assert_matches_oracle(res, orc)
    # and a workspace smaller than that partition is refused (reading A12)
    with pytest.raises(sd.SdbgError) as ei:
        run_gpu((bases2, offs2), k, 2, workspace_bytes=sd.sdbg_min_workspace())
    assert ei.value.name == "SDBG_E_WORKSPACE" and "largest l=8 partition" in str(ei.value)


def test_P9_reverse_complement_closure_of_the_gpu_output():
    """Pin P9 on the CUDA path alone (no oracle involved): the solid set is closed under reverse complement and
    cnt(e) = cnt(rc(e)); the rc of a key is recomputed here from the key's symbols."""
    from workloads import ReadGenerator, get_config
    for k in (21, 31, 40):
        bases, offs = ReadGenerator(get_config(1, scale=0.05)).host()
        res = run_gpu((bases, offs), k, 2)
        w = res.W_words
        vals = [int.from_bytes(b"".join(int(x).to_bytes(8, "big") for x in row), "big") for row in res.keys]
        pad = 64 * w - 2 * (k + 1)
        table = {}
        for v, m in zip(vals, res.mult):
            sym = [((v >> pad) >> (2 * (k - t))) & 3 for t in range(k + 1)]      # key symbols (e[k-1],...,e[0],e[k])
            e = sym[:k][::-1] + [sym[k]]                                         # edge e[0..k]
            table[tuple(e)] = int(m)
        for e, m in table.items():
            r = tuple(3 - x for x in reversed(e))
            assert table.get(r) == m, (k, e)


def test_k_schedule_on_one_resident_read_set():
    """The multi-k loop of the paper (options --k-min 27 --k-max 87 --k-step 10 at PAPER.md:82) as far as
    this path goes: reads are packed once and stay in HBM, sdbg_count_edges + sdbg_build run per k."""
    import torch
    import paper_1409_7208_b200 as sd
    from workloads import ReadGenerator, get_config
    cfg = get_config(2, scale=0.002)
    bases, offs = ReadGenerator(cfg).host()
    ctx = sd.Context(sd.sdbg_full_workspace(cfg.n_bases, 99))
    rd = sd.Reads(cfg.n_bases)
    sd.sdbg_pack_reads(ctx, torch.from_numpy(bases).cuda(), torch.from_numpy(offs.view(np.int64)).cuda(), cfg.n_reads, rd)
    for k in (27, 37, 47, 57, 67, 77, 87, 99):
        orc = run_oracle((bases, offs), k, 2)
        ed = sd.Edges(max(orc.n_solid, 1), k)
        st = sd.Stats(want_checksums=True)
        sd.sdbg_count_edges(ctx, rd, cfg.n_reads, k, 2, ed, st)
        g = sd.Graph(max(ed.n, 1))
        sd.sdbg_build(ctx, ed, sd.SDBG_SORTED, g)
        torch.cuda.synchronize()
        assert ed.n == orc.n_solid and st.n_distinct == orc.n_distinct and st.csum_raw == st.csum_distinct
        assert np.array_equal(ed.keys_np(), orc.keys) and np.array_equal(ed.mult_np(), orc.mult)
        assert np.array_equal(g.W_np(), orc.Wbyte) and np.array_equal(g.last_bits_np(), orc.last_bits)


def test_wide_range_code_path_at_small_size():
    """Ranges of 2^32 records and more use other kernels (wide look-back words, 64-bit run lengths); the option
    SDBG_OPT_FORCE_WIDE sends small inputs down that path (include/sdbg.h), so that it is covered here and not only by
    config 5 (tests/test_gpu_configs.py runs a range of more than 2^32 records for real)."""
    from workloads import ReadGenerator, get_config
    import paper_1409_7208_b200 as sd
    for k, scale in ((21, 0.3), (31, 0.1)):
        bases, offs = ReadGenerator(get_config(1, scale=scale)).host()
        orc = run_oracle((bases, offs), k, 2)
        assert_matches_oracle(run_gpu((bases, offs), k, 2, options=[sd.SDBG_OPT_FORCE_WIDE]), orc)
        assert_matches_oracle(run_gpu((bases, offs), k, 2, workspace_bytes=sd.sdbg_min_workspace()), orc)


@pytest.mark.parametrize("k", [1, 3, 7, 8, 9, 11, 12, 15, 16, 19, 20, 21, 23, 24, 27, 28, 30, 31, 32, 47, 64, 99])
def test_plain_path_without_statistics(k):
    """No checksums, no partition histogram: the extractor's plain path (both keys of a window in one 16-byte store;
    for one-word keys and k >= 8 the digit histograms of the node bytes counted per read position as differences over
    the key bytes). Every boundary of floor(k/4) and of the padding bytes is here; reads of ragged lengths, some
    shorter than a window, put many positions next to a read end."""
    import random
    from oracle import run_oracle
    from tests.gpu_util import run_gpu, assert_matches_oracle
    from tests.helpers import rc
    rng = random.Random(500 + k)
    src = ["".join(rng.choice("ACGT") for _ in range(rng.randint(k + 1, k + 300))) for _ in range(5)]
    reads = []
    for _ in range(300):
        s_ = rng.choice(src)
        a = rng.randint(0, len(s_)); b = min(len(s_), a + rng.randint(0, k + 80))
        reads.append(s_[a:b] if rng.random() < 0.5 else rc(s_[a:b]))
    for d in (1, 2):
        res = run_gpu(reads, k, d, checksums=False)
        assert_matches_oracle(res, run_oracle(reads, k, d), check_stats=False)


def _radix_launches(res):
    """Radix passes over all records since the context was created (launch accounting of sdbg_ctx_get_timing)."""
    return res.ctx.get_timing().launches["radix"]


@pytest.mark.parametrize("k", [15, 21, 31, 40, 70, 99])
def test_table_count_path_and_its_way_back(k):
    """The top-sort + table-count path (api_count.inc count_range_hash, hashcount.cu): records sorted by the most
    significant passes only, segments of whole buckets counted in shared-memory tables. Checked against the oracle and
    against the plain path (option SDBG_OPT_NO_TABLE_COUNT: every pass over every record) and the stable first pass
    (SDBG_OPT_STABLE_FIRST_PASS), statistics included; the number of radix launches says which path ran. Cases: (1) covered reads with one-mismatch
    copies, d = 2 and 3: the path completes with fewer passes than the key has bytes; (2) the all-ones key (T...T at
    k = 31 fills the word) and its all-zero twin; (3) a bucket longer than the search window (poly-A): overflow, the
    records are sorted the plain way from where the top passes left them; (4) reads over two letters only: far more
    distinct keys per bucket than a table holds: overflow; (5) every read twice at d = 2: half of the records of a
    segment are solid edges, more than its 1,024 sort places: overflow. Keys of several words (k = 40, 70, 99: whole
    records go through the top passes of the first key word, the tables hold fingerprints of whole keys and every record
    is compared with the one that installed its slot) run the same cases with longer reads; where the outcome depends on
    how the buckets fall, only the result is checked."""
    import os
    import random
    from oracle import run_oracle
    from tests.gpu_util import run_gpu, assert_matches_oracle
    from tests.helpers import rc
    rng = random.Random(1700 + k)
    P = (2 * (k + 1) + 7) // 8
    genome = "".join(rng.choice("ACGT") for _ in range(3000))
    covered = []
    L = 100 if k <= 31 else k + 60
    for _ in range(1500):
        a = rng.randint(0, len(genome) - L)
        x = list(genome[a:a + L])
        if rng.random() < 0.3:
            x[rng.randrange(L)] = rng.choice("ACGT")
        x = "".join(x)
        covered.append(x if rng.random() < 0.5 else rc(x))
    poly_t = covered + ["T" * (L - 30)] * 5 + ["GATTACA" + "T" * (L - 50)] * 3
    poly_a = covered + ["A" * (L + 50)] * 400
    two_letters = ["".join(rng.choice("AC") for _ in range(L + 20)) for _ in range(1200)]
    twice = ["".join(rng.choice("ACGT") for _ in range(L + 30)) for _ in range(600)] * 2
    multi = k > 31                                        # None: only the result is checked
    cases = [("covered", covered, 2, True), ("covered", covered, 3, True), ("poly_t", poly_t, 2, True),
             ("poly_a", poly_a, 2, False), ("two_letters", two_letters, 2, None if multi else False),
             ("twice", twice, 2, None if multi else False)]
    for name, reads, d, completes in cases:
        orc = run_oracle(reads, k, d)
        res = run_gpu(reads, k, d, checksums=False)
        assert_matches_oracle(res, orc, check_stats=True)
        n_hash = _radix_launches(res)
        if completes is True:
            assert 0 <= n_hash < P - 1, (name, k, d, n_hash)           # top passes only, the first of them fused with extraction
        elif completes is False:
            assert P <= n_hash < 2 * P, (name, k, d, n_hash)           # top passes, then all passes (the way back)
        import paper_1409_7208_b200 as sd
        for opt in (sd.SDBG_OPT_NO_TABLE_COUNT, sd.SDBG_OPT_STABLE_FIRST_PASS, sd.SDBG_OPT_NO_FUSED_EXTRACT):
            res2 = run_gpu(reads, k, d, checksums=False, options=[opt])
            assert_matches_oracle(res2, orc, check_stats=True)
            if opt == sd.SDBG_OPT_NO_TABLE_COUNT:
                assert _radix_launches(res2) == P, (name, k, d)
            assert res2.edges.n == res.edges.n
    if multi:   # keys that share their first word under the weak fingerprint: caught by the check, redone the plain way
        resw = run_gpu(covered, k, 2, checksums=False, options=[sd.SDBG_OPT_WEAK_FINGERPRINT])
        assert_matches_oracle(resw, run_oracle(covered, k, 2), check_stats=True)
        assert P <= _radix_launches(resw) < 2 * P, (k, _radix_launches(resw))
    # d = 1 keeps every distinct edge: the table count is not used, the records go through all passes exactly once
    res1 = run_gpu(covered, k, 1, checksums=False)
    assert_matches_oracle(res1, run_oracle(covered, k, 1), check_stats=True)
    assert _radix_launches(res1) == P
