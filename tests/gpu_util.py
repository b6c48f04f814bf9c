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
            n_calls=1, ctx=None, options=()):
    """reads: list[str] or (bases uint8, offsets uint64) numpy pair or (torch cuda bases, torch cuda offsets).
    options: SDBG_OPT_* switched on in the context made here (include/sdbg.h sdbg_ctx_set_option)."""
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
        for opt in options:
            ctx.set_option(opt, 1)
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


# ---- full-size configs: oracle-verified sampled l=8 partitions + global invariants (BASELINE.json north_star) ----------

SYM = "ACGT"


def bucket_prefix(b: int) -> str:
    """l=8 partition number (top 16 key bits) -> its 8 key-string symbols."""
    return "".join(SYM[(b >> (14 - 2 * t)) & 3] for t in range(8))


_PAR = {}


def _scan_part(args):
    from oracle import Oracle
    a, b = args
    bases, offs, k, prefixes = _PAR["bases"], _PAR["offs"], _PAR["k"], _PAR["prefixes"]
    o = Oracle(k, 1, prefixes)
    o.add_reads(bases[int(offs[a]):int(offs[b])], offs[a:b + 1] - offs[a])
    e = o.raw_edges()
    o.close()
    return e


def oracle_partitions(bases, offs, k, d, buckets, nproc=None):
    """The oracle restricted to the given l=8 partitions. Step 1 (the scan of the reads) runs in `nproc` forked
    processes over disjoint parts of the reads; steps 2-5 run in one oracle instance on the union of the kept records
    (oracle/sdbg_oracle.c header). Returns the OracleResult of the union (partitions concatenated in sorted order)."""
    import multiprocessing as mp
    import os
    from oracle import Oracle
    prefixes = [bucket_prefix(b) for b in sorted(buckets)]
    n = len(offs) - 1
    nproc = nproc or min(os.cpu_count() or 1, 16)
    parts = max(1, min(n, nproc * 4))
    cuts = [n * i // parts for i in range(parts + 1)]
    _PAR.update(bases=bases, offs=offs, k=k, prefixes=prefixes)
    parent = Oracle(k, d, prefixes)
    if nproc == 1:
        for ab in zip(cuts, cuts[1:]):
            parent.add_edges(_scan_part(ab))
    else:
        with mp.get_context("fork").Pool(nproc) as pool:
            for e in pool.imap(_scan_part, list(zip(cuts, cuts[1:]))):
                parent.add_edges(e)
    _PAR.clear()
    res = parent.finish(want_distinct=False)
    parent.close()
    return res


def run_gpu_workload(w, workspace_bytes=None, chunk_bases=1 << 30, keep_ascii=False):
    """Config-sized run through the C ABI: reads generated in HBM chunk by chunk and packed by appending calls,
    sdbg_count_edges (twice when the number of solid edges is not known: first with capacity 0), sdbg_build."""
    import torch
    from workloads import ReadGenerator
    gen = ReadGenerator(w)
    reads_per_chunk = max(1, chunk_bases // w.read_len)
    n_calls = (w.n_reads + reads_per_chunk - 1) // reads_per_chunk
    ws = workspace_bytes if workspace_bytes is not None else sd.sdbg_workspace_for_records(w.n_raw_edges, w.k)
    ctx = sd.Context(ws)
    rd = sd.Reads(w.n_bases, n_calls)
    buf = torch.empty(min(w.n_reads, reads_per_chunk) * w.read_len, dtype=torch.uint8, device="cuda")
    host = np.empty(w.n_bases, dtype=np.uint8) if keep_ascii else None
    for c in range(n_calls):
        r0, r1 = c * reads_per_chunk, min(w.n_reads, (c + 1) * reads_per_chunk)
        b, o = gen.device(r0, r1, out=buf)
        sd.sdbg_pack_reads(ctx, b, o, r1 - r0, rd)
        if keep_ascii:
            host[r0 * w.read_len:r1 * w.read_len] = b.cpu().numpy()
    del buf
    torch.cuda.empty_cache()
    st = sd.Stats(want_checksums=True, want_bucket_hist=True)
    probe = sd.Edges(0, w.k)
    try:
        sd.sdbg_count_edges(ctx, rd, rd.n_reads, w.k, w.d, probe, st)
    except sd.SdbgError as e:
        assert e.name == "SDBG_E_CAPACITY", e
    S = probe.n
    ed = sd.Edges(S, w.k)
    st = sd.Stats(want_checksums=True, want_bucket_hist=True)
    sd.sdbg_count_edges(ctx, rd, rd.n_reads, w.k, w.d, ed, st)
    assert ed.n == S
    g = sd.Graph(S)
    sd.sdbg_build(ctx, ed, sd.SDBG_SORTED, g)
    torch.cuda.synchronize()
    res = GpuResult()
    res.ctx, res.reads, res.edges, res.graph, res.stats, res.n, res.host_ascii = ctx, rd, ed, g, st, S, host
    return res


def _u64_sorted_view(t):
    """int64 tensor holding u64 bit patterns -> int64 tensor with the same order as the unsigned values."""
    return t ^ (-(2 ** 63))


# ---- multi-word keys as lists of int64 tensors holding u64 bit patterns (word 0 most significant); any device ------------

def _lsr(x, n):
    """Logical shift right of u64 bit patterns held in int64."""
    if n == 0:
        return x
    if n >= 64:
        return x * 0
    return (x >> n) & ((1 << (64 - n)) - 1)


def _shl(x, n):
    if n == 0:
        return x
    if n >= 64:
        return x * 0
    return x << n


def _mw_shl(words, nbits):
    """(w0:w1:...:w_{W-1}) << nbits, zeros shifted in."""
    W = len(words)
    q, r = divmod(nbits, 64)
    out = []
    for j in range(W):
        hi = words[j + q] if j + q < W else None
        lo = words[j + q + 1] if j + q + 1 < W else None
        v = _shl(hi, r) if hi is not None else words[0] * 0
        if r and lo is not None:
            v = v | _lsr(lo, 64 - r)
        out.append(v)
    return out


def _mw_shr(words, nbits):
    W = len(words)
    q, r = divmod(nbits, 64)
    out = []
    for j in range(W):
        lo = words[j - q] if j - q >= 0 else None
        hi = words[j - q - 1] if j - q - 1 >= 0 else None
        v = _lsr(lo, r) if lo is not None else words[0] * 0
        if r and hi is not None:
            v = v | _shl(hi, 64 - r)
        out.append(v)
    return out


def _s64(v):
    """Python int in [0, 2^64) -> the int64 with the same bit pattern."""
    v &= 2 ** 64 - 1
    return v - 2 ** 64 if v >= 2 ** 63 else v


def _rev2(x):
    """Reverses the order of the 32 two-bit groups of every u64 pattern."""
    for sh, m in ((2, 0x3333333333333333), (4, 0x0F0F0F0F0F0F0F0F), (8, 0x00FF00FF00FF00FF), (16, 0x0000FFFF0000FFFF)):
        x = (_lsr(x, sh) & m) | ((x & m) << sh)
    return _lsr(x, 32) | (x << 32)


def rc_key_words(words, k):
    """Key of rc(e) from the key of e, on the integer keys alone (tests/test_oracle_pins.py checks it against strings).
    Key symbols of e: s = (e[k-1], ..., e[0], e[k]); of rc(e): (c(s[k-2]), ..., c(s[0]), c(s[k]), c(s[k-1])), c = 3 - x
    ("useful identities")."""
    W = len(words)
    pad = 64 * W - 2 * (k + 1)
    R = [_rev2(x) for x in reversed(words)]              # (pad zeros, s[k], s[k-1], ..., s[0])
    X = _mw_shl(R, pad)                                  # (s[k], s[k-1], s[k-2], ..., s[0], zeros)
    T = [X[0] & _s64(0xF << 60)] + [x * 0 for x in X[1:]]   # the two leading symbols alone
    Y = _mw_shl(X, 4)                                    # (s[k-2], ..., s[0], 0, 0, zeros)
    Tm = _mw_shr(T, 2 * (k - 1))                         # (zeros, s[k], s[k-1]) at symbol places k-1, k
    out = []
    for q in range(W):
        nb = min(64, max(0, 2 * (k + 1) - 64 * q))       # significant bits of word q
        sig = _s64(((1 << nb) - 1) << (64 - nb)) if nb else 0
        out.append((Y[q] | Tm[q]) ^ sig)
    return out


_M1, _M2 = _s64(0xBF58476D1CE4E5B9), _s64(0x94D049BB133111EB)


def _mix64_t(z):
    z = (z ^ _lsr(z, 30)) * _M1
    z = (z ^ _lsr(z, 27)) * _M2
    return z ^ _lsr(z, 31)


def key_mix_t(words):
    """include/sdbg.h checksum of a key, on int64 tensors (wrapping arithmetic)."""
    h = words[0] * 0
    for x in words:
        h = _mix64_t(h ^ x)
    return h


def check_global_invariants(res, w):
    """Properties that hold at any size, evaluated on the device."""
    import torch
    st, ed, g, S, W = res.stats, res.edges, res.graph, res.n, res.edges.w
    k = w.k
    assert st.n_raw == w.n_raw_edges                                   # P3: N = 2 sum max(0, L - k)
    assert st.csum_raw == st.csum_distinct                             # P4: the sort/count lost or duplicated nothing
    assert st.n_solid == S and S <= st.n_distinct <= st.n_raw
    mult = ed.mult[:S]
    assert int(mult.to(torch.int64).sum()) == st.sum_solid_mult and int(mult.min()) >= w.d
    assert torch.equal(g.mult[:S], mult)
    keys = ed.keys[:S * W].view(S, W)
    # P5: strictly increasing multi-word keys; and nodes (top 2k bits) for P6
    gt = torch.zeros(S - 1, dtype=torch.bool, device="cuda")
    eq = torch.ones(S - 1, dtype=torch.bool, device="cuda")
    node_eq = torch.ones(S - 1, dtype=torch.bool, device="cuda")
    for q in range(W):
        col = _u64_sorted_view(keys[:, q].contiguous())
        a, b = col[:-1], col[1:]
        gt |= eq & (b > a)
        eq &= (b == a)
        nb = min(64, max(0, 2 * k - 64 * q))                          # bits of this word that belong to the node
        if nb == 64:
            node_eq &= (b == a)
        elif nb > 0:
            node_eq &= ((keys[1:, q] ^ keys[:-1, q]) >> (64 - nb)) == 0   # arithmetic shift: zero iff the top nb bits agree
        del col, a, b
    assert bool(gt.all()), "keys not strictly increasing"
    n_nodes = int((~node_eq).sum()) + 1
    lb = g.last_bits[:(S + 63) // 64]
    bits = ((lb.unsqueeze(1) >> torch.arange(64, device="cuda")) & 1).reshape(-1)[:S]
    assert int(bits.sum()) == n_nodes                                  # P6: one `last` per distinct node
    assert torch.equal(bits[:-1].bool(), ~node_eq) and int(bits[-1]) == 1
    del bits, gt, eq, node_eq
    Wb = g.W[:S]
    assert int(Wb.min()) >= 1 and int(Wb.max()) <= 8
    sym = (keys[:, W - 1] >> (64 * W - 2 * (k + 1))) & 3              # outgoing base = last symbol of the key
    assert torch.equal(((Wb - 1) & 3).to(torch.int64), sym)
    del sym
    # P7 (north_star): the minus flag is set iff an earlier edge sharing the (k-1)-suffix of the node has
    # the same outgoing base. Such edges share the top 2(k-1) key bits, so they are at most 15 places back (a group has
    # at most 4 x 4 edges): c = (top 2(k-1) bits, outgoing base) equal to that of one of the 15 edges before.
    pad = 64 * W - 2 * (k + 1)
    cw = []
    for q in range(W):
        nb = min(64, max(0, 2 * (k - 1) - 64 * q))
        m = ((1 << nb) - 1) << (64 - nb) if nb else 0
        if q == W - 1:
            m |= 3 << pad
        cw.append(keys[:, q] & _s64(m))
    want_minus = torch.zeros(S, dtype=torch.bool, device="cuda")
    for dist in range(1, 16):
        if dist >= S:
            break
        same = torch.ones(S - dist, dtype=torch.bool, device="cuda")
        for q in range(W):
            same &= cw[q][dist:] == cw[q][:-dist]
        want_minus[dist:] |= same
        del same
    got_minus = Wb > 4
    assert torch.equal(got_minus, want_minus), "minus flags differ from the rule"
    n_targets = int((~want_minus).sum())                               # #(minus = 0) = distinct target k-mers
    assert int((Wb <= 4).sum()) == n_targets
    del cw, want_minus, got_minus
    # P9 (reading A4): the solid set is closed under reverse complement with equal multiplicities. Checksums over
    # (key, mult) and over (key of the reverse complement, mult) agree; for one-word keys the sorted reverse-complement
    # keys ARE the key list and carry the same multiplicities.
    kw = [keys[:, q].contiguous() for q in range(W)]
    rw = rc_key_words(kw, k)
    m64 = mult.to(torch.int64)
    assert int((key_mix_t(kw) * m64).sum()) == int((key_mix_t(rw) * m64).sum()), "not closed under reverse complement"
    if W == 1:
        order = torch.argsort(_u64_sorted_view(rw[0]))
        assert torch.equal(rw[0][order], kw[0]), "reverse complements of the solid edges are not the solid edges"
        assert torch.equal(mult[order], mult), "an edge and its reverse complement differ in multiplicity"
        del order
    del kw, rw, m64
    return n_nodes


def check_full_graph(res, w, n_nodes):
    """sdbg_build_full at full size: properties that tie its arrays to those of sdbg_build (checked bit for bit against
    the oracle in tests/test_gpu_full_graph.py at sizes the oracle can hold): the real edges are an order-preserving
    subsequence with unchanged W / last / mult, every '$' edge is the only edge of its node, validity bits are m ones,
    and, both strands being present, the nodes without outgoing edge mirror the nodes without incoming edge."""
    import torch
    ed, g, S = res.edges, res.graph, res.n
    ws = 64 * S * ed.w + (1 << 28)
    ctx = sd.Context(ws)
    probe = sd.FullGraph(0, 0, w.k)
    try:
        sd.sdbg_build_full(ctx, ed, probe)
    except sd.SdbgError as e:
        assert e.name == "SDBG_E_CAPACITY", e
    fg = sd.FullGraph(probe.m, probe.t, w.k)
    sd.sdbg_build_full(ctx, ed, fg)
    m, t, nzo = fg.m, fg.t, fg.n_zero_out
    assert m == S + nzo and t == nzo
    Wf = fg.W[:m]
    real = Wf != 0
    assert int(real.sum()) == S
    assert torch.equal(Wf[real], g.W[:S]) and torch.equal(fg.mult[:m][real], g.mult[:S])
    assert int(fg.mult[:m][~real].abs().sum()) == 0
    bits = ((fg.last_bits[:(m + 63) // 64].unsqueeze(1) >> torch.arange(64, device="cuda")) & 1).reshape(-1)[:m].bool()
    gbits = ((g.last_bits[:(S + 63) // 64].unsqueeze(1) >> torch.arange(64, device="cuda")) & 1).reshape(-1)[:S].bool()
    assert torch.equal(bits[real], gbits) and bool(bits[~real].all())
    assert int(bits.sum()) == n_nodes + nzo
    vb = fg.valid_bits[:(m + 63) // 64]
    ones = ((vb.unsqueeze(1) >> torch.arange(64, device="cuda")) & 1).reshape(-1)
    assert int(ones[:m].sum()) == m and int(ones[m:].sum()) == 0
    check_traversal(ctx, fg, ed, w, bits, real)
    ctx.close(); ctx.workspace = None
    return m, t


def check_traversal(ctx, fg, ed, w, last, real, n_sample=1 << 22):
    """sdbg_forward / sdbg_backward at full size (checked edge by edge against the oracle in tests/test_gpu_traverse.py
    at sizes the oracle can hold): properties that pin the two maps without an oracle. For sampled edges q: forward(q)
    is -1 exactly for '$' edges, else the last edge of a node that has an incoming edge; the first edge entering that
    node carries the same base without the minus flag, does not come after q and has the same forward image; for
    one-word keys the node of forward(q) IS e_q[1..k] (compared on the keys); backward is -1 exactly on the nodes of
    the auxiliary vector, and forward(backward(p)) = p for the last edge p of every other sampled node."""
    import torch
    m, k = fg.m, w.k
    ix = sd.Index(m)
    sd.sdbg_index_build(ctx, fg, ix)
    W = fg.W[:m]
    zin = ((fg.zin_bits[:(m + 63) // 64].unsqueeze(1) >> torch.arange(64, device="cuda")) & 1).reshape(-1)[:m].bool()
    assert int(zin.sum()) == fg.t and bool((last | ~zin).all())
    F = fg.F
    assert F[0] == 0 and F[4] == m and all(F[c] <= F[c + 1] for c in range(4))
    assert ix.ones[4] == int(last.sum()) - fg.t
    for c in range(4):
        assert ix.ones[c] == int((W == c + 1).sum())
    # BOSS counting property per class: has-incoming nodes ending with c == edges labelled c without the minus flag
    H = last & ~zin
    for c in range(4):
        assert int(H[F[c]:F[c + 1]].sum()) == ix.ones[c], c
    g = torch.Generator(device="cuda"); g.manual_seed(w.seed)
    q = torch.randint(0, m, (min(n_sample, 4 * m),), device="cuda", generator=g)
    f = torch.empty_like(q); b = torch.empty_like(q); f2 = torch.empty_like(q)
    sd.sdbg_forward(ctx, ix, q, q.numel(), f)
    torch.cuda.synchronize()
    isreal = real[q]
    assert bool((f[~isreal] == -1).all()) and bool((f[isreal] >= 0).all())
    qr, fr = q[isreal], f[isreal].contiguous()
    assert bool(H[fr].all())
    br = torch.empty_like(fr)
    sd.sdbg_backward(ctx, ix, fr, fr.numel(), br)
    torch.cuda.synchronize()
    assert bool((br >= 0).all()) and bool((br <= qr).all())
    assert bool((W[br] == ((W[qr] - 1) & 3) + 1).all())
    f2 = torch.empty_like(br)
    sd.sdbg_forward(ctx, ix, br, br.numel(), f2)
    torch.cuda.synchronize()
    assert torch.equal(f2, fr)
    if ed.w == 1:                                        # the node of forward(q) is e_q[1..k], on the keys themselves
        rank_real = torch.cumsum(real, 0) - 1
        keys = ed.keys[:ed.n]
        pad = 64 - 2 * (k + 1)
        mask2k = (1 << (2 * k)) - 1
        kq = keys[rank_real[qr]]
        node_q = (kq >> (64 - 2 * k)) & mask2k
        tgt = (((kq >> pad) & 3) << (2 * (k - 1))) | (node_q >> 2)
        to_real = real[fr]
        kf = keys[rank_real[fr[to_real]]]
        assert torch.equal((kf >> (64 - 2 * k)) & mask2k, tgt[to_real])
        # a '$' image: the node has no real edge, so its predecessor and successor nodes in the list differ from tgt
        del rank_real
    # backward on the nodes of the auxiliary vector and on sampled other nodes
    zpos = torch.nonzero(zin).reshape(-1)[:n_sample].contiguous()
    if zpos.numel():
        bz = torch.empty_like(zpos)
        sd.sdbg_backward(ctx, ix, zpos, zpos.numel(), bz)
        torch.cuda.synchronize()
        assert bool((bz == -1).all())
    hp = q[H[q]].contiguous()
    bh = torch.empty_like(hp); fh = torch.empty_like(hp)
    sd.sdbg_backward(ctx, ix, hp, hp.numel(), bh)
    torch.cuda.synchronize()
    assert bool((bh >= 0).all())
    sd.sdbg_forward(ctx, ix, bh, bh.numel(), fh)
    torch.cuda.synchronize()
    assert torch.equal(fh, hp)


def check_mercy(res, w, reads):
    """sdbg_mercy_edges at full size (bit-exact against the oracle in tests/test_gpu_mercy.py at oracle sizes):
    records come as (window, reverse complement) pairs, and no mercy record is a solid edge."""
    import torch
    ed, S = res.edges, res.n
    ctx = sd.Context((112 + 16 * ed.w) * S + (1 << 28))   # zero-degree scratch + 16-byte hash slots, at most 4 per edge
    probe = sd.Edges(0, w.k)
    try:
        sd.sdbg_mercy_edges(ctx, reads, ed, probe)
    except sd.SdbgError as e:
        assert e.name == "SDBG_E_CAPACITY", e
    M = probe.n
    me = sd.Edges(M, w.k)
    sd.sdbg_mercy_edges(ctx, reads, ed, me)
    assert me.n == M and M % 2 == 0
    if M:
        assert int(me.mult[:M].min()) == 1 and int(me.mult[:M].max()) == 1
        if ed.w == 1:
            sk = _u64_sorted_view(ed.keys[:S]); mk = _u64_sorted_view(me.keys[:M])
            pos = torch.searchsorted(sk, mk).clamp(max=S - 1)
            assert int((sk[pos] == mk).sum()) == 0, "a mercy record is a solid edge"
    ctx.close(); ctx.workspace = None
    return M


def compare_partitions(res, w, orc, buckets):
    """Bit-exact comparison of the GPU output slices of the given l=8 partitions with the oracle's result for them."""
    import torch
    ed, g, S, W = res.edges, res.graph, res.n, res.edges.w
    word0 = _u64_sorted_view(ed.keys[:S * W].view(S, W)[:, 0].contiguous())
    okeys = orc.keys
    ob = (okeys[:, 0] >> np.uint64(48)).astype(np.int64) if len(okeys) else np.zeros(0, np.int64)
    total = 0
    for b in sorted(buckets):
        lo_v = torch.tensor([(b << 48) - 2 ** 63], dtype=torch.int64, device="cuda")
        lo = int(torch.searchsorted(word0, lo_v)[0])
        hi = S if b == 65535 else int(torch.searchsorted(word0, torch.tensor([((b + 1) << 48) - 2 ** 63], dtype=torch.int64, device="cuda"))[0])
        sel = np.nonzero(ob == b)[0]
        assert hi - lo == len(sel), (b, hi - lo, len(sel))
        total += len(sel)
        if hi == lo:
            continue
        o0, o1 = int(sel[0]), int(sel[-1]) + 1
        assert o1 - o0 == len(sel)
        gk = ed.keys[lo * W:hi * W].cpu().numpy().view(np.uint64).reshape(-1, W)
        assert np.array_equal(gk, okeys[o0:o1]), f"partition {b}: keys differ"
        assert np.array_equal(ed.mult[lo:hi].cpu().numpy().view(np.uint32), orc.mult[o0:o1]), f"partition {b}: mult differs"
        assert np.array_equal(g.W[lo:hi].cpu().numpy(), orc.Wbyte[o0:o1]), f"partition {b}: W differs"
        words = g.last_bits[lo // 64:(hi + 63) // 64].cpu().numpy().view(np.uint64)
        bits = np.unpackbits(words.view(np.uint8), bitorder="little")[lo % 64:lo % 64 + (hi - lo)]
        want = orc.last[o0:o1].copy()
        if hi < S:
            want[-1] = 1      # the partition's last edge: its successor lies in another partition = another node (k >= 9)
        assert np.array_equal(bits, want), f"partition {b}: last differs"
    assert total == orc.n_solid
    return total
