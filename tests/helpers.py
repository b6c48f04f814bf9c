"""Independent test-side restatements (brute force, de Bruijn sequences, checksum definition).
These share no code with oracle/ or the CUDA library; they exist to pin both."""
import numpy as np

CODE = {"A": 0, "C": 1, "G": 2, "T": 3}
COMP = {"A": "T", "C": "G", "G": "C", "T": "A"}


def rc(s):
    return "".join(COMP[c] for c in reversed(s))


def brute_force(reads, k, d):
    """Dict count + sorted() with the colex key + literal O(S^2) minus scan (pin P2)."""
    cnt = {}
    n = 0
    for r in reads:
        r = r.upper()
        for i in range(len(r) - k):
            e = r[i:i + k + 1]
            for x in (e, rc(e)):
                cnt[x] = cnt.get(x, 0) + 1
                n += 1
    distinct = sorted(cnt, key=lambda e: (e[:k][::-1], e[k]))
    S = [e for e in distinct if cnt[e] >= d]
    W = [e[k] for e in S]
    last = [1 if (i == len(S) - 1 or S[i + 1][:k] != S[i][:k]) else 0 for i in range(len(S))]
    minus = [1 if any(S[j][1:k] == S[i][1:k] and S[j][k] == S[i][k] for j in range(i)) else 0 for i in range(len(S))]
    return dict(n_raw=n, distinct=distinct, cnt=[cnt[e] for e in distinct], solid=S, mult=[cnt[e] for e in S],
                W=W, last=last, minus=minus)


def key_words(e, k):
    """Step-6 key of edge string e as a list of w python ints."""
    w = (2 * (k + 1) + 63) // 64
    sym = e[:k][::-1] + e[k]
    v = 0
    for c in sym:
        v = (v << 2) | CODE[c]
    v <<= 64 * w - 2 * (k + 1)
    return [(v >> (64 * (w - 1 - j))) & (2 ** 64 - 1) for j in range(w)]


def de_bruijn(alphabet, n):
    """Linearised de Bruijn sequence B(|alphabet|, n) by the Lyndon-word (FKM) construction, plus the
    n-1 wrap-around symbols, so that every n-mer occurs exactly once."""
    q = len(alphabet)
    a = [0] * (q * n)
    seq = []

    def db(t, p):
        if t > n:
            if n % p == 0:
                seq.extend(a[1:p + 1])
        else:
            a[t] = a[t - p]
            db(t + 1, p)
            for j in range(a[t - p] + 1, q):
                a[t] = j
                db(t + 1, t)

    db(1, 1)
    s = "".join(alphabet[i] for i in seq)
    return s + s[:n - 1]


_M1 = 0xBF58476D1CE4E5B9
_M2 = 0x94D049BB133111EB
_MASK = 2 ** 64 - 1


def mix64(z):
    z &= _MASK
    z = ((z ^ (z >> 30)) * _M1) & _MASK
    z = ((z ^ (z >> 27)) * _M2) & _MASK
    return z ^ (z >> 31)


def key_mix(words):
    """include/sdbg.h 'checksum of a key': h = 0; for each word, most significant first: h = mix64(h ^ word)."""
    h = 0
    for x in words:
        h = mix64(h ^ int(x))
    return h


def key_mix_np(keys):
    """vectorised key_mix over an (n, w) uint64 array."""
    keys = np.ascontiguousarray(keys, dtype=np.uint64)
    keys = keys.reshape(len(keys), keys.shape[1] if keys.ndim == 2 else 1)
    h = np.zeros(len(keys), dtype=np.uint64)
    with np.errstate(over="ignore"):
        for j in range(keys.shape[1]):
            z = h ^ keys[:, j]
            z = (z ^ (z >> np.uint64(30))) * np.uint64(_M1)
            z = (z ^ (z >> np.uint64(27))) * np.uint64(_M2)
            h = z ^ (z >> np.uint64(31))
    return h


def brute_force_full(reads, k, d):
    """The lossless extras of PAPER.md:31 (readings A18-A20) from brute_force(): sets and sorted() only."""
    b = brute_force(reads, k, d)
    S = b["solid"]
    src, tgt = {e[:k] for e in S}, {e[1:] for e in S}
    order = {"$": 0, "A": 1, "C": 2, "G": 3, "T": 4}
    zout = sorted(tgt - src, key=lambda v: v[::-1])
    zin = sorted(src - tgt, key=lambda v: v[::-1])
    F = sorted(S + [v + "$" for v in zout], key=lambda e: (e[:k][::-1], order[e[k]]))
    mult = dict(zip(S, b["mult"]))
    W, last, M = [], [], []
    for i, e in enumerate(F):
        last.append(1 if (i == len(F) - 1 or F[i + 1][:k] != e[:k]) else 0)
        minus = e[k] != "$" and any(F[j][1:k] == e[1:k] and F[j][k] == e[k] for j in range(i))
        W.append(0 if e[k] == "$" else order[e[k]] + (4 if minus else 0))
        M.append(mult.get(e, 0))
    return dict(F=F, W=W, last=last, mult=M, aux=zin, zout=zout)


def brute_force_mercy(reads, k, d):
    """Mercy-kmers of PAPER.md:35 (readings A21-A23) from brute_force(): sets and plain loops."""
    b = brute_force(reads, k, d)
    S = set(b["solid"])
    src, tgt = {e[:k] for e in S}, {e[1:] for e in S}
    no_out, no_in = tgt - src, src - tgt
    out = []
    for r in reads:
        r = r.upper()
        w = [r[i:i + k + 1] for i in range(len(r) - k)]
        i = 0
        while i < len(w):
            if w[i] in S:
                i += 1
                continue
            j = i
            while j + 1 < len(w) and w[j + 1] not in S:
                j += 1
            if i >= 1 and j + 1 < len(w) and w[i - 1][1:] in no_out and w[j + 1][:k] in no_in:
                for e in w[i:j + 1]:
                    out += [e, rc(e)]
            i = j + 1
    return out


def brute_force_navigation(F, aux, k):
    """forward / backward / zin / F-array of the full edge list F (strings, '$' for dummies) by loops over strings
    (readings A24-A26): nothing but comparisons of node strings."""
    m = len(F)
    zin = [1 if (F[i][:k] in set(aux) and (i == m - 1 or F[i + 1][:k] != F[i][:k])) else 0 for i in range(m)]
    Farr = [min([i for i in range(m) if F[i][k - 1] >= c], default=m) for c in "ACGT"] + [m]
    fwd, bwd = [], []
    for i in range(m):
        if F[i][k] == "$":
            fwd.append(-1)
        else:
            fwd.append(max(j for j in range(m) if F[j][:k] == F[i][1:]))
        inc = [j for j in range(m) if F[j][k] != "$" and F[j][1:] == F[i][:k]]
        bwd.append(min(inc) if inc else -1)
    return dict(zin=zin, F=Farr, forward=fwd, backward=bwd)


def boss_navigation(W, last, zin, Farr):
    """The same two maps from the succinct arrays alone, by the rank/select formulas of Bowe et al.
    adapted to the graph without incoming dummy edges (reading A26), with counting loops for rank and select:
      H[i] = last[i] and not zin[i]                 (last edge of a node that has an incoming edge)
      B_c[i] = (W[i] == c, minus flag clear)
      forward(i)  = select_H(rank_H(F[c]) + rank_{B_c}(i + 1)),   c = base of W[i]
      backward(j) = select_{B_c}(rank_H(p + 1) - rank_H(F[c])),   p = last edge of the node of j, c = its class in F."""
    m = len(W)
    H = [1 if (last[i] and not zin[i]) else 0 for i in range(m)]

    def rank(bits, x):
        return sum(bits[:x])

    def select(bits, r):
        seen = 0
        for i, b in enumerate(bits):
            seen += b
            if b and seen == r:
                return i
        raise AssertionError("select out of range")

    B = [[1 if W[i] == c + 1 else 0 for i in range(m)] for c in range(4)]
    fwd, bwd = [], []
    for i in range(m):
        if W[i] == 0:
            fwd.append(-1)
        else:
            c = (W[i] - 1) & 3
            fwd.append(select(H, rank(H, Farr[c]) + rank(B[c], i + 1)))
        p = i
        while not last[p]:
            p += 1
        if not H[p]:
            bwd.append(-1)
        else:
            c = max(c for c in range(4) if Farr[c] <= p)
            bwd.append(select(B[c], rank(H, p + 1) - rank(H, Farr[c])))
    return dict(forward=fwd, backward=bwd)
