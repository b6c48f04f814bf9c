"""CPU test of the fingerprint constants of common.cuh pair_key() (the one-word stand-in of a key of several words on the
table-count path, DESIGN.md §6 a4'). The form  sum_i  w_i * c_i + brev(w_i) * d_i  (mod 2^64, over the 32-bit halves w_i of
the key) is linear over Z / 2^64 in the halves and their bit reversals, so changing a set of key symbols changes it by ONE
amount whatever the two keys are. Two keys share a fingerprint only if that amount lies within 2^top_bits of zero (the
fingerprint is the form shifted right by top_bits <= 32; 24 on config 4). Sequencing reads are full of keys that differ in
one, two or three symbols (copies of an edge with errors), so none of those patterns may come that close: all of them are
enumerated here, for the constants parsed out of the header. (Patterns of four and more symbols behave like random
numbers: a meeting there is caught by the check in hashcount.cu and costs a slower run, never a wrong result.)"""
import os
import re

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
M = 1 << 64


def _constants():
    src = open(os.path.join(ROOT, "paper_1409_7208_b200", "csrc", "common.cuh")).read()
    body = src[src.index("pair_key(const u64"):]
    out = []
    for name in ("c", "d"):
        m = re.search(r"constexpr u32 %s\[8\] = \{([^}]*)\}" % name, body)
        out.append([int(x.strip().rstrip("u"), 16) for x in m.group(1).split(",")])
        assert len(out[-1]) == 8 and all(v & 1 for v in out[-1]) and len(set(out[-1])) == 8
    return out


def _single_changes(c, d):
    """the change of the form for every (half, symbol place, old symbol, new symbol); 12 per place, place = index // 12"""
    swap = lambda x: ((x & 1) << 1) | (x >> 1)           # a symbol's two bits as they stand in the reversed word
    out = []
    for h in range(8):
        for j in range(16):
            for s in range(4):
                for t in range(4):
                    if s != t:
                        out.append(((t - s) * 4 ** j * c[h] + (swap(t) - swap(s)) * (1 << (30 - 2 * j)) * d[h]) % M)
    return np.array(out, dtype=np.uint64)


def _near_zero(x, bits):
    return (x < np.uint64(1 << bits)) | (x > np.uint64(M - (1 << bits)))


def test_no_pattern_of_up_to_three_changed_symbols_cancels():
    c, d = _constants()
    one = _single_changes(c, d)
    n = len(one)
    assert n == 8 * 16 * 12
    bits = 30                                            # far above the 2^24 that matters on config 4
    assert not _near_zero(one, bits).any()
    place = np.arange(n) // 12
    two = (one[:, None] + one[None, :])[np.triu(place[:, None] != place[None, :], 1)]    # two different places
    assert not _near_zero(two, bits).any()
    two.sort()
    hits = 0                                             # three places: a pair within 2^bits of minus a single change
    for k in range(n):                                   # (a triple that repeats a place is a pair or a single change again)
        t = (-int(one[k])) % M
        lo, hi = (t - (1 << bits)) % M, (t + (1 << bits)) % M
        a, b = np.searchsorted(two, np.uint64(lo)), np.searchsorted(two, np.uint64(hi))
        hits += (b - a) if lo < hi else (len(two) - a) + b
    assert hits == 0


def test_the_form_is_what_the_header_computes():
    """pair_key restated on integers for random keys and changes: the difference of two keys' forms is the sum of the
    single changes of the symbols in which they differ (what the enumeration above relies on)."""
    c, d = _constants()
    rng = np.random.default_rng(5)

    def brev(x):
        return int("{:032b}".format(x)[::-1], 2)

    def form(halves):
        return sum(w * c[i] + brev(w) * d[i] for i, w in enumerate(halves)) % M

    one = _single_changes(c, d)
    for _ in range(200):
        halves = [int(x) for x in rng.integers(0, 1 << 32, size=8)]
        other = list(halves)
        want = 0
        for h, j in {(int(rng.integers(0, 8)), int(rng.integers(0, 16))) for _ in range(3)}:
            s = (halves[h] >> (2 * j)) & 3
            t = (s + 1 + int(rng.integers(0, 3))) & 3
            other[h] = (other[h] & ~(3 << (2 * j))) | (t << (2 * j))
            idx = ((h * 16 + j) * 4 + s) * 3 + (t if t < s else t - 1)
            want = (want + int(one[idx])) % M
        assert (form(other) - form(halves)) % M == want
