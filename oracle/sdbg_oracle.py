"""ctypes front-end of oracle/sdbg_oracle.c (the plain CPU definition; see that file's header for the
step-by-step citation of PAPER.md). TEST INFRASTRUCTURE ONLY — never imported by the product path."""
from __future__ import annotations

import ctypes
import os
import subprocess
from dataclasses import dataclass

import numpy as np

_DIR = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_DIR, "sdbg_oracle.c")
_SO = os.path.join(_DIR, "libsdbg_oracle.so")
_lib = None


def build_oracle_lib(force: bool = False) -> str:
    if force or not os.path.exists(_SO) or os.path.getmtime(_SRC) > os.path.getmtime(_SO):
        subprocess.check_call(["gcc", "-O2", "-std=c11", "-shared", "-fPIC", "-o", _SO, _SRC])
    return _SO


def _load():
    global _lib
    if _lib is None:
        L = ctypes.CDLL(build_oracle_lib())
        vp, u64, u32 = ctypes.c_void_p, ctypes.c_uint64, ctypes.c_uint32
        L.orc_new.argtypes = [u32, u32, ctypes.c_char_p, u32]; L.orc_new.restype = vp
        L.orc_add_edges.argtypes = [vp, vp, u64]; L.orc_add_edges.restype = ctypes.c_int
        L.orc_raw.argtypes = [vp]; L.orc_raw.restype = vp
        L.orc_free.argtypes = [vp]; L.orc_free.restype = None
        L.orc_add_reads.argtypes = [vp, vp, vp, u64]; L.orc_add_reads.restype = ctypes.c_int
        L.orc_finish.argtypes = [vp]; L.orc_finish.restype = ctypes.c_int
        for f in ("n_raw", "n_seen", "n_distinct", "n_solid", "sum_solid_mult"):
            getattr(L, "orc_" + f).argtypes = [vp]; getattr(L, "orc_" + f).restype = u64
        for f in ("sorted_raw", "distinct", "distinct_cnt", "solid", "mult", "W", "last", "minus"):
            getattr(L, "orc_" + f).argtypes = [vp]; getattr(L, "orc_" + f).restype = vp
        L.orc_encode_keys.argtypes = [vp, vp, u64, vp]; L.orc_encode_keys.restype = None
        L.orc_encode_graph.argtypes = [vp, vp, vp]; L.orc_encode_graph.restype = None
        L.orc_full_graph.argtypes = [vp]; L.orc_full_graph.restype = vp
        L.orc_full_free.argtypes = [vp]; L.orc_full_free.restype = None
        for f in ("m", "t", "n_zero_out"):
            getattr(L, "orc_full_" + f).argtypes = [vp]; getattr(L, "orc_full_" + f).restype = u64
        for f in ("edges", "W", "last", "mult", "aux"):
            getattr(L, "orc_full_" + f).argtypes = [vp]; getattr(L, "orc_full_" + f).restype = vp
        L.orc_mercy_scan.argtypes = [vp, vp, vp, u64]; L.orc_mercy_scan.restype = vp
        L.orc_mercy_n.argtypes = [vp]; L.orc_mercy_n.restype = u64
        L.orc_mercy_edges.argtypes = [vp]; L.orc_mercy_edges.restype = vp
        L.orc_mercy_free.argtypes = [vp]; L.orc_mercy_free.restype = None
        _lib = L
    return _lib


def _copy(ptr, n, dtype):
    if n == 0 or not ptr:
        return np.zeros(0, dtype=dtype)
    nbytes = n * np.dtype(dtype).itemsize
    return np.frombuffer(ctypes.string_at(ptr, nbytes), dtype=dtype).copy()


@dataclass
class OracleResult:
    k: int
    d: int
    n_raw: int             # records kept in step 1 (after the optional partition restriction)
    n_seen: int            # records of step 1 before that restriction (= N = 2*sum max(0, L_r-k))
    n_distinct: int
    n_solid: int
    sum_solid_mult: int
    distinct: np.ndarray       # (n_distinct, k+1) uint8 letters, sorted
    distinct_cnt: np.ndarray   # u32
    solid: np.ndarray          # (n_solid, k+1) uint8 letters, sorted
    mult: np.ndarray           # u32
    W: np.ndarray              # uint8 letters
    last: np.ndarray           # uint8 0/1
    minus: np.ndarray          # uint8 0/1
    # step-6 encodings
    keys: np.ndarray           # u64 (n_solid, w)
    distinct_keys: np.ndarray  # u64 (n_distinct, w)
    Wbyte: np.ndarray          # u8
    last_bits: np.ndarray      # u64 ceil(n_solid/64)

    @property
    def w(self) -> int:
        return (2 * (self.k + 1) + 63) // 64

    def solid_strings(self):
        return [bytes(r).decode() for r in self.solid]

    def distinct_strings(self):
        return [bytes(r).decode() for r in self.distinct]


class Oracle:
    """Steps 1-6 of sdbg_oracle.c. ``prefix``: optional 8-letter key-string prefix (one l=8 partition) or a list
    of them."""

    def __init__(self, k: int, d: int = 2, prefix=None):
        L = _load()
        self.k, self.d = int(k), int(d)
        plist = [prefix] if isinstance(prefix, str) else list(prefix or [])
        assert all(len(p) == 8 for p in plist)
        self._h = L.orc_new(self.k, self.d, "".join(plist).encode() if plist else None, len(plist))
        if not self._h:
            raise ValueError("oracle: invalid k/d/prefix")

    def add_reads(self, bases, offsets) -> None:
        """bases: bytes / uint8 array of the concatenated reads; offsets: n+1 uint64 starts."""
        b = np.frombuffer(bases, dtype=np.uint8) if isinstance(bases, (bytes, bytearray)) else np.ascontiguousarray(bases, dtype=np.uint8)
        o = np.ascontiguousarray(offsets, dtype=np.uint64)
        rc = _load().orc_add_reads(self._h, b.ctypes.data if b.size else None, o.ctypes.data, len(o) - 1)
        if rc == -2:
            raise ValueError("oracle: non-ACGT base")
        if rc != 0:
            raise MemoryError(f"oracle: error {rc}")

    def add_edges(self, edges: np.ndarray) -> None:
        """edges: (n, k+1) uint8 letters extracted earlier (see sdbg_oracle.c header)."""
        e = np.ascontiguousarray(edges, dtype=np.uint8).reshape(-1, self.k + 1)
        rc = _load().orc_add_edges(self._h, e.ctypes.data if e.size else None, len(e))
        if rc != 0:
            raise MemoryError(f"oracle: error {rc}")

    def raw_edges(self) -> np.ndarray:
        """The records step 1 has kept so far, (n, k+1) uint8 letters (call before finish)."""
        L = _load()
        return _copy(L.orc_raw(self._h), L.orc_n_raw(self._h) * (self.k + 1), np.uint8).reshape(-1, self.k + 1)

    def finish(self, want_distinct: bool = True) -> OracleResult:
        L = _load()
        rc = L.orc_finish(self._h)
        if rc != 0:
            raise MemoryError(f"oracle: error {rc}")
        h, k = self._h, self.k
        R, w = k + 1, (2 * (k + 1) + 63) // 64
        nd, ns = L.orc_n_distinct(h), L.orc_n_solid(h)
        keys = np.zeros(ns * w, dtype=np.uint64)
        L.orc_encode_keys(h, L.orc_solid(h), ns, keys.ctypes.data)
        dkeys = np.zeros(nd * w if want_distinct else 0, dtype=np.uint64)
        if want_distinct:
            L.orc_encode_keys(h, L.orc_distinct(h), nd, dkeys.ctypes.data)
        Wb = np.zeros(ns, dtype=np.uint8)
        lb = np.zeros((ns + 63) // 64, dtype=np.uint64)
        L.orc_encode_graph(h, Wb.ctypes.data, lb.ctypes.data)
        return OracleResult(
            k=k, d=self.d, n_raw=L.orc_n_raw(h), n_seen=L.orc_n_seen(h), n_distinct=nd, n_solid=ns,
            sum_solid_mult=L.orc_sum_solid_mult(h),
            distinct=_copy(L.orc_distinct(h), nd * R if want_distinct else 0, np.uint8).reshape(-1, R),
            distinct_cnt=_copy(L.orc_distinct_cnt(h), nd, np.uint32),
            solid=_copy(L.orc_solid(h), ns * R, np.uint8).reshape(-1, R),
            mult=_copy(L.orc_mult(h), ns, np.uint32), W=_copy(L.orc_W(h), ns, np.uint8),
            last=_copy(L.orc_last(h), ns, np.uint8), minus=_copy(L.orc_minus(h), ns, np.uint8),
            keys=keys.reshape(-1, w), distinct_keys=dkeys.reshape(-1, w), Wbyte=Wb, last_bits=lb)

    def full_graph(self) -> dict:
        """The lossless extras of PAPER.md:31 over the solid edges (call after finish): see sdbg_oracle.c.
        Returns m, t, n_zero_out, edges (m, k+1) letters with '$', W bytes, last 0/1, mult, aux (t, k) letters, and the
        encodings compared with the CUDA library: last_bits (LSB first), valid_bits (all ones), aux_bits (2 bits per
        base A0 C1 G2 T3, node i at stream bits [2k i, 2k (i+1)), stream bit 0 = most significant bit of word 0)."""
        L = _load()
        f = L.orc_full_graph(self._h)
        if not f:
            raise MemoryError("oracle: full graph")
        try:
            k, m, t = self.k, L.orc_full_m(f), L.orc_full_t(f)
            out = dict(m=m, t=t, n_zero_out=L.orc_full_n_zero_out(f),
                       edges=_copy(L.orc_full_edges(f), m * (k + 1), np.uint8).reshape(-1, k + 1),
                       W=_copy(L.orc_full_W(f), m, np.uint8), last=_copy(L.orc_full_last(f), m, np.uint8),
                       mult=_copy(L.orc_full_mult(f), m, np.uint32), aux=_copy(L.orc_full_aux(f), t * k, np.uint8).reshape(-1, k))
        finally:
            L.orc_full_free(f)
        lb = np.zeros((m + 63) // 64, dtype=np.uint64)
        vb = np.zeros((m + 63) // 64, dtype=np.uint64)
        for i in range(m):       # plain loops: this is the definition of the packing
            if out["last"][i]:
                lb[i // 64] |= np.uint64(1) << np.uint64(i % 64)
            vb[i // 64] |= np.uint64(1) << np.uint64(i % 64)
        code = {65: 0, 67: 1, 71: 2, 84: 3}
        ab = np.zeros((2 * k * t + 63) // 64, dtype=np.uint64)
        pos = 0
        for row in out["aux"]:
            for ch in row:
                ab[pos // 64] |= np.uint64(code[int(ch)]) << np.uint64(62 - pos % 64)
                pos += 2
        out.update(last_bits=lb, valid_bits=vb, aux_bits=ab)
        return out

    def mercy(self, bases, offsets):
        """Mercy-kmers of PAPER.md:35 (call after finish, with the reads again): dict with `edges` (n, k+1) letters in
        the order met (a multiset holding both strands) and `keys` (n, w) their step-6 keys."""
        L = _load()
        b = np.frombuffer(bases, dtype=np.uint8) if isinstance(bases, (bytes, bytearray)) else np.ascontiguousarray(bases, dtype=np.uint8)
        o = np.ascontiguousarray(offsets, dtype=np.uint64)
        m = L.orc_mercy_scan(self._h, b.ctypes.data if b.size else None, o.ctypes.data, len(o) - 1)
        if not m:
            raise MemoryError("oracle: mercy scan")
        try:
            n, k = L.orc_mercy_n(m), self.k
            w = (2 * (k + 1) + 63) // 64
            edges = _copy(L.orc_mercy_edges(m), n * (k + 1), np.uint8).reshape(-1, k + 1)
            keys = np.zeros(n * w, dtype=np.uint64)
            if n:
                L.orc_encode_keys(self._h, edges.ctypes.data, n, keys.ctypes.data)
        finally:
            L.orc_mercy_free(m)
        return dict(edges=edges, keys=keys.reshape(-1, w))

    def close(self):
        if self._h:
            _load().orc_free(self._h)
            self._h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass


def reads_to_arrays(reads):
    """list of str -> (uint8 bases, uint64 offsets) — plain concatenation."""
    offs = np.zeros(len(reads) + 1, dtype=np.uint64)
    for i, r in enumerate(reads):
        offs[i + 1] = offs[i] + np.uint64(len(r))
    return np.frombuffer("".join(reads).encode(), dtype=np.uint8), offs


def run_oracle(reads, k: int, d: int = 2, prefix=None) -> OracleResult:
    """reads: list of str, or a (bases, offsets) pair."""
    o = Oracle(k, d, prefix)
    try:
        if isinstance(reads, tuple):
            o.add_reads(*reads)
        else:
            o.add_reads(*reads_to_arrays(list(reads)))
        return o.finish()
    finally:
        o.close()
