"""ctypes binding of include/sdbg.h — same names, argument marshalling only.

PyTorch appears here for device memory and streams (plumbing): every buffer is a torch CUDA tensor owned by the
Python side, and the library receives raw device pointers. The product path fails loudly when ``csrc/libsdbg.so``
is missing or when there is no CUDA device; nothing here computes any step of the method on the host.
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

_DIR = os.path.dirname(os.path.abspath(__file__))
_LIB_PATH = os.path.join(_DIR, "csrc", "libsdbg.so")
_lib = None

SDBG_SORTED = 1
SDBG_NUM_BUCKETS = 65536
STATUS = {0: "SDBG_OK", -1: "SDBG_E_INVAL", -2: "SDBG_E_BADBASE", -3: "SDBG_E_CAPACITY", -4: "SDBG_E_WORKSPACE",
          -5: "SDBG_E_CUDA", -6: "SDBG_E_UNSUPPORTED"}
SDBG_OPT_FORCE_WIDE, SDBG_OPT_NO_TABLE_COUNT, SDBG_OPT_STABLE_FIRST_PASS, SDBG_OPT_NO_FUSED_EXTRACT, SDBG_OPT_WEAK_FINGERPRINT = 1, 2, 3, 4, 5
T_CLASSES = ("pack", "extract", "radix", "count", "emit", "other", "table")


class SdbgError(RuntimeError):
    def __init__(self, status: int, detail: str = ""):
        self.status = status
        self.name = STATUS.get(status, str(status))
        super().__init__(f"{self.name}: {detail}")


class _Reads(C.Structure):
    _fields_ = [("words", C.c_void_p), ("ends", C.c_void_p), ("slots_cap", C.c_uint64), ("n_reads", C.c_uint64),
                ("n_bases", C.c_uint64), ("n_slots", C.c_uint64)]


class _Edges(C.Structure):
    _fields_ = [("keys", C.c_void_p), ("mult", C.c_void_p), ("cap", C.c_uint64), ("n", C.c_uint64),
                ("k", C.c_uint32), ("w", C.c_uint32)]


class _Stats(C.Structure):
    _fields_ = [("n_raw", C.c_uint64), ("n_distinct", C.c_uint64), ("n_solid", C.c_uint64),
                ("sum_solid_mult", C.c_uint64), ("n_ranges", C.c_uint64), ("max_range_records", C.c_uint64),
                ("csum_raw", C.c_uint64), ("csum_distinct", C.c_uint64), ("want_checksums", C.c_uint32),
                ("reserved", C.c_uint32), ("bucket_hist", C.c_void_p)]


class _Graph(C.Structure):
    _fields_ = [("W", C.c_void_p), ("last_bits", C.c_void_p), ("mult", C.c_void_p), ("cap", C.c_uint64), ("n", C.c_uint64)]


class _FullGraph(C.Structure):
    _fields_ = [("W", C.c_void_p), ("last_bits", C.c_void_p), ("valid_bits", C.c_void_p), ("mult", C.c_void_p),
                ("aux_bits", C.c_void_p), ("cap", C.c_uint64), ("aux_cap", C.c_uint64), ("m", C.c_uint64),
                ("t", C.c_uint64), ("n_zero_out", C.c_uint64), ("zin_bits", C.c_void_p), ("F", C.c_uint64 * 5)]


class _Index(C.Structure):
    _fields_ = [("cells", C.c_void_p), ("bytes", C.c_uint64), ("m", C.c_uint64), ("n_cells", C.c_uint64),
                ("F", C.c_uint64 * 5), ("HF", C.c_uint64 * 5), ("ones", C.c_uint64 * 5), ("W", C.c_void_p),
                ("last_bits", C.c_void_p)]


class _Timing(C.Structure):
    _fields_ = [("ms", C.c_double * 7), ("launches", C.c_uint64 * 7), ("bytes", C.c_uint64 * 7)]


def lib_path() -> str:
    return _LIB_PATH


def lib():
    """Loads csrc/libsdbg.so (built by paper_1409_7208_b200.build / __graft_entry__.build). No fallback."""
    global _lib
    if _lib is None:
        if not os.path.exists(_LIB_PATH):
            raise RuntimeError(f"{_LIB_PATH} is missing: run `python -m paper_1409_7208_b200.build` "
                               "(or __graft_entry__.build()); there is no CPU fallback")
        L = C.CDLL(_LIB_PATH)
        vp, u64, u32, i32 = C.c_void_p, C.c_uint64, C.c_uint32, C.c_int
        L.sdbg_ctx_create.argtypes = [C.POINTER(vp), i32, vp, vp, u64]; L.sdbg_ctx_create.restype = i32
        L.sdbg_ctx_destroy.argtypes = [vp]; L.sdbg_ctx_destroy.restype = None
        L.sdbg_ctx_set_option.argtypes = [vp, i32, i32]; L.sdbg_ctx_set_option.restype = i32
        L.sdbg_unstable_radix_launches.argtypes = []; L.sdbg_unstable_radix_launches.restype = u64
        L.sdbg_strerror.argtypes = [i32]; L.sdbg_strerror.restype = C.c_char_p
        L.sdbg_last_error.argtypes = [vp]; L.sdbg_last_error.restype = C.c_char_p
        L.sdbg_read_slots.argtypes = [u64, u64]; L.sdbg_read_slots.restype = u64
        L.sdbg_pack_reads.argtypes = [vp, vp, vp, u64, C.POINTER(_Reads)]; L.sdbg_pack_reads.restype = i32
        L.sdbg_key_words.argtypes = [u32]; L.sdbg_key_words.restype = u32
        L.sdbg_full_workspace.argtypes = [u64, u32]; L.sdbg_full_workspace.restype = u64
        L.sdbg_min_workspace.argtypes = []; L.sdbg_min_workspace.restype = u64
        L.sdbg_workspace_for_records.argtypes = [u64, u32]; L.sdbg_workspace_for_records.restype = u64
        L.sdbg_count_edges.argtypes = [vp, C.POINTER(_Reads), u64, u32, u32, C.POINTER(_Edges), C.POINTER(_Stats)]
        L.sdbg_count_edges.restype = i32
        L.sdbg_count_edges_range.argtypes = [vp, C.POINTER(_Reads), u64, u32, u32, u32, u32, C.POINTER(_Edges), C.POINTER(_Stats)]
        L.sdbg_count_edges_range.restype = i32
        L.sdbg_bucket_hist.argtypes = [vp, C.POINTER(_Reads), u32, vp]; L.sdbg_bucket_hist.restype = i32
        L.sdbg_plan_shards.argtypes = [vp, u32, vp]; L.sdbg_plan_shards.restype = i32
        L.sdbg_plan_ranges.argtypes = [vp, u64, vp, u64]; L.sdbg_plan_ranges.restype = C.c_int64
        L.sdbg_build.argtypes = [vp, C.POINTER(_Edges), u32, C.POINTER(_Graph)]; L.sdbg_build.restype = i32
        L.sdbg_build_full.argtypes = [vp, C.POINTER(_Edges), C.POINTER(_FullGraph)]; L.sdbg_build_full.restype = i32
        L.sdbg_mercy_edges.argtypes = [vp, C.POINTER(_Reads), C.POINTER(_Edges), C.POINTER(_Edges)]; L.sdbg_mercy_edges.restype = i32
        L.sdbg_index_bytes.argtypes = [u64]; L.sdbg_index_bytes.restype = u64
        L.sdbg_index_build.argtypes = [vp, C.POINTER(_FullGraph), C.POINTER(_Index)]; L.sdbg_index_build.restype = i32
        L.sdbg_index_static_max_edges.argtypes = []; L.sdbg_index_static_max_edges.restype = u64
        L.sdbg_index_static_bytes.argtypes = [u64]; L.sdbg_index_static_bytes.restype = u64
        L.sdbg_index_build_static.argtypes = [vp, C.POINTER(_FullGraph), C.POINTER(_Index)]; L.sdbg_index_build_static.restype = i32
        L.sdbg_index_build_static_error.argtypes = []; L.sdbg_index_build_static_error.restype = C.c_char_p
        L.sdbg_forward.argtypes = [vp, C.POINTER(_Index), vp, u64, vp]; L.sdbg_forward.restype = i32
        L.sdbg_backward.argtypes = [vp, C.POINTER(_Index), vp, u64, vp]; L.sdbg_backward.restype = i32
        L.sdbg_ctx_set_timing.argtypes = [vp, i32]; L.sdbg_ctx_set_timing.restype = i32
        L.sdbg_ctx_get_timing.argtypes = [vp, C.POINTER(_Timing)]; L.sdbg_ctx_get_timing.restype = i32
        _lib = L
    return _lib


# ---- host-only helpers (no GPU needed) -----------------------------------------------------------------------------

def sdbg_unstable_radix_launches() -> int:
    return int(lib().sdbg_unstable_radix_launches())


def sdbg_strerror(status: int) -> str:
    return lib().sdbg_strerror(status).decode()


def sdbg_key_words(k: int) -> int:
    return lib().sdbg_key_words(k)


def sdbg_read_slots(n_bases: int, n_calls: int = 1) -> int:
    return lib().sdbg_read_slots(n_bases, n_calls)


def sdbg_full_workspace(n_bases: int, k: int) -> int:
    return lib().sdbg_full_workspace(n_bases, k)


def sdbg_workspace_for_records(n_records: int, k: int) -> int:
    return lib().sdbg_workspace_for_records(n_records, k)


def sdbg_min_workspace() -> int:
    return lib().sdbg_min_workspace()


def sdbg_plan_ranges(hist, capacity: int):
    """hist: 65536 counts (host). Returns a list of (lo, hi, records); raises SdbgError(SDBG_E_WORKSPACE)."""
    h = np.ascontiguousarray(hist, dtype=np.uint64)
    assert h.size == SDBG_NUM_BUCKETS
    out = np.zeros(3 * SDBG_NUM_BUCKETS, dtype=np.uint64)
    n = lib().sdbg_plan_ranges(h.ctypes.data, capacity, out.ctypes.data, SDBG_NUM_BUCKETS)
    if n < 0:
        raise SdbgError(int(n), "one l=8 partition exceeds the capacity")
    return [tuple(int(x) for x in out[3 * i:3 * i + 3]) for i in range(n)]


# ---- device objects ------------------------------------------------------------------------------------------------

def _torch():
    import torch
    if not torch.cuda.is_available():
        raise RuntimeError("libsdbg needs a CUDA device (sm_100a); there is no CPU fallback")
    return torch


class Context:
    """sdbg_ctx bound to the current torch CUDA device and stream, with a torch-owned workspace."""

    def __init__(self, workspace_bytes: int, device: int | None = None):
        torch = _torch()
        self.device = torch.cuda.current_device() if device is None else device
        workspace_bytes = max(int(workspace_bytes), sdbg_min_workspace())
        self.workspace = torch.empty(workspace_bytes, dtype=torch.uint8, device=f"cuda:{self.device}")
        self.stream = torch.cuda.current_stream(self.device)
        h = C.c_void_p()
        rc = lib().sdbg_ctx_create(C.byref(h), self.device, self.stream.cuda_stream, self.workspace.data_ptr(), workspace_bytes)
        if rc != 0:
            raise SdbgError(rc, sdbg_strerror(rc))
        self._h = h

    def check(self, rc: int):
        if rc != 0:
            raise SdbgError(rc, lib().sdbg_last_error(self._h).decode() or sdbg_strerror(rc))

    def set_option(self, option: int, value: int = 1):
        self.check(lib().sdbg_ctx_set_option(self._h, int(option), int(value)))

    def set_timing(self, on: bool):
        self.check(lib().sdbg_ctx_set_timing(self._h, 1 if on else 0))

    def get_timing(self) -> "Timing":
        t = _Timing()
        self.check(lib().sdbg_ctx_get_timing(self._h, C.byref(t)))
        return Timing({c: t.ms[i] for i, c in enumerate(T_CLASSES)}, {c: t.launches[i] for i, c in enumerate(T_CLASSES)},
                      {c: t.bytes[i] for i, c in enumerate(T_CLASSES)})

    def close(self):
        if getattr(self, "_h", None):
            lib().sdbg_ctx_destroy(self._h)
            self._h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass


class Timing:
    def __init__(self, ms, launches, bytes_):
        self.ms, self.launches, self.bytes = ms, launches, bytes_

    @property
    def total_launches(self) -> int:
        return sum(self.launches.values())


class Reads:
    """Device buffers of sdbg_reads, sized for n_bases bases packed in at most n_calls calls."""

    def __init__(self, n_bases: int, n_calls: int = 1, device=None):
        torch = _torch()
        slots = sdbg_read_slots(n_bases, n_calls)
        self.words = torch.empty(slots // 32, dtype=torch.int64, device=device or "cuda")
        self.ends = torch.empty(slots // 64, dtype=torch.int64, device=device or "cuda")
        self.c = _Reads(self.words.data_ptr(), self.ends.data_ptr(), slots, 0, 0, 0)

    n_reads = property(lambda self: self.c.n_reads)
    n_bases = property(lambda self: self.c.n_bases)


class Edges:
    def __init__(self, cap: int, k: int, device=None):
        torch = _torch()
        self.k, self.w = k, sdbg_key_words(k)
        self.keys = torch.empty(max(cap, 1) * self.w, dtype=torch.int64, device=device or "cuda")
        self.mult = torch.empty(max(cap, 1), dtype=torch.int32, device=device or "cuda")
        self.c = _Edges(self.keys.data_ptr(), self.mult.data_ptr(), cap, 0, k, self.w)

    n = property(lambda self: self.c.n)

    def keys_np(self) -> np.ndarray:
        return self.keys[: self.n * self.w].cpu().numpy().view(np.uint64).reshape(-1, self.w)

    def mult_np(self) -> np.ndarray:
        return self.mult[: self.n].cpu().numpy().view(np.uint32)


class Graph:
    def __init__(self, cap: int, device=None):
        torch = _torch()
        self.W = torch.empty(max(cap, 1), dtype=torch.uint8, device=device or "cuda")
        self.last_bits = torch.empty((max(cap, 1) + 63) // 64, dtype=torch.int64, device=device or "cuda")
        self.mult = torch.empty(max(cap, 1), dtype=torch.int32, device=device or "cuda")
        self.c = _Graph(self.W.data_ptr(), self.last_bits.data_ptr(), self.mult.data_ptr(), cap, 0)

    n = property(lambda self: self.c.n)

    def W_np(self):
        return self.W[: self.n].cpu().numpy()

    def last_bits_np(self):
        return self.last_bits[: (self.n + 63) // 64].cpu().numpy().view(np.uint64)

    def mult_np(self):
        return self.mult[: self.n].cpu().numpy().view(np.uint32)


class FullGraph:
    """Device buffers of sdbg_full_graph: cap edges, aux_cap zero-indegree nodes of k bases."""

    def __init__(self, cap: int, aux_cap: int, k: int, device=None):
        torch = _torch()
        dev = device or "cuda"
        self.k = k
        self.W = torch.empty(max(cap, 1), dtype=torch.uint8, device=dev)
        self.last_bits = torch.empty((max(cap, 1) + 63) // 64, dtype=torch.int64, device=dev)
        self.valid_bits = torch.empty((max(cap, 1) + 63) // 64, dtype=torch.int64, device=dev)
        self.mult = torch.empty(max(cap, 1), dtype=torch.int32, device=dev)
        self.aux_bits = torch.empty((2 * k * max(aux_cap, 1) + 63) // 64, dtype=torch.int64, device=dev)
        self.zin_bits = torch.empty((max(cap, 1) + 63) // 64, dtype=torch.int64, device=dev)
        self.c = _FullGraph(self.W.data_ptr(), self.last_bits.data_ptr(), self.valid_bits.data_ptr(), self.mult.data_ptr(),
                            self.aux_bits.data_ptr(), cap, aux_cap, 0, 0, 0, self.zin_bits.data_ptr())

    m = property(lambda self: self.c.m)
    t = property(lambda self: self.c.t)
    n_zero_out = property(lambda self: self.c.n_zero_out)

    def W_np(self):
        return self.W[: self.m].cpu().numpy()

    def mult_np(self):
        return self.mult[: self.m].cpu().numpy().view(np.uint32)

    def last_bits_np(self):
        return self.last_bits[: (self.m + 63) // 64].cpu().numpy().view(np.uint64)

    def valid_bits_np(self):
        return self.valid_bits[: (self.m + 63) // 64].cpu().numpy().view(np.uint64)

    def aux_bits_np(self):
        return self.aux_bits[: (2 * self.k * self.t + 63) // 64].cpu().numpy().view(np.uint64)

    def zin_bits_np(self):
        return self.zin_bits[: (self.m + 63) // 64].cpu().numpy().view(np.uint64)

    F = property(lambda self: [int(x) for x in self.c.F])


class Index:
    """Device block of sdbg_index for a graph of up to cap edges (rank/select cells; borrows the graph's W and last_bits)."""

    def __init__(self, cap: int, device=None):
        torch = _torch()
        nbytes = lib().sdbg_index_bytes(cap)
        self.cells = torch.empty((nbytes + 7) // 8, dtype=torch.int64, device=device or "cuda")
        self.c = _Index(self.cells.data_ptr(), nbytes)
        self.graph = None

    m = property(lambda self: self.c.m)
    ones = property(lambda self: [int(x) for x in self.c.ones])
    HF = property(lambda self: [int(x) for x in self.c.HF])


class Stats:
    def __init__(self, want_checksums: bool = False, want_bucket_hist: bool = False):
        self.c = _Stats()
        self.c.want_checksums = 1 if want_checksums else 0
        self.bucket_hist = None
        if want_bucket_hist:
            torch = _torch()
            self.bucket_hist = torch.zeros(SDBG_NUM_BUCKETS, dtype=torch.int64, device="cuda")
            self.c.bucket_hist = self.bucket_hist.data_ptr()

    def __getattr__(self, name):
        return getattr(self.__dict__["c"], name)


def _ptr(x):
    """torch tensor (CUDA or pinned/pageable CPU) or numpy array -> raw address; keeps no reference."""
    if x is None:
        return None
    if isinstance(x, np.ndarray):
        return x.ctypes.data
    return x.data_ptr()


def sdbg_pack_reads(ctx: Context, bases, offsets, n: int, out: Reads) -> None:
    """bases: uint8 ASCII (torch CUDA/CPU tensor or numpy array); offsets: n+1 uint64/int64, same space."""
    ctx.check(lib().sdbg_pack_reads(ctx._h, _ptr(bases), _ptr(offsets), n, C.byref(out.c)))


def sdbg_count_edges(ctx: Context, reads: Reads, n: int, k: int, d: int, out: Edges, stats: Stats | None = None) -> int:
    rc = lib().sdbg_count_edges(ctx._h, C.byref(reads.c), n, k, d, C.byref(out.c), C.byref(stats.c) if stats else None)
    ctx.check(rc)
    return out.c.n


def sdbg_count_edges_range(ctx: Context, reads: Reads, n: int, k: int, d: int, bucket_lo: int, bucket_hi: int, out: Edges,
                           stats: Stats | None = None) -> int:
    rc = lib().sdbg_count_edges_range(ctx._h, C.byref(reads.c), n, k, d, bucket_lo, bucket_hi, C.byref(out.c),
                                      C.byref(stats.c) if stats else None)
    ctx.check(rc)
    return out.c.n


def sdbg_bucket_hist(ctx: Context, reads: Reads, k: int, hist) -> None:
    """hist: 65,536 int64/uint64 on the device. Does not synchronise."""
    ctx.check(lib().sdbg_bucket_hist(ctx._h, C.byref(reads.c), k, _ptr(hist)))


def sdbg_plan_shards(hist: np.ndarray, n_shards: int) -> np.ndarray:
    """hist: 65,536 uint64 on the host -> n_shards + 1 partition bounds (uint32)."""
    h = np.ascontiguousarray(hist, dtype=np.uint64)
    assert h.size == SDBG_NUM_BUCKETS
    bounds = np.zeros(n_shards + 1, dtype=np.uint32)
    rc = lib().sdbg_plan_shards(h.ctypes.data, n_shards, bounds.ctypes.data)
    if rc != 0:
        raise SdbgError(rc, sdbg_strerror(rc))
    return bounds


def sdbg_mercy_edges(ctx: Context, reads: Reads, solid: Edges, out: Edges) -> int:
    ctx.check(lib().sdbg_mercy_edges(ctx._h, C.byref(reads.c), C.byref(solid.c), C.byref(out.c)))
    return out.c.n


def sdbg_build_full(ctx: Context, edges: Edges, out: FullGraph) -> int:
    ctx.check(lib().sdbg_build_full(ctx._h, C.byref(edges.c), C.byref(out.c)))
    return out.c.m


def sdbg_index_bytes(m: int) -> int:
    return lib().sdbg_index_bytes(m)


def sdbg_index_build(ctx: Context, graph: FullGraph, out: Index) -> None:
    ctx.check(lib().sdbg_index_build(ctx._h, C.byref(graph.c), C.byref(out.c)))
    out.graph = graph                                    # the index borrows W and last_bits


def sdbg_index_build_static(graph: FullGraph, out: Index, stream=None) -> None:
    """The index built with the library's static device scratch: no ctx, no workspace, no allocation (include/sdbg.h).
    stream: a torch.cuda.Stream or None (the default stream); synchronises it."""
    rc = lib().sdbg_index_build_static(stream.cuda_stream if stream is not None else None, C.byref(graph.c), C.byref(out.c))
    if rc != 0:
        raise SdbgError(rc, lib().sdbg_index_build_static_error().decode())
    out.graph = graph


def sdbg_forward(ctx: Context, index: Index, edge_idx, n: int, out) -> None:
    """edge_idx: n uint64/int64 on the device; out: n int64 on the device. Does not synchronise."""
    ctx.check(lib().sdbg_forward(ctx._h, C.byref(index.c), _ptr(edge_idx), n, _ptr(out)))


def sdbg_backward(ctx: Context, index: Index, edge_idx, n: int, out) -> None:
    ctx.check(lib().sdbg_backward(ctx._h, C.byref(index.c), _ptr(edge_idx), n, _ptr(out)))


def sdbg_build(ctx: Context, edges: Edges, flags: int, out: Graph) -> int:
    ctx.check(lib().sdbg_build(ctx._h, C.byref(edges.c), flags, C.byref(out.c)))
    return out.c.n
