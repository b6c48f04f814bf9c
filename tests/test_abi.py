"""CPU-side checks of the boundary: the C-ABI library builds for sm_100a, loads, exports every symbol that
include/sdbg.h declares, and its host-only logic (planner, sizing, error strings) behaves. No compute calls."""
import ctypes
import os
import re

import numpy as np
import pytest

import paper_1409_7208_b200 as sd
from paper_1409_7208_b200 import build as sdbuild

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module", autouse=True)
def _built():
    sdbuild.build()


def _declared_functions():
    src = open(os.path.join(ROOT, "include", "sdbg.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(sdbg_[a-z_0-9]+)\s*\(", src)))


def test_library_exports_every_declared_symbol():
    names = _declared_functions()
    assert {"sdbg_pack_reads", "sdbg_count_edges", "sdbg_build", "sdbg_ctx_create", "sdbg_plan_ranges"} <= set(names)
    L = ctypes.CDLL(sd.lib_path())
    for n in names:
        assert hasattr(L, n), f"{n} declared in include/sdbg.h but not exported"


def test_python_binding_has_the_same_names():
    for n in ("sdbg_pack_reads", "sdbg_count_edges", "sdbg_build", "sdbg_plan_ranges", "sdbg_key_words",
              "sdbg_read_slots", "sdbg_full_workspace", "sdbg_workspace_for_records", "sdbg_min_workspace", "sdbg_strerror"):
        assert callable(getattr(sd, n))


def test_host_helpers():
    assert [sd.sdbg_key_words(k) for k in (1, 21, 31, 32, 63, 64, 95, 96, 99, 127)] == [1, 1, 1, 2, 2, 3, 3, 4, 4, 4]
    assert sd.sdbg_strerror(0) == "ok" and "workspace" in sd.sdbg_strerror(-4)
    assert sd.sdbg_read_slots(100, 1) % 64 == 0 and sd.sdbg_read_slots(100, 1) >= 100 + 64 + 256
    # a single-range workspace grows with the key width and holds at least two key buffers
    w31, w99 = sd.sdbg_full_workspace(10 ** 6, 31), sd.sdbg_full_workspace(10 ** 6, 99)
    assert w31 >= 2 * 8 * 2 * 10 ** 6 and w99 >= 4 * (w31 - sd.sdbg_min_workspace())
    assert sd.sdbg_full_workspace(10 ** 6, 0) == 0 and sd.sdbg_full_workspace(10 ** 6, 128) == 0
    assert sd.sdbg_workspace_for_records(2 * 10 ** 6, 31) == w31 and sd.sdbg_workspace_for_records(10 ** 6, 31) < w31


def test_plan_ranges_greedy_consecutive():
    """A12: greedy maximal runs of consecutive l=8 partitions under the capacity."""
    rng = np.random.default_rng(5)
    h = rng.integers(0, 100, size=65536).astype(np.uint64)
    cap = 5000
    r = sd.sdbg_plan_ranges(h, cap)
    assert r[0][0] == 0 and r[-1][1] == 65536
    for (lo, hi, n), nxt in zip(r, r[1:] + [None]):
        assert n == int(h[lo:hi].sum()) <= cap
        if nxt is not None:
            assert nxt[0] == hi and n + int(h[hi]) > cap          # maximal: the next partition would not fit
    assert sd.sdbg_plan_ranges(h, int(h.sum())) == [(0, 65536, int(h.sum()))]
    z = np.zeros(65536, dtype=np.uint64)
    assert sd.sdbg_plan_ranges(z, 0) == [(0, 65536, 0)]
    h2 = z.copy(); h2[7] = 11
    with pytest.raises(sd.SdbgError) as ei:
        sd.sdbg_plan_ranges(h2, 10)
    assert ei.value.name == "SDBG_E_WORKSPACE"
    assert sd.sdbg_plan_ranges(h2, 11) == [(0, 65536, 11)]


def test_no_cpu_fallback_without_device():
    import torch
    if torch.cuda.is_available():
        pytest.skip("has a GPU")
    with pytest.raises(RuntimeError):
        sd.Context(1 << 26)
    # and the raw ABI refuses too
    h = ctypes.c_void_p()
    buf = ctypes.create_string_buffer(1 << 10)
    rc = sd.lib().sdbg_ctx_create(ctypes.byref(h), 0, None, ctypes.c_void_p(256 * ((ctypes.addressof(buf) + 255) // 256)), 1 << 30)
    assert rc == -5


def test_product_never_imports_the_oracle():
    for dirpath, _, files in os.walk(os.path.join(ROOT, "paper_1409_7208_b200")):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".inc", ".h")):
                txt = open(os.path.join(dirpath, f)).read()
                assert not re.search(r"^\s*(from|import)\s+oracle|#include\s+[\"<].*oracle", txt, flags=re.M), f
