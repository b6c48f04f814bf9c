"""Builds csrc/libsdbg.so in-tree with nvcc for sm_100a (cross-compiles without a GPU)."""
from __future__ import annotations

import os
import subprocess

_DIR = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(_DIR, "csrc")
LIB = os.path.join(CSRC, "libsdbg.so")
SOURCES = ["pack.cu", "extract.cu", "radix.cu", "count.cu", "hashcount.cu", "emit.cu", "dummies.cu", "mercy.cu", "rank.cu", "api.cu"]
NVCC_FLAGS = ["-O3", "-std=c++17", "-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo",
              "-Xcompiler", "-fPIC", "-shared"]


def _deps():
    d = [os.path.join(CSRC, f) for f in os.listdir(CSRC) if f.endswith((".cu", ".cuh", ".inc"))]
    d.append(os.path.join(os.path.dirname(_DIR), "include", "sdbg.h"))
    return d


def build(force: bool = False, extra_flags=()) -> str:
    if not force and os.path.exists(LIB) and all(os.path.getmtime(s) <= os.path.getmtime(LIB) for s in _deps()):
        return LIB
    cmd = ["nvcc", *NVCC_FLAGS, *extra_flags, "-o", LIB, *[os.path.join(CSRC, s) for s in SOURCES]]
    subprocess.check_call(cmd, cwd=CSRC)
    return LIB


if __name__ == "__main__":
    print(build(force=True))
