"""Builds csrc/libsdbg.so in-tree with nvcc for sm_100a (cross-compiles without a GPU).

Every .cu is compiled to an object of its own under csrc/build/ (recompiled only when the file, a header, an .inc or
the flags changed; the compilations run side by side), then the objects are linked into the shared library."""
from __future__ import annotations

import hashlib
import os
import subprocess
from concurrent.futures import ThreadPoolExecutor

_DIR = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(_DIR, "csrc")
OBJ = os.path.join(CSRC, "build")
LIB = os.path.join(CSRC, "libsdbg.so")
SOURCES = ["pack.cu", "extract.cu", "radix.cu", "count.cu", "hashcount.cu", "emit.cu", "dummies.cu", "mercy.cu", "rank.cu", "api.cu"]
NVCC_FLAGS = ["-O3", "-std=c++17", "-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-diag-suppress", "186",
              "-Xcompiler", "-fPIC"]


def _headers():
    d = [os.path.join(CSRC, f) for f in sorted(os.listdir(CSRC)) if f.endswith((".cuh", ".inc"))]
    d.append(os.path.join(os.path.dirname(_DIR), "include", "sdbg.h"))
    return d


def _stamp(src: str, flags) -> str:
    h = hashlib.sha256()
    for p in [os.path.join(CSRC, src), *_headers()]:
        with open(p, "rb") as f:
            h.update(f.read())
    h.update(" ".join(flags).encode())
    return h.hexdigest()[:16]


def build(force: bool = False, extra_flags=()) -> str:
    flags = [*NVCC_FLAGS, *extra_flags]
    os.makedirs(OBJ, exist_ok=True)
    jobs, objs = [], []
    for src in SOURCES:
        obj = os.path.join(OBJ, f"{src[:-3]}.{_stamp(src, flags)}.o")
        objs.append(obj)
        if force or not os.path.exists(obj):
            for old in os.listdir(OBJ):                  # objects of older versions of this source
                if old.startswith(src[:-3] + ".") and old.endswith(".o"):
                    os.remove(os.path.join(OBJ, old))
            jobs.append(["nvcc", *flags, "-c", os.path.join(CSRC, src), "-o", obj])
    if not jobs and os.path.exists(LIB) and all(os.path.getmtime(o) <= os.path.getmtime(LIB) for o in objs):
        return LIB
    with ThreadPoolExecutor(max_workers=min(len(jobs), os.cpu_count() or 1) or 1) as ex:
        for rc in ex.map(lambda c: subprocess.run(c, cwd=CSRC).returncode, jobs):
            if rc:
                raise RuntimeError("nvcc failed")
    subprocess.check_call(["nvcc", "-shared", "-gencode", "arch=compute_100a,code=sm_100a", "-o", LIB, *objs], cwd=CSRC)
    return LIB


if __name__ == "__main__":
    import sys
    print(build(force="--force" in sys.argv, extra_flags=[a for a in sys.argv[1:] if a.startswith("-D")]))
