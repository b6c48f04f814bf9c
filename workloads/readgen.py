"""ctypes front-ends of the two generator twins (host C, device CUDA). Inputs only."""
from __future__ import annotations

import ctypes
import os
import subprocess

import numpy as np

from .configs import Workload

_DIR = os.path.dirname(os.path.abspath(__file__))
_HOST_SO = os.path.join(_DIR, "libreadgen_host.so")
_CUDA_SO = os.path.join(_DIR, "libreadgen_cuda.so")


class _Params(ctypes.Structure):
    _fields_ = [("seed", ctypes.c_uint64), ("n_genomes", ctypes.c_uint64),
                ("read_len", ctypes.c_uint32), ("err_thr", ctypes.c_uint32)]


def _stale(so, srcs):
    return (not os.path.exists(so)) or any(os.path.getmtime(s) > os.path.getmtime(so) for s in srcs)


def build_host_lib(force: bool = False) -> str:
    srcs = [os.path.join(_DIR, "readgen_host.c"), os.path.join(_DIR, "readgen_core.h")]
    if force or _stale(_HOST_SO, srcs):
        subprocess.check_call(["gcc", "-O2", "-std=c11", "-shared", "-fPIC", "-o", _HOST_SO, srcs[0]])
    return _HOST_SO


def build_cuda_lib(force: bool = False) -> str:
    srcs = [os.path.join(_DIR, "readgen_cuda.cu"), os.path.join(_DIR, "readgen_core.h")]
    if force or _stale(_CUDA_SO, srcs):
        subprocess.check_call(["nvcc", "-O3", "-std=c++17", "-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo",
                               "-shared", "-Xcompiler", "-fPIC", "-o", _CUDA_SO, srcs[0]])
    return _CUDA_SO


class ReadGenerator:
    """Reads of one Workload. ``host(r0, r1)`` -> (uint8 ASCII array, uint64 offsets[r1-r0+1]);
    ``device(r0, r1)`` -> the same bytes as torch CUDA tensors, generated in HBM."""

    def __init__(self, w: Workload):
        self.w = w
        self.glen, self.cdf = w.tables()
        self.params = _Params(w.seed, w.n_genomes, w.read_len, int(w.err_rate * 2.0 ** 32))
        self._host = None
        self._cuda = None
        self._dev_tables = None

    def offsets(self, r0: int, r1: int) -> np.ndarray:
        return (np.arange(r1 - r0 + 1, dtype=np.uint64) * np.uint64(self.w.read_len))

    def host(self, r0: int = 0, r1: int | None = None):
        r1 = self.w.n_reads if r1 is None else r1
        if self._host is None:
            self._host = ctypes.CDLL(build_host_lib())
            self._host.rg_generate_host.argtypes = [ctypes.c_void_p] * 3 + [ctypes.c_uint64] * 2 + [ctypes.c_void_p]
            self._host.rg_generate_host.restype = None
        out = np.empty((r1 - r0) * self.w.read_len, dtype=np.uint8)
        self._host.rg_generate_host(ctypes.byref(self.params), self.glen.ctypes.data, self.cdf.ctypes.data,
                                    r0, r1, out.ctypes.data)
        return out, self.offsets(r0, r1)

    def device(self, r0: int = 0, r1: int | None = None, out=None):
        import torch
        r1 = self.w.n_reads if r1 is None else r1
        if self._cuda is None:
            if not os.path.exists(_CUDA_SO):
                raise RuntimeError(f"{_CUDA_SO} missing: run __graft_entry__.build() first")
            self._cuda = ctypes.CDLL(_CUDA_SO)
            self._cuda.rg_generate_device.argtypes = [ctypes.c_void_p] * 3 + [ctypes.c_uint64] * 2 + [ctypes.c_void_p] * 2
            self._cuda.rg_generate_device.restype = ctypes.c_int
            self._dev_tables = (torch.from_numpy(self.glen.view(np.int64)).cuda(),
                                torch.from_numpy(self.cdf.view(np.int64)).cuda())
        n = (r1 - r0) * self.w.read_len
        if out is None:
            out = torch.empty(n, dtype=torch.uint8, device="cuda")
        assert out.numel() >= n and out.is_cuda
        rc = self._cuda.rg_generate_device(ctypes.byref(self.params), self._dev_tables[0].data_ptr(),
                                           self._dev_tables[1].data_ptr(), r0, r1, out.data_ptr(),
                                           torch.cuda.current_stream().cuda_stream)
        if rc != 0:
            raise RuntimeError(f"rg_generate_device failed: cudaError {rc}")
        offs = torch.arange(r1 - r0 + 1, dtype=torch.int64, device="cuda") * self.w.read_len
        return out[:n], offs
