"""Seeded synthetic workloads (inputs only) shared by the CPU oracle and the CUDA path.

Nothing in this package performs any step of the SdBG method: it only produces ASCII reads
(bytes over ACGT) and their offsets, from a counter-based generator with a host twin (C) and a
device twin (CUDA) compiled from the same header, see ``readgen_core.h``.
"""
from .configs import Workload, get_config, CONFIG_NAMES  # noqa: F401
from .readgen import ReadGenerator, build_host_lib, build_cuda_lib  # noqa: F401
