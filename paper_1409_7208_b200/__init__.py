"""paper_1409_7208_b200 — thin Python binding of libsdbg (include/sdbg.h): the SdBG-construction hot path of
MEGAHIT (arxiv 1409.7208) as sm_100a CUDA kernels. Argument marshalling only; every step runs in the CUDA library.
There is no CPU fallback: without the built library or without a CUDA device the calls raise."""
from .binding import (  # noqa: F401
    SdbgError, Context, Reads, Edges, Graph, FullGraph, Index, Stats, Timing, lib, lib_path,
    sdbg_pack_reads, sdbg_count_edges, sdbg_build, sdbg_build_full, sdbg_mercy_edges, sdbg_plan_ranges,
    sdbg_index_bytes, sdbg_index_build, sdbg_index_build_static, sdbg_forward, sdbg_backward,
    sdbg_count_edges_range, sdbg_bucket_hist, sdbg_plan_shards,
    sdbg_key_words, sdbg_read_slots, sdbg_full_workspace, sdbg_workspace_for_records, sdbg_min_workspace, sdbg_strerror,
    sdbg_unstable_radix_launches,
    SDBG_SORTED, STATUS, SDBG_OPT_FORCE_WIDE, SDBG_OPT_NO_TABLE_COUNT, SDBG_OPT_STABLE_FIRST_PASS, SDBG_OPT_NO_FUSED_EXTRACT,
    SDBG_OPT_WEAK_FINGERPRINT,
)
