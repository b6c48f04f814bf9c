#!/usr/bin/env python
"""bench.py — (k+1)-mers sorted+counted per second on one B200 (BASELINE.json metric), through the C ABI.

A "step" is one pass of the whole hot path over one batch of synthetic reads:
sdbg_pack_reads -> sdbg_count_edges (extract, radix sort, count, solid filter) -> sdbg_build(SDBG_SORTED).
Default workload: BASELINE.json configs[1] (single bacterium, 5 Mbp, 150 bp reads at 50x, k=31, d=2).

  python bench.py [--gpus N] [--steps K] [--warmup W] [--config 1..4] [--impl reference]

`--impl reference` times the CPU oracle (oracle/, as it stands) on a bounded sample of the same workload.
With N>1 (torchrun) every rank runs an independent replica on its own GPU ("replicas only": the path does not
shard); value = records of all ranks / max-over-ranks time.
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "(k+1)-mers sorted+counted/sec"
UNIT = "edges/s"


def _peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        try:
            return float(json.load(open(p))["hbm_gbs"]), "measured (MEASURED_PEAKS.json)"
        except Exception:
            pass
    return 6650.0, "fallback (B200_PROFILING.md)"


def _traffic(workload_name, kernel_class):
    """DRAM bytes (read + write) per launch of a kernel class, from the committed ncu --set full capture of this
    workload (profiles/*_traffic.csv, newest round last; columns workload, kernel_class, dram_bytes_per_launch), or None."""
    import csv
    import glob
    val = None
    for p in sorted(glob.glob(os.path.join(ROOT, "profiles", "*_traffic.csv"))):
        try:
            for row in csv.DictReader(open(p)):
                if row.get("workload") == workload_name and row.get("kernel_class", "radix") == kernel_class:
                    val = int(row["dram_bytes_per_launch"])
        except Exception:
            pass
    return val


class ClockSampler(threading.Thread):
    """Samples SM clocks / throttle reasons while the timed region runs: NVML every 5 ms when the module is there,
    otherwise nvidia-smi (one process per sample, ~10 per second)."""
    Q = ("clocks.sm,clocks.max.sm,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")
    NAMES = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]

    def __init__(self, gpu_index):
        super().__init__(daemon=True)
        self.gpu, self.stop_flag, self.rows, self.source = gpu_index, threading.Event(), [], "nvidia-smi"
        self.mark0 = self.mark1 = None                   # sample counts at the start / end of the timed region

    def _nvml_loop(self):
        import pynvml as nv
        nv.nvmlInit()
        vis = os.environ.get("CUDA_VISIBLE_DEVICES", "")
        idx = self.gpu
        if vis and all(x.strip().isdigit() for x in vis.split(",")):
            idx = int(vis.split(",")[self.gpu])
        h = nv.nvmlDeviceGetHandleByIndex(idx)
        mx = float(nv.nvmlDeviceGetMaxClockInfo(h, nv.NVML_CLOCK_SM))
        bits = [getattr(nv, n) for n in ("nvmlClocksEventReasonHwSlowdown", "nvmlClocksEventReasonHwThermalSlowdown",
                                         "nvmlClocksEventReasonSwThermalSlowdown", "nvmlClocksEventReasonSwPowerCap")] \
            if hasattr(nv, "nvmlClocksEventReasonHwSlowdown") else \
            [nv.nvmlClocksThrottleReasonHwSlowdown, nv.nvmlClocksThrottleReasonHwThermalSlowdown,
             nv.nvmlClocksThrottleReasonSwThermalSlowdown, nv.nvmlClocksThrottleReasonSwPowerCap]
        get_reasons = getattr(nv, "nvmlDeviceGetCurrentClocksEventReasons", None) or nv.nvmlDeviceGetCurrentClocksThrottleReasons
        self.source = "nvml"
        while not self.stop_flag.is_set():
            r = get_reasons(h)
            self.rows.append([str(float(nv.nvmlDeviceGetClockInfo(h, nv.NVML_CLOCK_SM))), str(mx)] +
                             ["Active" if r & b else "Not Active" for b in bits])
            self.stop_flag.wait(0.005)

    def run(self):
        try:
            self._nvml_loop()
            return
        except Exception:
            self.source = "nvidia-smi"
        while not self.stop_flag.is_set():
            try:
                out = subprocess.run(["nvidia-smi", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits", "-i", str(self.gpu)],
                                     capture_output=True, text=True, timeout=5).stdout.strip()
                if out:
                    self.rows.append([x.strip() for x in out.split(",")])
            except Exception:
                pass
            self.stop_flag.wait(0.1)

    def mark(self, which):
        if which == 0:
            self.mark0 = len(self.rows)
        else:
            self.mark1 = len(self.rows)

    def summary(self):
        self.stop_flag.set()
        self.join(timeout=6)
        rows = self.rows
        if self.mark0 is not None and self.mark1 is not None and self.mark1 - self.mark0 >= 3:
            rows = rows[self.mark0:self.mark1]           # the timed region only (else everything seen, warm-up included)
        sm = sorted(float(r[0]) for r in rows if r and r[0].replace(".", "").isdigit())
        mx = [float(r[1]) for r in rows if len(r) > 1 and r[1].replace(".", "").isdigit()]
        reasons = sorted({n for r in rows if len(r) >= 6 for n, v in zip(self.NAMES, r[2:6]) if v.lower().startswith("active")})
        return {"sm_mhz": sm[len(sm) // 2] if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "reasons": reasons, "samples": len(rows), "source": self.source}


def run_reference(args, w):
    """The oracle, as it stands, on the host cores: each step = steps 1-6 on a bounded sample of the workload."""
    from oracle import run_oracle
    from workloads import ReadGenerator
    n_reads = min(w.n_reads, args.ref_reads)
    bases, offs = ReadGenerator(w).host(0, n_reads)
    n_rec = 2 * n_reads * max(0, w.read_len - w.k)
    for _ in range(args.warmup if args.warmup < 2 else 1):
        run_oracle((bases, offs), w.k, w.d)
    t0 = time.perf_counter()
    for _ in range(args.steps):
        run_oracle((bases, offs), w.k, w.d)
    dt = (time.perf_counter() - t0) / args.steps
    val = n_rec / dt
    sample = f"first {n_reads} reads of {w.name} ({n_rec} records) per step"
    line = {"impl": "reference", "metric": METRIC, "value": val, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": dt * 1e3, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "u64", "data": "synthetic",
            "config": {"workload": w.name, "k": w.k, "d": w.d, "read_len": w.read_len, "sample": sample},
            "cpu_baseline": {"value": val, "unit": UNIT, "cores": 1, "kind": "oracle", "sample": sample},
            "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}}
    print(json.dumps(line), flush=True)


def cpu_baseline(w, n_reads):
    """Oracle timed once on a bounded sample (rank 0, N=1 only): about 10-30 s of single-core CPU work."""
    from oracle import run_oracle
    from workloads import ReadGenerator
    n_reads = min(w.n_reads, n_reads)
    bases, offs = ReadGenerator(w).host(0, n_reads)
    n_rec = 2 * n_reads * max(0, w.read_len - w.k)
    t0 = time.perf_counter()
    run_oracle((bases, offs), w.k, w.d)
    dt = time.perf_counter() - t0
    return {"value": n_rec / dt, "unit": UNIT, "cores": 1, "kind": "oracle",
            "sample": f"first {n_reads} reads of {w.name} ({n_rec} records), {dt:.1f} s, single thread"}


def rank_seed(base_seed: int, rank: int) -> int:
    """Replicas only: every rank sorts its own read set."""
    return base_seed + 1000003 * rank


def max_over_ranks(values, device="cpu"):
    """Element-wise MAX of a list of floats over all ranks of the default process group (identity without one)."""
    import torch
    import torch.distributed as dist
    t = torch.tensor(list(values), dtype=torch.float64, device=device)
    if dist.is_available() and dist.is_initialized() and dist.get_world_size() > 1:
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return [float(x) for x in t]


def whole_job_value(records_per_rank: int, world: int, steps: int, ms_max: float) -> float:
    """Records all ranks processed / the slowest rank's time (weak scaling: per-rank work is fixed)."""
    return world * records_per_rank * steps / (ms_max * 1e-3)


NOMINAL_HBM_GBS = 8000.0    # the denominator BASELINE.json:north_star names ("~8 TB/s HBM3e peak")

KERNEL_OF_CLASS = {
    "pack": "pack_kernel + mark_ends_kernel",
    "extract": "extract_kernel",
    "radix": "onesweep_kernel (one LSD radix pass over all records)",
    "table": "hash_count_kernel (table count of the top-sorted records)",
    "count": "count step helpers (hash_bounds/scan/copy kernels, or the sweeps of count.cu)",
    "emit": "emit_kernel",
    "other": "memsets, histogram scan, gathers",
}


def full_lsd_model_bytes_per_record(k: int) -> int:
    """K (2P + 2) bytes per raw record for a full LSD sort with 8-bit digits (144 at k = 31)."""
    bits = 2 * (k + 1)
    K = 8 * ((bits + 63) // 64)
    P = sum(-(-min(64, bits - 64 * q) // 8) for q in range((bits + 63) // 64))
    return K * (2 * P + 2)


def roofline_blocks(tim, steps, ms_per_step, peak, peak_src, wl_name, k, value):
    """`roofline` for the kernel class with the largest share of the step, the same figures for the other classes, the
    whole step on the bytes the library accounted, and records/s against the full-LSD byte model."""
    per = {}
    for c in tim.ms:
        n, ms, by = tim.launches[c], tim.ms[c], tim.bytes[c]
        if n == 0 or ms <= 0:
            continue
        ach = by / (ms * 1e-3) / 1e9
        per[c] = {"kernel": KERNEL_OF_CLASS.get(c, c), "bound": "hbm", "achieved": ach, "peak": peak, "unit": "GB/s",
                  "frac": ach / peak, "frac_of_measured": ach / peak, "frac_of_nominal_8TBps": ach / NOMINAL_HBM_GBS,
                  "traffic": _traffic(wl_name, c), "peak_source": peak_src, "launches": int(n),
                  "avg_launch_ms": ms / n, "algorithmic_bytes_per_launch": by // n,
                  "ms_per_step": ms / steps, "share_of_step": ms / steps / ms_per_step}
    top = max(per, key=lambda c: per[c]["ms_per_step"])
    step_bytes = sum(tim.bytes.values()) / steps
    step_ach = step_bytes / (ms_per_step * 1e-3) / 1e9
    model = full_lsd_model_bytes_per_record(k)
    out = {
        "roofline": dict(per[top], kernel_class=top),
        "roofline_other_kernels": {c: v for c, v in per.items() if c != top},
        "roofline_step": {"bound": "hbm", "achieved": step_ach, "peak": peak, "unit": "GB/s", "frac": step_ach / peak,
                          "frac_of_nominal_8TBps": step_ach / NOMINAL_HBM_GBS,
                          "algorithmic_bytes_per_step": int(step_bytes), "bytes_per_record": None,
                          "note": "bytes the library accounted for every kernel of the step / device time of the step"},
        "records_per_s_vs_full_lsd_model": {
            "model_bytes_per_record": model, "model_records_per_s_at_measured_peak": peak * 1e9 / model,
            "ratio": value / (peak * 1e9 / model),
            "note": "SURVEY.md 8(d): a full LSD sort moves K(2P+2) bytes per record; this path moves fewer (top passes + table count)"},
    }
    return out


def device_steps(sd, torch, wl, args, steps, warmup, rank, world, local, barrier, sampler=None):
    """`steps` timed steps of the whole hot path with the ASCII reads resident in HBM. Returns (ms_total, timing, S,
    device tensors for the end-to-end leg)."""
    from workloads import ReadGenerator
    gen = ReadGenerator(wl)
    bases_d, offs_d = gen.device()
    torch.cuda.synchronize()
    n_reads, N = wl.n_reads, wl.n_raw_edges
    ws_bytes = int(args.workspace_gb * 2 ** 30) if args.workspace_gb else sd.sdbg_workspace_for_records(N, wl.k)
    ctx = sd.Context(ws_bytes)
    reads = sd.Reads(wl.n_bases)
    cap = N // wl.d
    if cap * (8 * wl.words_per_key + 10) > 40 * 2 ** 30:      # the safe bound N / d would not fit: ask for the count first
        sd.sdbg_pack_reads(ctx, bases_d, offs_d, n_reads, reads)
        probe = sd.Edges(0, wl.k)
        try:
            sd.sdbg_count_edges(ctx, reads, n_reads, wl.k, wl.d, probe, None)
        except sd.SdbgError as e:
            if e.name != "SDBG_E_CAPACITY":
                raise
        cap = probe.n + 1024
    edges = sd.Edges(cap, wl.k)
    graph = sd.Graph(cap)

    def step():
        reads.c.n_reads = reads.c.n_bases = reads.c.n_slots = 0
        sd.sdbg_pack_reads(ctx, bases_d, offs_d, n_reads, reads)
        if args.shard:     # replicated reads, each rank counts its range of l=8 partitions
            from paper_1409_7208_b200.shard import count_edges_sharded, gather_counts
            n_local, _ = count_edges_sharded(ctx, reads, n_reads, wl.k, wl.d, edges, rank, world)
            sd.sdbg_build(ctx, edges, sd.SDBG_SORTED, graph)
            gather_counts(n_local, device="cuda")        # offsets of the concatenation: the only exchange
            return edges.n
        sd.sdbg_count_edges(ctx, reads, n_reads, wl.k, wl.d, edges, None)
        sd.sdbg_build(ctx, edges, sd.SDBG_SORTED, graph)
        return edges.n

    S = 0
    for _ in range(max(warmup, 3)):
        S = step()
    ctx.get_timing()
    ctx.set_timing(True)
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    barrier()
    if sampler is not None:
        sampler.mark(0)
    ev0.record()
    for _ in range(steps):
        step()
    ev1.record()
    barrier()
    if sampler is not None:
        sampler.mark(1)
    ms_total = ev0.elapsed_time(ev1)
    tim = ctx.get_timing()
    ctx.set_timing(False)
    ctx.close(); ctx.workspace = None
    del reads, edges, graph
    torch.cuda.empty_cache()
    return ms_total, tim, S, bases_d, offs_d


def pcie_rates(torch, nbytes=256 << 20):
    """Measured host<->device copy rates of this box (pinned memory, one direction at a time), GB/s."""
    h = torch.empty(nbytes, dtype=torch.uint8, pin_memory=True)
    d = torch.empty(nbytes, dtype=torch.uint8, device="cuda")
    out = []
    for src, dst in ((h, d), (d, h)):
        dst.copy_(src, non_blocking=True)
        torch.cuda.synchronize()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        for _ in range(3):
            dst.copy_(src, non_blocking=True)
        e1.record()
        torch.cuda.synchronize()
        out.append(3 * nbytes / (e0.elapsed_time(e1) * 1e-3) / 1e9)
    return out


def run_gpu(args, w):
    import torch
    import torch.distributed as dist
    import paper_1409_7208_b200 as sd

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))

    # ---- inputs resident in HBM: every rank an independent replica (own seed) ------------------------------
    from dataclasses import replace
    wl = replace(w, seed=rank_seed(w.seed, rank)) if (rank and not args.shard) else w   # --shard: the same reads on every rank
    n_bases, n_reads = wl.n_bases, wl.n_reads
    N = wl.n_raw_edges
    K = 8 * wl.words_per_key

    def barrier():
        torch.cuda.synchronize()
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    sampler = ClockSampler(local)
    sampler.start()
    ms_total, tim, S, bases_d, offs_d = device_steps(sd, torch, wl, args, args.steps, args.warmup, rank, world, local, barrier, sampler)
    clocks = sampler.summary()

    # ---- end to end: HOST pinned buffers in, SdBG arrays out, copies inside the timed region ---------------------
    # Every step copies its reads from pinned host memory, runs the whole path and copies the SdBG arrays back; the
    # step is over when its results are on the host. `--e2e-pipelines P` (default 3) runs P such step loops at once,
    # each with its own context, stream, workspace and output buffers, fed by one host thread each, so that the copies
    # of one step overlap the kernels of another (PCIe is full duplex and idle while a step sorts).
    ms_e2e, e2e_steps, n_pipes = float("nan"), 0, 0
    h2d_gbs = d2h_gbs = None
    if not args.no_e2e and not args.shard:
        ws_bytes = sd.sdbg_workspace_for_records(N, wl.k)
        bases_h = torch.empty(n_bases, dtype=torch.uint8, pin_memory=True)
        offs_h = torch.empty(n_reads + 1, dtype=torch.int64, pin_memory=True)
        bases_h.copy_(bases_d); offs_h.copy_(offs_d)
        del bases_d, offs_d
        torch.cuda.empty_cache()
        h2d_gbs, d2h_gbs = pcie_rates(torch)
        free_b = torch.cuda.mem_get_info()[0]
        per_pipe = ws_bytes + n_bases // 2 + S * (K + 4 + 5 + 1) + (64 << 20)
        n_pipes = max(1, min(args.e2e_pipelines, int(free_b * 0.9 // per_pipe)))

        class Pipe:
            pass

        pipes = []
        for _ in range(n_pipes):
            pp = Pipe()
            pp.stream = torch.cuda.Stream()
            pp.copy_stream = torch.cuda.Stream()
            with torch.cuda.stream(pp.stream):
                pp.ctx = sd.Context(ws_bytes)
                pp.reads = sd.Reads(n_bases)
                pp.edges = sd.Edges(S + 1024, wl.k)
                pp.graph = sd.Graph(S + 1024)
            pp.out_W = torch.empty(S, dtype=torch.uint8, pin_memory=True)
            pp.out_last = torch.empty((S + 63) // 64, dtype=torch.int64, pin_memory=True)
            pp.out_mult = torch.empty(S, dtype=torch.int32, pin_memory=True)
            pp.out_keys = torch.empty(S * wl.words_per_key, dtype=torch.int64, pin_memory=True)
            pp.gpu_done = torch.cuda.Event()
            pp.done = torch.cuda.Event()
            pipes.append(pp)

        # one loop at a time in each phase: identical loops started together would otherwise stay in lockstep and share
        # the link and the SMs phase by phase; with the locks one loop sorts while another copies. The device-to-host
        # copy of a step runs on the pipe's copy stream behind an event, so the host thread never waits for the kernels
        # of its own step before it queues the copy, and the GPU lock is free as soon as the last kernel is queued.
        lock_in, lock_gpu, lock_out = threading.Lock(), threading.Lock(), threading.Lock()

        def e2e_loop(pp, n_steps, start_event):
            torch.cuda.set_device(local)
            with torch.cuda.stream(pp.stream):
                if start_event is not None:
                    pp.stream.wait_event(start_event)
                for _ in range(n_steps):
                    pp.reads.c.n_reads = pp.reads.c.n_bases = pp.reads.c.n_slots = 0
                    with lock_in:                        # host -> device copy of the reads (+ the pack kernel)
                        sd.sdbg_pack_reads(pp.ctx, bases_h, offs_h, n_reads, pp.reads)
                    with lock_gpu:                       # extract, sort, count (returns with the count), emit
                        sd.sdbg_count_edges(pp.ctx, pp.reads, n_reads, wl.k, wl.d, pp.edges, None)
                        sd.sdbg_build(pp.ctx, pp.edges, sd.SDBG_SORTED, pp.graph)
                        pp.gpu_done.record(pp.stream)
                    s_ = pp.edges.n
                    with lock_out:                       # device -> host copy of the SdBG arrays
                        pp.copy_stream.wait_event(pp.gpu_done)
                        with torch.cuda.stream(pp.copy_stream):
                            pp.out_W.copy_(pp.graph.W[:s_], non_blocking=True)
                            pp.out_last.copy_(pp.graph.last_bits[:(s_ + 63) // 64], non_blocking=True)
                            pp.out_mult.copy_(pp.graph.mult[:s_], non_blocking=True)
                            pp.out_keys.copy_(pp.edges.keys[:s_ * wl.words_per_key], non_blocking=True)
                        pp.copy_stream.synchronize()     # the step's results are on the host
                    pp.stream.wait_stream(pp.copy_stream)
                pp.done.record(pp.stream)

        def run_all(n_steps, start_event):
            ths = [threading.Thread(target=e2e_loop, args=(pp, n_steps, start_event)) for pp in pipes]
            for t in ths:
                t.start()
            for t in ths:
                t.join()

        run_all(1, None)                                 # warm-up: one step per pipeline
        per = (args.steps + n_pipes - 1) // n_pipes
        e2e_steps = per * n_pipes
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        barrier()
        e0.record()
        run_all(per, e0)
        for pp in pipes:
            torch.cuda.current_stream().wait_event(pp.done)
        e1.record()
        barrier()
        ms_e2e = e0.elapsed_time(e1) * args.steps / e2e_steps     # scaled to args.steps steps, as the other timings
        for pp in pipes:
            assert pp.edges.n == S
            pp.ctx.close(); pp.ctx.workspace = None
        del pipes, bases_h, offs_h
        torch.cuda.empty_cache()
    else:
        del bases_d, offs_d
        torch.cuda.empty_cache()
    h2d = n_bases + 8 * (n_reads + 1)
    d2h = S * (1 + 4 + K) + 8 * ((S + 63) // 64)

    # ---- the second headline config of SURVEY.md 8(d) (config 3: mock metagenome, k = 31) in the same process ------------
    also = {}
    if world == 1 and not args.shard and not args.no_also and args.config == 2:
        from workloads import get_config
        w3 = get_config(3)
        ms3, tim3, S3, b3, o3 = device_steps(sd, torch, w3, args, args.also_steps, 3, 0, 1, local, barrier, None)
        del b3, o3
        torch.cuda.empty_cache()
        peak3, src3 = _peaks()
        v3 = w3.n_raw_edges * args.also_steps / (ms3 * 1e-3)
        blk = {"ms_per_step": ms3 / args.also_steps, "value": v3, "unit": UNIT, "steps": args.also_steps, "warmup": 3,
               "raw_edges": w3.n_raw_edges, "solid_edges": int(S3), "k": w3.k, "d": w3.d,
               "kernel_ms_per_step": {c: tim3.ms[c] / args.also_steps for c in tim3.ms},
               "kernel_launches_per_step": {c: tim3.launches[c] / args.also_steps for c in tim3.launches}}
        blk.update(roofline_blocks(tim3, args.also_steps, ms3 / args.also_steps, peak3, src3, w3.name, w3.k, v3))
        also[w3.name] = blk

    ms_total, ms_e2e = max_over_ranks([ms_total, ms_e2e], device="cuda")
    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return

    peak, peak_src = _peaks()
    value = whole_job_value(N, 1 if args.shard else world, args.steps, ms_total)
    line = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world,
        "steps": args.steps, "warmup": max(args.warmup, 3), "ms_per_step": ms_total / args.steps,
        "higher_is_better": True, "scaling": "strong" if args.shard else "weak", "vs_baseline": None, "dtype": "u64", "data": "synthetic",
        "config": {"workload": wl.name, "k": wl.k, "d": wl.d, "reads": n_reads, "read_len": wl.read_len, "bases": n_bases,
                   "raw_edges": N, "solid_edges": int(S), "key_bytes": K, "parallelism": ("sharded by ranges of l=8 partitions, reads replicated" if args.shard else "replicas only" if world > 1 else "1 gpu"),
                   "l2": "inputs larger than L2 (keys %.2f GB, reads %.0f MB ASCII)" % (N * K / 1e9, n_bases / 1e6),
                   "workspace_gib": args.workspace_gb or None},
        "read_bases_per_s": (1 if args.shard else world) * n_bases * args.steps / (ms_total * 1e-3),
        "clocks": clocks,
        "e2e": {"value": whole_job_value(N, world, args.steps, ms_e2e), "unit": UNIT, "h2d_bytes_per_step": h2d,
                "d2h_bytes_per_step": d2h, "ms_per_step": ms_e2e / args.steps, "pipelines": n_pipes,
                "steps_timed": e2e_steps, "h2d_gbs_measured": h2d_gbs, "d2h_gbs_measured": d2h_gbs,
                "pcie_lower_bound_ms": (max(h2d / (h2d_gbs * 1e9), d2h / (d2h_gbs * 1e9)) * 1e3) if h2d_gbs and d2h_gbs else None},
        "gpu_launches": int(tim.total_launches),
        "kernel_ms_per_step": {c: tim.ms[c] / args.steps for c in tim.ms},
        "kernel_launches_per_step": {c: tim.launches[c] / args.steps for c in tim.launches},
    }
    line.update(roofline_blocks(tim, args.steps, ms_total / args.steps, peak, peak_src, wl.name, wl.k, value / (1 if args.shard else world)))
    if also:
        line["also"] = also
    if world == 1 and not args.no_cpu_baseline:
        line["cpu_baseline"] = cpu_baseline(wl, 2 * args.ref_reads)   # ~11 s of one host core (the reference arm: half of it per step)
    print(json.dumps(line), flush=True)
    if world > 1:
        dist.destroy_process_group()


def run_next_rows(args, w):
    """`--next`: the widened rows (DESIGN.md §0 f-1, f-2, f-3) on the same workload, timed by CUDA events around the
    C-ABI calls: sdbg_build_full, sdbg_mercy_edges, sdbg_index_build and the two
    traversal maps over the solid edges of one sdbg_count_edges run. Not part of
    the step that `value` measures."""
    import torch
    import paper_1409_7208_b200 as sd
    from workloads import ReadGenerator
    torch.cuda.set_device(0)
    bases_d, offs_d = ReadGenerator(w).device()
    N = w.n_raw_edges
    ctx = sd.Context(sd.sdbg_workspace_for_records(N, w.k))
    reads = sd.Reads(w.n_bases)
    sd.sdbg_pack_reads(ctx, bases_d, offs_d, w.n_reads, reads)
    edges = sd.Edges(N // w.d, w.k)
    sd.sdbg_count_edges(ctx, reads, w.n_reads, w.k, w.d, edges, None)
    S = edges.n

    def sized(call, make):
        probe = make(0)
        try:
            call(probe)
        except sd.SdbgError as e:
            if e.name != "SDBG_E_CAPACITY":
                raise
        return probe

    pf = sized(lambda g: sd.sdbg_build_full(ctx, edges, g), lambda c: sd.FullGraph(c, c, w.k))
    fg = sd.FullGraph(pf.m, pf.t, w.k)
    pm = sized(lambda e: sd.sdbg_mercy_edges(ctx, reads, edges, e), lambda c: sd.Edges(c, w.k))
    me = sd.Edges(pm.n, w.k)

    def timed(fn):
        for _ in range(2):
            fn()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        torch.cuda.synchronize()
        e0.record()
        for _ in range(args.steps):
            fn()
        e1.record()
        torch.cuda.synchronize()
        return e0.elapsed_time(e1) / args.steps

    ms_full = timed(lambda: sd.sdbg_build_full(ctx, edges, fg))
    ms_mercy = timed(lambda: sd.sdbg_mercy_edges(ctx, reads, edges, me))
    # traversal (f-3): index build, then 2^24 random forward / backward queries (indices and answers resident in HBM)
    ix = sd.Index(fg.m)
    ms_index = timed(lambda: sd.sdbg_index_build(ctx, fg, ix))
    nq = 1 << 24
    gen = torch.Generator(device="cuda"); gen.manual_seed(w.seed)
    q = torch.randint(0, max(int(fg.m), 1), (nq,), device="cuda", generator=gen)
    ans = torch.empty(nq, dtype=torch.int64, device="cuda")
    ms_fwd = timed(lambda: sd.sdbg_forward(ctx, ix, q, nq, ans))
    ms_bwd = timed(lambda: sd.sdbg_backward(ctx, ix, q, nq, ans))
    trav = {"index_build_ms": ms_index, "index_bytes": int(sd.sdbg_index_bytes(fg.m)), "queries": nq,
            "forward_ms": ms_fwd, "forward_queries_per_s": nq / (ms_fwd * 1e-3),
            "backward_ms": ms_bwd, "backward_queries_per_s": nq / (ms_bwd * 1e-3)}
    print(json.dumps({"impl": "next_rows", "config": {"workload": w.name, "k": w.k, "d": w.d, "solid_edges": int(S)},
                      "traversal": trav,
                      "sdbg_build_full": {"ms": ms_full, "m": int(fg.m), "t": int(fg.t), "dollar_edges": int(fg.n_zero_out),
                                          "solid_edges_per_s": S / (ms_full * 1e-3)},
                      "sdbg_mercy_edges": {"ms": ms_mercy, "mercy_records": int(me.n),
                                           "read_bases_per_s": w.n_bases / (ms_mercy * 1e-3)}}), flush=True)


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--config", type=int, default=2, help="BASELINE.json config number (1-5); default 2 = configs[1]; 5 (20 Gbp, "
                    "block-wise) needs --workspace-gb (default 100) and skips the end-to-end leg")
    ap.add_argument("--workspace-gb", type=float, default=0.0, help="workspace of the context in GiB (default: what holds all records in one range)")
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--ref-reads", type=int, default=40000, help="reads in the oracle's bounded sample")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true", help="development runs: skip the host-buffer end-to-end leg")
    ap.add_argument("--e2e-pipelines", type=int, default=3, help="concurrent host-to-host step loops of the end-to-end leg")
    ap.add_argument("--no-also", action="store_true", help="skip the config-3 sub-record of the default run")
    ap.add_argument("--also-steps", type=int, default=3, help="timed steps of the config-3 sub-record")
    ap.add_argument("--shard", action="store_true", help="strong scaling: every rank holds the same reads and counts its own range "
                    "of l=8 partitions (SURVEY.md §8(e)); default is independent replicas")
    ap.add_argument("--next", action="store_true", help="time the widened rows (sdbg_build_full, sdbg_mercy_edges) instead")
    args = ap.parse_args()
    from workloads import get_config
    w = get_config(args.config)
    if args.config == 5:
        args.no_e2e = True
        args.workspace_gb = args.workspace_gb or 100.0
    if args.next:
        if int(os.environ.get("RANK", "0")) == 0:
            run_next_rows(args, w)
        return
    if args.impl == "reference":
        if int(os.environ.get("RANK", "0")) == 0:
            run_reference(args, w)
        return
    run_gpu(args, w)


if __name__ == "__main__":
    main()
