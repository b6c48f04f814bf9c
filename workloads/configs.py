"""The five BASELINE.json configs as generator parameters.

Each stands in for a workload of the paper (E. coli isolate; Iowa prairie soil
metagenome); none of those datasets is reproduced here — genomes are iid-uniform ACGT.
"""
from __future__ import annotations

import math
from dataclasses import dataclass, replace

import numpy as np

from . import _hash

CONFIG_NAMES = {
    1: "cfg1_tiny_isolate_k21",
    2: "cfg2_single_bacterium_k31",
    3: "cfg3_mock_metagenome_k31",
    4: "cfg4_mock_metagenome_k99",
    5: "cfg5_soil_like_k21_blockwise",
}


@dataclass(frozen=True)
class Workload:
    name: str
    seed: int
    n_genomes: int
    genome_model: str       # "fixed" | "uniform_1_5M_lognormal_abund" | "lognormal_len_zipf_abund"
    genome_len: int         # for "fixed"; the scale unit otherwise
    read_len: int
    n_reads: int
    err_rate: float
    k: int
    d: int = 2

    @property
    def n_bases(self) -> int:
        return self.n_reads * self.read_len

    @property
    def n_raw_edges(self) -> int:
        """N = 2 * sum_r max(0, L_r - k)  (SURVEY.md §8 notation)."""
        return 2 * self.n_reads * max(0, self.read_len - self.k)

    @property
    def words_per_key(self) -> int:
        return (2 * (self.k + 1) + 63) // 64

    def scaled(self, f: float) -> "Workload":
        """Same shape at a fraction f of the size (genome lengths and read count both scaled)."""
        return replace(self, name=f"{self.name}@{f:g}", n_reads=max(1, int(round(self.n_reads * f))),
                       genome_len=max(self.read_len + 1, int(round(self.genome_len * f))))

    def tables(self):
        """(genome lengths u64[n], cumulative pick weights u64[n]) — built on the host in float64 and
        handed to both generator twins, so no device-side exp/log can diverge."""
        n, seed = self.n_genomes, self.seed
        g = np.arange(n, dtype=np.uint64)
        if self.genome_model == "fixed":
            glen = np.full(n, self.genome_len, dtype=np.uint64)
            abund = np.ones(n, dtype=np.float64)
        else:
            u1 = (_hash.rg_hash(seed, _hash.STREAM_TABLE, g, 1) >> np.uint64(11)).astype(np.float64) * 2.0 ** -53
            u2 = (_hash.rg_hash(seed, _hash.STREAM_TABLE, g, 2) >> np.uint64(11)).astype(np.float64) * 2.0 ** -53
            z = np.sqrt(-2.0 * np.log(1.0 - u1)) * np.cos(2.0 * math.pi * u2)   # Box-Muller, float64
            unit = self.genome_len
            if self.genome_model == "uniform_1_5M_lognormal_abund":
                span = np.uint64(4 * unit + 1)
                glen = np.uint64(unit) + _hash.rg_hash(seed, _hash.STREAM_TABLE, g, 0) % span
                abund = np.exp(1.5 * z)
            elif self.genome_model == "lognormal_len_zipf_abund":
                glen = np.maximum(np.rint(unit * np.exp(0.5 * z)), self.read_len + 1).astype(np.uint64)
                abund = (g.astype(np.float64) + 1.0) ** -1.2
            else:
                raise ValueError(self.genome_model)
        glen = np.maximum(glen, np.uint64(self.read_len + 1))
        wgt = abund * glen.astype(np.float64)
        cum = np.cumsum(wgt)
        frac = cum / cum[-1]
        cdf = np.array([min(int(f * 2.0 ** 64), 2 ** 64 - 1) for f in frac], dtype=np.uint64)
        cdf[-1] = np.uint64(2 ** 64 - 1)
        return np.ascontiguousarray(glen), np.ascontiguousarray(cdf)


_BASE = {
    1: Workload(CONFIG_NAMES[1], 140972081, 1, "fixed", 100_000, 100, 30_000, 0.005, 21),
    2: Workload(CONFIG_NAMES[2], 140972082, 1, "fixed", 5_000_000, 150, 1_666_667, 0.01, 31),
    3: Workload(CONFIG_NAMES[3], 140972083, 200, "uniform_1_5M_lognormal_abund", 1_000_000, 150, 13_333_333, 0.01, 31),
    4: Workload(CONFIG_NAMES[4], 140972083, 200, "uniform_1_5M_lognormal_abund", 1_000_000, 150, 13_333_333, 0.01, 99),
    5: Workload(CONFIG_NAMES[5], 140972085, 50_000, "lognormal_len_zipf_abund", 3_000_000, 100, 200_000_000, 0.005, 21),
}


def get_config(i: int, scale: float = 1.0) -> Workload:
    w = _BASE[i]
    return w if scale == 1.0 else w.scaled(scale)
