"""numpy restatement of rg_mix / rg_hash from readgen_core.h (used only to build the per-genome
tables on the host; checked against the C twin in tests/test_workloads.py)."""
import numpy as np

STREAM_GENOME, STREAM_READ, STREAM_ERR, STREAM_TABLE = 1, 2, 3, 4
_M1 = np.uint64(0xBF58476D1CE4E5B9)
_M2 = np.uint64(0x94D049BB133111EB)


def rg_mix(z):
    z = np.asarray(z, dtype=np.uint64)
    with np.errstate(over="ignore"):
        z = (z ^ (z >> np.uint64(30))) * _M1
        z = (z ^ (z >> np.uint64(27))) * _M2
        return z ^ (z >> np.uint64(31))


def rg_hash(seed, stream, a, b):
    with np.errstate(over="ignore"):
        h = rg_mix(np.uint64(seed) ^ rg_mix(np.uint64(stream + 1)))
        h = rg_mix(h + np.asarray(a, dtype=np.uint64))
        return rg_mix(h + np.asarray(b, dtype=np.uint64))
