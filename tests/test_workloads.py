"""The seeded input generator: host twin determinism and shape; device twin equality (gpu)."""
import ctypes

import numpy as np
import pytest

from workloads import ReadGenerator, build_host_lib, get_config
from workloads import _hash


def test_numpy_hash_equals_c_twin():
    L = ctypes.CDLL(build_host_lib())
    L.rg_hash_host.argtypes = [ctypes.c_uint64] * 4
    L.rg_hash_host.restype = ctypes.c_uint64
    for seed, s, a, b in [(1, 1, 0, 0), (140972083, 4, 199, 2), (2 ** 63 + 5, 3, 2 ** 40, 17)]:
        assert int(_hash.rg_hash(seed, s, a, b)) == L.rg_hash_host(seed, s, a, b)


def test_host_reads_are_deterministic_and_chunk_independent():
    g = ReadGenerator(get_config(1))
    a, oa = g.host(0, 500)
    b1, _ = g.host(0, 123)
    b2, _ = g.host(123, 500)
    assert np.array_equal(a, np.concatenate([b1, b2]))
    assert set(np.unique(a).tolist()) <= set(b"ACGT")
    assert list(oa[:3]) == [0, 100, 200] and oa[-1] == 500 * 100


def test_shape_of_config1():
    w = get_config(1)
    assert (w.n_reads, w.read_len, w.k, w.d, w.n_raw_edges) == (30000, 100, 21, 2, 4_740_000)
    g = ReadGenerator(w)
    a, _ = g.host(0, 4000)
    f = np.bincount(a, minlength=256)[[65, 67, 71, 84]] / a.size
    assert np.all(np.abs(f - 0.25) < 0.02)


def test_tables_of_metagenome_configs():
    for i, n in ((3, 200), (5, 50000)):
        w = get_config(i)
        glen, cdf = w.tables()
        assert len(glen) == n and np.all(np.diff(cdf.astype(np.float64)) >= 0) and int(cdf[-1]) == 2 ** 64 - 1
        assert int(glen.min()) > w.read_len
    glen, _ = get_config(3).tables()
    assert 1_000_000 <= int(glen.min()) and int(glen.max()) <= 5_000_000
    assert get_config(3).tables()[0].tobytes() == get_config(4).tables()[0].tobytes()   # cfg 4 = same read set
    assert get_config(2).n_raw_edges == 396_666_746


def test_error_rate_close_to_nominal():
    # two reads of the same genome position differ only by substitutions; estimate by regenerating with eps=0
    from dataclasses import replace
    w = get_config(2, scale=0.002)
    a, _ = ReadGenerator(w).host(0, 2000)
    b, _ = ReadGenerator(replace(w, err_rate=0.0)).host(0, 2000)
    rate = float((a != b).mean())
    assert 0.007 < rate < 0.013


@pytest.mark.gpu
def test_device_twin_equals_host_twin():
    for i, n in ((1, 3000), (3, 2000), (5, 2000)):
        g = ReadGenerator(get_config(i))
        h, oh = g.host(100, 100 + n)
        d, od = g.device(100, 100 + n)
        assert np.array_equal(h, d.cpu().numpy())
        assert np.array_equal(oh.astype(np.int64), od.cpu().numpy())
