"""Generator: frozen bytes (golden checksums), thread-count independence, the structural rules of SURVEY §8(d)."""
import json
import os
import sys

import numpy as np

from paper_2606_24647_b200 import datagen

HERE = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, os.path.join(HERE, "golden"))


def test_frozen_checksums():
    import make_generator_checksums as m
    with open(os.path.join(HERE, "golden", "generator_checksums.json")) as f:
        assert json.load(f) == json.loads(json.dumps(m.snapshot()))


def test_thread_count_independent():
    L = datagen.lib()
    n = 300_000
    a, b = np.empty(n, np.int64), np.empty(n, np.int64)
    L.gqgen_uniform_i64(5, 3, 90000, 10500000, n, a.ctypes.data, 1)
    L.gqgen_uniform_i64(5, 3, 90000, 10500000, n, b.ctypes.data, 7)
    assert np.array_equal(a, b) and a.min() >= 90000 and a.max() <= 10500000
    L.gqgen_zipf_keys(5, 4, 1000, n, a.ctypes.data, 1)
    L.gqgen_zipf_keys(5, 4, 1000, n, b.ctypes.data, 5)
    assert np.array_equal(a, b)


def test_fanout_rule_s15():
    t = datagen.make_config(3, scale=0.002)
    key, fk = t["dim"]["key"], t["fact"]["fk"]
    assert sorted(key.tolist()) == list(range(1, len(key) + 1))          # permutation of 1..n
    u, c = np.unique(fk, return_counts=True)
    assert len(u) == len(key) and c.min() >= 1 and c.max() <= 7 and c.sum() == len(fk) == 4 * len(key)
    tc = datagen.make_config(3, scale=0.002, clustered=True)
    assert np.array_equal(np.sort(fk), np.sort(tc["fact"]["fk"]))        # same multiset, different order
    assert np.all(np.diff(np.unique(tc["fact"]["fk"], return_index=True)[1]) != 0)


def test_zipf_rule_s16():
    n, N = 400_000, 5000
    k = datagen.zipf_keys(11, 15, N, n)
    assert k.min() >= 1 and k.max() <= N
    H = (1.0 / np.arange(1, N + 1)).sum()
    top_key = 1 + (0 * 2654435761) % N                                   # rank 1 -> key 1
    p = 1.0 / H
    assert abs((k == top_key).mean() - p) < 5 * (p * (1 - p) / n) ** 0.5
    r2 = 1 + (1 * 2654435761) % N
    assert abs((k == r2).mean() - p / 2) < 5 * (p / 2 / n) ** 0.5


def test_value_ranges():
    f = datagen.make_config(1, scale=0.1)["fact"]
    rng = dict(shipdate=(0, 2525), quantity=(1, 50), price=(90000, 10500000), discount=(0, 10), tax=(0, 8),
               flagA=(0, 2), flagB=(0, 1))
    for c, (lo, hi) in rng.items():
        assert lo <= f[c].min() and f[c].max() <= hi
        if hi - lo < 3000:
            assert f[c].min() == lo and f[c].max() == hi
    assert f["shipdate"].dtype == np.int32 and f["flagA"].dtype == np.int8 and f["price"].dtype == np.int64
