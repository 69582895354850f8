"""CPU-only checks of the boundary: libgq.so loads, exports every symbol include/gq.h declares, validates arguments
that need no device, and the plan compiler emits sm_100a kernels for the five benchmark plan shapes (no GPU needed)."""
import ctypes as C
import os
import re

import pytest

from paper_2606_24647_b200 import build as gqbuild

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def gq():
    gqbuild.build()
    from paper_2606_24647_b200 import gq as m
    return m


def test_exports_every_declared_symbol(gq):
    hdr = open(os.path.join(ROOT, "include", "gq.h")).read()
    hdr = re.sub(r"/\*.*?\*/", "", hdr, flags=re.S)
    declared = sorted(set(re.findall(r"\b(gq_[a-z_0-9]+)\s*\(", hdr)))
    assert declared, "no declarations parsed"
    L = gq.lib()
    missing = [s for s in declared if not hasattr(L, s)]
    assert not missing, missing
    assert sorted(gq.SYMBOLS) == declared


def test_status_strings_and_workspace_queries(gq):
    L = gq.lib()
    assert L.gq_status_str(0) == b"GQ_OK" and L.gq_status_str(3) == b"GQ_ERR_CAPACITY"
    n = C.c_size_t()
    assert L.gq_hash_build_workspace(7_480_000, 0, C.byref(n)) == 0
    assert 7_480_000 * 8 / 0.71 <= n.value <= 7_480_000 * 8 / 0.65   # C3: key-only slots, larger than L2: load factor 0.7, no power-of-two rounding
    assert L.gq_hash_build_workspace(10, 1, C.byref(n)) == 0 and n.value >= 1024 * 16
    assert L.gq_hash_build_workspace(-1, 0, C.byref(n)) == 1
    assert L.gq_hash_build_workspace(10, 9, C.byref(n)) == 1
    assert L.gq_hash_aggregate_workspace(50_000_000, 1, 5, C.byref(n)) == 0
    assert n.value >= (1 << 26) * 48                      # C5: 2^26 slots of key + 5 aggregates
    assert L.gq_hash_aggregate_workspace(0, 1, 5, C.byref(n)) == 1
    assert L.gq_topk_scratch_bytes() > 0


def test_plan_compiler_emits_sm100_tma_kernels(gq, tmp_path):
    I8, I32, I64 = gq.I8, gq.I32, gq.I64
    col = lambda i: ("col", i)
    L = gq.lib()
    L.gq_set_kernel_cache_dir(str(tmp_path).encode())
    try:
        path = gq.precompile_pipeline([I32, I64, I64, I64], 60_000_000,
                                      preds=[(0, "range_co", 730, 1095), (1, "range_cc", 5, 7), (2, "lt", 24)],
                                      exprs=[[col(3), col(1), ("mul",)]], keys=[], aggs=[("sum", 0), ("count",)])
        assert os.path.exists(path) and os.path.exists(path.replace(".cubin", ".cu"))
        src = open(path.replace(".cubin", ".cu")).read()
        assert "cp.async.bulk.shared::cluster.global.mbarrier" in src and "gq_pass" in src
        blob = open(path, "rb").read()
        assert blob[:4] == b"\x7fELF" and b"gq_scan" in blob
        # malformed plans are rejected at plan time
        with pytest.raises(gq.GqError):
            gq.precompile_pipeline([I32], 10, exprs=[[("add",)]], aggs=[("sum", 0)])
        with pytest.raises(gq.GqError):
            gq.precompile_pipeline([I32], 10, preds=[(3, "lt", 1)], aggs=[("count",)])
        with pytest.raises(gq.GqError):   # i64 + i32 key tuple needs a declared dependent key (S17)
            gq.precompile_pipeline([I64, I32], 10, keys=[0, 1], aggs=[("count",)], max_groups=100)
        gq.precompile_pipeline([I64, I32], 10, keys=[0, 1], ndependent=1, aggs=[("count",)], max_groups=100)
    finally:
        L.gq_set_kernel_cache_dir(None)


def test_plan_compiler_covers_probes_of_duplicate_key_tables(gq):
    # one-row-at-a-time row code (a probed table may hold duplicate keys): every consumer compiles (no GPU needed)
    I8, I32, I64 = gq.I8, gq.I32, gq.I64
    col = lambda i: ("col", i)
    multi, uniq = gq.describe_table([I32], unique=False), gq.describe_table([I32], unique=True)
    ex, ag = [[col(2), col(3), ("mul",)]], [("sum", 0), ("count",)]
    for kw in (dict(keys=[], max_groups=1), dict(keys=[1], max_groups=6), dict(keys=[0], max_groups=100_000),
               dict(keys=[0, 3], ndependent=1, max_groups=100_000, check_dependent=True)):
        assert os.path.exists(gq.precompile_pipeline([I64, I8, I64], 1_000_000, probes=[(multi, 0)], exprs=ex, aggs=ag, **kw))
    # multiset step followed by a unique step whose key is the group key: hashed group-by, not direct aggregation
    assert os.path.exists(gq.precompile_pipeline([I64, I64, I64], 1_000_000, probes=[(multi, 0), (uniq, 1)], exprs=ex,
                                                 keys=[1], aggs=ag, max_groups=100_000))
    assert os.path.exists(gq.precompile_build([I64, I64], 1_000_000, probes=[(multi, 0)], key=1, payload=[2]))
    assert os.path.exists(gq.precompile_materialise([I64, I64], 1_000_000, probes=[(multi, 0)], exprs=[[col(2)], [col(1)]]))


def test_plan_compiler_covers_direct_address_tables(gq):
    # GQ_F_DENSE_KEYS tables (bitmap + payload rows indexed by key - key_min): build, probe in both row-code forms,
    # direct aggregation through the matched index; the flag needs GQ_F_UNIQUE_KEYS
    I8, I32, I64 = gq.I8, gq.I32, gq.I64
    col = lambda i: ("col", i)
    dense, multi = gq.describe_table([I32], unique=True, dense=True), gq.describe_table([I32], unique=False)
    ag = [("sum", 0), ("count",)]
    assert os.path.exists(gq.precompile_build([I64, I32], 1_000_000, preds=[(1, "lt", 5)], key=0, payload=[1], unique=True,
                                              dense_range=(1, 1_000_000)))
    assert os.path.exists(gq.precompile_build([I64, I64, I32], 1_000_000, probes=[(multi, 0)], key=1, payload=[2], unique=True,
                                              dense_range=(-5, 5)))
    for kw in (dict(keys=[], max_groups=1), dict(keys=[1], max_groups=6), dict(keys=[0], max_groups=100_000),
               dict(keys=[0, 3], ndependent=1, max_groups=100_000)):
        assert os.path.exists(gq.precompile_pipeline([I64, I8, I64], 1_000_000, probes=[(dense, 0)], exprs=[[col(2)]], aggs=ag, **kw))
    assert os.path.exists(gq.precompile_pipeline([I64, I64, I64], 1_000_000, probes=[(multi, 0), (dense, 1)], exprs=[[col(2)]],
                                                 keys=[1], aggs=ag, max_groups=100_000))
    assert os.path.exists(gq.precompile_materialise([I64, I64], 1_000_000, probes=[(dense, 0)], exprs=[[col(2)], [col(1)]]))
    with pytest.raises(gq.GqError):
        gq.precompile_build([I64], 100, key=0, unique=False, dense_range=(0, 10))
    n = C.c_size_t()
    L = gq.lib()
    assert L.gq_hash_build_workspace_dense(1, 15_000_000, 8_000_000, 1, C.byref(n)) == 0
    assert n.value >= 15_000_000 // 4 + 15_000_000 * 8 + 8_000_000 * 8
    assert L.gq_hash_build_workspace_dense(5, 4, 0, 0, C.byref(n)) == 1


def test_options(gq):
    L = gq.lib()
    assert L.gq_set_option(b"part_min_rows", 4096) == 0 and L.gq_set_option(b"part_min_rows", -1) == 0
    assert L.gq_set_option(b"no_such_option", 1) == 1 and L.gq_set_option(None, 1) == 1


def test_no_device_context_fails_loudly(gq):
    import torch
    if torch.cuda.is_available():
        pytest.skip("GPU present")
    with pytest.raises(RuntimeError):
        gq.Context()
