"""Parity of the CUDA path against the CPU oracle, element by element, through the C ABI (-m gpu).

Integer outputs are compared bit-exact after sorting by key; AVG doubles at 1e-12 relative (north_star)."""
import os

import numpy as np
import pytest

import oracle
import plans
from golden_util import load, table
from paper_2606_24647_b200 import datagen

pytestmark = pytest.mark.gpu
G = load()


@pytest.fixture(scope="module")
def gqm():
    from paper_2606_24647_b200 import build as gqbuild
    gqbuild.build()
    from paper_2606_24647_b200 import gq
    return gq


@pytest.fixture(scope="module")
def ctx(gqm):
    return gqm.Context()


def check(plan, ctx, avgs=(), out_capacity=None):
    import gqrun
    exp = oracle.run_query(plan)
    got = gqrun.run_query(plan, ctx=ctx, avgs=avgs, out_capacity=out_capacity)
    assert got["n"] == exp.nrows
    assert len(got["cols"]) == len(exp.cols)
    for c, (g, e) in enumerate(zip(got["cols"], exp.cols)):
        assert np.array_equal(g, e), f"column {c} differs"
    return exp, got


# ------------------------------------------------------------------ worked examples through the GPU
def test_golden_T1_to_T5(ctx):
    t = table(G["T1"]["cols"], G["T1"]["rows"])
    f = dict(shipdate=t["shipdate"], quantity=t["qty"], price=t["price"], discount=t["disc"], tax=t["tax"],
             flagA=t["flagA"], flagB=t["flagB"])
    exp, got = check(plans.plan_c1({"fact": f}), ctx, avgs=[(0, 4), (1, 4)])
    assert [list(map(int, r)) for r in zip(*got["cols"])] == G["T1"]["expect"]
    assert list(got["avgs"][0]) == G["T1"]["expect_avg_qty"] and list(got["avgs"][1]) == G["T1"]["expect_avg_price"]
    t = table(G["T2"]["cols"], G["T2"]["rows"])
    f = dict(shipdate=t["shipdate"], discount=t["disc"], quantity=t["qty"], price=t["price"])
    exp, got = check(plans.plan_c2({"fact": f}), ctx)
    assert [int(c[0]) for c in got["cols"]] == G["T2"]["expect"][0]
    d, f = table(G["T3"]["dim_cols"], G["T3"]["dim"]), table(G["T3"]["fact_cols"], G["T3"]["fact"])
    t3 = {"dim": d, "fact": dict(fk=f["fk"], shipdate=f["shipdate"], price=f["price"], discount=f["disc"])}
    check(plans.plan_c3(t3), ctx)
    exp, got = check(plans.plan_c3(t3, topk=10), ctx)
    assert [list(map(int, r)) for r in zip(*got["cols"])] == G["T3"]["expect_topk"]
    c, o, f = (table(G["T4"][k + "_cols"], G["T4"][k]) for k in ("cust", "orders", "fact"))
    t4 = {"cust": c, "orders": o, "fact": dict(fk=f["fk"], shipdate=f["shipdate"], price=f["price"], discount=f["disc"])}
    exp, got = check(plans.plan_c4(t4), ctx)
    assert [list(map(int, r)) for r in zip(*got["cols"])] == G["T4"]["expect"]
    t = table(G["T5"]["cols"], G["T5"]["rows"])
    f = dict(key=t["key"], shipdate=t["shipdate"], price=t["price"], quantity=t["qty"])
    exp, got = check(plans.plan_c5({"fact": f}), ctx)          # INT64_MIN / INT64_MAX / -1 / 0 keys (S14)
    assert [list(map(int, r)) for r in zip(*got["cols"])] == G["T5"]["expect"]


def _rows(cols):
    return [list(map(int, r)) for r in zip(*cols)]


def test_golden_T6_topk_ties(ctx):
    # S11 ties through every top-k route: direct (slot-indexed) state, hashed state, packed two-key state (signed
    # second key), and a low-cardinality state finished with top-k
    import gqrun
    from test_oracle_pins import t6_plans
    t, pair = t6_plans()
    for k in (3, 4, 10):
        exp, got = check(plans.plan_c3(t, topk=k), ctx, out_capacity=k)
        assert _rows(got["cols"]) == G["T6"][f"expect_top{k}"]
    plan = plans.plan_c3(t)
    tables = gqrun.build_tables(ctx, plan)
    st = ctx.aggregate(None, gqrun.dev(plan["table"]), preds=plan["preds"], probes=[(tables[0], 0)], exprs=plan["exprs"],
                       keys=plan["keys"], aggs=plan["aggs"], max_groups=100)          # hashed route (table-agnostic workspace)
    r = ctx.aggregate_finish(st, capacity=3, topk=3, topk_agg=0)
    ctx.sync()
    assert int(r["n"].item()) == 3
    assert _rows([r["keys"][0].cpu().numpy()] + [a.cpu().numpy() for a in r["aggs"]])[:3] == G["T6"]["expect_top3"]
    for k in (3, 5):
        for mg in (5000, 6):
            exp, got = check(dict(pair(k), max_groups=mg), ctx, out_capacity=k)
            assert _rows(got["cols"]) == G["T6"][f"expect_pair_top{k}"]


def test_golden_T7_wrapping_sums(ctx):
    # S6: running sums wrap modulo 2^64 on every aggregation route (RED.ADD at L2, thread-private cells, registers)
    from test_oracle_pins import t7_plan
    rows = G["T7"]["rows"]
    for mg in (5000, 4):                                          # high-cardinality table / low-cardinality fused finaliser
        exp, got = check(t7_plan(rows, max_groups=mg), ctx)
        assert _rows(got["cols"]) == G["T7"]["expect"] and exp.overflow
    exp, got = check(t7_plan(rows, keys=()), ctx)                 # key-less: registers -> shuffle -> last-CTA merge
    assert _rows(got["cols"]) == G["T7"]["expect_global"]
    t = table(G["T7"]["cols"], rows)                              # direct aggregation: group key = key of a unique probe
    dim = dict(table=[np.array([4, 2, 1, 3, 9], np.int64)], preds=[], probes=[], key=0, payload=[], unique=True)
    plan = dict(builds=[dim], table=[t["key"], t["v"]], preds=[], probes=[(0, 0)], exprs=[[("col", 1)]], keys=[0],
                aggs=[("sum", 0), ("min", 0), ("max", 0), ("count",)], max_groups=5)
    exp, got = check(plan, ctx)
    assert _rows(got["cols"]) == G["T7"]["expect"]
    # many rows: 2^20 + 3 rows of 2^62 on one key wrap the sum 2^18 times; hot-key / warp-level paths included
    n = (1 << 22) + 3
    k = np.where(np.arange(n) % 4 == 0, 1, np.arange(n) % 1000 + 2).astype(np.int64)
    v = np.where(k == 1, 1 << 62, 3).astype(np.int64)
    for mg in (2000, 0):
        plan = dict(table=[k, v], preds=[], exprs=[[("col", 1)]], keys=[0] if mg else [], aggs=[("sum", 0), ("count",)],
                    max_groups=max(mg, 1))
        exp, got = check(plan, ctx)
        assert exp.overflow


# ------------------------------------------------------------------ configs at sizes spanning many tiles + ragged tail
@pytest.mark.parametrize("cfg,scale", [(1, 1.0), (1, 0.0371), (2, 0.0333333), (3, 0.02), (4, 0.02), (5, 0.003), (5, 0.0101)])
def test_config_small(ctx, cfg, scale):
    t = datagen.make_config(cfg, scale=scale)
    plan = plans.PLANS[cfg](t)
    avgs = [(0, 4), (1, 4)] if cfg == 1 else ()
    exp, got = check(plan, ctx, avgs=avgs)
    if cfg == 1:
        for j, s in enumerate((2, 3)):
            want = np.array([oracle.avg(int(a), int(b)) for a, b in zip(exp.cols[s], exp.cols[6])])
            assert np.allclose(got["avgs"][j], want, rtol=1e-12, atol=0) and np.array_equal(got["avgs"][j], want)
    if cfg == 3:
        check(plans.plan_c3(t, topk=10), ctx)
        assert int(got["cols"][2].sum()) == exp.input_rows      # join cardinality = sum of COUNT (I2)


def test_clustered_fact_variant(ctx):
    a = datagen.make_config(3, scale=0.01)
    b = datagen.make_config(3, scale=0.01, clustered=True)
    # same fk multiset in a different row order (the other fact columns are drawn by row index, so the two results
    # differ from each other; each must equal the oracle's on its own table)
    check(plans.plan_c3(a), ctx)
    check(plans.plan_c3(b), ctx)


# ------------------------------------------------------------------ standalone operators
def _sorted_rows(cols):
    a = np.stack(cols, axis=1) if len(cols[0]) else np.zeros((0, len(cols)), np.int64)
    return a[np.lexsort(a.T[::-1])] if len(a) else a


@pytest.mark.parametrize("n", [0, 1, 15, 16, 17, 511, 512, 513, 2047, 2048, 2049, 100_003, 1_300_021])
def test_filter_project_sizes(ctx, n):
    import gqrun
    rng = np.random.default_rng(n + 1)
    a = rng.integers(-100, 100, n).astype(np.int8)
    b = rng.integers(0, 2526, n).astype(np.int32)
    c = rng.integers(-2**40, 2**40, n).astype(np.int64)
    preds = [(1, "range_co", 300, 2000), (0, "ne", 3)]
    exprs = [[("col", 2), ("col", 0), ("mul",), ("col", 1), ("add",)], [("col", 1)], [("const", 7), ("col", 2), ("sub",)]]
    exp = oracle.filter_project([a, b, c], preds, exprs)
    outs, count = ctx.filter_project(gqrun.dev([a, b, c]), preds, exprs)
    ctx.sync()
    k = int(count.item())
    assert k == exp.nrows
    got = [o[:k].cpu().numpy() for o in outs]
    assert np.array_equal(_sorted_rows(got), _sorted_rows(exp.cols))


@pytest.mark.parametrize("unique", [False, True])
def test_hash_build_probe_materialising_join(ctx, unique):
    import gqrun
    rng = np.random.default_rng(5 + unique)
    nb, npr = 70_001, 300_007
    bkey = (rng.permutation(200_000)[:nb] if unique else rng.integers(0, 30_000, nb)).astype(np.int64)
    bval = rng.integers(0, 2406, nb).astype(np.int32)
    bpay = rng.integers(-2**50, 2**50, nb).astype(np.int64)
    pkey = rng.integers(-500, 210_000 if unique else 31_000, npr).astype(np.int64)     # dangling fks too (S4)
    pval = rng.integers(0, 2526, npr).astype(np.int32)
    pairs = oracle.join_pairs([bkey, bval], [(1, "lt", 1200)], 0, [pkey, pval], [(1, "gt", 1200)], 0)
    want = [pkey[pairs.cols[0]], pval[pairs.cols[0]].astype(np.int64) * 3 + bval[pairs.cols[1]], bpay[pairs.cols[1]]]
    tb = ctx.hash_build(gqrun.dev([bkey, bval, bpay]), preds=[(1, "lt", 1200)], key=0, payload=[1, 2], unique=unique)
    exprs = [[("col", 0)], [("col", 1), ("const", 3), ("mul",), ("col", 2), ("add",)], [("col", 3)]]
    outs, count = ctx.hash_probe(gqrun.dev([pkey, pval]), [(1, "gt", 1200)], [(tb, 0)], exprs, capacity=pairs.nrows + 10)
    cnt = ctx.table_count(tb)
    ctx.sync()
    assert int(cnt.item()) == int((bval < 1200).sum())
    k = int(count.item())
    assert k == pairs.nrows > 0
    assert np.array_equal(_sorted_rows([o[:k].cpu().numpy() for o in outs]), _sorted_rows(want))


def test_join_sentinel_and_extreme_keys(ctx):
    import gqrun
    I = np.iinfo(np.int64)
    bkey = np.array([I.min, I.min, I.max, -1, 0, 5, 5], dtype=np.int64)
    bpay = np.arange(7, dtype=np.int64) * 10
    pkey = np.array([I.min, 0, 5, 7, I.max, -1, I.min], dtype=np.int64)
    pid = np.arange(7, dtype=np.int64)
    pairs = oracle.join_pairs([bkey, bpay], [], 0, [pkey, pid], [], 0)
    bf = oracle.join_pairs([bkey, bpay], [], 0, [pkey, pid], [], 0, bruteforce=True)
    assert pairs.nrows == bf.nrows == 2 * 2 + 1 + 2 + 1 + 1
    tb = ctx.hash_build(gqrun.dev([bkey, bpay]), key=0, payload=[1])
    outs, count = ctx.hash_probe(gqrun.dev([pkey, pid]), [], [(tb, 0)], [[("col", 1)], [("col", 2)]], capacity=64)
    ctx.sync()
    k = int(count.item())
    assert k == pairs.nrows
    assert np.array_equal(_sorted_rows([o[:k].cpu().numpy() for o in outs]),
                          _sorted_rows([pid[pairs.cols[0]], bpay[pairs.cols[1]]]))


# ------------------------------------------------------------------ streaming of batches (S18)
@pytest.mark.parametrize("k", [1, 2, 7, 64])
def test_streaming_batches_invariance(ctx, k):
    import gqrun
    t = datagen.make_config(5, scale=0.001)
    plan = plans.plan_c5(t)
    exp = oracle.run_query(plan)
    cols = gqrun.dev(plan["table"])
    n = len(plan["table"][0])
    cuts = sorted(set([0, n] + [int(x) // 16 * 16 for x in np.linspace(0, n, k + 1)[1:-1]]))   # 16-row cuts keep 16 B alignment
    st = None
    for lo, hi in zip(cuts[:-1], cuts[1:]):
        st = ctx.aggregate(st, [c[lo:hi] for c in cols], preds=plan["preds"], exprs=plan["exprs"], keys=plan["keys"],
                           aggs=plan["aggs"], max_groups=plan["max_groups"])
    r = ctx.aggregate_finish(st, capacity=exp.nrows + 5)
    ctx.sync()
    ng = int(r["n"].item())
    assert ng == exp.nrows
    got = gqrun.sort_rows([r["keys"][0][:ng].cpu().numpy()] + [a[:ng].cpu().numpy() for a in r["aggs"]], 1)
    for g, e in zip(got, exp.cols):
        assert np.array_equal(g, e)


def test_build_streaming_batches(ctx):
    import gqrun
    t = datagen.make_config(3, scale=0.01)
    plan = plans.plan_c3(t)
    exp = oracle.run_query(plan)
    b = plan["builds"][0]
    cols = gqrun.dev(b["table"])
    n = len(b["table"][0]); h = n // 32 * 16
    tb = ctx.hash_build([c[:h] for c in cols], preds=b["preds"], key=0, unique=True, max_rows=n, finish=False)
    tb = ctx.hash_build([c[h:] for c in cols], preds=b["preds"], key=0, unique=True, table=tb, finish=True)
    p = gqrun.prepare(ctx, plan, [tb])
    p.run(); ctx.sync()
    r = p.result()
    got = gqrun.sort_rows([r["keys"][0].cpu().numpy()] + [a.cpu().numpy() for a in r["aggs"]], 1)
    for g, e in zip(got, exp.cols):
        assert np.array_equal(g, e)


# ------------------------------------------------------------------ adversarial aggregation inputs
def test_all_same_key_and_all_distinct(ctx):
    n = 200_003
    v = np.arange(n, dtype=np.int64) - 1000
    for keys in (np.full(n, 77, np.int64), np.arange(n, dtype=np.int64) * 2654435761 % (1 << 40)):
        for mg in (n, 4):         # high-card table path and (when it fits) the low-card shared-memory path
            if mg == 4 and len(np.unique(keys)) > 4:
                continue
            plan = dict(table=[keys, v], preds=[], exprs=[[("col", 1)]], keys=[0],
                        aggs=[("sum", 0), ("min", 0), ("max", 0), ("count",)], max_groups=mg)
            check(plan, ctx)


def test_two_packed_keys_i32_i8_and_negative_values(ctx):
    rng = np.random.default_rng(3)
    n = 150_001
    k0 = rng.integers(-3, 4, n).astype(np.int32)
    k1 = rng.integers(-2, 3, n).astype(np.int8)
    v = rng.integers(-10**12, 10**12, n).astype(np.int64)
    for mg in (35, 5000):
        plan = dict(table=[k0, k1, v], preds=[], exprs=[[("col", 2)]], keys=[0, 1],
                    aggs=[("sum", 0), ("min", 0), ("max", 0), ("count",)], max_groups=mg)
        check(plan, ctx)


def test_colliding_keys_and_full_load(ctx):
    # keys that collide under Fibonacci hashing of the folded key: equal low 32 bits after folding => same bucket run
    n = 3000
    base = np.arange(n, dtype=np.int64)
    keys = (base << 32) ^ base            # x ^ (x >> 32) == base<<32: tiny products' top bits cluster
    v = np.ones(n, np.int64)
    plan = dict(table=[keys, v], preds=[], exprs=[[("col", 1)]], keys=[0], aggs=[("sum", 0), ("count",)], max_groups=n)
    check(plan, ctx)
    # table at its maximum permitted load: capacity 4096 slots, 3072 = 0.75 * 4096 groups
    keys = np.random.default_rng(1).permutation(1 << 20)[:3072].astype(np.int64)
    plan = dict(table=[keys, np.ones(3072, np.int64)], preds=[], exprs=[[("col", 1)]], keys=[0],
                aggs=[("sum", 0)], max_groups=3072)
    check(plan, ctx)


def test_hot_key_path_negative_values_and_filtered_hot_keys(ctx):
    # >= 2^22 rows switches the heavy-hitter pass on: skewed keys, negative values (carry logic of the split 32-bit
    # shared-memory adds), MIN/MAX, and one hot key whose rows are ALL filtered out (it must not appear as a group)
    rng = np.random.default_rng(11)
    n = (1 << 22) + 12_345
    hot = np.array([7, -3, 2**40 + 1, 123456789, 99], dtype=np.int64)
    keys = np.where(rng.random(n) < 0.6, hot[rng.integers(0, 5, n)], rng.integers(0, 3_000_000, n)).astype(np.int64)
    v = rng.integers(-2**45, 2**45, n).astype(np.int64)
    f = rng.integers(0, 100, n).astype(np.int32)
    f[keys == 99] = 1000                                          # hot key 99 never passes the filter
    plan = dict(table=[keys, v, f], preds=[(2, "lt", 90)], exprs=[[("col", 1)]], keys=[0],
                aggs=[("sum", 0), ("min", 0), ("max", 0), ("count",)], max_groups=3_100_000)
    exp, got = check(plan, ctx)
    assert 99 not in set(got["cols"][0].tolist()) and 7 in set(got["cols"][0].tolist())


def test_empty_and_filtered_out_inputs(ctx):
    t = datagen.make_config(2, scale=0.0005)
    plan = plans.plan_c2(t)
    plan["preds"] = [(0, "lt", -5)]
    exp, got = check(plan, ctx)                                   # global group present with (0, 0)  (S9)
    assert [int(c[0]) for c in got["cols"]] == [0, 0]
    t5 = datagen.make_config(5, scale=0.0001)
    plan = plans.plan_c5(t5)
    plan["preds"] = [(1, "lt", -5)]
    exp, got = check(plan, ctx)
    assert got["n"] == 0


# ------------------------------------------------------------------ error model (gq.h "Errors")
def test_capacity_and_duplicate_errors_are_sticky_and_clearable(gqm):
    import gqrun
    ctx = gqm.Context()
    keys = np.arange(5000, dtype=np.int64)
    plan = dict(table=[keys, keys], preds=[], exprs=[[("col", 1)]], keys=[0], aggs=[("sum", 0)], max_groups=100)
    p = gqrun.prepare(ctx, plan, [], out_capacity=5000)
    p.run()
    with pytest.raises(gqm.GqError) as e:
        ctx.sync()
    assert e.value.status == 3                                   # GQ_ERR_CAPACITY: never a silent partial result
    with pytest.raises(gqm.GqError):
        ctx.sync()                                               # sticky
    ctx.clear_error(); ctx.sync()
    dup = np.array([1, 2, 3, 2], dtype=np.int64)
    ctx.hash_build(gqrun.dev([dup]), key=0, unique=True)
    with pytest.raises(gqm.GqError) as e:
        ctx.sync()
    assert e.value.status == 6                                   # GQ_ERR_DUPLICATE_KEY: the flag is verified, not trusted
    ctx.clear_error(); ctx.sync()
    # output capacity too small
    plan = dict(table=[keys, keys], preds=[], exprs=[[("col", 1)]], keys=[0], aggs=[("sum", 0)], max_groups=5000)
    p = gqrun.prepare(ctx, plan, [], out_capacity=10)
    p.run()
    with pytest.raises(gqm.GqError):
        ctx.sync()
    ctx.clear_error(); ctx.sync()
    with pytest.raises(gqm.GqError):                             # host-detectable: misaligned column pointer
        ctx.filter_project([gqrun.dev([np.arange(64, dtype=np.int64)])[0][1:]], [], [[("col", 0)]])


def test_two_contexts_two_streams(gqm):
    import torch
    import gqrun
    t = datagen.make_config(3, scale=0.01)
    plan = plans.plan_c3(t)
    exp = oracle.run_query(plan)
    s1, s2 = torch.cuda.Stream(), torch.cuda.Stream()
    c1, c2 = gqm.Context(stream=s1), gqm.Context(stream=s2)
    torch.cuda.synchronize()
    tabs = gqrun.build_tables(c1, plan)                          # built on stream 1 ...
    torch.cuda.synchronize()                                     # (inputs were uploaded on other streams)
    p1 = gqrun.prepare(c1, plan, tabs)
    p2 = gqrun.prepare(c2, plan, tabs)                           # ... probed on stream 2: waits on the build event
    torch.cuda.synchronize()
    p1.run(); p2.run()
    c1.sync(); c2.sync()
    for p in (p1, p2):
        r = p.result()
        got = gqrun.sort_rows([r["keys"][0].cpu().numpy()] + [a.cpu().numpy() for a in r["aggs"]], 1)
        for g, e in zip(got, exp.cols):
            assert np.array_equal(g, e)


def test_host_pipeline_matches(ctx):
    import torch
    import gqrun
    t = datagen.make_config(2, scale=0.02)
    plan = plans.plan_c2(t)
    exp = oracle.run_query(plan)
    cols = [torch.from_numpy(np.ascontiguousarray(c)).pin_memory() for c in plan["table"]]
    p = gqrun.prepare(ctx, plan, [], cols=cols)
    p.run_host(chunk_rows=100_000)
    r = p.result()
    assert r["n"] == 1 and [int(a[0]) for a in r["aggs"]] == [int(c[0]) for c in exp.cols]
