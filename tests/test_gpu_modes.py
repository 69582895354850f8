"""Aggregation modes, state merge and growth (-m gpu, PAPER.md:154 / :125-127): metamorphic tests
against the oracle's invariant I6 — aggregating the parts and merging equals aggregating the whole."""
import numpy as np
import pytest

import oracle

pytestmark = pytest.mark.gpu
I64_MIN = np.iinfo(np.int64).min


@pytest.fixture(scope="module")
def gqm():
    from paper_2606_24647_b200 import build as gqbuild
    gqbuild.build()
    from paper_2606_24647_b200 import gq
    return gq


def _finish(ctx, st, nkeys, cap):
    import gqrun
    r = ctx.aggregate_finish(st, capacity=cap)
    ctx.sync()
    n = int(r["n"].item())
    cols = [k[:n].cpu().numpy().astype(np.int64) for k in r["keys"]] + [a[:n].cpu().numpy() for a in r["aggs"]]
    return n, gqrun.sort_rows(cols, nkeys)


def _equal(exp, n, cols):
    assert n == exp.nrows
    for c, (g, e) in enumerate(zip(cols, exp.cols)):
        assert np.array_equal(g, e), f"column {c} differs"


def _data(rng, n, ngroups):
    k = rng.integers(-ngroups // 2, ngroups // 2, n).astype(np.int64) * 10007
    k[::911] = I64_MIN                                           # the reserved bit pattern (side slot)
    dep = (k % 97).astype(np.int32)
    v = rng.integers(-10**9, 10**9, n).astype(np.int64)
    w = rng.integers(0, 9, n).astype(np.int8)
    return [k, dep, v, w]


AGGS = [("sum", 0), ("min", 0), ("max", 1), ("count",), ("sum", 1)]
EXPRS = [[("col", 2)], [("col", 2), ("col", 3), ("mul",)]]


@pytest.mark.parametrize("shape", ["highcard", "highcard_dep", "lowcard", "global"])
def test_merging_the_states_of_two_streams_equals_the_whole(gqm, shape):
    import gqrun
    import torch
    rng = np.random.default_rng(61)
    n = 400_003
    cols = _data(rng, n, 30_000 if shape.startswith("highcard") else 20)
    if shape == "lowcard":
        cols[0] = (cols[3] % 5).astype(np.int64) - 2
    keys, ndep, mg = {"highcard": ([0], 0, 40_000), "highcard_dep": ([0, 1], 1, 40_000), "lowcard": ([0], 0, 8), "global": ([], 0, 1)}[shape]
    plan = dict(table=cols, preds=[(3, "lt", 8)], exprs=EXPRS, keys=keys, ndependent=ndep, aggs=AGGS, max_groups=mg)
    exp = oracle.run_query(plan)
    kw = dict(preds=plan["preds"], exprs=EXPRS, keys=keys, ndependent=ndep, aggs=AGGS, max_groups=mg)
    cut = 200_000 // 16 * 16
    c1 = gqm.Context()
    s2 = torch.cuda.Stream()
    with torch.cuda.stream(s2):
        c2 = gqm.Context(0, stream=s2)
        d2 = gqrun.dev(cols)
        st2 = c2.aggregate(None, [c[cut:] for c in d2], **kw)
        st2 = c2.aggregate(st2, [c[cut - 4096:cut] for c in d2], **kw)       # a second batch into the same state
    d1 = gqrun.dev(cols)
    st1 = c1.aggregate(None, [c[:cut - 4096] for c in d1], **kw)
    c2.sync()                                                    # pipeline boundary: the other stream's state is complete
    c1.aggregate_merge(st1, st2)
    assert int(c1.aggregate_count(st1).item()) == exp.nrows
    _equal(exp, *_finish(c1, st1, len(keys), exp.nrows + 4))
    # the source state is unchanged: it still finishes to its own part
    part = oracle.run_query(dict(plan, table=[c[cut - 4096:] for c in cols]))
    _equal(part, *_finish(c2, st2, len(keys), part.nrows + 4))
    # states of different shapes are refused
    other = c1.aggregate(None, [c[:1024] for c in d1], preds=[], exprs=EXPRS, keys=keys, ndependent=ndep, aggs=AGGS[:2], max_groups=mg)
    with pytest.raises(gqm.GqError):
        c1.aggregate_merge(st1, other)


def test_merging_direct_aggregation_states(gqm):
    import gqrun
    rng = np.random.default_rng(62)
    nb, nf = 30_000, 300_000
    bkeys = rng.permutation(4 * nb)[:nb].astype(np.int64)
    attr = rng.integers(0, 100, nb).astype(np.int32)
    fk = rng.integers(-5, 4 * nb + 5, nf).astype(np.int64)
    v = rng.integers(-5000, 5000, nf).astype(np.int64)
    for dense in (None, (0, 4 * nb - 1)):
        b = dict(table=[bkeys, attr], preds=[(1, "lt", 70)], key=0, payload=[1], unique=True)
        if dense:
            b["dense_range"] = dense
        plan = dict(builds=[b], table=[fk, v], preds=[], probes=[(0, 0)], exprs=[[("col", 1)]], keys=[0, 2], ndependent=1,
                    aggs=[("sum", 0), ("max", 0)], max_groups=nb)            # no COUNT: the hidden touch word merges too
        exp = oracle.run_query(plan)
        ctx = gqm.Context()
        tables = gqrun.build_tables(ctx, plan)
        d = gqrun.dev(plan["table"])
        kw = dict(preds=[], probes=[(tables[0], 0)], exprs=plan["exprs"], keys=plan["keys"], ndependent=1, aggs=plan["aggs"],
                  max_groups=nb, plan_aware_workspace=True)
        cut = 160_000
        sa = ctx.aggregate(None, [c[:cut] for c in d], **kw)
        sb = ctx.aggregate(None, [c[cut:] for c in d], **kw)
        ctx.aggregate_merge(sa, sb)
        assert int(ctx.aggregate_count(sa).item()) == exp.nrows
        _equal(exp, *_finish(ctx, sa, 2, exp.nrows + 4))


def test_partial_then_final_through_intermediate_rows(gqm):
    # three "workers" aggregate their shard (mode Partial = the plain output without AVG); their output rows, concatenated,
    # are aggregated again in mode Final, where COUNT sums the partial counts
    import gqrun
    import torch
    rng = np.random.default_rng(63)
    n = 300_000
    cols = _data(rng, n, 5000)
    plan = dict(table=cols, preds=[(3, "ne", 4)], exprs=EXPRS, keys=[0, 1], ndependent=1, aggs=AGGS, max_groups=6000)
    exp = oracle.run_query(plan)
    ctx = gqm.Context()
    parts = []
    for lo, hi in ((0, 99_984), (99_984, 200_000), (200_000, n)):
        got = gqrun.run_query(dict(plan, table=[c[lo:hi] for c in cols]), ctx=ctx)
        parts.append(got["cols"])
    inter = [np.concatenate([p[j] for p in parts]) for j in range(len(parts[0]))]       # key, dep, sum, min, max, count, sum2
    inter[1] = inter[1].astype(np.int32)
    fexprs = [[("col", j)] for j in range(2, 7)]
    faggs = [("sum", 0), ("min", 1), ("max", 2), ("count", 3), ("sum", 4)]
    st = ctx.aggregate(None, gqrun.dev(inter), exprs=fexprs, keys=[0, 1], ndependent=1, aggs=faggs, max_groups=6000, final_mode=True)
    _equal(exp, *_finish(ctx, st, 2, exp.nrows + 4))
    # and fused: gq_pipeline in mode Final is the same plan with the flag (here through the streaming entry point on two batches)
    st = None
    d = gqrun.dev(inter)
    half = len(inter[0]) // 2 // 16 * 16
    for sl in (slice(0, half), slice(half, None)):
        st = ctx.aggregate(st, [c[sl] for c in d], exprs=fexprs, keys=[0, 1], ndependent=1, aggs=faggs, max_groups=6000, final_mode=True)
    _equal(exp, *_finish(ctx, st, 2, exp.nrows + 4))


def test_state_growth_by_rehash(gqm):
    # a streaming group-by whose group count outgrows its table ("dynamic hash table expansion"): the planner
    # re-hashes the state into a larger table when the rows fed so far could exceed max_groups — no device round trip
    import gqrun
    rng = np.random.default_rng(64)
    n = 500_000
    cols = _data(rng, n, 120_000)
    plan = dict(table=cols, preds=[], exprs=EXPRS, keys=[0, 1], ndependent=1, aggs=AGGS, max_groups=200_000)
    exp = oracle.run_query(plan)
    ctx = gqm.Context()
    d = gqrun.dev(cols)
    kw = dict(exprs=EXPRS, keys=[0, 1], ndependent=1, aggs=AGGS)
    st, fed, cap = None, 0, 4096
    for lo in range(0, n, 50_000 - 50_000 % 16):
        hi = min(n, lo + 50_000 - 50_000 % 16)
        while st is not None and fed + (hi - lo) > cap:           # groups <= rows fed: grow before the batch that could overflow
            cap *= 8
            ctx.aggregate_rehash(st, cap)
        st = ctx.aggregate(st, [c[lo:hi] for c in d], max_groups=max(cap, hi - lo), **kw)
        if fed == 0:
            cap = max(cap, hi - lo)
        fed += hi - lo
    assert int(ctx.aggregate_count(st).item()) == exp.nrows
    _equal(exp, *_finish(ctx, st, 2, exp.nrows + 4))
    # without growth the same stream of batches overflows the table: a sticky error, never a wrong answer
    c2 = gqm.Context()
    st = None
    for lo in range(0, n, 100_000):
        st = c2.aggregate(st, [c[lo:lo + 100_000] for c in d], max_groups=4096, **kw)
    with pytest.raises(gqm.GqError) as e:
        c2.sync()
    assert e.value.status == 3
    c2.clear_error(); c2.sync()
    # low-cardinality and key-less states do not grow
    small = ctx.aggregate(None, [c[:1024] for c in d], exprs=EXPRS, keys=[], aggs=AGGS, max_groups=1)
    with pytest.raises(gqm.GqError):
        ctx.aggregate_rehash(small, 100)


def test_degenerate_inputs(gqm):
    # empty build side, one-key range, every row filtered out, empty states merged: the degenerate cases of the new paths
    import gqrun
    import torch
    from paper_2606_24647_b200 import gq
    ctx = gqm.Context()
    rng = np.random.default_rng(65)
    fk = rng.integers(-3, 4, 10_000).astype(np.int64)
    v = rng.integers(0, 100, 10_000).astype(np.int64)
    # (a) dense table whose build batch has no surviving row; range of a single key
    for bkeys, preds, rng_ in ((np.array([1, 2, 3], np.int64), [(0, "gt", 100)], (0, 5)), (np.array([2], np.int64), [], (2, 2))):
        b = dict(table=[bkeys], preds=preds, key=0, payload=[], unique=True, dense_range=rng_)
        plan = dict(builds=[b], table=[fk, v], preds=[], probes=[(0, 0)], exprs=[[("col", 1)]], keys=[0], aggs=[("sum", 0), ("count",)],
                    max_groups=8)
        exp = oracle.run_query(plan)
        got = gqrun.run_query(plan, ctx=ctx)
        assert got["n"] == exp.nrows and all(np.array_equal(g, e) for g, e in zip(got["cols"], exp.cols))
    # (b) partitioned shared-memory aggregation with every row filtered out, and with one surviving row
    try:
        gq.set_option("part_min_table_mb", 0); gq.set_option("part_min_rows", 4096); gq.set_option("hot_min_rows", 4096)
        k = rng.integers(0, 1000, 50_000).astype(np.int64)
        w = np.zeros(50_000, np.int64); w[777] = 5
        for lim in (9, 3):
            plan = dict(table=[k, w], preds=[(1, "gt", lim)], exprs=[[("col", 1)]], keys=[0], aggs=[("sum", 0), ("min", 0), ("count",)],
                        max_groups=100_000)
            exp = oracle.run_query(plan)
            got = gqrun.run_query(plan, ctx=ctx)
            assert got["n"] == exp.nrows == (0 if lim == 9 else 1)
            assert all(np.array_equal(g, e) for g, e in zip(got["cols"], exp.cols))
    finally:
        gq.set_option("part_min_table_mb", -1); gq.set_option("part_min_rows", -1); gq.set_option("hot_min_rows", -1)
    # (c) merging an empty state, into an empty state; counting an empty state
    d = gqrun.dev([fk, v])
    kw = dict(exprs=[[("col", 1)]], keys=[0], aggs=[("sum", 0), ("count",)], max_groups=1000)
    full = ctx.aggregate(None, d, **kw)
    empty = ctx.aggregate(None, [c[:0] for c in d], **kw)
    empty2 = ctx.aggregate(None, [c[:0] for c in d], **kw)
    assert int(ctx.aggregate_count(empty).item()) == 0
    ctx.aggregate_merge(full, empty)
    ctx.aggregate_merge(empty2, full)
    exp = oracle.run_query(dict(table=[fk, v], **kw))
    for st in (full, empty2):
        _equal(exp, *_finish(ctx, st, 1, 100))
    # (d) order by on a single row and on all-equal keys with limit 1
    idx, outs = ctx.order_by(gqrun.dev([np.array([7], np.int64)]), [(0, True)])
    ctx.sync()
    assert idx.cpu().tolist() == [0] and outs[0].cpu().tolist() == [7]
