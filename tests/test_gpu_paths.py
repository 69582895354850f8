"""Parity of the specialised kernel paths against the CPU oracle (-m gpu): direct (slot-indexed) aggregation, the
finaliser fused into the scan kernel, low-cardinality key tables with 64-bit keys, join tables at full load."""
import numpy as np
import pytest

import oracle
import plans
from paper_2606_24647_b200 import datagen

pytestmark = pytest.mark.gpu
I64_MIN = np.iinfo(np.int64).min


@pytest.fixture(scope="module")
def ctx():
    from paper_2606_24647_b200 import build as gqbuild
    gqbuild.build()
    from paper_2606_24647_b200 import gq
    return gq.Context()


def run(plan, ctx, **kw):
    import gqrun
    exp = oracle.run_query(plan)
    got = gqrun.run_query(plan, ctx=ctx, **kw)
    assert got["n"] == exp.nrows
    for c, (g, e) in enumerate(zip(got["cols"], exp.cols)):
        assert np.array_equal(g, e), f"column {c} differs"
    return exp, got


def _join_plan(nb, nf, rng, aggs, with_dep=False, extra_keys=()):
    """dim(key unique [, attr]) JOIN fact(fk, v) GROUP BY fk [, attr]."""
    bkeys = np.concatenate([rng.permutation(4 * nb)[:nb].astype(np.int64) - nb, np.array(extra_keys, np.int64)])
    attr = rng.integers(-1000, 1000, len(bkeys)).astype(np.int32)
    bsel = rng.integers(0, 2, len(bkeys)).astype(np.int8)
    fk = rng.choice(np.concatenate([bkeys, np.array([7 * nb + 1, 7 * nb + 2], np.int64)]), nf).astype(np.int64)
    v = rng.integers(-5000, 5000, nf).astype(np.int64)
    fsel = rng.integers(0, 4, nf).astype(np.int32)
    build = dict(table=[bkeys, attr, bsel], preds=[(2, "eq", 1)], key=0, payload=[1] if with_dep else [], unique=True)
    return dict(builds=[build], table=[fk, v, fsel], preds=[(2, "lt", 3)], probes=[(0, 0)], exprs=[[("col", 1)]],
                keys=[0, 3] if with_dep else [0], ndependent=1 if with_dep else 0, aggs=aggs, max_groups=len(bkeys))


@pytest.mark.parametrize("with_dep", [False, True])
@pytest.mark.parametrize("aggs", [[("sum", 0), ("count",)], [("min", 0), ("max", 0), ("sum", 0)]])
def test_direct_aggregation_pipeline(ctx, with_dep, aggs):
    # group key = key of a unique-key probe step: the pipeline aggregates into an array indexed by the matched slot.
    # Second aggregate list has no COUNT(*): a hidden touch word marks the groups. INT64_MIN is a build key (S14).
    rng = np.random.default_rng(5)
    plan = _join_plan(20_000, 300_000, rng, aggs, with_dep, extra_keys=[I64_MIN, np.iinfo(np.int64).max])
    run(plan, ctx)


def test_direct_equals_hashed_standalone_and_streams(ctx):
    import gqrun
    rng = np.random.default_rng(6)
    plan = _join_plan(5_000, 120_000, rng, [("sum", 0), ("count",)])
    exp = oracle.run_query(plan)
    tables = gqrun.build_tables(ctx, plan)
    cols = gqrun.dev(plan["table"])
    n = len(plan["table"][0])
    for aware in (False, True):                    # hashed state vs direct state, three batches each
        st = None
        for lo, hi in ((0, 40_000), (40_000, 40_016), (40_016, n)):
            st = ctx.aggregate(st, [c[lo:hi] for c in cols], preds=plan["preds"], probes=[(tables[0], 0)],
                               exprs=plan["exprs"], keys=plan["keys"], aggs=plan["aggs"], max_groups=plan["max_groups"],
                               plan_aware_workspace=aware)
        r = ctx.aggregate_finish(st, capacity=exp.nrows + 3)
        ctx.sync()
        ng = int(r["n"].item())
        assert ng == exp.nrows
        got = gqrun.sort_rows([r["keys"][0][:ng].cpu().numpy()] + [a[:ng].cpu().numpy() for a in r["aggs"]], 1)
        for g, e in zip(got, exp.cols):
            assert np.array_equal(g, e)


def test_direct_topk(ctx):
    rng = np.random.default_rng(7)
    plan = _join_plan(3_000, 50_000, rng, [("sum", 0), ("count",)])
    plan["topk"], plan["topk_agg"] = 10, 0
    run(plan, ctx, out_capacity=10)


@pytest.mark.parametrize("k", [1, 10, 32])
def test_topk_admission_bound_ties_and_both_merge_paths(ctx, k):
    # top-k finaliser: (a) every group has the same ordering aggregate — the sampled admission bound equals that value,
    # every warp list of pass 1 fills up and the merge takes its sorted-list path, the key order decides; (b) distinct
    # values over a table far larger than the sample — few entries survive the bound, the merge ranks them by counting;
    # (c) fewer groups than k
    rng = np.random.default_rng(70 + k)
    n = 400_000
    keys = rng.permutation(1 << 21)[:n].astype(np.int64) - 5000
    ones = np.ones(n, np.int64)
    plan = dict(table=[keys, ones], preds=[], exprs=[[("col", 1)]], keys=[0], aggs=[("sum", 0), ("count",)],
                max_groups=n, topk=k, topk_agg=0)
    exp, got = run(plan, ctx, out_capacity=k)
    assert np.array_equal(got["cols"][0], np.sort(keys)[:k])
    vals = rng.integers(-10**12, 10**12, n).astype(np.int64)
    vals[rng.integers(0, n, 50)] = vals.max()                      # ties at the top
    run(dict(plan, table=[keys, vals]), ctx, out_capacity=k)
    run(dict(plan, table=[keys[:5], vals[:5]], max_groups=8), ctx, out_capacity=k)


def test_join_table_at_full_load_and_all_misses(ctx):
    rng = np.random.default_rng(8)
    nb = 50_000
    bkeys = rng.permutation(1 << 22)[:nb].astype(np.int64)
    fk = np.concatenate([bkeys, bkeys + (1 << 23)])           # second half matches nothing
    v = np.ones(len(fk), np.int64)
    build = dict(table=[bkeys], preds=[], key=0, payload=[], unique=True, max_rows=nb)   # exactly the hinted rows
    plan = dict(builds=[build], table=[fk, v], preds=[], probes=[(0, 0)], exprs=[[("col", 1)]], keys=[0],
                aggs=[("sum", 0), ("count",)], max_groups=nb)
    exp, got = run(plan, ctx)
    assert exp.nrows == nb and int(got["cols"][2].sum()) == nb


@pytest.mark.parametrize("n", [1, 255, 1024, 1025, 5000, 200_003])
def test_fused_finaliser_lowcard_sizes(ctx, n):
    # one-kernel pipeline (scan + in-kernel finaliser): tail-only inputs, one CTA, many CTAs
    plan = plans.plan_c1(datagen.make_config(1, scale=n / 1_000_000))
    exp, got = run(plan, ctx, avgs=[(0, 4), (1, 4)])
    for a, (s, c) in zip(got["avgs"], [(2, 6), (3, 6)]):
        ref = np.array([oracle.avg(int(x), int(y)) for x, y in zip(exp.cols[s], exp.cols[c])])
        assert np.allclose(a, ref, rtol=1e-12, atol=0)


def test_fused_finaliser_global_no_passing_rows_and_repeat(ctx):
    import gqrun
    plan = plans.plan_c2(datagen.make_config(2, scale=0.002))
    plan["preds"] = [(0, "lt", -5)]                           # nothing passes: one row (0, 0)   (S9)
    exp, got = run(plan, ctx)
    assert [int(c[0]) for c in got["cols"]] == [0, 0]
    plan = plans.plan_c2(datagen.make_config(2, scale=0.01))
    p = gqrun.prepare(ctx, plan, [])
    exp = oracle.run_query(plan)
    for _ in range(5):                                        # the ticket counter must return to zero every run
        p.run()
        ctx.sync()
        r = p.result()
        assert r["n"] == 1 and [int(a[0]) for a in r["aggs"]] == [int(c[0]) for c in exp.cols]


def test_lowcard_wide_keys_reserved_pattern_and_many_groups(ctx):
    rng = np.random.default_rng(9)
    n = 70_000
    pool = np.array([I64_MIN, -1, 0, 1, 1 << 40, np.iinfo(np.int64).max, 12345678901234], np.int64)
    k = pool[rng.integers(0, len(pool), n)]
    v = rng.integers(-100, 100, n).astype(np.int64)
    plan = dict(table=[k, v], preds=[(1, "ne", 3)], exprs=[[("col", 1)]], keys=[0],
                aggs=[("sum", 0), ("min", 0), ("max", 0), ("count",)], max_groups=len(pool))
    run(plan, ctx)
    # 24 groups over two packed narrow keys; also streamed in batches into a (non-fused) low-cardinality state
    a = rng.integers(-3, 3, n).astype(np.int8)
    b = rng.integers(10, 14, n).astype(np.int32)
    plan = dict(table=[a, b, v], preds=[], exprs=[[("col", 2)]], keys=[0, 1], aggs=[("sum", 0), ("count",)], max_groups=24)
    exp, _ = run(plan, ctx)
    import gqrun
    cols = gqrun.dev(plan["table"])
    st = None
    for lo, hi in ((0, 4096), (4096, 4112), (4112, n)):
        st = ctx.aggregate(st, [c[lo:hi] for c in cols], exprs=plan["exprs"], keys=plan["keys"], aggs=plan["aggs"], max_groups=24)
    r = ctx.aggregate_finish(st, capacity=30)
    ctx.sync()
    ng = int(r["n"].item())
    got = gqrun.sort_rows([kk[:ng].cpu().numpy().astype(np.int64) for kk in r["keys"]] + [x[:ng].cpu().numpy() for x in r["aggs"]], 2)
    for g, e in zip(got, exp.cols):
        assert np.array_equal(g, e)


def test_lowcard_more_groups_than_declared_is_an_error():
    from paper_2606_24647_b200 import gq
    import gqrun
    c = gq.Context()
    k = (np.arange(5000) % 9).astype(np.int8)
    plan = dict(table=[k, np.ones(5000, np.int64)], preds=[], exprs=[[("col", 1)]], keys=[0], aggs=[("sum", 0)], max_groups=6)
    p = gqrun.prepare(c, plan, [])
    p.run()
    with pytest.raises(gq.GqError) as e:
        c.sync()
    assert e.value.status == 3                                 # GQ_ERR_CAPACITY, sticky
    c.clear_error()
    plan["max_groups"] = 9
    p = gqrun.prepare(c, plan, [])
    p.run()
    c.sync()                                                   # and the ticket counter survived the failed run
    assert p.result()["n"] == 9


def test_lowcard_single_int8_key_with_negative_values(ctx):
    # {key32, gid} entries of the shared-memory key table: a sign-extended -1 must not be mistaken for an EMPTY entry
    import gqrun
    rng = np.random.default_rng(21)
    n = 90_001
    k = rng.choice(np.array([-128, -1, 0, 5, 127], np.int8), n)
    v = rng.integers(-1000, 1000, n).astype(np.int64)
    plan = dict(table=[k, v], preds=[], exprs=[[("col", 1)]], keys=[0], aggs=[("sum", 0), ("min", 0), ("max", 0), ("count",)],
                max_groups=5)
    exp, got = run(plan, ctx)                                  # fused one-kernel pipeline
    assert set(got["cols"][0].tolist()) == {-128, -1, 0, 5, 127}
    cols = gqrun.dev(plan["table"])
    st = None
    for lo, hi in ((0, 4096), (4096, n)):                      # streaming state (global table behind the shared cells)
        st = ctx.aggregate(st, [c[lo:hi] for c in cols], exprs=plan["exprs"], keys=[0], aggs=plan["aggs"], max_groups=5)
    r = ctx.aggregate_finish(st, capacity=8)
    ctx.sync()
    ng = int(r["n"].item())
    got = gqrun.sort_rows([r["keys"][0][:ng].cpu().numpy().astype(np.int64)] + [a[:ng].cpu().numpy() for a in r["aggs"]], 1)
    for g, e in zip(got, exp.cols):
        assert np.array_equal(g, e)
    # only -1 present: the one key that used to vanish
    plan = dict(table=[np.full(5000, -1, np.int8), np.ones(5000, np.int64)], preds=[], exprs=[[("col", 1)]], keys=[0],
                aggs=[("sum", 0)], max_groups=3)
    exp, got = run(plan, ctx)
    assert got["n"] == 1 and int(got["cols"][1][0]) == 5000


# ------------------------------------------------------------------ probes of tables with duplicate keys (multiset, S3)
def _multiset_plan(rng, nb, nf, keys, aggs, max_groups, ndependent=0, dup=4):
    """fact(fk, grp8, v) JOIN build(key with duplicates, attr) — every matching pair counts (inner join)."""
    bkey = rng.integers(0, nb // dup, nb).astype(np.int64) * 3 - 100          # ~dup rows per key, some keys absent
    attr = (bkey % 17).astype(np.int32)                                       # functionally dependent on the key
    bsel = rng.integers(0, 3, nb).astype(np.int8)
    fk = (rng.integers(-20, nb // dup + 20, nf).astype(np.int64)) * 3 - 100   # dangling fks too (S4)
    grp = rng.integers(-2, 3, nf).astype(np.int8)
    v = rng.integers(-10**9, 10**9, nf).astype(np.int64)
    build = dict(table=[bkey, attr, bsel], preds=[(2, "ne", 0)], probes=[], key=0, payload=[1], unique=False)
    return dict(builds=[build], table=[fk, grp, v], preds=[(2, "gt", -900_000_000)], probes=[(0, 0)],
                exprs=[[("col", 2), ("col", 3), ("mul",)], [("col", 3)]], keys=keys, ndependent=ndependent, aggs=aggs,
                max_groups=max_groups)


@pytest.mark.parametrize("consumer", ["global", "lowcard", "highcard", "highcard_dep"])
def test_fused_pipeline_over_duplicate_key_build(ctx, consumer):
    rng = np.random.default_rng(31)
    aggs = [("sum", 0), ("min", 1), ("max", 0), ("count",)]
    keys, mg, ndep = {"global": ([], 1, 0), "lowcard": ([1], 5, 0), "highcard": ([0], 30_000, 0),
                      "highcard_dep": ([0, 3], 30_000, 1)}[consumer]
    plan = _multiset_plan(rng, 40_000, 250_003, keys, aggs, mg, ndep)
    exp, got = run(plan, ctx)
    assert exp.input_rows > 250_003                              # rows really fan out
    assert int(got["cols"][-1].sum()) == exp.input_rows          # I2: join cardinality


def test_fused_pipeline_over_duplicate_key_build_large_and_chained(ctx):
    import gqrun
    rng = np.random.default_rng(32)
    # >= 2^22 fact rows: the size at which unique-probe plans switch the heavy-hitter pass on (it must stay off here)
    plan = _multiset_plan(rng, 60_000, (1 << 22) + 777, [0], [("sum", 0), ("count",)], 40_000, dup=3)
    exp, got = run(plan, ctx)
    assert int(got["cols"][-1].sum()) == exp.input_rows
    # chained join THROUGH a multiset table: orders-like build probes the duplicate-key table, fact probes the result
    nb = 20_000
    ckey = rng.integers(0, 3000, nb).astype(np.int64)                          # duplicates
    cval = rng.integers(0, 5, nb).astype(np.int8)
    okey = rng.permutation(50_000).astype(np.int64)
    ocust = rng.integers(-10, 3100, 50_000).astype(np.int64)
    fk = rng.integers(0, 52_000, 300_001).astype(np.int64)
    v = rng.integers(0, 10**6, 300_001).astype(np.int64)
    b0 = dict(table=[ckey, cval], preds=[(1, "lt", 2)], probes=[], key=0, payload=[1], unique=False)
    b1 = dict(table=[okey, ocust], preds=[], probes=[(0, 1)], key=0, payload=[2], unique=False,   # fans out: NOT unique,
              max_rows=400_000)                                     # and more rows are inserted than the batch has
    plan = dict(builds=[b0, b1], table=[fk, v], preds=[], probes=[(1, 0)], exprs=[[("col", 1), ("col", 2), ("add",)]],
                keys=[0], aggs=[("sum", 0), ("count",)], max_groups=60_000)
    exp, got = run(plan, ctx)
    assert exp.input_rows > 0 and int(got["cols"][-1].sum()) == exp.input_rows
    # and a unique dimension joined after the multiset step, grouped by the dimension's key (no direct aggregation here)
    dkey = np.arange(-2, 3, dtype=np.int64)
    plan = _multiset_plan(rng, 30_000, 200_000, [1], [("sum", 0), ("count",)], 10_000)
    plan["builds"].append(dict(table=[dkey], preds=[], probes=[], key=0, payload=[], unique=True))
    plan["probes"].append((1, 1))
    run(plan, ctx)


# ------------------------------------------------------------------ direct-address (dense-key) join tables
def _with_dense(plan, ranges):
    import copy
    q = copy.copy(plan)
    q["builds"] = [dict(b, dense_range=r) if r is not None else b for b, r in zip(plan["builds"], ranges)]
    return q


@pytest.mark.parametrize("cfg", [3, 4])
def test_direct_address_tables_config_shapes(ctx, cfg):
    # C3 / C4 with the planner's column statistics (min/max of the build keys) declared: bitmap membership, payload rows
    # and the direct aggregation indexed by key - key_min; the hashed route on the same plan must agree (both == oracle)
    t = datagen.make_config(cfg, scale=0.01)
    plan = plans.PLANS[cfg](t)
    dense = _with_dense(plan, [(int(b["table"][b["key"]].min()), int(b["table"][b["key"]].max())) for b in plan["builds"]])
    run(dense, ctx)
    run(plan, ctx)
    if cfg == 3:
        top = dict(dense, topk=10, topk_agg=0)
        exp, got = run(top, ctx)
        assert got["n"] == 10


def test_direct_address_tables_adversarial(ctx):
    import gqrun
    from paper_2606_24647_b200 import gq
    rng = np.random.default_rng(51)
    # keys around zero incl. negatives, range much wider than the rows present, probes far outside the range (wrap-around of
    # key - key_min), payload that is the dependent group key, a ragged fact tail
    nb, nf = 20_001, 300_007
    bkeys = (rng.permutation(60_000)[:nb].astype(np.int64) - 30_000)
    attr = rng.integers(-1000, 1000, nb).astype(np.int32)
    bsel = rng.integers(0, 2, nb).astype(np.int8)
    fk = rng.integers(-40_000, 40_000, nf).astype(np.int64)
    fk[::97] = I64_MIN; fk[1::97] = np.iinfo(np.int64).max
    v = rng.integers(-5000, 5000, nf).astype(np.int64)
    b = dict(table=[bkeys, attr, bsel], preds=[(2, "eq", 1)], key=0, payload=[1], unique=True, dense_range=(-30_000, 29_999))
    for keys, ndep, mg in (([0, 2], 1, nb), ([0], 0, nb), ([], 0, 1), ([2], 0, 2100)):
        plan = dict(builds=[b], table=[fk, v], preds=[], probes=[(0, 0)], exprs=[[("col", 1)], [("col", 1), ("col", 2), ("mul",)]],
                    keys=keys, ndependent=ndep, aggs=[("sum", 0), ("min", 1), ("max", 0), ("count",)], max_groups=mg)
        exp, got = run(plan, ctx)
        assert exp.nrows > 0
    # materialising probe (inner join as output columns) through a dense table
    tb = ctx.hash_build(gqrun.dev(b["table"]), preds=b["preds"], key=0, payload=[1], unique=True, dense_range=b["dense_range"])
    assert int(ctx.table_count(tb).item()) == int((bsel == 1).sum())
    outs, count = ctx.hash_probe(gqrun.dev([fk, v]), [], [(tb, 0)], [[("col", 0)], [("col", 2)], [("col", 1)]], capacity=nf)
    ctx.sync()
    n = int(count.item())
    got = np.stack([o[:n].cpu().numpy() for o in outs], 1)
    pairs = oracle.join_pairs([bkeys, attr, bsel], [(2, "eq", 1)], 0, [fk, v], [], 0)
    ref = np.stack([fk[pairs.cols[0]], attr[pairs.cols[1]].astype(np.int64), v[pairs.cols[0]]], 1)
    assert n == pairs.nrows > 0 and np.array_equal(got[np.lexsort(got.T[::-1])], ref[np.lexsort(ref.T[::-1])])
    # streaming batches into one dense table; a multiset step in front of a dense step (one-row-at-a-time row code)
    h = gqrun.dev(b["table"])
    tb2 = ctx.hash_build([c[:7008] for c in h], preds=b["preds"], key=0, payload=[1], unique=True, dense_range=b["dense_range"], finish=False,
                         max_rows=nb)                              # the row bound covers ALL batches (default: this batch's rows)
    ctx.hash_build([c[7008:] for c in h], preds=b["preds"], key=0, payload=[1], unique=True, dense_range=b["dense_range"], table=tb2)
    assert int(ctx.table_count(tb2).item()) == int((bsel == 1).sum())
    mkey = rng.integers(0, 300, 5000).astype(np.int64)
    mval = rng.integers(-30_000, 30_000, 5000).astype(np.int64)
    f2 = rng.integers(0, 320, 50_000).astype(np.int64)
    plan = dict(builds=[dict(table=[mkey, mval], preds=[], key=0, payload=[1], unique=False), b], table=[f2, v[:50_000]], preds=[],
                probes=[(0, 0), (1, 2)], exprs=[[("col", 1), ("col", 3), ("add",)]], keys=[2], aggs=[("sum", 0), ("count",)], max_groups=nb)
    run(plan, ctx)
    # the declarations are verified on the device: a key outside the range, a repeated key
    c2 = gq.Context()
    c2.hash_build(gqrun.dev([bkeys]), key=0, unique=True, dense_range=(-30_000, 20_000))
    with pytest.raises(gq.GqError) as e:
        c2.sync()
    assert e.value.status == 9                                  # GQ_ERR_KEY_RANGE
    c2.clear_error(); c2.sync()
    dup = bkeys.copy(); dup[5] = dup[9000]
    c2.hash_build(gqrun.dev([dup]), key=0, unique=True, dense_range=(-30_000, 29_999))
    with pytest.raises(gq.GqError) as e:
        c2.sync()
    assert e.value.status == 6                                  # GQ_ERR_DUPLICATE_KEY
    c2.clear_error(); c2.sync()
    c2.hash_build(gqrun.dev([bkeys]), key=0, unique=True, dense_range=(-30_000, 29_999), max_rows=100)
    with pytest.raises(gq.GqError) as e:                        # more build rows than max_build_rows promised
        c2.sync()
    assert e.value.status == 3                                  # GQ_ERR_CAPACITY
    c2.clear_error(); c2.sync()
    tb3 = c2.hash_build(gqrun.dev([bkeys]), key=0, unique=True, dense_range=(-30_000, 29_999), finish=False)
    with pytest.raises(gq.GqError):                             # probing a dense table before gq_hash_build_finish
        c2.hash_probe(gqrun.dev([fk, v]), [], [(tb3, 0)], [[("col", 0)]], capacity=nf)


def test_check_dependent_flag_catches_a_false_declaration(ctx):
    # S17: a key declared functionally dependent is stored, not hashed. With GQ_F_CHECK_DEPENDENT a false declaration
    # is a sticky error instead of silently merged groups; a true one gives the oracle's tuple-grouped result.
    import gqrun
    from paper_2606_24647_b200 import gq
    rng = np.random.default_rng(41)
    n = 120_000
    k = rng.integers(0, 5000, n).astype(np.int64)
    dep_true = (k * 7 % 1000).astype(np.int32)
    v = rng.integers(0, 100, n).astype(np.int64)
    plan = dict(table=[k, dep_true, v], preds=[], exprs=[[("col", 2)]], keys=[0, 1], ndependent=1,
                aggs=[("sum", 0), ("count",)], max_groups=6000)
    exp = oracle.run_query(plan)
    for force_part in (False, True):
        if force_part:
            gq.set_option("part_min_table_mb", 0); gq.set_option("part_min_rows", 4096)
        try:
            c = gq.Context()
            p2 = c.prepare_pipeline(gqrun.dev(plan["table"]), exprs=plan["exprs"], keys=[0, 1], ndependent=1, aggs=plan["aggs"],
                                    max_groups=6000, check_dependent=True)
            p2.run(); c.sync()
            r = p2.result()
            got = gqrun.sort_rows([x.cpu().numpy().astype(np.int64) for x in r["keys"]] + [a.cpu().numpy() for a in r["aggs"]], 2)
            assert r["n"] == exp.nrows and all(np.array_equal(g, e) for g, e in zip(got, exp.cols))
            dep_false = dep_true.copy()
            dep_false[n // 2] += 1                                  # ONE row breaks the dependency
            p3 = c.prepare_pipeline(gqrun.dev([k, dep_false, v]), exprs=plan["exprs"], keys=[0, 1], ndependent=1,
                                    aggs=plan["aggs"], max_groups=6000, check_dependent=True)
            p3.run()
            with pytest.raises(gq.GqError) as e:
                c.sync()
            assert e.value.status == 8                              # GQ_ERR_DEPENDENT_KEY
            c.clear_error(); c.sync()
        finally:
            gq.set_option("part_min_table_mb", -1); gq.set_option("part_min_rows", -1)


# ------------------------------------------------------------------ radix-clustered (partitioned) aggregation
@pytest.fixture
def force_partition():
    # planner thresholds that switch the partitioned path on for tables and batches the oracle can check in seconds
    from paper_2606_24647_b200 import gq
    gq.set_option("part_min_table_mb", 0)
    gq.set_option("part_min_rows", 4096)
    yield
    gq.set_option("part_min_table_mb", -1)
    gq.set_option("part_min_rows", -1)


@pytest.mark.parametrize("scale", [0.003, 0.0101])
def test_partitioned_aggregation_c5_shape(ctx, force_partition, scale):
    plan = plans.plan_c5(datagen.make_config(5, scale=scale))
    l0 = ctx.launch_count()
    run(plan, ctx)
    assert ctx.launch_count() - l0 >= 4          # init, scan (pass A), partitioned upsert (pass B), finalise


def test_partitioned_aggregation_skew_overflow_reserved_key_and_dependent_key(ctx, force_partition):
    rng = np.random.default_rng(11)
    n = 300_000
    # one key owns 60 % of the rows (its partition overflows -> in-kernel fallback), plus the reserved bit pattern
    k = rng.integers(0, 50_000, n).astype(np.int64) * 7919
    k[rng.random(n) < 0.6] = 123456789
    k[::1000] = I64_MIN
    dep = (k % 1000).astype(np.int32)              # functionally dependent on the key
    v = rng.integers(-1000, 1000, n).astype(np.int64)
    w = rng.integers(0, 5, n).astype(np.int64)
    plan = dict(table=[k, dep, v, w], preds=[(3, "lt", 4)], exprs=[[("col", 2)], [("col", 3)]], keys=[0, 1], ndependent=1,
                aggs=[("sum", 0), ("min", 0), ("max", 1), ("count",), ("sum", 1)], max_groups=60_000)
    run(plan, ctx)


def test_partitioned_shared_memory_aggregation_shapes(ctx, force_partition):
    # gq_pipeline's single-batch path (scatter -> directory -> shared-memory aggregation per partition): packed two-key
    # groups with signed narrow keys, AVG, a probe step in front, and a batch that is only a ragged tail
    rng = np.random.default_rng(12)
    n = 260_007
    a = rng.integers(-300, 300, n).astype(np.int32)
    b = rng.integers(-100, 100, n).astype(np.int8)
    v = rng.integers(-10**11, 10**11, n).astype(np.int64)
    plan = dict(table=[a, b, v], preds=[(2, "ne", 5)], exprs=[[("col", 2)], [("col", 2), ("col", 0), ("mul",)]], keys=[0, 1],
                aggs=[("sum", 0), ("count",), ("min", 1), ("max", 0)], max_groups=130_000)
    l0 = ctx.launch_count()
    exp, got = run(plan, ctx, avgs=[(0, 1)])
    assert ctx.launch_count() - l0 == 6          # merge-table init, scan+scatter, directory x2, shared-memory aggregation, merge emit
    ref = np.array([oracle.avg(int(x), int(y)) for x, y in zip(exp.cols[2], exp.cols[3])])
    assert np.array_equal(got["avgs"][0], ref)
    rngj = np.random.default_rng(13)
    plan = _join_plan(9_000, 200_000, rngj, [("sum", 0), ("count",)])
    plan["keys"] = [1]; plan["max_groups"] = 20_000                      # group by a non-join column: hashed, partitioned
    run(plan, ctx)
    plan = plans.plan_c5(datagen.make_config(5, scale=0.00001))          # 6000 rows: tail-only batches still work
    plan["max_groups"] = 10_000
    run(plan, ctx)


def test_partitioned_shared_memory_aggregation_heavy_keys_and_many_groups(ctx, force_partition):
    rng = np.random.default_rng(14)
    # (a) heavy partitions are cut into segments whose partial groups meet in the global merge table: one key owns 55 %
    # of 1.5 M rows, another 20 %, plus the reserved bit pattern and a dependent key
    n = 1_500_000
    k = rng.integers(0, 40_000, n).astype(np.int64) * 104729
    u = rng.random(n)
    k[u < 0.55] = 987654321
    k[(u >= 0.55) & (u < 0.75)] = -5
    k[::997] = I64_MIN
    dep = (k % 1000).astype(np.int32)
    v = rng.integers(-10**6, 10**6, n).astype(np.int64)
    plan = dict(table=[k, dep, v], preds=[], exprs=[[("col", 2)]], keys=[0, 1], ndependent=1,
                aggs=[("sum", 0), ("min", 0), ("max", 0), ("count",)], max_groups=45_000)
    exp, got = run(plan, ctx)
    assert int(got["cols"][-1].max()) > 800_000
    # (b) far more distinct keys than max_groups promised: partitions overflow their shared-memory table and their key
    # range is halved (second hash) until it fits -- slower, never wrong
    n = 700_000
    k = rng.permutation(5_000_000)[:n].astype(np.int64) - 2_000_000
    plan = dict(table=[k, np.ones(n, np.int64)], preds=[], exprs=[[("col", 1)]], keys=[0], aggs=[("sum", 0), ("count",)],
                max_groups=100_000)
    exp, got = run(plan, ctx, out_capacity=n)
    assert got["n"] == n


def test_partitioned_shared_memory_aggregation_hot_keys_and_sub_passes(ctx, force_partition):
    # pass A aggregates the batch's most frequent keys in shared memory (they never become records; their groups reach
    # the output through the merge table), and with fewer pass-A partitions than key ranges pass B runs sub-passes
    from paper_2606_24647_b200 import gq
    rng = np.random.default_rng(15)
    n = 900_000
    k = (rng.zipf(1.3, n) % 300_000).astype(np.int64) * 7 - 1000          # a few very hot keys, a long tail
    k[::5000] = I64_MIN
    v = rng.integers(-10**9, 10**9, n).astype(np.int64)
    w = rng.integers(0, 50, n).astype(np.int64)
    plan = dict(table=[k, v, w], preds=[(2, "lt", 45)], exprs=[[("col", 1)], [("col", 2)]], keys=[0],
                aggs=[("sum", 0), ("sum", 1), ("min", 0), ("max", 0), ("count",)], max_groups=300_000)
    try:
        gq.set_option("hot_min_rows", 4096)
        for lp, cl in ((14, 2), (6, 2), (5, 1), (14, 1)):           # with and without thread-block clusters in pass A
            gq.set_option("psa_max_log2_partitions", lp)
            gq.set_option("psa_cluster", cl)
            for th in (512, 1024):
                gq.set_option("psa_threads", th)
                l0 = ctx.launch_count()
                exp, got = run(plan, ctx)
                assert ctx.launch_count() - l0 == 11     # + table init and four kernels of the heavy-hitter sampling
                assert int(got["cols"][-1].max()) > 100_000
        # more keys reach the sampling threshold than the hot set holds (3000 equally frequent keys + a long tail): the
        # selection raises its threshold past all of them and fills the list from the bin below it
        gq.set_option("psa_max_log2_partitions", -1); gq.set_option("psa_threads", 0)
        k2 = rng.integers(0, 3000, n).astype(np.int64) * 11 - 5000
        k2[::7] = rng.integers(10**6, 10**6 + 200_000, len(k2[::7]))
        run(dict(plan, table=[k2, v, w]), ctx)
    finally:
        gq.set_option("hot_min_rows", -1); gq.set_option("psa_max_log2_partitions", -1); gq.set_option("psa_threads", 0)
        gq.set_option("psa_cluster", 2)


def test_clustered_direct_aggregation(ctx, force_partition):
    # direct aggregation (group = matched slot / rank of a probed unique table) with its REDs clustered by slice of the
    # accumulator array: records appended per slice by the scan, applied slice by slice — hashed and direct-address tables,
    # a dependent key, a plan without COUNT (hidden touch word), MIN/MAX, overflowing record buffers (in-place fallback)
    from paper_2606_24647_b200 import gq
    rng = np.random.default_rng(16)
    try:
        gq.set_option("dpart_min_acc_mb", 0)
        for aggs in ([("sum", 0), ("count",)], [("sum", 0), ("min", 0), ("max", 0)]):
            plan = _join_plan(120_000, 700_001, rng, aggs, with_dep=True)
            l0 = ctx.launch_count()
            run(plan, ctx)
            assert ctx.launch_count() - l0 == 6      # join table init, build, accumulator init, scan + append, apply, finalise
            dense = dict(plan, builds=[dict(plan["builds"][0], dense_range=(int(plan["builds"][0]["table"][0].min()),
                                                                           int(plan["builds"][0]["table"][0].max())))])
            run(dense, ctx)
        # one key receives 70 % of the rows: its slice's record buffer overflows, the rest is aggregated in place
        plan = _join_plan(50_000, 600_000, rng, [("sum", 0), ("count",)])
        hot = plan["builds"][0]["table"][0][plan["builds"][0]["table"][2] == 1][0]
        fk = plan["table"][0].copy()
        fk[rng.random(len(fk)) < 0.7] = hot
        plan["table"][0] = fk
        exp, got = run(plan, ctx)
        assert int(got["cols"][-1].max()) > 300_000
    finally:
        gq.set_option("dpart_min_acc_mb", -1)


def test_partitioned_aggregation_streams_batches(ctx, force_partition):
    import gqrun
    plan = plans.plan_c5(datagen.make_config(5, scale=0.004))
    exp = oracle.run_query(plan)
    cols = gqrun.dev(plan["table"])
    n = len(plan["table"][0])
    st = None
    for lo, hi in ((0, n // 2 // 16 * 16), (n // 2 // 16 * 16, n - 160), (n - 160, n)):   # last batch takes the plain path
        st = ctx.aggregate(st, [c[lo:hi] for c in cols], preds=plan["preds"], exprs=plan["exprs"], keys=plan["keys"],
                           aggs=plan["aggs"], max_groups=plan["max_groups"], plan_aware_workspace=True)
    r = ctx.aggregate_finish(st, capacity=exp.nrows + 5)
    ctx.sync()
    ng = int(r["n"].item())
    assert ng == exp.nrows
    got = gqrun.sort_rows([r["keys"][0][:ng].cpu().numpy()] + [a[:ng].cpu().numpy() for a in r["aggs"]], 1)
    for g, e in zip(got, exp.cols):
        assert np.array_equal(g, e)


def test_pipeline_is_cuda_graph_capturable():
    # every call only enqueues on the context's stream (no allocation, no host sync): a whole build + pipeline sequence
    # can be captured into a CUDA graph and replayed (operators return immediately)
    import torch
    import gqrun
    from paper_2606_24647_b200 import gq
    s = torch.cuda.Stream()
    with torch.cuda.stream(s):
        c = gq.Context(0, stream=s)
        plan = plans.plan_c3(datagen.make_config(3, scale=0.01))
        exp = oracle.run_query(plan)
        bcols = [gqrun.dev(b["table"]) for b in plan["builds"]]
        tables = gqrun.build_tables(c, plan, device_tables=bcols)      # warm-up run compiles / loads the kernels
        ws = [t.workspace for t in tables]
        p = gqrun.prepare(c, plan, tables)
        p.run()
        c.sync()
        g = torch.cuda.CUDAGraph()
        # (no cyclic garbage collection inside the capture: a context of an earlier test collected there would cudaFree,
        # which invalidates a capture in progress)
        import gc
        gc.collect(); gc.disable()
        try:
            with torch.cuda.graph(g, stream=s):
                tables = gqrun.build_tables(c, plan, device_tables=bcols, workspaces=ws)
                pr, _ = p.m.probes([(tables[bi], kc) for bi, kc in plan["probes"]])
                p.plan.agg.probes = pr
                p.run()
        finally:
            gc.enable()
        for _ in range(3):
            for a in p.aggs:
                a.zero_()
            g.replay()
            torch.cuda.synchronize()
            r = p.result()
            got = gqrun.sort_rows([r["keys"][0].cpu().numpy()] + [a.cpu().numpy() for a in r["aggs"]], 1)
            assert r["n"] == exp.nrows
            for x, e in zip(got, exp.cols):
                assert np.array_equal(x, e)
