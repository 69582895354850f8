"""Pins the CPU oracle to things other than itself (CPU only; -m "not gpu").

  * hand-computed worked examples T1-T5 (tests/golden/worked_examples.json)
  * brute-force nested-loop join == hash-multimap join (definition 3)
  * pandas / numpy group-by + merge as an independent third opinion (special cases reducing to library routines)
  * invariants I1-I7 and closed-form pass fractions of the seeded generator
  * adversarial inputs: duplicate build keys, dangling fks, sentinel-valued keys, wrapping products
"""
import numpy as np
import pandas as pd
import pytest

import oracle
import plans
from golden_util import load, table
from paper_2606_24647_b200 import datagen

G = load()


def _cols(res):
    return [list(map(int, c)) for c in res.cols]


def _rows(res):
    return [list(map(int, r)) for r in zip(*res.cols)] if res.nrows else []


# ------------------------------------------------------------------ worked examples
def test_T1_filter_lowcard_groupby():
    t = table(G["T1"]["cols"], G["T1"]["rows"])
    f = dict(shipdate=t["shipdate"], quantity=t["qty"], price=t["price"], discount=t["disc"], tax=t["tax"],
             flagA=t["flagA"], flagB=t["flagB"])
    r = oracle.run_query(plans.plan_c1({"fact": f}))
    assert _rows(r) == G["T1"]["expect"]
    assert r.input_rows == G["T1"]["rows_passing"] == sum(row[-1] for row in _rows(r))
    assert not r.overflow
    for g, row in enumerate(_rows(r)):
        assert oracle.avg(row[2], row[6]) == G["T1"]["expect_avg_qty"][g]
        assert oracle.avg(row[3], row[6]) == G["T1"]["expect_avg_price"][g]


def test_T2_selective_filter_global_sum():
    t = table(G["T2"]["cols"], G["T2"]["rows"])
    f = dict(shipdate=t["shipdate"], discount=t["disc"], quantity=t["qty"], price=t["price"])
    r = oracle.run_query(plans.plan_c2({"fact": f}))
    assert _rows(r) == G["T2"]["expect"]


def _t3():
    d = table(G["T3"]["dim_cols"], G["T3"]["dim"])
    f = table(G["T3"]["fact_cols"], G["T3"]["fact"])
    return {"dim": d, "fact": dict(fk=f["fk"], shipdate=f["shipdate"], price=f["price"], discount=f["disc"])}


def test_T3_join_groupby_topk():
    r = oracle.run_query(plans.plan_c3(_t3()))
    assert _rows(r) == G["T3"]["expect"]
    assert r.input_rows == G["T3"]["join_rows"]
    r = oracle.run_query(plans.plan_c3(_t3(), topk=10))
    assert _rows(r) == G["T3"]["expect_topk"]
    r = oracle.run_query(plans.plan_c3(_t3(), topk=1))
    assert _rows(r) == G["T3"]["expect_topk"][:1]


def test_T4_chained_join():
    c = table(G["T4"]["cust_cols"], G["T4"]["cust"])
    o = table(G["T4"]["orders_cols"], G["T4"]["orders"])
    f = table(G["T4"]["fact_cols"], G["T4"]["fact"])
    t = {"cust": c, "orders": o, "fact": dict(fk=f["fk"], shipdate=f["shipdate"], price=f["price"], discount=f["disc"])}
    r = oracle.run_query(plans.plan_c4(t))
    assert _rows(r) == G["T4"]["expect"]
    assert r.input_rows == G["T4"]["join_rows"]


def test_T5_extreme_keys_min_max():
    t = table(G["T5"]["cols"], G["T5"]["rows"])
    f = dict(key=t["key"], shipdate=t["shipdate"], price=t["price"], quantity=t["qty"])
    r = oracle.run_query(plans.plan_c5({"fact": f}))
    assert _rows(r) == G["T5"]["expect"]
    assert r.input_rows == G["T5"]["rows_passing"]


def t6_plans():
    d, f = table(G["T6"]["dim_cols"], G["T6"]["dim"]), table(G["T6"]["fact_cols"], G["T6"]["fact"])
    t = {"dim": d, "fact": dict(fk=f["fk"], shipdate=f["shipdate"], price=f["price"], discount=f["disc"])}
    p = table(G["T6"]["pair_cols"], G["T6"]["pair_rows"])
    pair = lambda k: dict(table=[p["a"], p["b"], p["v"]], preds=[], exprs=[[("col", 2)]], keys=[0, 1],
                          aggs=[("sum", 0)], topk=k, topk_agg=0, max_groups=5000)
    return t, pair


def test_T6_topk_ties_are_decided_by_the_key():
    # S11: (aggregate desc, key tuple asc). Keys 3, 5, 9 tie at 1000 and k = 3 cuts through the tie; reversing the
    # oracle's tie-break (or comparing keys unsigned) changes these lists.
    t, pair = t6_plans()
    r = oracle.run_query(plans.plan_c3(t))
    assert _rows(r) == G["T6"]["expect"] and r.input_rows == G["T6"]["join_rows"]
    for k in (3, 4, 10):
        assert _rows(oracle.run_query(plans.plan_c3(t, topk=k))) == G["T6"][f"expect_top{k}"]
    for k in (3, 5):
        assert _rows(oracle.run_query(pair(k))) == G["T6"][f"expect_pair_top{k}"]


def t7_plan(rows, keys=(0,), max_groups=5000):
    t = table(G["T7"]["cols"], rows)
    aggs = [("sum", 0), ("min", 0), ("max", 0), ("count",)] if keys else [("sum", 0), ("count",)]
    return dict(table=[t["key"], t["v"]], preds=[], exprs=[[("col", 1)]], keys=list(keys), aggs=aggs, max_groups=max_groups)


def test_T7_running_sum_wraps_and_is_flagged():
    # S6: the running SUM wraps modulo 2^64 and the __int128 shadow raises the flag; no single value overflows here
    r = oracle.run_query(t7_plan(G["T7"]["rows"]))
    assert _rows(r) == G["T7"]["expect"] and r.overflow == bool(G["T7"]["expect_overflow"])
    g = oracle.run_query(t7_plan(G["T7"]["rows"], keys=()))
    assert _rows(g) == G["T7"]["expect_global"] and g.overflow
    n = oracle.run_query(t7_plan(G["T7"]["rows_no_wrap"]))
    assert _rows(n) == G["T7"]["expect_no_wrap"] and not n.overflow      # INT64_MAX reached exactly: no wrap, no flag


# ------------------------------------------------------------------ joins: brute force, duplicates, dangling
@pytest.mark.parametrize("seed", [1, 2, 3])
def test_join_equals_bruteforce_with_duplicates_and_dangling(seed):
    rng = np.random.default_rng(seed)
    nb, npr = 700, 1500
    bkey = rng.integers(0, 300, nb).astype(np.int64)        # duplicates on the build side (S3)
    bval = rng.integers(0, 2406, nb).astype(np.int32)
    pkey = rng.integers(-50, 400, npr).astype(np.int64)     # some fks match nothing (S4)
    pval = rng.integers(0, 2526, npr).astype(np.int32)
    a = oracle.join_pairs([bkey, bval], [(1, "lt", 1200)], 0, [pkey, pval], [(1, "gt", 1200)], 0)
    b = oracle.join_pairs([bkey, bval], [(1, "lt", 1200)], 0, [pkey, pval], [(1, "gt", 1200)], 0, bruteforce=True)
    assert a.nrows == b.nrows > 0
    assert _cols(a) == _cols(b)
    # third opinion: pandas merge cardinality (I2)
    B = pd.DataFrame(dict(k=bkey, v=bval)).query("v < 1200")
    P = pd.DataFrame(dict(k=pkey, v=pval)).query("v > 1200")
    assert len(P.merge(B, on="k", how="inner")) == a.nrows
    # the query path over the same join: COUNT(*) summed over groups == join cardinality
    q = dict(builds=[dict(table=[bkey, bval], preds=[(1, "lt", 1200)], probes=[], key=0, payload=[1])],
             table=[pkey, pval], preds=[(1, "gt", 1200)], probes=[(0, 0)], exprs=[[("col", 2)]], keys=[0],
             aggs=[("count",), ("sum", 0)])
    r = oracle.run_query(q)
    assert r.input_rows == a.nrows == int(r.cols[1].sum())
    M = P.merge(B, on="k", how="inner").groupby("k").agg(n=("v_y", "size"), s=("v_y", "sum")).sort_index()
    assert list(M.index) == list(r.cols[0]) and list(M.n) == list(r.cols[1]) and list(M.s) == list(r.cols[2])


# ------------------------------------------------------------------ third opinion on the configs (pandas / numpy)
def test_c1_vs_pandas():
    t = datagen.make_config(1, scale=0.2)
    r = oracle.run_query(plans.plan_c1(t))
    f = pd.DataFrame(t["fact"]).query("shipdate <= 2430")
    f["dp"] = f.price * (100 - f.discount)
    f["ch"] = f.dp * (100 + f.tax)
    g = f.groupby(["flagA", "flagB"]).agg(q=("quantity", "sum"), p=("price", "sum"), dp=("dp", "sum"),
                                          ch=("ch", "sum"), n=("price", "size")).sort_index().reset_index()
    assert r.nrows == len(g) == 6
    for c, name in enumerate(["flagA", "flagB", "q", "p", "dp", "ch", "n"]):
        assert list(g[name]) == list(r.cols[c])
    assert r.input_rows == len(f) and not r.overflow                          # I1
    assert abs(len(f) / len(t["fact"]["price"]) - 2431 / 2526) < 5 * (0.0362 / 2e5) ** 0.5   # closed form, 5 sigma


def test_c2_vs_numpy():
    t = datagen.make_config(2, scale=0.02)
    f = t["fact"]
    r = oracle.run_query(plans.plan_c2(t))
    m = (f["shipdate"] >= 730) & (f["shipdate"] < 1095) & (f["discount"] >= 5) & (f["discount"] <= 7) & (f["quantity"] < 24)
    assert _rows(r) == [[int((f["price"][m] * f["discount"][m]).sum()), int(m.sum())]]
    n = len(m)
    p = (365 / 2526) * (3 / 11) * (23 / 50)
    assert abs(m.sum() - n * p) < 5 * (n * p * (1 - p)) ** 0.5                  # closed form, 5 sigma


def test_c3_vs_pandas_and_invariants():
    t = datagen.make_config(3, scale=0.004)
    r = oracle.run_query(plans.plan_c3(t))
    D = pd.DataFrame(t["dim"]).query("orderdate < 1200")
    F = pd.DataFrame(t["fact"]).query("shipdate > 1200")
    M = F.merge(D, left_on="fk", right_on="key", how="inner")
    M["dp"] = M.price * (100 - M.discount)
    g = M.groupby("key").agg(s=("dp", "sum"), n=("dp", "size")).sort_index()
    assert list(g.index) == list(r.cols[0]) and list(g.s) == list(r.cols[1]) and list(g.n) == list(r.cols[2])
    assert r.input_rows == len(M) == int(r.cols[2].sum())                      # I1, I2
    assert r.cols[2].min() >= 1 and r.cols[2].max() <= 7 and r.nrows <= len(D)  # I4
    top = oracle.run_query(plans.plan_c3(t, topk=10))
    exp = g.reset_index().sort_values(["s", "key"], ascending=[False, True]).head(10)
    assert list(exp.key) == list(top.cols[0]) and list(exp.s) == list(top.cols[1])


def test_c4_vs_pandas_and_invariants():
    t = datagen.make_config(4, scale=0.004)
    r = oracle.run_query(plans.plan_c4(t))
    Cc = pd.DataFrame(t["cust"]).query("segment == 1")
    O = pd.DataFrame(t["orders"]).query("orderdate < 1200").merge(Cc, left_on="custkey", right_on="key")
    F = pd.DataFrame(t["fact"]).query("shipdate > 1200").merge(O, left_on="fk", right_on="orderkey")
    F["dp"] = F.price * (100 - F.discount)
    g = F.groupby(["orderkey", "orderdate"]).agg(s=("dp", "sum"), n=("dp", "size")).sort_index().reset_index()
    assert r.nrows == len(g) > 0
    for c, name in enumerate(["orderkey", "orderdate", "s", "n"]):
        assert list(g[name]) == list(r.cols[c])
    assert r.input_rows == len(F)
    # I4: every emitted (orderkey, orderdate) is the orders table's pair
    od = dict(zip(t["orders"]["orderkey"].tolist(), t["orders"]["orderdate"].tolist()))
    assert all(od[int(k)] == int(d) for k, d in zip(r.cols[0], r.cols[1]))


def test_c5_vs_pandas_and_invariants():
    t = datagen.make_config(5, scale=0.0005)
    r = oracle.run_query(plans.plan_c5(t))
    F = pd.DataFrame(t["fact"]).query("shipdate < 2000")
    g = F.groupby("key").agg(sp=("price", "sum"), sq=("quantity", "sum"), mn=("price", "min"), mx=("price", "max"),
                             n=("price", "size")).sort_index().reset_index()
    for c, name in enumerate(["key", "sp", "sq", "mn", "mx", "n"]):
        assert list(g[name]) == list(r.cols[c])
    # I3: MIN <= SUM/COUNT <= MAX, sums add up to the global sum
    assert np.all(r.cols[3] * r.cols[5] <= r.cols[1]) and np.all(r.cols[1] <= r.cols[4] * r.cols[5])
    assert int(r.cols[1].sum()) == int(F.price.sum()) and r.input_rows == len(F)


# ------------------------------------------------------------------ invariants I5-I7, special cases
def test_filter_true_false_and_empty():
    t = datagen.make_config(2, scale=0.001)
    f = t["fact"]
    cols = [f["shipdate"], f["discount"], f["quantity"], f["price"]]
    allp = oracle.run_query(dict(table=cols, preds=[], exprs=[[("col", 3)]], keys=[], aggs=[("sum", 0), ("count",)]))
    assert _rows(allp) == [[int(f["price"].sum()), len(f["price"])]]                       # I5
    none = oracle.run_query(dict(table=cols, preds=[(0, "lt", -1)], exprs=[[("col", 3)]], keys=[],
                                 aggs=[("sum", 0), ("count",)]))
    assert _rows(none) == [[0, 0]]                                                         # S9 global
    noneg = oracle.run_query(dict(table=cols, preds=[(0, "lt", -1)], exprs=[[("col", 3)]], keys=[1],
                                  aggs=[("sum", 0), ("count",)]))
    assert noneg.nrows == 0                                                                # S9 grouped
    empty = oracle.run_query(dict(table=[c[:0] for c in cols], preds=[], exprs=[[("col", 3)]], keys=[1],
                                  aggs=[("sum", 0)]))
    assert empty.nrows == 0


def test_batch_split_permutation_and_partial_merge_invariance():
    t = datagen.make_config(5, scale=0.0002)
    base = oracle.run_query(plans.plan_c5(t))
    n = len(t["fact"]["key"])
    perm = np.random.default_rng(7).permutation(n)
    tp = {"fact": {k: v[perm] for k, v in t["fact"].items()}}
    assert _cols(oracle.run_query(plans.plan_c5(tp))) == _cols(base)                       # I7
    # I6: aggregate the two halves separately, merge (Partial -> Final), compare
    merged = {}
    for lo, hi in [(0, n // 3), (n // 3, n)]:
        part = oracle.run_query(plans.plan_c5({"fact": {k: v[lo:hi] for k, v in t["fact"].items()}}))
        for row in _rows(part):
            m = merged.setdefault(row[0], [0, 0, 2**63 - 1, -2**63, 0])
            m[0] += row[1]; m[1] += row[2]; m[2] = min(m[2], row[3]); m[3] = max(m[3], row[4]); m[4] += row[5]
    assert [[k] + v for k, v in sorted(merged.items())] == _rows(base)


def test_bounds_inclusive_exclusive():
    x = np.array([4, 5, 6, 7, 8], dtype=np.int32)
    one = np.ones(5, dtype=np.int64)
    def cnt(pred):
        return int(oracle.run_query(dict(table=[x, one], preds=[pred], exprs=[], keys=[], aggs=[("count",)])).cols[0][0])
    assert [cnt((0, "lt", 6)), cnt((0, "le", 6)), cnt((0, "gt", 6)), cnt((0, "ge", 6)), cnt((0, "eq", 6)),
            cnt((0, "ne", 6)), cnt((0, "range_co", 5, 7)), cnt((0, "range_cc", 5, 7))] == [2, 3, 2, 3, 1, 4, 2, 3]


def test_wrapping_products_flag_overflow():
    a = np.array([2**62, -3, 5], dtype=np.int64)
    b = np.array([4, 2**62, 7], dtype=np.int64)
    r = oracle.filter_project([a, b], [], [[("col", 0), ("col", 1), ("mul",)], [("col", 0), ("col", 1), ("sub",)]])
    assert r.overflow
    def wrap(x):                                                                           # low 64 bits, two's complement
        x %= 2**64
        return x - 2**64 if x >= 2**63 else x
    assert list(map(int, r.cols[0])) == [wrap(2**64), wrap(-3 * 2**62), 35] == [0, 2**62, 35]
    assert list(map(int, r.cols[1])) == [2**62 - 4, -3 - 2**62, -2]
    r2 = oracle.filter_project([a[2:], b[2:]], [], [[("col", 0), ("col", 1), ("mul",)]])
    assert not r2.overflow


def test_filter_project_keeps_input_order_and_signed_narrow_types():
    d = np.array([-128, -1, 0, 127], dtype=np.int8)
    v = np.array([10, 20, 30, 40], dtype=np.int32)
    r = oracle.filter_project([d, v], [(0, "lt", 0)], [[("col", 1), ("col", 0), ("add",)]])
    assert list(map(int, r.cols[0])) == [10 - 128, 19]                                      # S21 sign extension


def test_no_overflow_in_configs():
    # S6: the int128 shadow must stay silent on the config value ranges (max product 1.134e11 per row)
    for cfg, sc in [(1, 0.05), (3, 0.001), (5, 0.0001)]:
        t = datagen.make_config(cfg, scale=sc)
        assert not oracle.run_query(plans.PLANS[cfg](t)).overflow


# ------------------------------------------------------------------ ORDER BY / LIMIT
def test_T8_order_by_worked_example_with_ties():
    t = table(G["T8"]["cols"], G["T8"]["rows"])
    cols = [t["a"], t["b"]]
    r = oracle.order_by(cols, [tuple(k) for k in G["T8"]["keys"]])
    assert list(r.cols[0]) == G["T8"]["expect_index"] and list(r.cols[1]) == G["T8"]["expect_a"] and list(r.cols[2]) == G["T8"]["expect_b"]
    assert list(oracle.order_by(cols, [tuple(k) for k in G["T8"]["keys"]], limit=4).cols[0]) == G["T8"]["expect_index_limit4"]
    assert list(oracle.order_by(cols, [tuple(k) for k in G["T8"]["keys_b_desc_only"]]).cols[0]) == G["T8"]["expect_index_b_desc"]
    assert list(oracle.order_by(cols, []).cols[0]) == list(range(6))                # no keys: input order


def test_order_by_equals_numpy_lexsort():
    # an independent library routine: np.lexsort is stable and sorts by the LAST key first; a descending signed key is
    # its bitwise complement (-x - 1: order reversed, no overflow at INT64_MIN)
    rng = np.random.default_rng(81)
    n = 20_000
    a = rng.integers(-4, 4, n).astype(np.int8)
    b = rng.integers(-50, 50, n).astype(np.int32)
    c = rng.integers(-2**62, 2**62, n).astype(np.int64)
    c[::7] = c[0]; c[5] = np.iinfo(np.int64).min; c[6] = np.iinfo(np.int64).max
    for keys in ([(0, False)], [(0, True), (1, False)], [(2, True)], [(1, True), (0, True), (2, False)]):
        r = oracle.order_by([a, b, c], keys)
        cols = [a, b, c]
        lex = [np.arange(n)] + [(~cols[k].astype(np.int64) if d else cols[k].astype(np.int64)) for k, d in reversed(keys)]
        want = np.lexsort(tuple(lex))
        assert np.array_equal(r.cols[0], want)
        for j in range(3):
            assert np.array_equal(r.cols[1 + j], cols[j][want].astype(np.int64))
        lim = oracle.order_by([a, b, c], keys, limit=137)
        assert lim.nrows == 137 and np.array_equal(lim.cols[0], want[:137])
    # invariants: a permutation; adjacent rows are in order
    r = oracle.order_by([a, b, c], [(1, False), (2, True)])
    assert np.array_equal(np.sort(r.cols[0]), np.arange(n))
    kb, kc = r.cols[2], r.cols[3]
    assert np.all((kb[:-1] < kb[1:]) | ((kb[:-1] == kb[1:]) & (kc[:-1] >= kc[1:])))


# ------------------------------------------------------------------ hash partitioning
def test_hash_partition_murmur3_finaliser_vectors():
    # the published MurmurHash3 fmix64 vectors fmix64(0) = 0 and fmix64(1) = 0xB456BCFC34C2CB2C, reached through the seed:
    # a single key k gives h = fmix64(0x9E3779B97F4A7C15 xor k). nparts = 2^16 exposes the top 16 bits of h.
    seed = 0x9E3779B97F4A7C15
    k0 = np.array([seed], dtype=np.uint64).view(np.int64)                 # h = fmix64(0) = 0
    k1 = np.array([seed ^ 1], dtype=np.uint64).view(np.int64)             # h = fmix64(1)
    assert list(oracle.hash_partition([k0], [0], 1 << 16).cols[0]) == [0]
    assert list(oracle.hash_partition([k0], [0], 7).cols[0]) == [0]
    assert list(oracle.hash_partition([k1], [0], 1 << 16).cols[0]) == [0xB456]
    assert list(oracle.hash_partition([k1], [0], 256).cols[0]) == [0xB4]
    assert list(oracle.hash_partition([k1], [0], 3).cols[0]) == [(0xB456BCFC * 3) >> 32]   # floor(h_hi * nparts / 2^32)


def test_hash_partition_invariants():
    rng = np.random.default_rng(91)
    n = 30_000
    a = rng.integers(-100, 100, n).astype(np.int8)
    b = rng.integers(-5000, 5000, n).astype(np.int32)
    c = rng.integers(-2**62, 2**62, n).astype(np.int64)
    cols = [a, b, c]
    for keys, nparts in (([1], 8), ([0, 1], 7), ([2], 256), ([1, 2, 0], 3)):
        r = oracle.hash_partition(cols, keys, nparts)
        dest, row = r.cols[0], r.cols[1]
        assert r.nrows == n and np.array_equal(np.sort(row), np.arange(n))                 # a permutation of the rows
        for j in range(3):
            assert np.array_equal(r.cols[2 + j], cols[j][row].astype(np.int64))            # whole rows move together
        assert dest.min() >= 0 and dest.max() < nparts and np.all(dest[1:] >= dest[:-1])   # destination-major
        same = dest[1:] == dest[:-1]
        assert np.all(row[1:][same] > row[:-1][same])                                      # input order inside one
        # the destination is a function of the key tuple alone: not of the other columns, not of the row's position
        dest_of_row = np.empty(n, np.int64); dest_of_row[row] = dest
        perm = rng.permutation(n)
        other = [rng.integers(-9, 9, n).astype(x.dtype) if j not in keys else x for j, x in enumerate(cols)]
        r2 = oracle.hash_partition([x[perm] for x in other], keys, nparts)
        d2 = np.empty(n, np.int64); d2[r2.cols[1]] = r2.cols[0]
        assert np.array_equal(d2, dest_of_row[perm])
        seen = {}
        for kt, d in zip(zip(*[cols[k].tolist() for k in keys]), dest_of_row.tolist()):
            assert seen.setdefault(kt, d) == d                                             # equal keys, equal destination
    # one destination: the input, in order; empty input: empty output
    r = oracle.hash_partition(cols, [2], 1)
    assert np.array_equal(r.cols[1], np.arange(n)) and not r.cols[0].any()
    assert oracle.hash_partition([c[:0]], [0], 4).nrows == 0
    # floor(h_hi * nparts / 2^32): halving a power-of-two partition count merges neighbouring destinations
    d16 = np.empty(n, np.int64); r16 = oracle.hash_partition(cols, [2], 16); d16[r16.cols[1]] = r16.cols[0]
    d8 = np.empty(n, np.int64); r8 = oracle.hash_partition(cols, [2], 8); d8[r8.cols[1]] = r8.cols[0]
    assert np.array_equal(d16 >> 1, d8)


def test_hash_partition_balance_and_bigint_restatement():
    # consecutive integers (the worst input for a weak mix) spread evenly: chi-square of the destination sizes against
    # the uniform law, 7 degrees of freedom / 6: far below 40 (p < 1e-6) for a good mix, in the thousands for a bad one
    n = 400_000
    k = np.arange(n, dtype=np.int64) - 1000
    for nparts in (8, 7):
        sizes = np.bincount(oracle.hash_partition([k], [0], nparts).cols[0], minlength=nparts)
        chi2 = float(((sizes - n / nparts) ** 2 / (n / nparts)).sum())
        assert chi2 < 40.0, (nparts, sizes)
    # Python integers (no wrap-around, masked by hand) against the C arithmetic: negative keys sign-extended from narrow
    # types, several keys chained
    M = (1 << 64) - 1
    def fmix(x):
        x ^= x >> 33; x = (x * 0xff51afd7ed558ccd) & M; x ^= x >> 33; x = (x * 0xc4ceb9fe1a85ec53) & M; x ^= x >> 33
        return x
    a = np.array([-128, -1, 0, 1, 127, -77], np.int8)
    b = np.array([-2**31, -1, 0, 5, 2**31 - 1, 123456], np.int32)
    c = np.array([-2**63, -1, 0, 2**63 - 1, 42, -42], np.int64)
    for keys, nparts in (([0], 5), ([1], 256), ([2], 1000), ([0, 1, 2], 13), ([2, 0], 64)):
        r = oracle.hash_partition([a, b, c], keys, nparts)
        got = np.empty(6, np.int64); got[r.cols[1]] = r.cols[0]
        for i in range(6):
            h = 0x9E3779B97F4A7C15
            for kc in keys:
                h = fmix(h ^ (int([a, b, c][kc][i]) & M))
            assert got[i] == ((h >> 32) * nparts) >> 32
