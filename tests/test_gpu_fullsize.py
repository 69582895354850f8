"""Full-size parity (-m gpu): BASELINE.json's C2-C5 at their full row counts, in the launch configuration bench.py
times (same cardinality hints, same pipelines). The WHOLE result table is compared with the oracle's through the digests
of tests/golden/fullsize_digests.json (written by tests/golden/make_fullsize_digests.py from oracle/ + datagen only: group
count, rows fed to GROUP BY, and per output column in key order the wrapping sum, xor and SHA-256 — SURVEY §8(c) "full
table exact"). When a digest differs, the older checks localise it: (a) invariants computed from the inputs with plain
numpy selections and wrapping sums (I1/I3), (b) SAMPLED groups compared one by one with the oracle run on exactly the
input rows that can contribute to them (selecting rows is input preparation; all arithmetic is the oracle's)."""
import json
import os

from golden_util import digest_columns

with open(os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden", "fullsize_digests.json")) as _f:
    DIGESTS = json.load(_f)


def _check_digest(cfg, got):
    d = DIGESTS[f"C{cfg}"]
    assert got["n"] == d["ngroups"], f"C{cfg}: {got['n']} groups, the oracle has {d['ngroups']}"
    mine = digest_columns(got["cols"])
    for c, (a, b) in enumerate(zip(mine, d["columns"])):
        assert a == b, f"C{cfg}: output column {c} differs from the oracle's full table (digest)"
    assert len(mine) == len(d["columns"])

import numpy as np
import pytest

import oracle
import plans
from paper_2606_24647_b200 import datagen

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def ctx():
    from paper_2606_24647_b200 import build as gqbuild
    gqbuild.build()
    from paper_2606_24647_b200 import gq
    return gq.Context()


def _wsum(a):
    return int(np.sum(a.astype(np.uint64), dtype=np.uint64).astype(np.int64))


def _gpu(plan, ctx, out_capacity=None):
    import gqrun
    import torch
    got = gqrun.run_query(plan, ctx=ctx, out_capacity=out_capacity)
    torch.cuda.empty_cache()
    return got


def _dense(plan, sel):
    """bench.py's timed configuration: every build declared GQ_F_DENSE_KEYS over the min/max of its key column (column
    statistics), its row bound from the predicates' selectivities + 10 %."""
    for b, s in zip(plan["builds"], sel):
        k = b["table"][b["key"]]
        b["dense_range"] = (int(k.min()), int(k.max()))
        b["max_rows"] = int(len(k) * s * 1.1) + 1024
    plan["max_groups"] = plan["builds"][-1]["max_rows"]
    return plan


def _sample_check(plan, got, nkeys_out, rows_of, rng, nsample=48):
    """Oracle on the rows that can reach `nsample` sampled output groups (plus keys that produced no group)."""
    keys = got["cols"][0]
    pick = np.unique(np.concatenate([keys[rng.integers(0, len(keys), nsample)], keys[:4], keys[-4:]]))
    sub = rows_of(pick)
    exp = oracle.run_query(sub)
    sel = np.isin(keys, pick)
    assert exp.nrows == int(sel.sum())
    for c in range(len(exp.cols)):
        assert np.array_equal(got["cols"][c][sel], exp.cols[c]), f"sampled groups: column {c} differs"
    assert not exp.overflow


def test_c2_full_size(ctx):
    plan = plans.plan_c2(datagen.make_config(2))
    got = _gpu(plan, ctx)
    _check_digest(2, got)
    assert int(got["cols"][1][0]) == DIGESTS["C2"]["input_rows"]


def test_c3_full_size(ctx):
    t = datagen.make_config(3)
    plan = plans.plan_c3(t)
    plan["builds"][0]["max_rows"] = int(len(t["dim"]["key"]) * 0.55) + 1024          # bench.py's hints
    plan["max_groups"] = plan["builds"][0]["max_rows"]
    got = _gpu(plan, ctx)
    d, f = t["dim"], t["fact"]
    assert int(got["cols"][2].sum()) == DIGESTS["C3"]["input_rows"]
    dkeys = d["key"][d["orderdate"] < 1200]
    live = (f["shipdate"] > 1200) & np.isin(f["fk"], dkeys)
    assert int(got["cols"][2].sum()) == int(live.sum())                               # I1/I2: sum of COUNT = join cardinality
    assert _wsum(got["cols"][1]) == _wsum(f["price"][live] * (100 - f["discount"][live]))   # I3
    assert got["n"] == len(np.unique(f["fk"][live]))
    assert got["cols"][2].min() >= 1 and got["cols"][2].max() <= 7                    # I4: 1..7 fact rows per key

    def rows_of(pick):
        fm, dm = np.isin(f["fk"], pick), np.isin(d["key"], pick)
        sub = plans.plan_c3({"dim": {k: v[dm] for k, v in d.items()}, "fact": {k: v[fm] for k, v in f.items()}})
        return sub
    _sample_check(plan, got, 1, rows_of, np.random.default_rng(3))
    _check_digest(3, got)                                                              # the whole 6.5 M-row table
    # top-10 through the top-k finaliser = the oracle's top-10 (sum desc, key asc), in order
    top = _gpu(dict(plan, topk=10, topk_agg=0), ctx, out_capacity=10)
    assert [[int(c[i]) for c in top["cols"]] for i in range(top["n"])] == DIGESTS["C3"]["top10"]
    # and with the build side sized from its INPUT row count (no selectivity knowledge): same table
    plan_ub = plans.plan_c3(t)
    _check_digest(3, _gpu(plan_ub, ctx))
    # bench.py's timed configuration: a direct-address table from the build key's min/max statistics (GQ_F_DENSE_KEYS)
    plan_d = _dense(plans.plan_c3(t), [1200 / 2406])
    _check_digest(3, _gpu(plan_d, ctx))
    top = _gpu(dict(plan_d, topk=10, topk_agg=0), ctx, out_capacity=10)
    assert [[int(c[i]) for c in top["cols"]] for i in range(top["n"])] == DIGESTS["C3"]["top10"]


def test_c4_full_size(ctx):
    t = datagen.make_config(4)
    plan = plans.plan_c4(t)
    for b, h in zip(plan["builds"], (0.22, 0.11)):
        b["max_rows"] = int(len(b["table"][0]) * h) + 1024
    plan["max_groups"] = plan["builds"][-1]["max_rows"]
    got = _gpu(plan, ctx)
    c, o, f = t["cust"], t["orders"], t["fact"]
    ck = c["key"][c["segment"] == 1]
    om = (o["orderdate"] < 1200) & np.isin(o["custkey"], ck)
    live = (f["shipdate"] > 1200) & np.isin(f["fk"], o["orderkey"][om])
    assert int(got["cols"][3].sum()) == int(live.sum())
    assert _wsum(got["cols"][2]) == _wsum(f["price"][live] * (100 - f["discount"][live]))
    assert got["n"] == len(np.unique(f["fk"][live]))
    # I4: every emitted (orderkey, orderdate) pair is the orders table's pair
    srt = np.argsort(o["orderkey"])
    pos = srt[np.searchsorted(o["orderkey"][srt], got["cols"][0])]
    assert np.array_equal(o["orderdate"][pos].astype(np.int64), got["cols"][1])

    def rows_of(pick):
        fm, omk = np.isin(f["fk"], pick), np.isin(o["orderkey"], pick)
        cm = np.isin(c["key"], o["custkey"][omk])
        return plans.plan_c4({"cust": {k: v[cm] for k, v in c.items()}, "orders": {k: v[omk] for k, v in o.items()},
                              "fact": {k: v[fm] for k, v in f.items()}})
    _sample_check(plan, got, 2, rows_of, np.random.default_rng(4))
    _check_digest(4, got)                                                              # the whole 1.3 M-row table
    _check_digest(4, _gpu(plans.plan_c4(t), ctx))                                      # upper-bound sizing: same table
    _check_digest(4, _gpu(_dense(plans.plan_c4(t), [1 / 5, (1200 / 2406) / 5]), ctx))                              # bench.py's configuration: direct-address tables


def test_c5_full_size(ctx):
    t = datagen.make_config(5)
    plan = plans.plan_c5(t, max_groups=datagen.ROWS[5]["keys"])                       # bench.py: the key-domain bound
    got = _gpu(plan, ctx)                                                             # radix-clustered path at this size
    f = t["fact"]
    live = f["shipdate"] < 2000
    assert int(got["cols"][5].sum()) == int(live.sum())                               # I1
    assert _wsum(got["cols"][1]) == _wsum(f["price"][live]) and _wsum(got["cols"][2]) == _wsum(f["quantity"][live])   # I3
    assert int(got["cols"][3].min()) == int(f["price"][live].min()) and int(got["cols"][4].max()) == int(f["price"][live].max())
    assert np.all(got["cols"][3] * got["cols"][5] <= got["cols"][1]) and np.all(got["cols"][1] <= got["cols"][4] * got["cols"][5])
    assert np.all(np.diff(got["cols"][0]) > 0)                                        # distinct keys (sorted output)

    def rows_of(pick):
        m = np.isin(f["key"], pick)
        return plans.plan_c5({"fact": {k: v[m] for k, v in f.items()}}, max_groups=len(pick))
    rng = np.random.default_rng(5)
    keys = got["cols"][0]
    hot = keys[np.argsort(got["cols"][5])[-6:]]                                       # the most frequent keys too
    pick_extra = np.concatenate([hot, keys[rng.integers(0, len(keys), 40)]])
    sub = rows_of(np.unique(pick_extra))
    exp = oracle.run_query(sub)
    sel = np.isin(keys, pick_extra)
    assert exp.nrows == int(sel.sum())
    for c in range(len(exp.cols)):
        assert np.array_equal(got["cols"][c][sel], exp.cols[c]), f"sampled groups: column {c} differs"
    _check_digest(5, got)                                                              # the whole 34.2 M-row table
