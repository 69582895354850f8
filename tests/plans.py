"""Neutral (library-free) descriptions of the five BASELINE.json configs as query plans.

A plan is plain Python data (see oracle/__init__.py for the format); tests hand the same plan to the oracle and, via
``tests/gqrun.py``, to the CUDA library.  Nothing here computes anything.
"""
from __future__ import annotations

# expression helpers (postfix)
def col(i): return ("col", i)
def const(v): return ("const", v)
ADD, SUB, MUL = ("add",), ("sub",), ("mul",)


def disc_price(price, disc):            # price*(100-discount)
    return [col(price), const(100), col(disc), SUB, MUL]


def charge(price, disc, tax):           # price*(100-discount)*(100+tax)
    return disc_price(price, disc) + [const(100), col(tax), ADD, MUL]


def plan_c1(t):
    """C1: fused filter + low-cardinality group-by (BASELINE.json configs[0])."""
    f = t["fact"]
    cols = [f["shipdate"], f["quantity"], f["price"], f["discount"], f["tax"], f["flagA"], f["flagB"]]
    return dict(table=cols, preds=[(0, "le", 2430)],
                exprs=[[col(1)], [col(2)], disc_price(2, 3), charge(2, 3, 4)],
                keys=[5, 6], aggs=[("sum", 0), ("sum", 1), ("sum", 2), ("sum", 3), ("count",)], max_groups=6)


def plan_c2(t):
    """C2: selective filter + global SUM(price*discount) (configs[1])."""
    f = t["fact"]
    cols = [f["shipdate"], f["discount"], f["quantity"], f["price"]]
    return dict(table=cols, preds=[(0, "range_co", 730, 1095), (1, "range_cc", 5, 7), (2, "lt", 24)],
                exprs=[[col(3), col(1), MUL]], keys=[], aggs=[("sum", 0), ("count",)], max_groups=1)


def plan_c3(t, topk=0):
    """C3: dim JOIN fact, group by key, SUM(price*(100-discount)), COUNT; top-10 by sum (configs[2])."""
    d, f = t["dim"], t["fact"]
    b = dict(table=[d["key"], d["orderdate"]], preds=[(1, "lt", 1200)], probes=[], key=0, payload=[], unique=True)
    cols = [f["fk"], f["shipdate"], f["price"], f["discount"]]
    return dict(builds=[b], table=cols, preds=[(1, "gt", 1200)], probes=[(0, 0)], exprs=[disc_price(2, 3)],
                keys=[0], aggs=[("sum", 0), ("count",)], topk=topk, topk_agg=0, max_groups=len(d["key"]))


def plan_c4(t):
    """C4: cust -> orders -> fact chain, group by (orderkey, orderdate) (configs[3])."""
    c, o, f = t["cust"], t["orders"], t["fact"]
    b0 = dict(table=[c["key"], c["segment"]], preds=[(1, "eq", 1)], probes=[], key=0, payload=[], unique=True)
    b1 = dict(table=[o["orderkey"], o["custkey"], o["orderdate"]], preds=[(2, "lt", 1200)], probes=[(0, 1)], key=0,
              payload=[2], unique=True)
    cols = [f["fk"], f["shipdate"], f["price"], f["discount"]]
    # fact row = 4 own columns ++ payload (orderdate) of build 1 at index 4
    return dict(builds=[b0, b1], table=cols, preds=[(1, "gt", 1200)], probes=[(1, 0)], exprs=[disc_price(2, 3)],
                keys=[0, 4], ndependent=1, aggs=[("sum", 0), ("count",)], max_groups=len(o["orderkey"]))


def plan_c5(t, max_groups=None):
    """C5: Zipf-skewed high-cardinality group-by with five aggregates (configs[4])."""
    f = t["fact"]
    cols = [f["key"], f["shipdate"], f["price"], f["quantity"]]
    return dict(table=cols, preds=[(1, "lt", 2000)], exprs=[[col(2)], [col(3)]], keys=[0],
                aggs=[("sum", 0), ("sum", 1), ("min", 0), ("max", 0), ("count",)],
                max_groups=max_groups if max_groups is not None else len(f["key"]))


PLANS = {1: plan_c1, 2: plan_c2, 3: plan_c3, 4: plan_c4, 5: plan_c5}
