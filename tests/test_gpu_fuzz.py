"""Randomised plan shapes (-m gpu): seeded random filters, projections, join chains (hash tables with unique or duplicate
keys, direct-address tables) and group-bys of every kind, each compared element by element with the oracle. Every plan
shape is compiled by the plan compiler on the spot, so this also exercises code-generation paths no hand-written test
names."""
import numpy as np
import pytest

import oracle

pytestmark = pytest.mark.gpu
DT = [np.int8, np.int32, np.int64]
OPS = ["lt", "le", "gt", "ge", "eq", "ne", "range_co", "range_cc"]


@pytest.fixture(scope="module")
def ctx():
    from paper_2606_24647_b200 import build as gqbuild
    gqbuild.build()
    from paper_2606_24647_b200 import gq
    return gq.Context()


def _col(rng, n, dt, lo=None, hi=None):
    info = np.iinfo(dt)
    lo = max(info.min, -50 if lo is None else lo)
    hi = min(info.max, 50 if hi is None else hi)
    return rng.integers(lo, hi + 1, n).astype(dt)


def _pred(rng, c):
    """a predicate most rows pass (columns hold -50..50), so that the plans keep rows to join and group"""
    op = OPS[rng.integers(0, len(OPS))]
    if op in ("lt", "le"):
        return (c, op, int(rng.integers(0, 45)))
    if op in ("gt", "ge"):
        return (c, op, int(rng.integers(-45, 0)))
    if op == "eq":
        return (c, op, int(rng.integers(-3, 3)))
    if op == "ne":
        return (c, op, int(rng.integers(-50, 50)))
    return (c, op, int(rng.integers(-45, -5)), int(rng.integers(5, 45)))


def _expr(rng, ncols, depth=0):
    """postfix token list over columns [0, ncols)"""
    r = rng.random()
    if depth >= 2 or r < 0.35:
        return [("col", int(rng.integers(0, ncols)))] if rng.random() < 0.8 else [("const", int(rng.integers(-1000, 1000)))]
    op = [("add",), ("sub",), ("mul",)][rng.integers(0, 3)]
    return _expr(rng, ncols, depth + 1) + _expr(rng, ncols, depth + 1) + [op]


def _random_plan(seed):
    rng = np.random.default_rng(seed)
    n = int(rng.choice([0, 1, 777, 5000, 40_000, 150_001], p=[0.04, 0.04, 0.12, 0.3, 0.3, 0.2]))
    ncols = int(rng.integers(2, 6))
    cols = [_col(rng, n, DT[rng.integers(0, 3)]) for _ in range(ncols)]
    preds = [_pred(rng, int(rng.integers(0, ncols))) for _ in range(int(rng.integers(0, 3)))]
    builds, probes, width = [], [], ncols
    for _ in range(int(rng.integers(0, 3))):                        # 0..2 join steps
        nb = int(rng.choice([1, 50, 3000], p=[0.1, 0.3, 0.6]))
        kind = rng.choice(["unique", "dense", "multi"])
        bkey = (rng.permutation(200)[:min(nb, 200)] - 100).astype(np.int64) if kind != "multi" else _col(rng, nb, np.int64, -60, 60)
        nb = len(bkey)
        pay = _col(rng, nb, DT[rng.integers(0, 3)])
        bsel = _col(rng, nb, np.int8, 0, 9)
        b = dict(table=[bkey, pay, bsel], preds=[(2, "lt", 9)], key=0, payload=[1] if rng.random() < 0.7 else [], unique=kind != "multi",
                 max_rows=nb)
        if kind == "dense":
            b["dense_range"] = (-100, 99)
        builds.append(b)
        kc = int(rng.integers(0, width))
        probes.append((len(builds) - 1, kc))
        width += len(b["payload"])
    exprs = [_expr(rng, width) for _ in range(int(rng.integers(1, 4)))]
    aggs = []
    for _ in range(int(rng.integers(1, 5))):
        a = rng.choice(["sum", "min", "max", "count"])
        aggs.append(("count",) if a == "count" else (str(a), int(rng.integers(0, len(exprs)))))
    shape = rng.choice(["global", "lowcard", "highcard", "highcard2"])
    plan = dict(builds=builds, table=cols, preds=preds, probes=probes, exprs=exprs, aggs=aggs)
    if shape == "global":
        plan.update(keys=[], max_groups=1)
    elif shape == "lowcard":
        small = [c for c in range(ncols) if cols[c].dtype != np.int64]
        if not small:
            cols[0] = _col(rng, n, np.int8, -3, 3)
            small = [0]
        k = int(rng.choice(small))
        cols[k] = (cols[k] % 7).astype(cols[k].dtype)               # <= 13 distinct values
        plan.update(keys=[k], max_groups=16)
    else:
        keys = [int(rng.integers(0, width))]
        if shape == "highcard2":
            k2 = int(rng.integers(0, ncols))
            if cols[k2].dtype == np.int64:
                cols[k2] = cols[k2].astype(np.int32)
            if keys[0] < ncols and cols[keys[0]].dtype == np.int64:
                cols[keys[0]] = cols[keys[0]].astype(np.int32)
            keys = keys + [k2] if keys[0] != k2 else keys
        plan.update(keys=keys, max_groups=max(64, 101 * 101 + 10))
    return plan


@pytest.mark.parametrize("seed", range(64))
def test_random_plan_equals_oracle(ctx, seed):
    import gqrun
    from paper_2606_24647_b200 import gq
    plan = _random_plan(1000 + seed)
    exp = oracle.run_query(plan)
    try:
        got = gqrun.run_query(plan, ctx=ctx, out_capacity=max(1, exp.nrows) + 3)
    except gq.GqError as e:
        # the only legal refusals: a key tuple wider than 64 bits without a declared dependent key (S17)
        assert e.status == 2 and "dependent" in str(e), str(e)
        return
    assert got["n"] == exp.nrows, f"seed {seed}: {got['n']} groups, oracle {exp.nrows}"
    for c, (g, e) in enumerate(zip(got["cols"], exp.cols)):
        assert np.array_equal(g, e), f"seed {seed}: column {c} differs"
