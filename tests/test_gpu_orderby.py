"""OrderBy / TopN (-m gpu): gq_order_by against the oracle's std::stable_sort, element by element.
The order is total (ties broken by input position), so row numbers and gathered columns are compared bit-exactly."""
import numpy as np
import pytest

import oracle
from golden_util import load, table

pytestmark = pytest.mark.gpu
G = load()


@pytest.fixture(scope="module")
def ctx():
    from paper_2606_24647_b200 import build as gqbuild
    gqbuild.build()
    from paper_2606_24647_b200 import gq
    return gq.Context()


def check(ctx, cols, keys, limit=0, gather=True):
    import gqrun
    exp = oracle.order_by(cols, keys, limit)
    index, outs = ctx.order_by(gqrun.dev(cols), keys, limit=limit, gather=gather)
    ctx.sync()
    assert index.numel() == exp.nrows
    assert np.array_equal(index.cpu().numpy(), exp.cols[0]), f"row order differs (keys {keys}, limit {limit})"
    if gather:
        for j, o in enumerate(outs):
            assert o.dtype == gqrun.dev([cols[j][:1]])[0].dtype
            assert np.array_equal(o.cpu().numpy().astype(np.int64), exp.cols[1 + j]), f"gathered column {j} differs"


def test_T8_worked_example(ctx):
    t = table(G["T8"]["cols"], G["T8"]["rows"])
    cols = [t["a"], t["b"]]
    check(ctx, cols, [tuple(k) for k in G["T8"]["keys"]])
    check(ctx, cols, [tuple(k) for k in G["T8"]["keys"]], limit=4)
    check(ctx, cols, [tuple(k) for k in G["T8"]["keys_b_desc_only"]])
    check(ctx, cols, [])
    import gqrun
    index, _ = ctx.order_by(gqrun.dev(cols), [tuple(k) for k in G["T8"]["keys"]], limit=4, gather=False)
    ctx.sync()
    assert index.cpu().tolist() == G["T8"]["expect_index_limit4"]


@pytest.mark.parametrize("n", [1, 2, 255, 256, 257, 2048, 2049, 5000, 70_001, 300_007])
def test_sizes_dtypes_and_ties(ctx, n):
    rng = np.random.default_rng(n)
    a = rng.integers(-3, 3, n).astype(np.int8)                      # heavy ties
    b = rng.integers(-1000, 1000, n).astype(np.int32)
    c = rng.integers(-2**62, 2**62, n).astype(np.int64)
    c[::5] = c[0]
    if n > 10:
        c[3], c[4] = np.iinfo(np.int64).min, np.iinfo(np.int64).max
        b[7], b[8] = np.iinfo(np.int32).min, np.iinfo(np.int32).max
        a[1], a[2] = -128, 127
    for keys in ([(0, False)], [(2, True)], [(0, True), (1, False)], [(1, False), (0, True), (2, True)]):
        check(ctx, [a, b, c], keys)
    check(ctx, [a, b, c], [(2, False), (1, True)], limit=max(1, n // 3))
    check(ctx, [a, b, c], [(0, False)], limit=n + 5)                # limit beyond the row count: all rows


def test_topn_selects_candidates_on_device(ctx):
    # limit << rows takes the radix-select path: candidates are picked on keys[0] in two 12-bit levels, also when the
    # threshold falls inside a long run of equal keys (the tie is then decided by the later keys / input position)
    rng = np.random.default_rng(91)
    n = 1_000_003
    wide = rng.integers(-2**40, 2**40, n).astype(np.int64)
    narrow = rng.integers(0, 50, n).astype(np.int32)                # 20 000 rows per value: the top-100 all tie on it
    tiny = rng.integers(-2, 2, n).astype(np.int8)
    other = rng.integers(-10**6, 10**6, n).astype(np.int64)
    for keys, limit in (([(0, True)], 10), ([(0, False)], 1000), ([(1, False), (3, True)], 100), ([(2, True), (0, False)], 4096),
                        ([(1, True)], 100_000), ([(3, False), (1, False)], 1)):
        check(ctx, [wide, narrow, tiny, other], keys, limit=limit)
    # keys that share a long prefix of bits: small non-negative int64 values (prices, counts), values that differ only in
    # their low bits, and both with ties at the threshold — the select's two levels start below the common prefix
    price = rng.integers(0, 10**7, n).astype(np.int64)
    offset = (2**50 + rng.integers(0, 1000, n)).astype(np.int64)
    negs = (-(2**40) - rng.integers(0, 5000, n)).astype(np.int64)
    for keys, limit in (([(0, True)], 100), ([(0, False)], 100), ([(1, False), (0, True)], 64), ([(2, True)], 3000), ([(2, False), (1, True)], 7)):
        check(ctx, [price, offset, negs, other], keys, limit=limit)
    same = np.full(200_000, 7, np.int64)                            # one key value only: every row is a candidate
    check(ctx, [same, other[:200_000]], [(0, True)], limit=5)
    check(ctx, [same, other[:200_000]], [(0, False), (1, True)], limit=5)


def test_order_by_the_output_of_a_group_by(ctx):
    # the plan shape of PAPER.md Fig. 2: HashAggregation -> OrderBy/TopN over its output columns (several sort keys,
    # any k: the top-k finaliser of gq_hash_aggregate_finish handles one aggregate and k <= 32)
    import gqrun
    import plans
    from paper_2606_24647_b200 import datagen
    plan = plans.plan_c3(datagen.make_config(3, scale=0.01))
    exp = oracle.run_query(plan)
    got = gqrun.run_query(plan, ctx=ctx)
    cols = [got["cols"][2], got["cols"][1], got["cols"][0]]        # count, sum, key
    check(ctx, cols, [(0, True), (1, True), (2, False)], limit=500)
    top = oracle.run_query(dict(plan, topk=10, topk_agg=0))
    index, outs = ctx.order_by(gqrun.dev([got["cols"][1], got["cols"][0]]), [(0, True), (1, False)], limit=10)
    ctx.sync()
    assert np.array_equal(outs[1].cpu().numpy(), top.cols[0]) and np.array_equal(outs[0].cpu().numpy(), top.cols[1])


def test_order_by_errors(ctx):
    import gqrun
    from paper_2606_24647_b200 import gq
    cols = gqrun.dev([np.arange(10, dtype=np.int64)])
    with pytest.raises(gq.GqError):
        ctx.order_by(cols, [(3, False)])
    index, outs = ctx.order_by(gqrun.dev([np.zeros(0, np.int64)]), [(0, False)])
    assert index.numel() == 0


def test_passes_over_constant_bytes_are_skipped_on_the_device(ctx):
    # a radix pass over a byte in which all keys agree is skipped by the kernels themselves, and which of the two buffers
    # holds the data is derived from the keys' bit masks: key columns with 0, 1, 2, 3 and 8 live bytes, in every order,
    # so that the number of executed passes is odd and even, also on the TopN path and in the static-scratch entry point
    import torch
    import gqrun
    rng = np.random.default_rng(123)
    n = 150_001
    const = np.full(n, -12345, np.int64)                                     # no live byte: nothing moves
    one = rng.integers(0, 200, n).astype(np.int64)                           # 1 live byte
    two = (2**45 + rng.integers(0, 60_000, n)).astype(np.int64)              # 2 live bytes below a constant prefix
    three = rng.integers(0, 2**24, n).astype(np.int32)                       # 3 of 4
    full = rng.integers(-2**63, 2**63 - 1, n).astype(np.int64)               # all 8
    mid = ((rng.integers(0, 256, n).astype(np.int64) << 24) + 7)             # one live byte in the middle
    cols = [const, one, two, three, full, mid]
    for keys in ([(0, False)], [(1, True)], [(2, False)], [(3, True)], [(4, False)], [(5, False)],
                 [(1, False), (2, True)], [(2, True), (1, False), (0, True)], [(5, True), (3, False)], [(3, False), (5, True), (1, True)],
                 [(0, True), (4, True)], [(1, False), (5, False), (2, False), (3, False)]):
        check(ctx, cols, keys)
        check(ctx, cols, keys, limit=50)                                     # TopN path (n >= 2^16, limit * 8 < n)
    small = [c[:100_000] for c in cols]
    dcols = gqrun.dev(small)
    for keys in ([(0, False)], [(1, True), (5, False)], [(2, False), (3, True), (1, False)]):
        exp = oracle.order_by(small, keys, 0)
        index = torch.empty(100_000, dtype=torch.int64, device="cuda")
        ctx.order_by_static(dcols, keys, 0, index)
        ctx.sync()
        assert np.array_equal(index.cpu().numpy(), exp.cols[0])


@pytest.mark.parametrize("n", [3, 6, 100, 1000, 2047, 2048])
def test_small_inputs_take_one_launch(ctx, n):
    # up to 2048 rows: one CTA sorts the row numbers in shared memory (comparator over the key columns) and gathers the
    # outputs — one launch instead of the radix path's >= 27; heavy ties (stability), every dtype, limits
    import gqrun
    rng = np.random.default_rng(1000 + n)
    a = rng.integers(-2, 2, n).astype(np.int8)
    b = rng.integers(-3, 3, n).astype(np.int32)
    c = rng.integers(-2**62, 2**62, n).astype(np.int64)
    c[::4] = c[0]
    cols = [a, b, c]
    for keys, limit in (([(0, False), (1, True)], 0), ([(2, True)], 0), ([(1, True), (0, False), (2, False)], max(1, n // 2)), ([], 0), ([(0, True)], 1)):
        check(ctx, cols, keys, limit=limit)
    dcols = gqrun.dev(cols)
    l0 = ctx.launch_count()
    ctx.order_by(dcols, [(0, False), (2, True)], limit=0, gather=True)
    ctx.sync()
    assert ctx.launch_count() - l0 == 1
