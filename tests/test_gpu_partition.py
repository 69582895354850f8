"""Hash partitioning (-m gpu): gq_hash_partition (the GPU side of PartitionedOutput; PAPER.md:160,
:174) against the oracle's definition, element by element. Destination-major with input order inside a destination is a
unique result, so offsets, row numbers and every moved column are compared bit-exactly."""
import numpy as np
import pytest

import oracle

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def ctx():
    from paper_2606_24647_b200 import build as gqbuild
    gqbuild.build()
    from paper_2606_24647_b200 import gq
    return gq.Context()


def check(ctx, cols, key_cols, nparts):
    import gqrun
    exp = oracle.hash_partition(cols, key_cols, nparts)
    outs, offsets, rows = ctx.hash_partition(gqrun.dev(cols), key_cols, nparts, want_rows=True)
    ctx.sync()
    n = len(cols[0])
    want_off = np.searchsorted(exp.cols[0], np.arange(nparts + 1), side="left")     # first output row of every destination
    assert np.array_equal(offsets.cpu().numpy(), want_off), f"offsets differ (n {n}, keys {key_cols}, nparts {nparts})"
    assert np.array_equal(rows.cpu().numpy(), exp.cols[1]), f"row order differs (n {n}, keys {key_cols}, nparts {nparts})"
    for j, o in enumerate(outs):
        assert o.numel() == n and np.array_equal(o.cpu().numpy().astype(np.int64), exp.cols[2 + j]), f"column {j} differs"
    return offsets.cpu().numpy()


def _cols(n, seed):
    rng = np.random.default_rng(seed)
    a = rng.integers(-100, 100, n).astype(np.int8)
    b = rng.integers(-50_000, 50_000, n).astype(np.int32)
    c = rng.integers(-2**62, 2**62, n).astype(np.int64)
    d = np.arange(n, dtype=np.int64) * 3 - 7
    return [a, b, c, d]


@pytest.mark.parametrize("n", [1, 31, 32, 33, 127, 128, 129, 4096, 4097, 75_777, 1_000_003])
def test_sizes_span_chunks_and_ragged_tails(ctx, n):
    cols = _cols(n, n)
    check(ctx, cols, [1], 8)
    check(ctx, cols, [2, 0], 7)


@pytest.mark.parametrize("nparts", [1, 2, 3, 16, 64, 255, 256])
def test_destination_counts(ctx, nparts):
    cols = _cols(200_001, nparts)
    off = check(ctx, cols, [2], nparts)
    assert off[0] == 0 and off[-1] == 200_001
    check(ctx, cols, [0], nparts)                       # 200 distinct int8 keys: many empty destinations


def test_key_dtypes_multi_key_and_degenerate_inputs(ctx):
    cols = _cols(50_000, 5)
    for keys in ([0], [1], [2], [3], [0, 1, 2, 3], [3, 3], [1, 0, 1, 0, 1, 0, 1, 0]):
        check(ctx, cols, keys, 13)
    # every row to one destination; extreme values; the seed itself (h = fmix64(0) = 0: destination 0)
    one = [np.full(70_000, 42, np.int64), np.arange(70_000, dtype=np.int32)]
    off = check(ctx, one, [0], 32)
    assert np.count_nonzero(np.diff(off)) == 1
    ext = np.array([np.iinfo(np.int64).min, np.iinfo(np.int64).max, -1, 0, 1] * 100, np.int64)
    ext[::7] = np.array([0x9E3779B97F4A7C15], np.uint64).view(np.int64)[0]
    check(ctx, [ext, np.arange(500, dtype=np.int8)], [0], 5)
    check(ctx, [ext, np.arange(500, dtype=np.int8)], [0], 1 << 8)


def test_empty_input_and_argument_errors(ctx):
    import torch
    from paper_2606_24647_b200 import gq
    outs, offsets, rows = ctx.hash_partition([torch.empty(0, dtype=torch.int64, device="cuda")], [0], 4, want_rows=True)
    ctx.sync()
    assert offsets.cpu().tolist() == [0, 0, 0, 0, 0]
    col = torch.arange(100, dtype=torch.int64, device="cuda")
    for keys, nparts, what in (([0], 257, "GQ_ERR_UNSUPPORTED"), ([0], 0, "GQ_ERR_INVALID_ARG"), ([1], 4, "GQ_ERR_INVALID_ARG"),
                               ([], 4, "GQ_ERR_INVALID_ARG"), ([0] * 9, 4, "GQ_ERR_INVALID_ARG")):
        with pytest.raises(gq.GqError) as ei:
            ctx.hash_partition([col], keys, nparts)
        assert what in str(ei.value), (keys, nparts, str(ei.value))
    ctx.sync()
    check(ctx, [col.cpu().numpy()], [0], 4)             # the context stays usable


def test_partitions_feed_partial_to_final_aggregation(ctx):
    # the use the paper makes of it: Partial aggregation -> partition the partial groups by key ->
    # (exchange) -> Final aggregation per destination. Here the "exchange" is a slice: every destination's Final result
    # must be exactly the oracle's groups whose key maps to that destination, and together they are the whole answer.
    import torch
    import gqrun
    rng = np.random.default_rng(12)
    n, nparts = 300_000, 4
    k = (rng.zipf(1.4, n) % 20_000).astype(np.int64) - 3000
    v = rng.integers(-10**6, 10**6, n).astype(np.int64)
    plan = dict(table=[k, v], preds=[], exprs=[[("col", 1)]], keys=[0], aggs=[("sum", 0), ("count",), ("min", 0), ("max", 0)],
                max_groups=20_000)
    whole = oracle.run_query(plan)
    dest_of = {}
    part = oracle.hash_partition([whole.cols[0]], [0], nparts)
    for d, r in zip(part.cols[0], part.cols[1]):
        dest_of[int(whole.cols[0][r])] = int(d)
    # two "workers" aggregate half of the rows each (Partial), each partitions its partial groups, destination d gets both
    halves = []
    for sl in (slice(0, n // 2 + 16), slice(n // 2 + 16, n)):
        p = dict(plan, table=[k[sl], v[sl]])
        r = gqrun.run_query(p, ctx=ctx)
        cols = [torch.from_numpy(c).cuda() for c in r["cols"]]
        outs, offsets, _ = ctx.hash_partition(cols, [0], nparts)
        ctx.sync()
        halves.append(([o.cpu().numpy() for o in outs], offsets.cpu().numpy()))
    seen = 0
    for d in range(nparts):
        recv = [np.concatenate([h[0][j][h[1][d]:h[1][d + 1]] for h in halves]) for j in range(5)]
        final = dict(table=recv, preds=[], exprs=[[("col", 1)], [("col", 2)], [("col", 3)], [("col", 4)]], keys=[0],
                     aggs=[("sum", 0), ("sum", 1), ("min", 2), ("max", 3)], max_groups=20_000)
        got = gqrun.run_query(final, ctx=ctx)
        sel = np.array([dest_of[int(x)] == d for x in whole.cols[0]])
        assert got["n"] == int(sel.sum())
        for j in range(5):
            assert np.array_equal(got["cols"][j], whole.cols[j][sel]), f"destination {d}, column {j}"
        seen += got["n"]
    assert seen == whole.nrows


@pytest.mark.parametrize("nparts", [5, 200])
def test_count_then_scatter_into_destination_buffers(ctx, nparts):
    # the fused partition + transfer protocol on one GPU: three "senders" (batches) count, the counts are laid out per
    # destination (sender after sender: what an exchange of counts gives every rank), then every sender scatters straight
    # into the destinations' own buffers — separate allocations here, peer-mapped memory on several GPUs. Destination d
    # must end up with exactly the oracle's rows of destination d: by sender, input order inside a sender.
    import torch
    import gqrun
    rng = np.random.default_rng(21)
    sizes = (70_001, 4_097, 33)                                    # (200 destinations: the 512-thread kernels)
    senders = []
    for i, n in enumerate(sizes):
        cols = _cols(n, 300 + i)
        cols[2][::3] = cols[2][0]                                   # repeated keys across senders meet on one destination
        senders.append(cols)
    keys = [2, 0]
    dcols = [gqrun.dev(c) for c in senders]
    counts, wss = [], []
    for dc in dcols:
        c, ws = ctx.hash_partition_count(dc, keys, nparts)
        counts.append(c); wss.append(ws)
    ctx.sync()
    cm = torch.stack(counts).cpu().numpy()                           # [sender][destination]
    exp = [oracle.hash_partition(c, keys, nparts) for c in senders]
    for s, e in enumerate(exp):
        assert np.array_equal(cm[s], np.bincount(e.cols[0], minlength=nparts))
    row0 = np.cumsum(cm, axis=0) - cm                                # first row of sender s in destination d's buffers
    total = cm.sum(axis=0)
    dst = [[torch.full((int(total[d]) + 16,), -99, dtype=c.dtype, device="cuda") for c in dcols[0]] for d in range(nparts)]
    for s, dc in enumerate(dcols):
        ctx.hash_partition_scatter_to(dc, keys, nparts, wss[s], dst, torch.from_numpy(row0[s].copy()).cuda())
    ctx.sync()
    for d in range(nparts):
        for j in range(4):
            want = np.concatenate([e.cols[2 + j][e.cols[0] == d] for e in exp])
            got = dst[d][j].cpu().numpy().astype(np.int64)
            assert np.array_equal(got[:len(want)], want), f"destination {d}, column {j}"
            assert np.all(got[len(want):] == -99)                    # nothing written past the destination's rows
    # an empty sender and argument errors
    from paper_2606_24647_b200 import gq
    c0, ws0 = ctx.hash_partition_count([t[:0] for t in dcols[0]], keys, nparts)
    ctx.sync()
    assert c0.cpu().tolist() == [0] * nparts
    with pytest.raises(gq.GqError):
        ctx.hash_partition_count(dcols[0], [9], nparts)
