"""Exchange of hash-partitioned batches between ranks (paper_2606_24647_b200/exchange.py; SURVEY §8(e), NEXT-4;
PAPER.md:154, :160-174) on CPU: world_size 2 over gloo. The partitions come from the oracle's hash_partition (the CUDA
kernel is compared with it in tests/test_gpu_partition.py), so this file checks the host logic alone: counts first, then
one all-to-all of unequal splits per column, rows ordered by sender then input order — and that Partial -> partition ->
exchange -> Final over two ranks gives exactly the single-process answer."""
import os
import sys

import numpy as np
import torch
import torch.distributed as td
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
N, WORLD = 40_000, 2


def _table(rank):
    rng = np.random.default_rng(100 + rank)
    k = (rng.zipf(1.5, N) % 3000).astype(np.int64) - 500
    a = rng.integers(-100, 100, N).astype(np.int8)
    b = rng.integers(-10**6, 10**6, N).astype(np.int32)
    v = rng.integers(-10**9, 10**9, N).astype(np.int64)
    return [k, a, b, v]


def _partial_plan(cols):
    return dict(table=[cols[0], cols[3]], preds=[], exprs=[[("col", 1)]], keys=[0],
                aggs=[("sum", 0), ("count",), ("min", 0), ("max", 0)], max_groups=4000)


def _worker(rank, world, port, out):
    sys.path.insert(0, ROOT)
    sys.path.insert(0, os.path.join(ROOT, "tests"))
    import oracle
    from paper_2606_24647_b200 import exchange
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    td.init_process_group("gloo", rank=rank, world_size=world)
    try:
        # (1) raw rows: partition this rank's table by its key column, exchange, return what arrived
        cols = _table(rank)
        part = oracle.hash_partition(cols, [0], world)
        offsets = np.searchsorted(part.cols[0], np.arange(world + 1))
        packed = [torch.from_numpy(part.cols[2 + j].astype(c.dtype)) for j, c in enumerate(cols)]
        got, counts = exchange.exchange_partitioned(packed, torch.from_numpy(offsets), None)
        # (2) Partial -> partition the partial groups -> exchange -> Final
        pr = oracle.run_query(_partial_plan(cols))
        ppart = oracle.hash_partition(pr.cols, [0], world)
        poff = np.searchsorted(ppart.cols[0], np.arange(world + 1))
        recv, _ = exchange.exchange_partitioned([torch.from_numpy(ppart.cols[2 + j]) for j in range(5)], list(poff), None)
        recv = [r.numpy() for r in recv]
        final = oracle.run_query(dict(table=recv, preds=[], exprs=[[("col", 1)], [("col", 2)], [("col", 3)], [("col", 4)]],
                                      keys=[0], aggs=[("sum", 0), ("sum", 1), ("min", 2), ("max", 3)], max_groups=4000))
        # (3) argument checks are local (no collective is entered)
        bad = 0
        for off in ([0, 1], [1, 2, 3], [0, 5, 3]):
            try:
                exchange.exchange_partitioned([torch.zeros(8, dtype=torch.int64)], off, None)
            except ValueError:
                bad += 1
        # (4) layout of the fused variant: every rank announces its counts, gets the first row of its runs
        mine = torch.from_numpy(np.diff(offsets).astype(np.int64))
        row0, rc = exchange.exchange_layout(mine, None)
        out.put((rank, [g.numpy() for g in got], counts.tolist(), [c.copy() for c in final.cols], bad, row0.tolist(), rc.tolist()))
        td.barrier()
    finally:
        td.destroy_process_group()


def test_two_ranks_exchange_rows_and_partial_groups():
    sys.path.insert(0, ROOT)
    import oracle
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = 31000 + os.getpid() % 2000
    ps = [ctx.Process(target=_worker, args=(r, WORLD, port, q)) for r in range(WORLD)]
    for p in ps:
        p.start()
    res = sorted((q.get(timeout=180) for _ in ps), key=lambda x: x[0])
    for p in ps:
        p.join(timeout=60)
        assert p.exitcode == 0
    tables = [_table(r) for r in range(WORLD)]
    dests = []
    for t in tables:                                       # destination of every input row of every sender
        part = oracle.hash_partition(t, [0], WORLD)
        d = np.empty(N, np.int64); d[part.cols[1]] = part.cols[0]
        dests.append(d)
    whole = oracle.run_query(_partial_plan([np.concatenate([t[j] for t in tables]) for j in range(4)]))
    whole_part = oracle.hash_partition([whole.cols[0]], [0], WORLD)
    owner = np.empty(whole.nrows, np.int64); owner[whole_part.cols[1]] = whole_part.cols[0]
    seen = 0
    cm = np.array([[int((dests[s] == d).sum()) for d in range(WORLD)] for s in range(WORLD)])     # [sender][destination]
    for rank, got, counts, final_cols, bad, row0, rc in res:
        assert bad == 3
        assert row0 == (np.cumsum(cm, axis=0) - cm)[rank].tolist() and rc == cm[:, rank].tolist()
        assert counts == [int((dests[s] == rank).sum()) for s in range(WORLD)]
        for j in range(4):                                 # rows by sender, input order inside a sender, whole rows together
            want = np.concatenate([tables[s][j][dests[s] == rank] for s in range(WORLD)])
            assert got[j].dtype == tables[0][j].dtype and np.array_equal(got[j], want), f"rank {rank} column {j}"
        sel = owner == rank                                # this rank's Final groups = the whole answer's groups it owns
        assert len(final_cols[0]) == int(sel.sum())
        for j in range(5):
            assert np.array_equal(final_cols[j], whole.cols[j][sel]), f"rank {rank} final column {j}"
        seen += len(final_cols[0])
    assert seen == whole.nrows
