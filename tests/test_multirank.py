"""N > 1 accounting of bench.py (replicas only) on CPU: world_size 2 over gloo."""
import os
import sys

import torch
import torch.distributed as td
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _worker(rank, world, port, out):
    sys.path.insert(0, ROOT)
    import bench
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    td.init_process_group("gloo", rank=rank, world_size=world)
    assert bench.dist()[:2] == (world, rank)
    local_ms = 10.0 if rank == 0 else 25.0                     # the slower rank decides the job's time
    ms, value = bench.whole_job_value(local_ms, 1000, 5, td)
    out.put((rank, ms, value))
    td.barrier()
    td.destroy_process_group()


def test_replicas_take_max_over_ranks_and_sum_rows():
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = 29500 + os.getpid() % 2000
    ps = [ctx.Process(target=_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in ps:
        p.start()
    res = sorted(q.get(timeout=120) for _ in ps)
    for p in ps:
        p.join(timeout=60)
        assert p.exitcode == 0
    for _, ms, value in res:
        assert ms == 5.0                                       # max(10, 25) / 5 steps
        assert value == 2 * 1000 / 5.0 * 1e3                   # both ranks' rows over the slower rank's time


def test_single_process_value():
    sys.path.insert(0, ROOT)
    import bench
    assert bench.whole_job_value(8.0, 400, 4) == (2.0, 400 / 2.0 * 1e3)
    assert bench.parse_configs("1,1x64,5", 0.5) == [("C1", 1, 1.0), ("C1x64", 1, 64.0), ("C5", 5, 0.5)]
