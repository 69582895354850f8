"""hash_exchange on the GPU with ONE rank over NCCL (-m gpu; this box has one GPU): gq_hash_partition feeds
torch.distributed.all_to_all_single from device memory. With world_size 1 every row's destination is rank 0, so the call
must return the input, in input order, through the real kernel + NCCL path. The two-rank logic is covered on CPU
(tests/test_exchange.py), the kernel for up to 256 destinations in tests/test_gpu_partition.py. Collected late on purpose:
a box without a working NCCL must not hide the kernel tests (the run uses pytest -x)."""
import os

import numpy as np
import pytest

pytestmark = pytest.mark.gpu


def test_single_rank_hash_exchange_returns_the_input():
    import torch
    import torch.distributed as td
    from paper_2606_24647_b200 import build as gqbuild
    gqbuild.build()
    from paper_2606_24647_b200 import exchange, gq
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(33000 + os.getpid() % 2000))
    torch.cuda.set_device(0)
    td.init_process_group("nccl", rank=0, world_size=1)
    try:
        ctx = gq.Context()
        rng = np.random.default_rng(3)
        n = 300_001
        cols = [rng.integers(-2**62, 2**62, n).astype(np.int64), rng.integers(-100, 100, n).astype(np.int8),
                rng.integers(-10**6, 10**6, n).astype(np.int32)]
        dcols = [torch.from_numpy(c).cuda() for c in cols]
        for _ in range(2):
            got, counts = exchange.hash_exchange(ctx, dcols, [0, 2])
            ctx.sync()
            torch.cuda.synchronize()
            assert counts.tolist() == [n]
            for g, c in zip(got, cols):
                assert g.dtype == torch.from_numpy(c[:1]).dtype and np.array_equal(g.cpu().numpy(), c)
        # the fused variant: counts -> layout (all-gather) -> the scatter stores into the destination's own buffers
        recv = [[torch.full((n + 8,), -5, dtype=c.dtype, device="cuda") for c in dcols]]
        for _ in range(2):
            rc = exchange.hash_exchange_fused(ctx, dcols, [0, 2], recv)
            assert rc.tolist() == [n]
            for g, c in zip(recv[0], cols):
                assert np.array_equal(g[:n].cpu().numpy(), c) and bool((g[n:] == -5).all())
        with pytest.raises(ValueError):
            exchange.hash_exchange_fused(ctx, dcols, [0], [[torch.empty(10, dtype=c.dtype, device="cuda") for c in dcols]])
    finally:
        td.destroy_process_group()
