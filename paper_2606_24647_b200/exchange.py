"""Exchange of hash-partitioned column batches between the ranks of a torch.distributed group (SURVEY §8(e), §8(f)
NEXT-4; CudfPartitionedOutput -> exchange -> consumer). One process per GPU; NCCL over NVLink 5 /
NVSwitch on GPUs, gloo for the CPU tests of this host logic.

The data path is: gq_hash_partition (CUDA, csrc/gq_sort.cu) packs every destination's rows into one contiguous range of
the output columns -> the per-destination row counts are exchanged (one small all-to-all: the "metadata" message of
PAPER.md:174) -> every packed column is exchanged with ONE all-to-all of unequal splits, straight from / into device
memory ("cudf columns gathered into contiguous memory", no host staging). What a rank receives is ordered by sending
rank, and inside one sender by that sender's input order: the result is unique.

Nothing here computes: partitioning happens in the CUDA kernel, this module only moves bytes. north_star keeps the
benchmarked path on one GPU ("replicas only"); this is the building block of the paper's
Partial -> exchange -> Final split, exercised by tests/test_exchange.py (world_size 2, gloo) and, with one rank, on the GPU.
"""
from __future__ import annotations

import torch
import torch.distributed as td


def exchange_partitioned(cols, offsets, group=None):
    """cols: this rank's packed columns (rows of destination d = cols[c][offsets[d]:offsets[d + 1]], d = rank in the
    group); offsets: int64[world + 1] tensor (any device) or sequence. -> (received columns, recv_counts): the rows every
    rank sent to this one, by sending rank; recv_counts[s] = rows that came from rank s. Collective: all ranks call it
    with the same number and dtypes of columns."""
    world = td.get_world_size(group)
    off = offsets.detach().to("cpu", torch.int64) if torch.is_tensor(offsets) else torch.tensor(list(offsets), dtype=torch.int64)
    if off.numel() != world + 1:
        raise ValueError(f"offsets must hold world_size + 1 = {world + 1} entries, got {off.numel()}")
    send_counts = off[1:] - off[:-1]
    if int(off[0]) != 0 or bool((send_counts < 0).any()):
        raise ValueError("offsets must start at 0 and be non-decreasing")
    for c in cols:
        if c.numel() < int(off[-1]):
            raise ValueError("a column is shorter than offsets[-1]")
    dev = cols[0].device if cols else torch.device("cpu")
    recv_counts = torch.empty(world, dtype=torch.int64, device=dev)
    td.all_to_all_single(recv_counts, send_counts.to(dev), group=group)          # metadata first: how much to expect
    recv_counts = recv_counts.cpu()
    n_in = int(recv_counts.sum())
    outs = []
    for c in cols:
        eb = c.element_size()
        send = c.contiguous().view(torch.uint8)[: int(off[-1]) * eb]              # raw bytes: any column dtype, any backend
        recv = torch.empty(n_in * eb, dtype=torch.uint8, device=c.device)
        td.all_to_all_single(recv, send, output_split_sizes=[int(x) * eb for x in recv_counts],
                             input_split_sizes=[int(x) * eb for x in send_counts], group=group)
        outs.append(recv.view(c.dtype))
    return outs, recv_counts


def hash_exchange(ctx, cols, key_cols, group=None):
    """PartitionedOutput + exchange in one call: hash-partition the device columns `cols` by `key_cols` to world_size
    destinations (gq_hash_partition: equal keys meet on one rank, whoever sends them) and exchange the packed ranges.
    -> (received columns, recv_counts). The partition kernel and the collectives are ordered on the context's stream."""
    world = td.get_world_size(group)
    outs, offsets, _ = ctx.hash_partition(cols, key_cols, world)
    with torch.cuda.stream(ctx.stream):
        return exchange_partitioned(outs, offsets, group)
