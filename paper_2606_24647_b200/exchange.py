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


def exchange_layout(counts, group=None):
    """Phase between gq_hash_partition_count and gq_hash_partition_scatter_to: all ranks share their per-destination row
    counts (one all-gather of world int64s per rank); receiver d lays the senders out one after the other. counts:
    int64[world] tensor of this rank. -> (row0 int64[world] CPU tensor: the row of destination d's buffers where THIS
    rank's run starts; recv_counts int64[world] CPU tensor: rows every sender will write into THIS rank's buffers)."""
    world, rank = td.get_world_size(group), td.get_rank(group)
    c = counts.detach().to(torch.int64).reshape(-1)
    if c.numel() != world:
        raise ValueError(f"counts must hold world_size = {world} entries, got {c.numel()}")
    allc = torch.empty(world * world, dtype=torch.int64, device=c.device)
    td.all_gather_into_tensor(allc, c.contiguous(), group=group)
    m = allc.cpu().reshape(world, world)                     # [sender][destination]
    row0 = m[:rank].sum(dim=0) if rank > 0 else torch.zeros(world, dtype=torch.int64)
    return row0, m[:, rank].clone()


def hash_exchange_fused(ctx, cols, key_cols, peer_cols, group=None):
    """Partition fused with its transfer (gq.h: gq_hash_partition_count / _scatter_to): no packed send buffer and no
    all-to-all of the data — after the counts have been shared, the scatter kernel stores every destination's run
    straight into that destination's receive buffers. peer_cols[d][c]: destination d's buffer for column c as a tensor
    THIS process can write — on several GPUs the peers' memory mapped over NVLink (CUDA IPC / symmetric memory; peer_cols
    [rank] are this rank's own buffers), allocated by the caller with room for what exchange_layout announces.
    -> recv_counts (CPU int64[world]): rows[sum(recv_counts[:s]) ...] of this rank's buffers came from sender s. On return
    every rank's scatter has completed (stream synchronised, then a barrier): the receive buffers may be read."""
    world = td.get_world_size(group)
    if len(peer_cols) != world or any(len(p) != len(cols) for p in peer_cols):
        raise ValueError("peer_cols must be [world_size][number of columns]")
    counts, ws = ctx.hash_partition_count(cols, key_cols, world)
    row0, recv_counts = exchange_layout(counts, group)
    for d in range(world):
        need = int(row0[d]) + int(counts[d])
        if any(t.numel() < need or t.dtype != c.dtype for t, c in zip(peer_cols[d], cols)):
            raise ValueError(f"destination {d}: receive buffers too small or of the wrong dtype (need {need} rows)")
    ctx.hash_partition_scatter_to(cols, key_cols, world, ws, peer_cols, row0.to(cols[0].device))
    ctx.sync()
    td.barrier(group=group)
    return recv_counts
