"""NEXT-2: the paper's distributed scheme on several GPUs of one node.

PAPER.md:103 (Section 3.3): the master counts the partition sizes, every worker holds a full copy of the
reads, gets "a contiguous range of partitions" of about equal total size, sorts it on its own, and "the
pieces can be sent back to the master node" where they are "simply concatenated".  Here every
rank computes the same partition sizes redundantly (one scan, cheaper than a broadcast round trip), a plan made with
shard_index / shard_count sorts only its range and writes it at its final position of the output, and the single
exchange step is an all-gather of the (padded) pieces over torch.distributed (NCCL on GPUs, gloo on CPU tensors in
the tests).  Argument marshalling and the collective only: all arithmetic of the method stays in libcxbwt.so.
"""
from __future__ import annotations

import torch
import torch.distributed as dist


def piece_table(offset: int, count: int, device, group=None) -> list[tuple[int, int]]:
    """(offset, count) of every rank's piece, in rank order (one tiny all-gather)."""
    world = dist.get_world_size(group)
    mine = torch.tensor([int(offset), int(count)], dtype=torch.int64, device=device)
    table = [torch.empty_like(mine) for _ in range(world)]
    dist.all_gather(table, mine, group=group)
    return [(int(t[0]), int(t[1])) for t in table]


def check_pieces(pieces: list[tuple[int, int]], n_total: int) -> None:
    """The pieces of ranks 0..W-1 must tile [0, N) in rank order (concatenation gives the BWT)."""
    at = 0
    for r, (o, c) in enumerate(pieces):
        if c < 0 or (c > 0 and o != at):
            raise RuntimeError(f"shard pieces do not tile the output: rank {r} wrote [{o}, {o + c}), expected to start at {at}")
        at += c
    if at != n_total:
        raise RuntimeError(f"shard pieces cover {at} of {n_total} positions")


def exchange_pieces(out: torch.Tensor, offset: int, count: int, group=None) -> list[tuple[int, int]]:
    """All-gather-v of the BWT pieces, in place: on return every rank holds the whole of `out`.

    out[offset : offset + count] is this rank's piece (cx_bwt_stats_t.shard_offset / shard_suffixes).  Pieces have
    different lengths (partition ranges are equal only roughly), so every rank sends its piece padded to the
    longest one in ONE all_gather_into_tensor and copies the others' pieces from the gathered rows to their places --
    N bytes in total (plus padding), bandwidth-trivial next to the sort."""
    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size(group) == 1:
        check_pieces([(offset, count)], out.numel())
        return [(offset, count)]
    world = dist.get_world_size(group)
    me = dist.get_rank(group)
    pieces = piece_table(offset, count, out.device, group)
    check_pieces(pieces, out.numel())
    longest = max(c for _, c in pieces)
    if longest == 0:
        return pieces
    send = torch.zeros(longest, dtype=out.dtype, device=out.device)
    if count:
        send[:count] = out[offset:offset + count]
    rows = torch.empty(world * longest, dtype=out.dtype, device=out.device)
    dist.all_gather_into_tensor(rows, send, group=group)
    for r, (o, c) in enumerate(pieces):
        if c and r != me:
            out[o:o + c] = rows[r * longest: r * longest + c]
    return pieces


def build_sharded(plan, packed: torch.Tensor, offsets: torch.Tensor, n_reads: int, out: torch.Tensor, group=None, stream=None):
    """cx_bwt_build on this rank's partition range, then the exchange.  `plan` was made with shard_index = this rank's
    index in `group` and shard_count = the group's size; every rank passes the same reads."""
    plan.build(packed, offsets, n_reads, out, stream=stream)
    st = plan.stats()
    return exchange_pieces(out, st["shard_offset"], st["shard_suffixes"], group)
