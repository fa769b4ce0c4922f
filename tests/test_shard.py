"""NEXT-2: partition-range sharding (the paper's distributed scheme, Section 3.3).

GPU part (one GPU): the W shards of a collection are built one after another into one output buffer; their pieces must
tile [0, N) in shard order and the buffer must equal the oracle's BWT byte for byte ("each partition gives
a portion of the BWT, which can be simply concatenated").  CPU part: the exchange step (all-gather-v of the pieces) with
two gloo processes."""
import os

import numpy as np
import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

import oracle
from workloads import generate as gen

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _sharded_bwt(coll, world, **opts):
    import paper_1401_7457_b200 as cx
    n_reads, total, N = coll.n_reads, coll.total_bases, coll.n_suffixes
    dev = torch.device("cuda")
    a = torch.from_numpy(coll.ascii).to(dev)
    off = torch.from_numpy(coll.offsets.astype(np.int64)).to(dev)
    packed = cx.cx_pack_reads(a) if total else torch.zeros(1, dtype=torch.int64, device=dev)
    out = torch.full((N,), ord("?"), dtype=torch.uint8, device=dev)
    opts.setdefault("max_read_len", max(coll.max_read_len, 1))
    pieces = []
    for k in range(world):
        plan = cx.Plan(n_reads, total, shard_index=k, shard_count=world, **opts)
        plan.build(packed, off, n_reads, out)
        torch.cuda.synchronize()
        st = plan.stats()
        pieces.append((st["shard_offset"], st["shard_suffixes"]))
        # a shard writes nothing outside its piece
        lo, n = pieces[-1]
        assert not bool((out[lo + n:] != ord("?")).any()), f"shard {k} of {world} wrote past its piece"
        plan.free()
    cx.check_pieces(pieces, N)
    return out.cpu().numpy(), pieces


@pytest.mark.gpu
@pytest.mark.parametrize("world", [2, 3, 8])
def test_shards_concatenate_to_the_oracle_bwt_config1(world):
    c = gen.config(0, 0.3)
    want = oracle.bwt(c.ascii, c.offsets)
    got, pieces = _sharded_bwt(c, world)
    assert np.array_equal(got, want)
    sizes = [n for _, n in pieces]
    assert max(sizes) - min(sizes) <= 2 * (c.n_suffixes // 4096 + c.n_reads)   # "roughly equal total size": within a partition or two


@pytest.mark.gpu
@pytest.mark.parametrize("idx,scale,world,opts", [
    (1, 0.02, 4, {}),                                     # deep ties (100x coverage)
    (2, 0.002, 5, {"max_batch_suffixes": 30_000}),        # several batches inside each shard
    (3, 0.0005, 3, {"prefix_len": 2}),                    # ragged lengths, 64-bit ids at full size; few, large partitions
    (1, 0.01, 2, {"prefix_len": 1, "max_batch_suffixes": 20_000}),   # oversize partitions refined inside a shard
])
def test_shards_of_config_shapes(idx, scale, world, opts):
    c = gen.config(idx, scale)
    want = oracle.bwt(c.ascii, c.offsets)
    got, _ = _sharded_bwt(c, world, **opts)
    assert np.array_equal(got, want)


@pytest.mark.gpu
def test_more_shards_than_partitions_and_degenerate_inputs():
    # homopolymers: a handful of non-empty partitions, most shards get nothing
    c = gen.from_strings(["A" * 60] * 40 + ["", "C", "AAC"])
    want = oracle.bwt(c.ascii, c.offsets)
    got, pieces = _sharded_bwt(c, 16, prefix_len=3)
    assert np.array_equal(got, want)
    assert sum(1 for _, n in pieces if n == 0) > 0
    got, _ = _sharded_bwt(gen.from_strings(["ACGT", "TAGT", "GGAA"]), 2)        # Figure 1
    assert got.tobytes() == b"TTAAG$TAG$CAGG$"


@pytest.mark.gpu
def test_bad_shard_options_are_rejected():
    import paper_1401_7457_b200 as cx
    with pytest.raises(cx.CxError):
        cx.Plan(10, 100, shard_index=2, shard_count=2)


# ---- the exchange step on CPU: two gloo ranks ---------------------------------------------------------
def _worker(rank, world, port, q):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    import sys
    sys.path.insert(0, ROOT)
    from paper_1401_7457_b200 import shard
    dist.init_process_group("gloo", rank=rank, world_size=world)
    full = (torch.arange(1000, dtype=torch.int64) * 7 % 251).to(torch.uint8)
    cuts = [0, 377, 1000]                                   # pieces of different lengths
    out = torch.zeros(1000, dtype=torch.uint8)
    lo, hi = cuts[rank], cuts[rank + 1]
    out[lo:hi] = full[lo:hi]                                # what this rank's build wrote
    pieces = shard.exchange_pieces(out, lo, hi - lo)
    ok = bool(torch.equal(out, full))
    # pieces that do not tile the output are refused on every rank
    try:
        shard.exchange_pieces(out, lo + (1 if rank else 0), hi - lo)
        refused = False
    except RuntimeError:
        refused = True
    dist.barrier()
    dist.destroy_process_group()
    q.put((rank, ok, pieces, refused))


def test_exchange_pieces_two_gloo_ranks():
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = 31500 + os.getpid() % 2000
    procs = [ctx.Process(target=_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    res = sorted(q.get(timeout=120) for _ in procs)
    for p in procs:
        p.join(60)
        assert p.exitcode == 0
    for rank, ok, pieces, refused in res:
        assert ok and refused and pieces == [(0, 377), (377, 623)]


def _worker3(rank, world, port, q):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    import sys
    sys.path.insert(0, ROOT)
    from paper_1401_7457_b200 import shard
    dist.init_process_group("gloo", rank=rank, world_size=world)
    full = (torch.arange(5003, dtype=torch.int64) * 13 % 241).to(torch.uint8)
    cuts = [0, 4000, 4000, 5003]                            # a long piece, an EMPTY one, a short one: padding and skipping
    out = torch.full((5003,), 255, dtype=torch.uint8)
    lo, hi = cuts[rank], cuts[rank + 1]
    out[lo:hi] = full[lo:hi]
    pieces = shard.exchange_pieces(out, lo, hi - lo)
    dist.barrier()
    dist.destroy_process_group()
    q.put((rank, bool(torch.equal(out, full)), pieces))


def test_exchange_pieces_three_gloo_ranks_one_empty_piece():
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = 35500 + os.getpid() % 2000
    procs = [ctx.Process(target=_worker3, args=(r, 3, port, q)) for r in range(3)]
    for p in procs:
        p.start()
    res = sorted(q.get(timeout=120) for _ in procs)
    for p in procs:
        p.join(60)
        assert p.exitcode == 0
    for rank, ok, pieces in res:
        assert ok and pieces == [(0, 4000), (4000, 0), (4000, 1003)]


def test_check_pieces():
    from paper_1401_7457_b200 import shard
    shard.check_pieces([(0, 5), (5, 0), (5, 7)], 12)
    shard.check_pieces([(12, 0), (0, 12)], 12)              # an empty piece may sit anywhere
    for bad in ([(0, 5), (6, 6)], [(0, 5), (5, 6)], [(1, 11)]):
        with pytest.raises(RuntimeError):
            shard.check_pieces(bad, 12)


@pytest.mark.gpu
def test_shards_stream_to_pinned_host_and_slice_the_end_marker_partition():
    """Pinned-host output (a9) inside a shard, and m1 below n_reads so that the partition of bare end-markers (identical
    suffixes) is cut into slices of the listing order inside the shard that owns it."""
    import paper_1401_7457_b200 as cx
    c = gen.config(1, 0.005)                                   # 5,000 reads
    want = oracle.bwt(c.ascii, c.offsets)
    a = torch.from_numpy(c.ascii).cuda()
    off = torch.from_numpy(c.offsets.astype(np.int64)).cuda()
    packed = cx.cx_pack_reads(a)
    out = torch.full((c.n_suffixes,), ord("?"), dtype=torch.uint8).pin_memory()
    pieces = []
    for k in range(3):
        p = cx.Plan(c.n_reads, c.total_bases, max_read_len=100, max_batch_suffixes=3_000, out_is_host_pinned=1, shard_index=k, shard_count=3)
        p.build(packed, off, c.n_reads, out)
        torch.cuda.synchronize()
        st = p.stats()
        pieces.append((st["shard_offset"], st["shard_suffixes"]))
        assert st["n_batches"] > 3
        p.free()
    cx.check_pieces(pieces, c.n_suffixes)
    assert np.array_equal(out.numpy(), want)


# ---- build_sharded end to end on CPU: two gloo ranks, a stand-in plan that writes the oracle's piece ----------------
class _PieceWriter:
    """Stands in for cx.Plan on a machine without a GPU: `build` writes this rank's piece of a BWT computed by the oracle
    (cut at a fixed position) and `stats` reports it, which is all build_sharded needs to drive the exchange."""

    def __init__(self, full, lo, hi):
        self.full, self.lo, self.hi = full, lo, hi

    def build(self, packed, offsets, n_reads, out, stream=None):
        out[self.lo:self.hi] = self.full[self.lo:self.hi]

    def stats(self):
        return {"shard_offset": self.lo, "shard_suffixes": self.hi - self.lo}


def _sharded_worker(rank, world, port, q):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    import sys
    sys.path.insert(0, ROOT)
    from paper_1401_7457_b200 import shard
    dist.init_process_group("gloo", rank=rank, world_size=world)
    c = gen.config(0, 0.01)                                                  # every rank holds the same reads
    full = torch.from_numpy(oracle.bwt(c.ascii, c.offsets))
    cut = [0, c.n_suffixes // 3, c.n_suffixes]
    out = torch.zeros(c.n_suffixes, dtype=torch.uint8)
    pieces = shard.build_sharded(_PieceWriter(full, cut[rank], cut[rank + 1]), None, None, c.n_reads, out)
    ok = bool(torch.equal(out, full))
    dist.barrier()
    dist.destroy_process_group()
    q.put((rank, ok, pieces == [(cut[0], cut[1] - cut[0]), (cut[1], cut[2] - cut[1])]))


def test_build_sharded_two_gloo_ranks_with_a_stand_in_plan():
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = 33500 + os.getpid() % 2000
    procs = [ctx.Process(target=_sharded_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    res = sorted(q.get(timeout=180) for _ in procs)
    for p in procs:
        p.join(60)
        assert p.exitcode == 0
    assert all(ok and pieces_ok for _, ok, pieces_ok in res)
