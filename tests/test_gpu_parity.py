"""Parity of the CUDA path (through the C ABI) against the CPU oracle, element by element, on the
same seeded inputs.  Integer/byte work: the bar is bit-exact.  Needs a B200: `pytest -m gpu`."""
import itertools
import os

import numpy as np
import pytest
import torch

import oracle
from tests import bwt_checks as chk
from workloads import generate as gen

pytestmark = pytest.mark.gpu


def gpu_bwt(coll, **opts):
    import paper_1401_7457_b200 as cx
    opts.setdefault("max_read_len", max(coll.max_read_len, 1))
    return cx.bwt_of_collection(coll.ascii, coll.offsets, **opts)


def assert_parity(coll, **opts):
    want = oracle.bwt(coll.ascii, coll.offsets)
    got = gpu_bwt(coll, **opts)
    assert got.shape == want.shape
    if not np.array_equal(got, want):
        bad = np.flatnonzero(got != want)
        raise AssertionError(f"{coll.name} {opts}: {bad.size} of {want.size} symbols differ, first at {bad[:5]}: "
                             f"got {got[bad[:5]].tobytes()} want {want[bad[:5]].tobytes()}")


# ---- the paper's worked example and the closed forms ---------------------------------------------

def test_figure1():
    got = gpu_bwt(gen.from_strings(["ACGT", "TAGT", "GGAA"]))
    assert got.tobytes() == b"TTAAG$TAG$CAGG$"          # PAPER.md:59, Figure 1


@pytest.mark.parametrize("reads,want", [
    (["ACGT"] * 3, "TTT$$$AAACCCGGG"),
    (["A", "AA", "AAA"], "AAA$AA$A$"),
    (["", "A", ""], "$A$$"),
    ([""], "$"),
    (["T"], "T$"),
])
def test_closed_forms(reads, want):
    assert gpu_bwt(gen.from_strings(reads)).tobytes().decode() == want


def test_empty_collection():
    import paper_1401_7457_b200 as cx
    assert cx.bwt_of_collection(np.zeros(0, np.uint8), np.zeros(1, np.uint64)).size == 0


def test_all_small_collections_two_letters():
    words = [""] + ["".join(w) for L in range(1, 4) for w in itertools.product("AC", repeat=L)]
    for reads in itertools.product(words, repeat=2):
        c = gen.from_strings(list(reads))
        assert gpu_bwt(c).tobytes().decode() == oracle.bwt_of_strings(list(reads)), reads


@pytest.mark.parametrize("seed", range(40))
def test_random_ragged_collections(seed):
    c = gen.random_collection(seed, n_reads=1 + (seed * 37) % 300, max_len=1 + (seed * 13) % 140,
                              alphabet=["ACGT", "GT", "A", "CGT", "AC"][seed % 5])
    assert_parity(c)
    assert_parity(c, small_group_max=1)                 # global re-key path only
    assert_parity(c, key_bases=7 + seed % 20, prefix_len=1 + seed % 7)
    assert_parity(c, finish_slots=[2, 4][seed % 2], key_bases=[0, 9][seed % 3 == 0])      # window width of the register refinement fixed


def test_homopolymer_reads_one_giant_group():
    c = gen.from_strings(["A" * 100] * 700 + ["A" * 37] * 50 + ["C" * 64] * 3)
    assert_parity(c)
    assert_parity(c, small_group_max=1)
    assert_parity(c, small_group_max=16)


@pytest.mark.parametrize("id64", [False, True])
def test_global_path_shares_the_buffers_of_the_first_sort(id64):
    """Tie groups above the block kernel's limit go through rounds of re-key, sort, write back.  That path owns no buffers:
    its (key, position) pairs ping-pong between the two key buffers and the spare id buffer (two position arrays in it with
    8-byte ids, the second in `pos` with 4-byte ids), and the gathered ids pass through whichever key buffer is free.  Batch
    sizes that are odd, a multiple of 4 plus 1, 2, 3 (where the second position array starts) and one that makes nearly
    every suffix active; several rounds (groups of 900 equal suffixes of 300 bases: the window of a round is 27 bases)."""
    rng = np.random.default_rng(5)
    unit = "".join(rng.choice(list("ACGT"), 300))
    reads = [unit] * 900 + [unit[:170]] * 300 + ["".join(rng.choice(list("ACGT"), 80)) for _ in range(50)]
    c = gen.from_strings(reads)
    extra = dict(max_read_len=0) if id64 else {}
    assert_parity(c, **extra)
    for m1 in (c.n_suffixes, c.n_suffixes // 2 + 1, c.n_suffixes // 3 + 2, c.n_suffixes // 5 + 3):
        assert_parity(c, max_batch_suffixes=m1, **extra)
    assert_parity(c, small_group_max=1, max_batch_suffixes=c.n_suffixes // 2 + 3, **extra)


@pytest.mark.parametrize("case", range(5))
def test_split_pairs_of_64_bit_keys_and_ids(case):
    """Batches of a multi-batch plan with 64-bit keys (19 bases) and 64-bit ids go through the sort as 12-byte pairs: the key
    above the id's high part in the 64-bit word, the id's low word as the value; the listing writes them, the probe, the warp
    and the block kernel read them, and groups left to the global path get their ids assembled into another buffer.
    Collections with every group size (singletons, <= 64, 65..256, above 256), ragged reads, a scaled configs[3]."""
    rng = np.random.default_rng(300 + case)
    if case == 0:
        c = gen.random_collection(11, 400, 120)
    elif case == 1:
        unit = "".join(rng.choice(list("ACGT"), 200))
        c = gen.from_strings([unit] * 700 + [unit[40:]] * 100 + [unit[:90]] * 30 + ["".join(rng.choice(list("ACGT"), 60)) for _ in range(200)])
    elif case == 2:
        genome = np.frombuffer(b"ACGT", np.uint8)[rng.integers(0, 4, 900)]
        c = gen.from_strings(["".join(map(chr, genome[s:s + 100])) for s in rng.integers(0, 800, 3000)])     # groups of 2..200
    elif case == 3:
        c = gen.config(3, 0.0003)
    else:
        c = gen.from_strings(["AC" * 70] * 150 + ["ACGT"] * 40 + [""] * 3 + ["T"])
    N = c.n_suffixes
    base = dict(key_bases=19, max_read_len=0)
    assert_parity(c, max_batch_suffixes=N // 3 + 1, **base)
    assert_parity(c, max_batch_suffixes=N // 7 + 2, finish_slots=4, **base)
    assert_parity(c, max_batch_suffixes=N // 2 + 3, small_group_max=1, **base)
    assert_parity(c, max_batch_suffixes=N // 4 + 1, small_group_max=100, key_bases=29, max_read_len=0)     # 60-bit keys: 4-bit split


def test_long_reads_and_tandem_repeats():
    c = gen.from_strings(["ACGT" * 200, "ACGT" * 150 + "T", "CGTA" * 180, "G" * 900, ""] * 7)
    assert_parity(c)


# ---- config shapes ---------------------------------------------------------------------------------

def test_config1_full():
    c = gen.config(0)
    assert_parity(c)                                     # 1,010,000 suffixes, spans many tiles + ragged tail


@pytest.mark.parametrize("idx,scale", [(1, 0.02), (2, 0.002), (3, 0.0005), (4, 0.000002)])
def test_config_shapes_scaled(idx, scale):
    c = gen.config(idx, scale)
    assert_parity(c)
    assert_parity(c, finish_slots=4)
    assert_parity(c, finish_slots=2)


def test_config2_full_size_every_suffix():
    """configs[1] (1.01e8 suffixes) at full size, EVERY output symbol compared with the oracle: the 16 two-base prefix ranges
    through the range-restricted oracle (each a contiguous piece of B_R; one range per host thread -- the C
    oracle runs outside the GIL), the one-base suffixes "X$" from the definition (identical strings, ordered by read index,
    PAPER.md:55) and the n end-marker suffixes by the first-n rule; plus counts and LF inversion of 20,000 reads."""
    import concurrent.futures as cf
    c = gen.config(1)
    got = gpu_bwt(c)
    chk.check_all(got, c, lf_sample=20_000)                  # includes the first-n rule: positions [0, n)
    covered = c.n_reads
    prefixes = [a + b for a in "ACGT" for b in "ACGT"]
    oracle.build()
    with cf.ThreadPoolExecutor(max_workers=os.cpu_count() or 1) as pool:
        res = list(pool.map(lambda pfx: oracle.bwt_with_prefix(c.ascii, c.offsets, pfx), prefixes))
    where = dict(zip(prefixes, res))
    for pfx, (off, want) in where.items():
        assert np.array_equal(got[off:off + want.size], want), f"configs[1]: slice of prefix {pfx} differs"
        covered += want.size
    # suffixes of exactly one base X: they sit immediately before the "XA" range, in read order; each is preceded by the
    # base before the read's last base (reads are 100 bp here)
    off64 = c.offsets.astype(np.int64)
    last = c.ascii[off64[1:] - 1]
    before_last = c.ascii[off64[1:] - 2]
    for x in "ACGT":
        sel = last == ord(x)
        cnt = int(sel.sum())
        end = where[x + "A"][0]
        assert np.array_equal(got[end - cnt:end], before_last[sel]), f"configs[1]: the one-base suffixes {x}$ differ"
        covered += cnt
    assert covered == c.n_suffixes                           # every position of the output was compared


@pytest.mark.parametrize("read_len", [200, 400, 1000])
def test_longer_reads_table4_shape(read_len):
    # NEXT-3: the paper's read-length experiment (Table 4) at reduced scale; deeper refinement
    c = gen.table4(read_len, 0.0002)
    assert_parity(c)
    assert_parity(c, small_group_max=1)


def test_one_long_read_and_word_aligned_lengths():
    # a single 200 kbp read (18 position bits; the textbook BWT of S$), then reads whose lengths sit on packed-word edges
    rng = np.random.default_rng(5)
    long_read = "".join("ACGT"[i] for i in rng.integers(0, 4, 200_000))
    assert_parity(gen.from_strings([long_read]))
    assert_parity(gen.from_strings([long_read[:70_000], long_read[:70_000], "ACGT" * 8000]), max_batch_suffixes=30_000, prefix_len=3)
    edge = ["".join("ACGT"[i] for i in rng.integers(0, 4, n)) for n in (31, 32, 33, 63, 64, 65, 0, 1, 96, 128, 127, 57, 58, 14, 15, 71, 72)] * 9
    assert_parity(gen.from_strings(edge))
    assert_parity(gen.from_strings(edge), max_batch_suffixes=700, prefix_len=2)


def test_empty_reads_everywhere():
    reads = ["", "", "ACGTACGT", "", "T", "", ""] * 300 + [""] * 500
    assert_parity(gen.from_strings(reads))
    assert_parity(gen.from_strings(reads), max_batch_suffixes=1000)     # fewer than n_reads: the end-marker partition is sliced
    assert_parity(gen.from_strings([""] * 5000), max_batch_suffixes=999)


def test_eight_byte_ids():
    c = gen.config(1, 0.02)
    assert_parity(c, max_read_len=0)                     # unknown read length -> 64-bit suffix ids
    import paper_1401_7457_b200 as cx
    p = cx.Plan(c.n_reads, c.total_bases)
    a = torch.from_numpy(c.ascii).cuda()
    out = torch.empty(c.n_suffixes, dtype=torch.uint8, device="cuda")
    p.build(cx.cx_pack_reads(a), torch.from_numpy(c.offsets.astype(np.int64)).cuda(), c.n_reads, out)
    assert p.stats()["id_bytes"] == 8


@pytest.mark.parametrize("m1", [12_000, 70_000, 400_000])
def test_multiple_batches(m1):
    c = gen.config(2, 0.001)                             # ~1.01e6 suffixes
    assert_parity(c, max_batch_suffixes=m1, prefix_len=5)
    assert_parity(c, max_batch_suffixes=m1, prefix_len=6, out_is_host_pinned=0, small_group_max=1)


def test_pinned_host_output_streams_batches():
    import paper_1401_7457_b200 as cx
    c = gen.config(1, 0.01)
    want = oracle.bwt(c.ascii, c.offsets)
    a = torch.from_numpy(c.ascii).cuda()
    off = torch.from_numpy(c.offsets.astype(np.int64)).cuda()
    p = cx.Plan(c.n_reads, c.total_bases, max_read_len=100, max_batch_suffixes=150_000, out_is_host_pinned=1)
    out = torch.empty(c.n_suffixes, dtype=torch.uint8).pin_memory()
    p.build(cx.cx_pack_reads(a), off, c.n_reads, out)
    assert p.stats()["n_batches"] > 3
    assert np.array_equal(out.numpy(), want)


# ---- NEXT-1: partitions larger than a batch are partitioned again by their next l characters ------------

def _stats_of(coll, **opts):
    import paper_1401_7457_b200 as cx
    p = cx.Plan(coll.n_reads, coll.total_bases, max_read_len=max(coll.max_read_len, 1), **opts)
    out = torch.empty(coll.n_suffixes, dtype=torch.uint8, device="cuda")
    a = torch.from_numpy(coll.ascii).cuda()
    packed = cx.cx_pack_reads(a) if coll.total_bases else torch.zeros(1, dtype=torch.int64, device="cuda")
    p.build(packed, torch.from_numpy(coll.offsets.astype(np.int64)).cuda(), coll.n_reads, out)
    return out.cpu().numpy(), p.stats()


@pytest.mark.parametrize("m1", [1000, 150, 37])
def test_homopolymer_collection_with_tiny_batches(m1):
    # every suffix falls in the AAAAAA partition or a partition of identical short suffixes: refinement down to the
    # read length, and (m1 < n_reads) partitions of identical suffixes cut into slices of the listing order
    c = gen.from_strings(["A" * 100] * 200)
    got, st = _stats_of(c, max_batch_suffixes=m1)
    assert np.array_equal(got, oracle.bwt(c.ascii, c.offsets))
    assert st["refined_partitions"] >= 10 and st["n_batches"] > 10


def test_tandem_repeats_and_duplicates_with_tiny_batches():
    c = gen.from_strings(["ACGT" * 50] * 40 + ["CGTA" * 30 + "T"] * 25 + ["G" * 77] * 30 + ["", "A", "AC"] * 20)
    for m1 in (500, 90):
        got, st = _stats_of(c, max_batch_suffixes=m1, prefix_len=3)
        assert np.array_equal(got, oracle.bwt(c.ascii, c.offsets)), m1
        assert st["refined_partitions"] > 0


@pytest.mark.parametrize("idx,scale,m1,ell", [(1, 0.01, 20_000, 2), (2, 0.001, 9_000, 1), (3, 0.0003, 30_000, 2)])
def test_config_shapes_with_forced_refinement(idx, scale, m1, ell):
    c = gen.config(idx, scale)
    got, st = _stats_of(c, max_batch_suffixes=m1, prefix_len=ell)
    assert np.array_equal(got, oracle.bwt(c.ascii, c.offsets))
    assert st["refined_partitions"] > 0


@pytest.mark.parametrize("seed", range(12))
def test_random_skewed_collections_with_tiny_batches(seed):
    c = gen.random_collection(100 + seed, n_reads=20 + (seed * 29) % 200, max_len=1 + (seed * 17) % 120, alphabet=["A", "AC", "ACGT", "GT"][seed % 4])
    for m1 in (64, 11):
        got, _ = _stats_of(c, max_batch_suffixes=m1, prefix_len=1 + seed % 4, small_group_max=[0, 1][seed % 2])
        assert np.array_equal(got, oracle.bwt(c.ascii, c.offsets)), (seed, m1)


def test_bad_offsets_and_oversize_input_are_reported_not_executed():
    import paper_1401_7457_b200 as cx
    c = gen.config(1, 0.002)
    a = torch.from_numpy(c.ascii).cuda()
    packed = cx.cx_pack_reads(a)
    out = torch.empty(c.n_suffixes, dtype=torch.uint8, device="cuda")
    good = torch.from_numpy(c.offsets.astype(np.int64)).cuda()
    for kind in ("decreasing", "nonzero_start"):
        off = good.clone()
        if kind == "decreasing":
            off[5] = off[7] + 3
        else:
            off[0] = 1
        p = cx.Plan(c.n_reads, c.total_bases, max_read_len=100)
        with pytest.raises(cx.CxError) as e:
            p.build(packed, off, c.n_reads, out)
        assert e.value.code == cx.binding.CX_ERR_ARG
        p.build(packed, good, c.n_reads, out)                # the plan is still usable
        assert np.array_equal(out.cpu().numpy(), oracle.bwt(c.ascii, c.offsets))
    small = cx.Plan(c.n_reads, c.total_bases // 2, max_read_len=100)      # planned for half the bases
    with pytest.raises(cx.CxError) as e:
        small.build(packed, good, c.n_reads, out)
    assert e.value.code == cx.binding.CX_ERR_ARG


def test_default_workspace_gives_one_batch():
    """cx_bwt_workspace_bytes sizes the workspace for one batch; the plan must then really take one
    (the listing scan that also counts partition sizes depends on it)."""
    import paper_1401_7457_b200 as cx
    c = gen.config(2, 0.002)
    p = cx.Plan(c.n_reads, c.total_bases, max_read_len=100)
    out = torch.empty(c.n_suffixes, dtype=torch.uint8, device="cuda")
    p.build(cx.cx_pack_reads(torch.from_numpy(c.ascii).cuda()), torch.from_numpy(c.offsets.astype(np.int64)).cuda(), c.n_reads, out)
    st = p.stats()
    assert st["n_batches"] == 1 and st["max_batch"] == c.n_suffixes
    assert np.array_equal(out.cpu().numpy(), oracle.bwt(c.ascii, c.offsets))


def test_plan_reuse_many_builds_and_side_stream():
    """One plan, many builds of different collections (more than 255 radix passes in total, so the look-back epoch of
    the tile states wraps), on a non-default stream."""
    import paper_1401_7457_b200 as cx
    colls = [gen.config(1, 0.003), gen.config(2, 0.0008), gen.random_collection(3, 150, 90), gen.from_strings(["A" * 100] * 300),
             gen.config(0, 0.3), gen.from_strings(["ACGT", "TAGT", "GGAA"])]
    wants = [oracle.bwt(c.ascii, c.offsets) for c in colls]
    max_reads = max(c.n_reads for c in colls)
    max_bases = max(c.total_bases for c in colls)
    plan = cx.Plan(max_reads, max_bases, max_read_len=100)
    stream = torch.cuda.Stream()
    passes = 0
    with torch.cuda.stream(stream):
        for it in range(14):
            for c, want in zip(colls, wants):
                a = torch.from_numpy(c.ascii).cuda()
                off = torch.from_numpy(c.offsets.astype(np.int64)).cuda()
                out = torch.empty(c.n_suffixes, dtype=torch.uint8, device="cuda")
                plan.build(cx.cx_pack_reads(a, stream=stream), off, c.n_reads, out, stream=stream)
                stream.synchronize()
                assert np.array_equal(out.cpu().numpy(), want), (it, c.name)
                passes += plan.stats()["sort_passes"]
    assert passes > 255


def test_deterministic():
    c = gen.config(2, 0.001)
    assert np.array_equal(gpu_bwt(c), gpu_bwt(c))


# ---- single steps ------------------------------------------------------------------------------------

def test_pack_matches_numpy_and_rejects_bad_bases():
    import paper_1401_7457_b200 as cx
    for n in (0, 1, 31, 32, 33, 1000, 100_003):
        codes = np.random.default_rng(n).integers(0, 4, n).astype(np.uint8)
        ascii_ = np.frombuffer(b"ACGT", np.uint8)[codes]
        if n == 0:
            continue
        padded = np.zeros((n + 31) // 32 * 32, dtype=np.uint64)
        padded[:n] = codes
        want = np.zeros(padded.size // 32, dtype=np.uint64)
        for j in range(32):
            want |= padded[j::32] << np.uint64(62 - 2 * j)
        got = cx.cx_pack_reads(torch.from_numpy(ascii_.copy()).cuda()).cpu().numpy().view(np.uint64)
        assert np.array_equal(got, want), n
        # unaligned input pointer
        buf = torch.zeros(n + 3, dtype=torch.uint8, device="cuda")
        buf[3:] = torch.from_numpy(ascii_.copy()).cuda()
        assert np.array_equal(cx.cx_pack_reads(buf[3:]).cpu().numpy().view(np.uint64), want)
    for bad in (b"ACGN", b"acgt", b"AC$T" * 100):
        with pytest.raises(cx.CxError) as e:
            cx.cx_pack_reads(torch.from_numpy(np.frombuffer(bad, np.uint8).copy()).cuda())
        assert e.value.code == cx.binding.CX_ERR_BAD_BASE


@pytest.mark.parametrize("n,bits,vb", [(1, 64, 4), (1000, 64, 4), (5000, 13, 8), (300_001, 63, 4), (1_000_003, 40, 8),
                                       (2_000_000, 8, 4)])
def test_sort_pairs_against_torch_stable_sort(n, bits, vb):
    import paper_1401_7457_b200 as cx
    g = torch.Generator(device="cuda").manual_seed(n)
    keys = torch.randint(-2**63, 2**63 - 1, (n,), dtype=torch.int64, device="cuda", generator=g)
    if bits < 64:
        keys = keys & ((1 << bits) - 1)
    if n > 1000:
        m = keys[1::3].numel()
        keys[::3][:m] = keys[1::3]                       # plenty of duplicates: stability matters
    vals = torch.arange(n, device="cuda", dtype=torch.int32 if vb == 4 else torch.int64)
    ks, vs = cx.cx_sort_pairs(keys, vals, 0, bits)
    # reference order: unsigned 64-bit compare == signed compare after flipping the sign bit
    order = torch.sort(keys ^ (-2**63), stable=True).indices
    assert torch.equal(ks, keys[order])
    assert torch.equal(vs.long(), order)


def test_partition_sizes_match_linear_scan():
    """P6 / Fig. 2 step 1: the histogram equals a plain count over the reads."""
    import paper_1401_7457_b200 as cx
    c = gen.config(3, 0.0001)
    ell = 4
    p = cx.Plan(c.n_reads, c.total_bases, max_read_len=c.max_read_len, prefix_len=ell)
    out = torch.empty(c.n_suffixes, dtype=torch.uint8, device="cuda")
    p.build(cx.cx_pack_reads(torch.from_numpy(c.ascii).cuda()), torch.from_numpy(c.offsets.astype(np.int64)).cuda(), c.n_reads, out)
    got = p.histogram()
    want = np.zeros(4 ** ell * (ell + 1), dtype=np.uint64)
    code = {65: 0, 67: 1, 71: 2, 84: 3}
    for i in range(c.n_reads):
        r = c.ascii[int(c.offsets[i]):int(c.offsets[i + 1])]
        for q in range(len(r) + 1):
            s = r[q:q + ell]
            k = 0
            for ch in s:
                k = k * 4 + code[int(ch)]
            k <<= 2 * (ell - len(s))
            want[k * (ell + 1) + len(s)] += 1
    assert np.array_equal(got, want)
    # partitions are contiguous and ordered in the output: per-partition symbol multiset check
    chk.check_all(out.cpu().numpy(), c)


def test_read_longer_than_2_pow_21_in_tie_groups():
    """A read of 2.2 Mbp whose suffixes sit in tie groups with short reads copied out of it: the in-block refinement must
    carry 'bases left' beyond 21 bits (a 21-bit field silently corrupted the emitted symbols)."""
    rng = np.random.default_rng(21)
    long_read = "".join(np.frombuffer(b"ACGT", np.uint8)[rng.integers(0, 4, 2_200_000)].tobytes().decode())
    reads = [long_read, long_read[100:160], long_read[100:160], long_read[5000:5100], long_read[2_199_900:], ""]
    assert_parity(gen.from_strings(reads))


# ---- NEXT-4: packed output, two symbols per byte (include/cx_bwt.h, opts.out_bits = 4) -----------------------------------

def _unpack4(packed: np.ndarray, n: int) -> np.ndarray:
    codes = np.stack([packed >> 4, packed & 15], 1).reshape(-1)[:n]
    assert codes.max(initial=0) <= 4
    return np.frombuffer(b"$ACGT", np.uint8)[codes]


@pytest.mark.parametrize("opts", [dict(), dict(max_batch_suffixes=70_001, prefix_len=5), dict(max_batch_suffixes=33_333, small_group_max=1),
                                  dict(max_batch_suffixes=150_001, out_is_host_pinned=1), dict(out_is_host_pinned=1)])
def test_packed_output_four_bits_per_symbol(opts):
    import paper_1401_7457_b200 as cx
    for c in (gen.config(2, 0.001), gen.from_strings(["ACGT", "TAGT", "GGAA"]), gen.random_collection(9, 301, 77)):   # N even, 15, odd
        want = oracle.bwt(c.ascii, c.offsets)
        N = c.n_suffixes
        p = cx.Plan(c.n_reads, c.total_bases, max_read_len=max(c.max_read_len, 1), out_bits=4, **opts)
        out = torch.full(((N + 1) // 2,), 0xEE, dtype=torch.uint8)
        out = out.pin_memory() if opts.get("out_is_host_pinned") else out.cuda()
        a = torch.from_numpy(c.ascii).cuda()
        p.build(cx.cx_pack_reads(a), torch.from_numpy(c.offsets.astype(np.int64)).cuda(), c.n_reads, out)
        torch.cuda.synchronize()
        got = out.cpu().numpy()
        assert np.array_equal(_unpack4(got, N), want), (c.name, opts)
        if N & 1:
            assert got[-1] & 15 == 0                      # the unused low nibble of the last byte
    with pytest.raises(cx.CxError):
        cx.Plan(100, 1000, out_bits=4, shard_index=0, shard_count=2)
    with pytest.raises(cx.CxError):
        cx.Plan(100, 1000, out_bits=3)


@pytest.mark.parametrize("L", [15, 16, 17, 31, 32, 33, 63, 64, 65, 95, 96, 97, 126, 127, 128, 200])
def test_equal_length_reads_at_the_kernel_dispatch_boundaries(L):
    """Collections of equal-length reads take their own scan kernels: one read per thread for 16 <= L <= 127 (a 128-bit mask per
    thread: positions 31/32, 63/64, 95/96 cross its words; L = 127 fills it), the 8192-slot walk otherwise.  Single batch (fused
    listing), several batches (count + select), 64-bit ids and two shards; 700 reads = two full tiles of 256 and a ragged one.
    Reads are copies from a short genome: deep ties, duplicates."""
    rng = np.random.default_rng(1000 + L)
    genome = np.frombuffer(b"ACGT", np.uint8)[rng.integers(0, 4, 3 * L + 40)]
    starts = rng.integers(0, genome.size - L + 1, 700)
    reads = ["".join(map(chr, genome[s:s + L])) for s in starts]
    c = gen.from_strings(reads)
    assert_parity(c)
    assert_parity(c, max_batch_suffixes=c.n_suffixes // 5 + 1, prefix_len=3)
    assert_parity(c, max_batch_suffixes=c.n_suffixes // 3 + 1, max_read_len=0)      # unknown read length: 64-bit ids
    import paper_1401_7457_b200 as cx
    want = oracle.bwt(c.ascii, c.offsets)
    a = torch.from_numpy(c.ascii).cuda()
    off = torch.from_numpy(c.offsets.astype(np.int64)).cuda()
    packed = cx.cx_pack_reads(a)
    out = torch.zeros(c.n_suffixes, dtype=torch.uint8, device="cuda")
    for k in range(2):
        p = cx.Plan(c.n_reads, c.total_bases, max_read_len=L, shard_index=k, shard_count=2)
        p.build(packed, off, c.n_reads, out)
        p.free()
    assert np.array_equal(out.cpu().numpy(), want)


@pytest.mark.parametrize("L", [16, 24, 37, 100, 127])
def test_equal_length_reads_in_many_small_batches(L):
    """A batch that is a short range of partitions: the select scan finds the positions whose first two bases fit the range
    with word-wide bit operations (24 positions per 32-base window: L = 24, 37 end a window early) and tests only those
    exactly; a wider range takes the plain walk.  Random reads (every l-mer about equally often) and copies from a short
    genome (few, heavy partitions); prefix lengths 2 (the two bases are the whole partition code), 6 and 7."""
    rng = np.random.default_rng(4000 + L)
    random_reads = ["".join(rng.choice(list("ACGT"), L)) for _ in range(600)]
    genome = np.frombuffer(b"ACGT", np.uint8)[rng.integers(0, 4, 2 * L + 30)]
    copies = ["".join(map(chr, genome[s:s + L])) for s in rng.integers(0, genome.size - L + 1, 300)]
    for reads in (random_reads, random_reads[:257] + copies):
        c = gen.from_strings(reads)
        assert_parity(c, max_batch_suffixes=c.n_suffixes // 40 + 1)
        assert_parity(c, max_batch_suffixes=c.n_suffixes // 150 + 1, prefix_len=7)
        assert_parity(c, max_batch_suffixes=c.n_suffixes // 9 + 1, prefix_len=2)


def test_host_pipeline_overlapped_builds_match_the_oracle():
    """HostPipeline: five DIFFERENT collections (sizes differ, one is a single read, two are tie-heavy) through two sets of
    buffers with the copies of neighbouring builds overlapped; every output compared with the oracle at every position.  A
    stale buffer, a missed event or a result taken before its copy finished shows up as another collection's bytes."""
    import paper_1401_7457_b200 as cx
    rng = np.random.default_rng(77)
    colls = [gen.random_collection(1, 300, 90), gen.from_strings(["ACGTACGTACGTAACC"]),
             gen.from_strings(["".join(rng.choice(list("AC"), 60)) for _ in range(400)]),
             gen.config(0, 0.1), gen.from_strings(["GATTACA" * 9] * 70 + ["GATTACA" * 5])]
    max_reads, max_bases = max(c.n_reads for c in colls), max(c.total_bases for c in colls)
    plan = cx.Plan(max_reads, max_bases)
    pipe = cx.HostPipeline(plan, max_reads, max_bases)
    items = [(torch.from_numpy(c.ascii.copy()).pin_memory(), torch.from_numpy(c.offsets.astype(np.int64)).pin_memory(), c.n_reads) for c in colls]
    n = 0
    for c, got in zip(colls, pipe.run(items)):
        assert np.array_equal(got.numpy().copy(), oracle.bwt(c.ascii, c.offsets)), f"collection {n}"
        n += 1
    assert n == len(colls)
    assert list(pipe.run([])) == []
    plan.free()
    for bad in (dict(out_is_host_pinned=1), dict(out_bits=4)):
        p2 = cx.Plan(10, 100, **bad)
        with pytest.raises(cx.CxError):
            cx.HostPipeline(p2, 10, 100)
        p2.free()


def test_bad_finish_slots_option_is_rejected():
    import paper_1401_7457_b200 as cx
    with pytest.raises(cx.CxError):
        cx.Plan(100, 1000, finish_slots=3)
