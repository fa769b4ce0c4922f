"""Pins for the CPU oracle (oracle/cx_oracle.c) against things other than itself:
the paper's worked example, closed forms, brute force, invariants, LF inversion and a reduction to
a textbook suffix array.  CPU only."""
import itertools
import os

import numpy as np
import pytest

import oracle
from workloads import generate as gen
from tests import bwt_checks as chk

GOLDEN = os.path.join(os.path.dirname(__file__), "golden", "figure1.txt")


def _figure1():
    reads, bwt, suffixes = None, None, []
    for line in open(GOLDEN):
        if line.startswith("#") or not line.strip():
            continue
        tag, *rest = line.split()
        if tag == "reads":
            reads = rest
        elif tag == "bwt":
            bwt = rest[0]
        elif tag == "suffix":
            suffixes.append(rest[0])
    return reads, bwt, suffixes


# ---- P1: Figure 1, PAPER.md:57-67 -------------------------------------------------------------

def test_figure1_bwt_and_sorted_suffixes():
    reads, bwt, suffixes = _figure1()
    coll = gen.from_strings(reads)
    got, order = oracle.bwt(coll.ascii, coll.offsets, return_order=True)
    assert got.tobytes().decode() == bwt == "TTAAG$TAG$CAGG$"
    spelled = [reads[int(i)][int(p):] + "$" for i, p in order]
    assert spelled == suffixes
    # terminator order: equal suffixes appear by read index
    assert [tuple(map(int, o)) for o in order[:3]] == [(0, 4), (1, 4), (2, 4)]
    assert [tuple(map(int, o)) for o in order[10:12]] == [(0, 2), (1, 2)]   # the two "GT$": C then A


# ---- P2: closed forms ---------------------------------------------------------------------------

def test_duplicate_reads_repeat_each_symbol():
    # k copies of X: every symbol of the single-read BWT of X repeated k times in place
    for x in ["ACGT", "GATTACA", "TTTT", "C", ""]:
        single = oracle.bwt_of_strings([x])
        for k in (2, 3, 5):
            assert oracle.bwt_of_strings([x] * k) == "".join(c * k for c in single)
    assert oracle.bwt_of_strings(["ACGT"] * 3) == "TTT$$$AAACCCGGG"


def test_homopolymers_of_different_lengths():
    # suffixes: $0 $1 $2 | A$0 A$1 A$2 | AA$1 AA$2 | AAA$2  -> preceding symbols
    assert oracle.bwt_of_strings(["A", "AA", "AAA"]) == "AAA$AA$A$"
    assert oracle.bwt_of_strings(["AAA", "AA", "A"]) == "AAA" + "AA$" + "A$" + "$"
    assert oracle.bwt_of_strings(["T", "TT"]) == "TT$T$"


def test_empty_reads_and_empty_collection():
    assert oracle.bwt_of_strings([]) == ""
    assert oracle.bwt_of_strings([""]) == "$"
    assert oracle.bwt_of_strings(["", "A", ""]) == "$A$$"


def test_single_read_is_textbook_bwt():
    # n = 1: B is the classic BWT of S$ (rotation sort), e.g. the textbook "banana"-style check on DNA
    for s in ["GATTACA", "ACGTACGT", "AAAAC", "T"]:
        t = s + "$"
        rots = sorted(range(len(t)), key=lambda k: t[k:] + t[:k])
        assert oracle.bwt_of_strings([s]) == "".join(t[k - 1] for k in rots)


def test_rejects_non_acgt():
    for bad in ["ACGN", "acgt", "AC$T", "AC T"]:
        with pytest.raises(oracle.OracleError) as e:
            oracle.bwt_of_strings([bad])
        assert e.value.code == oracle.BAD_BASE


# ---- P3: brute force on hand-enumerable collections ---------------------------------------------

def _brute(reads):
    """Independent few-line restatement of PAPER.md:55: a suffix is a tuple of (rank, tiebreak)
    symbols; the end-marker of read i is (0, i); bases are (1..4, 0)."""
    rank = {"A": 1, "C": 2, "G": 3, "T": 4}
    sufs = []
    for i, r in enumerate(reads):
        for p in range(len(r) + 1):
            key = tuple((rank[c], 0) for c in r[p:]) + ((0, i),)
            sufs.append((key, "$" if p == 0 else r[p - 1]))
    return "".join(c for _, c in sorted(sufs))


def test_brute_force_all_small_collections_two_letters():
    words = [""] + ["".join(w) for L in range(1, 4) for w in itertools.product("AC", repeat=L)]   # 15 words
    for k in (1, 2, 3):
        for reads in itertools.product(words, repeat=k):
            assert oracle.bwt_of_strings(list(reads)) == _brute(reads), reads


def test_brute_force_random_four_letters():
    for seed in range(300):
        c = gen.random_collection(seed, n_reads=1 + seed % 7, max_len=1 + seed % 9,
                                  alphabet=["ACGT", "GT", "A", "CGT"][seed % 4])
        assert oracle.bwt(c.ascii, c.offsets).tobytes().decode() == _brute(c.strings())


# ---- P4: invariants + LF inversion --------------------------------------------------------------

@pytest.mark.parametrize("idx,scale", [(0, 0.05), (1, 0.002), (2, 0.0005), (3, 0.0002)])
def test_invariants_and_lf_inversion_on_config_shapes(idx, scale):
    c = gen.config(idx, scale)
    b = oracle.bwt(c.ascii, c.offsets)
    chk.check_all(b, c)


def test_lf_inversion_with_empty_and_duplicate_reads():
    c = gen.from_strings(["", "ACGT", "ACGT", "", "CGT", "T", "ACGT", ""])
    chk.check_all(oracle.bwt(c.ascii, c.offsets), c)


# ---- P5: reduction to a generic integer-alphabet suffix array -----------------------------------

def _via_suffix_array(reads):
    n = len(reads)
    code = {"A": n, "C": n + 1, "G": n + 2, "T": n + 3}
    text = []
    for i, r in enumerate(reads):
        text += [code[c] for c in r] + [i]          # terminator of read i is the integer i
    sa = sorted(range(len(text)), key=lambda k: text[k:])          # textbook suffix array
    sym = {v: k for k, v in code.items()}
    out = []
    for k in sa:
        prev = text[k - 1] if k > 0 else 0         # wrap-around and every terminator map to '$'
        out.append(sym.get(prev, "$") if k > 0 else "$")
    return "".join(out)


def test_matches_generic_suffix_array():
    for seed in range(200):
        c = gen.random_collection(1000 + seed, n_reads=1 + seed % 9, max_len=12, alphabet="ACGT"[: 1 + seed % 4])
        assert oracle.bwt(c.ascii, c.offsets).tobytes().decode() == _via_suffix_array(c.strings())
    c = gen.config(1, 0.0003)       # overlapping reads from a genome, duplicates included
    assert oracle.bwt(c.ascii, c.offsets).tobytes().decode() == _via_suffix_array(c.strings())


# ---- P6 / PAPER.md:73: partitions concatenate -----------------------------------------------------

def test_prefix_slices_concatenate_to_full_bwt():
    c = gen.config(2, 0.0003)
    full = oracle.bwt(c.ascii, c.offsets)
    covered = np.zeros(full.shape[0], dtype=bool)
    prev_end = None
    for p in ["".join(w) for w in itertools.product("ACGT", repeat=2)]:
        off, sl = oracle.bwt_with_prefix(c.ascii, c.offsets, p)
        assert np.array_equal(full[off:off + sl.shape[0]], sl)
        assert not covered[off:off + sl.shape[0]].any()
        covered[off:off + sl.shape[0]] = True
        if prev_end is not None:
            assert off >= prev_end
        prev_end = off + sl.shape[0]
    # what is left are exactly the suffixes shorter than 2 symbols: "$" and "x$": (1 + 1) per read
    assert int((~covered).sum()) == 2 * c.n_reads
    off, sl = oracle.bwt_with_prefix(c.ascii, c.offsets, "")
    assert off == 0 and np.array_equal(sl, full)


def test_generators_are_deterministic_and_acgt_only():
    a, b = gen.config(3, 0.0002), gen.config(3, 0.0002)
    assert np.array_equal(a.ascii, b.ascii) and np.array_equal(a.offsets, b.offsets)
    assert set(np.unique(a.ascii)) <= set(b"ACGT")
    lens = np.diff(a.offsets.astype(np.int64))
    assert lens.min() >= 50 and lens.max() <= 250
    c2 = gen.config(1, 0.001)
    assert len(set(c2.strings())) < c2.n_reads       # 100x coverage: exact duplicate reads exist


def test_listed_form_equals_full_and_prefix_forms():
    """cx_oracle_bwt_of_listed: listing every suffix gives B_R; listing those with a prefix gives the prefix slice;
    dropping the reads that own no listed suffix (indices kept in order) changes nothing."""
    c = gen.config(2, 0.0003)
    off = c.offsets.astype(np.int64)
    every = np.array([(i, p) for i in range(c.n_reads) for p in range(int(off[i + 1] - off[i]) + 1)], dtype=np.uint64)
    got, order = oracle.bwt_of_listed(c.ascii, c.offsets, every[::-1])          # any input order
    want, want_order = oracle.bwt(c.ascii, c.offsets, return_order=True)
    assert np.array_equal(got, want) and np.array_equal(order, want_order)
    text = c.ascii.tobytes()
    for pfx in (b"AC", b"TTG", b"G"):
        sel = np.array([(i, p) for i, p in every.tolist() if text[off[i] + p: min(off[i] + p + len(pfx), off[i + 1])] == pfx],
                       dtype=np.uint64).reshape(-1, 2)
        _, want_slice = oracle.bwt_with_prefix(c.ascii, c.offsets, pfx.decode())
        got_slice, _ = oracle.bwt_of_listed(c.ascii, c.offsets, sel)
        assert np.array_equal(got_slice, want_slice)
        # sub-collection of the owning reads only
        owners = np.unique(sel[:, 0]).astype(np.int64)
        sub_off = np.zeros(owners.size + 1, dtype=np.uint64)
        sub_off[1:] = np.cumsum(off[owners + 1] - off[owners])
        sub_text = np.concatenate([c.ascii[off[i]:off[i + 1]] for i in owners]) if owners.size else np.zeros(0, np.uint8)
        remap = sel.copy()
        remap[:, 0] = np.searchsorted(owners, sel[:, 0].astype(np.int64))
        got_sub, _ = oracle.bwt_of_listed(sub_text, sub_off, remap)
        assert np.array_equal(got_sub, want_slice)
