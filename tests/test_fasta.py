"""NEXT-4: FASTA ingest.  CPU part: the oracle parser against a hand-enumerated fixture, special cases and round trips
of the seeded writer.  GPU part: cx_fasta_parse (through the C ABI) against the oracle, byte for byte, and the whole
path FASTA text -> BWT against the oracle's BWT."""
import os

import numpy as np
import pytest

import oracle
from oracle import fasta as ofa
from workloads import generate as gen

GOLD = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden")


def _expected():
    lines = open(os.path.join(GOLD, "fasta_small.expected")).read().split("\n")
    return [l.encode() for l in lines if not l.startswith("#")][:-1]      # the file ends with a newline


# ---- oracle pins (CPU) ---------------------------------------------------------------------------------
def test_oracle_parser_on_hand_enumerated_fixture():
    text = open(os.path.join(GOLD, "fasta_small.fa"), "rb").read()
    reads, orphans = ofa.parse_fasta(text)
    assert reads == _expected() == [b"ACGT", b"TAGT", b"", b"GGAA"] and orphans == 0


@pytest.mark.parametrize("text,reads,orphans", [
    (b"", [], 0),
    (b"\n\n", [], 0),
    (b">only a header", [b""], 0),
    (b">a\n>b\n", [b"", b""], 0),
    (b">a\nAC\nGT", [b"ACGT"], 0),
    (b">a\r\nAC\r\n\r\nGT\r\n", [b"ACGT"], 0),
    (b"ACGT\n>a\nTT\n", [b"TT"], 4),                       # sequence before any header belongs to no read
    (b">a\nAC>GT\n", [b"AC>GT"], 0),                       # '>' is a header mark only at the start of a line
    (b">a\nAC\n >b\nGT\n", [b"AC >bGT"], 0),               # not at the start: a sequence line (pack will reject the bytes)
])
def test_oracle_parser_special_cases(text, reads, orphans):
    assert ofa.parse_fasta(text) == (reads, orphans)


@pytest.mark.parametrize("width,crlf,final,seed", [(0, False, True, None), (7, False, False, 1), (60, True, True, 2), (1, True, False, 3)])
def test_oracle_parser_round_trips_the_writer(width, crlf, final, seed):
    c = gen.random_collection(5 + width, n_reads=200, max_len=150)
    text = gen.to_fasta(c, line_width=width, crlf=crlf, final_newline=final, seed=seed)
    bases, offsets, orphans = ofa.parse_fasta_arrays(text)
    assert orphans == 0 and np.array_equal(bases, c.ascii) and np.array_equal(offsets, c.offsets)
    # invariant: the bases are exactly the bytes of non-header lines other than line ends
    payload = sum(len(l.replace(b"\r", b"")) for l in text.split(b"\n") if l[:1] != b">")
    assert payload == bases.size


# ---- parity of the CUDA path (GPU) ------------------------------------------------------------------------
def _gpu_parse(text: bytes):
    import torch
    import paper_1401_7457_b200 as cx
    t = torch.from_numpy(np.frombuffer(text, dtype=np.uint8).copy()).cuda() if text else torch.zeros(0, dtype=torch.uint8, device="cuda")
    bases, offsets = cx.cx_fasta_parse(t)
    return bases.cpu().numpy(), offsets.cpu().numpy().astype(np.uint64)


def _assert_parse_parity(text: bytes):
    want_b, want_o, orphans = ofa.parse_fasta_arrays(text)
    assert orphans == 0
    got_b, got_o = _gpu_parse(text)
    assert np.array_equal(got_o, want_o), (got_o[:8], want_o[:8])
    assert np.array_equal(got_b, want_b)


@pytest.mark.gpu
def test_parse_fixture_and_special_cases():
    _assert_parse_parity(open(os.path.join(GOLD, "fasta_small.fa"), "rb").read())
    for text in (b"", b"\n\n", b">only a header", b">a\n>b\n", b">a\nAC\nGT", b">a\r\nAC\r\n\r\nGT\r\n", b">a\nAC>GT\n", b">\n", b">a\n" + b"ACGT" * 5000):
        _assert_parse_parity(text)


@pytest.mark.gpu
@pytest.mark.parametrize("width,crlf,final,seed", [(0, False, True, None), (7, False, False, 1), (60, True, True, 2), (1, True, False, 3),
                                                   (4096, False, True, 4), (16, False, True, 5)])
def test_parse_random_collections(width, crlf, final, seed):
    for k, (n_reads, max_len) in enumerate([(1, 1), (300, 140), (5000, 260), (40, 30000)]):      # lines longer than several tiles too
        c = gen.random_collection(100 * width + k, n_reads=n_reads, max_len=max_len)
        _assert_parse_parity(gen.to_fasta(c, line_width=width, crlf=crlf, final_newline=final, seed=seed))


@pytest.mark.gpu
def test_parse_text_at_unaligned_address_and_ragged_tail():
    import torch
    import paper_1401_7457_b200 as cx
    c = gen.config(0, 0.05)
    text = gen.to_fasta(c, line_width=33, seed=7)
    for skew in (1, 5, 15):
        buf = torch.zeros(len(text) + 32, dtype=torch.uint8, device="cuda")
        view = buf[skew:skew + len(text)]
        view.copy_(torch.from_numpy(np.frombuffer(text, dtype=np.uint8).copy()))
        bases, offsets = cx.cx_fasta_parse(view)
        assert np.array_equal(bases.cpu().numpy(), c.ascii) and np.array_equal(offsets.cpu().numpy().astype(np.uint64), c.offsets)


@pytest.mark.gpu
def test_orphan_bytes_and_too_many_reads_are_reported():
    import torch
    import paper_1401_7457_b200 as cx
    t = torch.from_numpy(np.frombuffer(b"ACGT\n>a\nTT\n", dtype=np.uint8).copy()).cuda()
    with pytest.raises(cx.CxError):
        cx.cx_fasta_parse(t)
    t = torch.from_numpy(np.frombuffer(b">a\nA\n>b\nC\n>c\nG\n", dtype=np.uint8).copy()).cuda()
    with pytest.raises(cx.CxError):
        cx.cx_fasta_parse(t, max_reads=2)
    bases, offsets = cx.cx_fasta_parse(t, max_reads=3)
    assert bases.cpu().numpy().tobytes() == b"ACG" and offsets.tolist() == [0, 1, 2, 3]


@pytest.mark.gpu
def test_fasta_text_to_bwt_end_to_end():
    import paper_1401_7457_b200 as cx
    assert cx.bwt_of_fasta(open(os.path.join(GOLD, "fasta_small.fa"), "rb").read()).tobytes() == oracle.bwt_of_strings(["ACGT", "TAGT", "", "GGAA"]).encode()
    assert cx.bwt_of_fasta(b">r0\nACGT\n>r1\nTAGT\n>r2\nGGAA\n").tobytes() == b"TTAAG$TAG$CAGG$"      # Figure 1
    c = gen.config(1, 0.01)
    got = cx.bwt_of_fasta(gen.to_fasta(c, line_width=60, crlf=True, seed=11))
    assert np.array_equal(got, oracle.bwt(c.ascii, c.offsets))
    with pytest.raises(cx.CxError):
        cx.bwt_of_fasta(b">r0\nACNT\n")                      # A8: bytes outside ACGT are rejected by the pack step


@pytest.mark.gpu
def test_parse_texts_around_the_tile_size():
    """Texts of exactly one tile (16 KB), one byte less and one more; a header and a CRLF pair straddling a tile edge;
    a tile of nothing but line ends."""
    tile = 16384
    for n in (tile - 1, tile, tile + 1, 2 * tile, 2 * tile + 17):
        body = (b"ACGT" * (n // 4 + 1))[:n - 3]
        _assert_parse_parity(b">x\n" + body)                                   # one read, no final newline, n bytes in all
    head = b">" + b"h" * 40 + b"\n"
    for cut in range(tile - 45, tile + 3, 7):                                 # the header line slides across the tile edge
        pre = (b">a\n" + b"ACGT" * (tile // 4))[:cut - 1] + b"\n"
        _assert_parse_parity(pre + head + b"GGAA\r\nTT\r\n")
    _assert_parse_parity(b">a\nAC" + b"\r\n" * (tile // 2 + 5) + b"GT\n>b\n" + b"\n" * tile + b"T")
