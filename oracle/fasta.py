"""CPU oracle of the FASTA ingest step (NEXT-4) -- TEST INFRASTRUCTURE, not product (same rules as oracle/__init__.py).

The paper says only that "the input was in FASTA format" and that reads consist of {A, C, G, T}; the
grammar below is the reading DESIGN.md section 16 takes, written out line by line:

  * the text is split at every b"\\n" (a last line without one is still a line);
  * a line whose first byte is b">" is a header: it opens a new read and contributes nothing else;
  * any other line is a sequence line: its bytes with every b"\\r" removed are appended to the open read;
  * sequence bytes met before the first header belong to no read: they are returned as `orphans`.

Pinned by a hand-enumerated fixture (tests/golden/fasta_small.fa / .expected), by special cases (empty text, empty
reads, wrapped lines, CRLF, no final newline) and by round trips of a seeded writer that lives with the generators.
"""
from __future__ import annotations

import numpy as np


def parse_fasta(text: bytes):
    """-> (list of reads as bytes, number of orphan bytes)."""
    reads: list[bytearray] = []
    orphans = 0
    for line in bytes(text).split(b"\n"):
        if line[:1] == b">":
            reads.append(bytearray())
            continue
        payload = line.replace(b"\r", b"")
        if reads:
            reads[-1] += payload
        else:
            orphans += len(payload)
    return [bytes(r) for r in reads], orphans


def parse_fasta_arrays(text: bytes):
    """-> (bases uint8[total], offsets uint64[n_reads + 1], orphans): the layout cx_pack_reads / cx_bwt_build take."""
    reads, orphans = parse_fasta(text)
    offsets = np.zeros(len(reads) + 1, dtype=np.uint64)
    if reads:
        offsets[1:] = np.cumsum([len(r) for r in reads], dtype=np.uint64)
    bases = np.frombuffer(b"".join(reads), dtype=np.uint8).copy()
    return bases, offsets, orphans
