"""Seeded synthetic read collections (inputs only; none of the method's arithmetic lives here).

Both the CPU oracle (``oracle/``) and the CUDA path (``paper_1401_7457_b200``) are fed from this
module and from nothing else they share.  A collection is plain data: the reads as one contiguous
ASCII byte array over ``ACGT`` (no terminators stored) plus ``n_reads + 1`` base offsets.

Every random choice is a pure function ``H(seed, stream, counter)`` of a SplitMix64-style 64-bit
mixer, so any read of any config can be regenerated anywhere without storing the collection.

The five recipes stand in for the paper's workload -- subsets of the "Asian YH" human short reads,
100 bp, ACGT only, 100M/500M/1000M reads (Section 4; Table 1) --
which is not available here.  Shapes follow BASELINE.json ``configs[0..4]``; the concrete draws are
the ones listed in SURVEY.md Section 8(d) and restated in DESIGN.md ("Input recipe").
"""
from __future__ import annotations

from dataclasses import dataclass

import numpy as np

_U64 = np.uint64
_GOLD = _U64(0x9E3779B97F4A7C15)
_M1 = _U64(0xBF58476D1CE4E5B9)
_M2 = _U64(0x94D049BB133111EB)

BASE_SEED = 0x14017457
ASCII_OF_CODE = np.frombuffer(b"ACGT", dtype=np.uint8)


def mix64(z: np.ndarray) -> np.ndarray:
    """SplitMix64 finaliser on uint64 arrays (wrapping arithmetic)."""
    z = np.asarray(z, dtype=_U64)
    z = (z ^ (z >> _U64(30))) * _M1
    z = (z ^ (z >> _U64(27))) * _M2
    return z ^ (z >> _U64(31))


def H(seed: int, stream: int, counter) -> np.ndarray:
    """Counter-based generator: ``mix64(mix64(seed + GOLD*(stream+1)) + GOLD*(counter+1))``."""
    with np.errstate(over="ignore"):
        s = mix64(np.array([(seed + 0x9E3779B97F4A7C15 * (stream + 1)) & 0xFFFFFFFFFFFFFFFF], dtype=_U64))[0]
        c = np.asarray(counter, dtype=_U64)
        return mix64(s + _GOLD * (c + _U64(1)))


@dataclass
class Collection:
    """A read collection: ``ascii[offsets[i]:offsets[i+1]]`` is read ``i`` (bytes over ``ACGT``)."""

    ascii: np.ndarray      # uint8[total_bases]
    offsets: np.ndarray    # uint64[n_reads + 1], offsets[0] = 0, non-decreasing
    name: str = ""

    @property
    def n_reads(self) -> int:
        return int(self.offsets.shape[0] - 1)

    @property
    def total_bases(self) -> int:
        return int(self.offsets[-1])

    @property
    def n_suffixes(self) -> int:
        return self.total_bases + self.n_reads

    @property
    def max_read_len(self) -> int:
        if self.n_reads == 0:
            return 0
        return int(np.max(np.diff(self.offsets.astype(np.int64))))

    def read(self, i: int) -> str:
        return self.ascii[int(self.offsets[i]):int(self.offsets[i + 1])].tobytes().decode("ascii")

    def strings(self) -> list[str]:
        return [self.read(i) for i in range(self.n_reads)]


def from_strings(reads: list[str], name: str = "") -> Collection:
    lens = np.array([len(r) for r in reads], dtype=np.uint64)
    offsets = np.zeros(len(reads) + 1, dtype=np.uint64)
    np.cumsum(lens, out=offsets[1:])
    ascii_ = np.frombuffer("".join(reads).encode("ascii"), dtype=np.uint8).copy()
    return Collection(ascii_, offsets, name)


# ----------------------------------------------------------------------------------------------
# genomes (arrays of codes 0..3)
# ----------------------------------------------------------------------------------------------

def _iid_codes(seed: int, stream: int, start: int, count: int) -> np.ndarray:
    out = np.empty(count, dtype=np.uint8)
    step = 1 << 22
    for a in range(0, count, step):
        b = min(count, a + step)
        out[a:b] = (H(seed, stream, np.arange(start + a, start + b, dtype=_U64)) & _U64(3)).astype(np.uint8)
    return out


def _substitute(codes: np.ndarray, draws: np.ndarray, rate_num: int, rate_den: int) -> np.ndarray:
    """Replace a base by one of the three OTHER bases with probability rate_num/rate_den."""
    thresh = _U64((rate_num << 32) // rate_den)
    hit = (draws & _U64(0xFFFFFFFF)) < thresh
    shift = ((draws >> _U64(32)) % _U64(3) + _U64(1)).astype(np.uint8)
    return np.where(hit, (codes + shift) & 3, codes).astype(np.uint8)


def repeat_genome(seed: int, G: int) -> np.ndarray:
    """configs[3] genome: iid background, 5 % covered by copies of 20 repeat elements at 2 % divergence."""
    g = _iid_codes(seed, 1, 0, G)
    n_elem = 20
    elem_len = (300 + H(seed, 6, np.arange(n_elem)) % _U64(5701)).astype(np.int64)   # uniform in [300, 6000]
    elem_len = np.minimum(elem_len, max(1, G // 8))
    elems = [_iid_codes(seed, 7, e * 8192, int(elem_len[e])) for e in range(n_elem)]
    target = G // 20
    pasted = 0
    c = 0
    while pasted < target:
        e = c % n_elem
        L = int(elem_len[e])
        pos = int(H(seed, 8, np.array([c]))[0] % _U64(G - L + 1))
        copy = _substitute(elems[e], H(seed, 10, c * 8192 + np.arange(L)), 2, 100)
        g[pos:pos + L] = copy
        pasted += L
        c += 1
    return g


# ----------------------------------------------------------------------------------------------
# read samplers
# ----------------------------------------------------------------------------------------------

def _sample_reads(seed: int, genome: np.ndarray, n_reads: int, len_lo: int, len_hi: int,
                  both_strands: bool, err_num: int, err_den: int, name: str) -> Collection:
    G = genome.shape[0]
    idx = np.arange(n_reads, dtype=_U64)
    if len_lo == len_hi:
        lens = np.full(n_reads, len_lo, dtype=np.int64)
    else:
        lens = (len_lo + H(seed, 5, idx) % _U64(len_hi - len_lo + 1)).astype(np.int64)
    lens = np.minimum(lens, G)
    offsets = np.zeros(n_reads + 1, dtype=np.uint64)
    np.cumsum(lens.astype(np.uint64), out=offsets[1:])
    total = int(offsets[-1])
    out = np.empty(total, dtype=np.uint8)
    starts = (H(seed, 2, idx) % (_U64(G) - lens.astype(_U64) + _U64(1))).astype(np.int64)
    strand = (H(seed, 3, idx) & _U64(1)).astype(np.uint8) if both_strands else np.zeros(n_reads, np.uint8)
    chunk = 1 << 18
    for a in range(0, n_reads, chunk):
        b = min(n_reads, a + chunk)
        ln = lens[a:b]
        o0 = int(offsets[a])
        tot = int(offsets[b]) - o0
        if tot == 0:
            continue
        rid = np.repeat(np.arange(a, b, dtype=np.int64), ln)              # read of each base
        k = np.arange(tot, dtype=np.int64) - (offsets[a:b].astype(np.int64) - o0)[rid - a]   # position in read
        st = strand[rid]
        # forward: genome[start + k]; reverse complement: 3 - genome[start + len - 1 - k]
        gpos = np.where(st == 0, starts[rid] + k, starts[rid] + lens[rid] - 1 - k)
        codes = genome[gpos]
        codes = np.where(st == 0, codes, 3 - codes).astype(np.uint8)
        if err_num:
            codes = _substitute(codes, H(seed, 4, rid.astype(_U64) * _U64(256) + k.astype(_U64)), err_num, err_den)
        out[o0:o0 + tot] = ASCII_OF_CODE[codes]
    return Collection(out, offsets, name)


def config(index: int, scale: float = 1.0, seed: int | None = None) -> Collection:
    """BASELINE.json ``configs[index]`` (0-based), optionally scaled down with coverage preserved.

    ``scale`` multiplies the number of reads and the genome length; read lengths, strand mix and
    error rates are unchanged, so tie depth and group sizes keep the full config's structure.
    """
    if seed is None:
        seed = BASE_SEED + index
    if index == 0:      # 10,000 x 100 bp iid
        n, m = max(1, int(round(10_000 * scale))), 100
        codes = _iid_codes(seed, 0, 0, n * m)
        offsets = (np.arange(n + 1, dtype=np.uint64) * np.uint64(m))
        return Collection(ASCII_OF_CODE[codes], offsets, f"C1x{scale:g}")
    if index == 1:      # 1M x 100 bp, 1 Mbp genome, forward only, no errors
        G, n = max(200, int(round(1_000_000 * scale))), max(1, int(round(1_000_000 * scale)))
        return _sample_reads(seed, _iid_codes(seed, 1, 0, G), n, 100, 100, False, 0, 1, f"C2x{scale:g}")
    if index == 2:      # 10M x 100 bp, 33 Mbp genome, both strands, 1 % substitutions
        G, n = max(200, int(round(33_000_000 * scale))), max(1, int(round(10_000_000 * scale)))
        return _sample_reads(seed, _iid_codes(seed, 1, 0, G), n, 100, 100, True, 1, 100, f"C3x{scale:g}")
    if index == 3:      # 40M x 50..250 bp, 50 Mbp repeat genome, both strands, 0.5 %
        G, n = max(8000, int(round(50_000_000 * scale))), max(1, int(round(40_000_000 * scale)))
        return _sample_reads(seed, repeat_genome(seed, G), n, 50, 250, True, 5, 1000, f"C4x{scale:g}")
    if index == 4:      # 1G x 100 bp, 3.3 Gbp genome, both strands, 1 %
        G, n = max(200, int(round(3_300_000_000 * scale))), max(1, int(round(1_000_000_000 * scale)))
        return _sample_reads(seed, _iid_codes(seed, 1, 0, G), n, 100, 100, True, 1, 100, f"C5x{scale:g}")
    raise ValueError("config index must be 0..4")


def table4(read_len: int, scale: float = 1.0, seed: int | None = None) -> Collection:
    """Stand-in for the paper's read-length experiment (Table 4; Section 4.3): equal
    total bases (1e10 at scale 1) in reads of 100, 200 or 400 bp -- 100M x 100, 50M x 200, 25M x 400 in the paper.
    Same structure as configs[2]: 30x over an iid genome, both strands, 1 % substitutions."""
    if seed is None:
        seed = BASE_SEED + 40 + read_len
    total = max(read_len, int(round(10_000_000_000 * scale)))
    n = max(1, total // read_len)
    G = max(2 * read_len, total // 30)
    return _sample_reads(seed, _iid_codes(seed, 1, 0, G), n, read_len, read_len, True, 1, 100, f"T4-{read_len}x{scale:g}")


def random_collection(seed: int, n_reads: int, max_len: int, alphabet: str = "ACGT",
                      min_len: int = 0) -> Collection:
    """Small adversarial collections for tests: short alphabets and ragged (possibly empty) reads."""
    idx = np.arange(n_reads, dtype=_U64)
    lens = (min_len + H(seed, 20, idx) % _U64(max_len - min_len + 1)).astype(np.int64)
    offsets = np.zeros(n_reads + 1, dtype=np.uint64)
    np.cumsum(lens.astype(np.uint64), out=offsets[1:])
    total = int(offsets[-1])
    letters = np.frombuffer(alphabet.encode("ascii"), dtype=np.uint8)
    draws = H(seed, 21, np.arange(total, dtype=_U64)) % _U64(len(letters))
    return Collection(letters[draws.astype(np.int64)], offsets, f"rand{seed}")


# ----------------------------------------------------------------------------------------------
# FASTA text of a collection (input of the ingest step, NEXT-4; "The input was in FASTA format")
# ----------------------------------------------------------------------------------------------
def to_fasta(coll: Collection, line_width: int = 0, crlf: bool = False, final_newline: bool = True, seed: int | None = None) -> bytes:
    """One record per read: a '>' header line, then the bases on lines of at most `line_width` bytes (0: one line;
    an empty read has no sequence line).  With a seed, header texts vary in length and a few blank lines are strewn in
    (both legal under the grammar of DESIGN.md section 16)."""
    eol = b"\r\n" if crlf else b"\n"
    parts = []
    draws = H(seed, 9, np.arange(coll.n_reads, dtype=np.uint64)) if seed is not None else None
    for i in range(coll.n_reads):
        r = coll.ascii[int(coll.offsets[i]):int(coll.offsets[i + 1])].tobytes()
        if draws is None:
            parts.append(b">r%d" % i)
        else:
            d = int(draws[i])
            parts.append(b">read_%d %s" % (i, b"x" * (d % 23)))
            if d % 11 == 0:
                parts.append(eol)      # a blank line after the header
        parts.append(eol)
        if r:
            if line_width:
                parts.append(eol.join(r[k:k + line_width] for k in range(0, len(r), line_width)))
            else:
                parts.append(r)
            parts.append(eol)
    text = b"".join(parts)
    if not final_newline and text.endswith(eol):
        text = text[:-len(eol)]
    return text
