"""Output-side checks that hold for any valid collection BWT: symbol counts,
terminator count, the first-n rule and LF-mapping inversion.  Independent of both the oracle and the
CUDA path: they only look at a BWT byte array and at the input reads."""
from __future__ import annotations

import numpy as np

SYMS = b"$ACGT"


def symbol_counts(b: np.ndarray) -> dict:
    cnt = np.bincount(b, minlength=256)
    return {chr(s): int(cnt[s]) for s in SYMS}


def check_counts(bwt: np.ndarray, coll) -> None:
    """length N, exactly n_reads '$', each base as often as in the input, nothing else."""
    assert bwt.shape[0] == coll.n_suffixes
    got = symbol_counts(bwt)
    want = symbol_counts(coll.ascii) if coll.total_bases else {chr(s): 0 for s in SYMS}
    want["$"] = coll.n_reads
    assert got == want
    assert sum(got.values()) == bwt.shape[0]


def check_first_n(bwt: np.ndarray, coll) -> None:
    """The n end-marker suffixes sort first, by read index, so the first n output
    symbols are the last base of each read in read order ('$' for an empty read)."""
    n = coll.n_reads
    off = coll.offsets.astype(np.int64)
    lens = np.diff(off)
    last = np.where(lens > 0, coll.ascii[np.maximum(off[1:] - 1, 0)] if coll.total_bases else ord("$"), ord("$"))
    assert np.array_equal(bwt[:n], last.astype(np.uint8))


class LF:
    """LF-mapping over a multi-string BWT: row k holds symbol c = B[k]; the suffix that starts with
    that occurrence of c sits at row C[c] + occ(c, k)."""

    def __init__(self, bwt: np.ndarray):
        self.b = bwt
        cnt = np.bincount(bwt, minlength=256)
        self.C = {}
        acc = 0
        for s in SYMS:
            self.C[s] = acc
            acc += int(cnt[s])
        self.pos = {s: np.flatnonzero(bwt == s) for s in SYMS[1:]}

    def invert(self, read_ids: np.ndarray, max_len: int) -> list[bytes]:
        """Reconstruct the given reads: start at row i (the $_i suffix), walk until '$'."""
        rows = np.asarray(read_ids, dtype=np.int64).copy()
        alive = np.ones(rows.shape[0], dtype=bool)
        out = [bytearray() for _ in range(rows.shape[0])]
        for _ in range(max_len + 1):
            if not alive.any():
                break
            sym = self.b[rows]
            alive &= sym != ord("$")
            nxt = rows.copy()
            for s in SYMS[1:]:
                m = alive & (sym == s)
                if m.any():
                    nxt[m] = self.C[s] + np.searchsorted(self.pos[s], rows[m], side="left")
            for j in np.flatnonzero(alive):
                out[j].append(int(sym[j]))
            rows = nxt
        assert not alive.any(), "walk did not reach '$' within max_len+1 steps"
        return [bytes(reversed(o)) for o in out]


def check_lf_inversion(bwt: np.ndarray, coll, read_ids=None) -> None:
    ids = np.arange(coll.n_reads) if read_ids is None else np.asarray(read_ids)
    if ids.size == 0:
        return
    got = LF(bwt).invert(ids, coll.max_read_len)
    for j, i in enumerate(ids):
        want = coll.ascii[int(coll.offsets[i]):int(coll.offsets[i + 1])].tobytes()
        assert got[j] == want, f"LF inversion of read {i} gave {got[j]!r}, want {want!r}"


def check_all(bwt: np.ndarray, coll, lf_sample: int | None = None, seed: int = 1) -> None:
    check_counts(bwt, coll)
    check_first_n(bwt, coll)
    if lf_sample is None or lf_sample >= coll.n_reads:
        check_lf_inversion(bwt, coll)
    else:
        rng = np.random.default_rng(seed)
        check_lf_inversion(bwt, coll, np.sort(rng.choice(coll.n_reads, lf_sample, replace=False)))
