"""The same seeded recipes as ``workloads/generate.py``, evaluated with torch tensor ops so that the
large configs (configs[3], configs[4]) can be produced chunk by chunk straight into device memory:
the 100 GB ASCII form of configs[4] never exists at once.  Inputs only -- none of the method's
arithmetic lives here.  ``tests/test_generators.py`` checks, on CPU tensors, that every function
below returns exactly what the numpy module returns.

64-bit unsigned arithmetic is spelled with int64 tensors: multiplication and addition wrap the same
way, right shifts are made logical with a mask, and ``x mod m`` is taken limb-wise.
"""
from __future__ import annotations

import torch

from . import generate as gen

_M1 = -4658895280553007687      # 0xBF58476D1CE4E5B9 as int64
_M2 = -7723592293110705685      # 0x94D049BB133111EB as int64
_GOLD = -7046029254386353131    # 0x9E3779B97F4A7C15 as int64


def _lsr(z: torch.Tensor, k: int) -> torch.Tensor:
    return (z >> k) & ((1 << (64 - k)) - 1)


def mix64(z: torch.Tensor) -> torch.Tensor:
    z = (z ^ _lsr(z, 30)) * _M1
    z = (z ^ _lsr(z, 27)) * _M2
    return z ^ _lsr(z, 31)


def _seed_stream(seed: int, stream: int) -> int:
    """mix64(seed + GOLD * (stream + 1)) as a Python int in int64 range (host arithmetic, one value)."""
    import numpy as np
    with np.errstate(over="ignore"):
        s = gen.mix64(np.array([(seed + 0x9E3779B97F4A7C15 * (stream + 1)) & 0xFFFFFFFFFFFFFFFF], dtype=np.uint64))[0]
    s = int(s)
    return s - (1 << 64) if s >= (1 << 63) else s


def H(seed: int, stream: int, counter: torch.Tensor) -> torch.Tensor:
    """``generate.H`` on an int64 tensor of counters; the result holds the uint64 bit pattern."""
    return mix64(_seed_stream(seed, stream) + _GOLD * (counter + 1))


def umod(x: torch.Tensor, m) -> torch.Tensor:
    """(x as uint64) mod m for 0 < m < 2^32, m an int or an int64 tensor."""
    hi = _lsr(x, 32)
    lo = x & 0xFFFFFFFF
    if isinstance(m, int):
        assert 0 < m < (1 << 32)
        return ((hi % m) * ((1 << 32) % m) + lo % m) % m
    return ((hi % m) * ((1 << 32) % m) + lo % m) % m


def iid_codes(seed: int, stream: int, start: int, count: int, device, chunk: int = 1 << 26) -> torch.Tensor:
    out = torch.empty(count, dtype=torch.uint8, device=device)
    for a in range(0, count, chunk):
        b = min(count, a + chunk)
        c = torch.arange(start + a, start + b, dtype=torch.int64, device=device)
        out[a:b] = (H(seed, stream, c) & 3).to(torch.uint8)
    return out


def substitute(codes: torch.Tensor, draws: torch.Tensor, rate_num: int, rate_den: int) -> torch.Tensor:
    thresh = (rate_num << 32) // rate_den
    hit = (draws & 0xFFFFFFFF) < thresh
    shift = (umod(_lsr(draws, 32), 3) + 1).to(torch.uint8)
    return torch.where(hit, (codes + shift) & 3, codes)


class ReadRecipe:
    """Parameters of ``generate._sample_reads`` for one config, with the genome already on `device`."""

    def __init__(self, index: int, scale: float = 1.0, seed: int | None = None, device="cpu"):
        self.index = index
        self.seed = gen.BASE_SEED + index if seed is None else seed
        self.device = torch.device(device)
        if index == 1:
            G, n, lo, hi, both, en, ed = max(200, int(round(1_000_000 * scale))), max(1, int(round(1_000_000 * scale))), 100, 100, False, 0, 1
        elif index == 2:
            G, n, lo, hi, both, en, ed = max(200, int(round(33_000_000 * scale))), max(1, int(round(10_000_000 * scale))), 100, 100, True, 1, 100
        elif index == 3:
            G, n, lo, hi, both, en, ed = max(8000, int(round(50_000_000 * scale))), max(1, int(round(40_000_000 * scale))), 50, 250, True, 5, 1000
        elif index == 4:
            G, n, lo, hi, both, en, ed = max(200, int(round(3_300_000_000 * scale))), max(1, int(round(1_000_000_000 * scale))), 100, 100, True, 1, 100
        else:
            raise ValueError("ReadRecipe covers configs[1..4]")
        self.G, self.n_reads, self.len_lo, self.len_hi, self.both, self.err_num, self.err_den = G, n, lo, hi, both, en, ed
        if index == 3:
            self.genome = torch.from_numpy(gen.repeat_genome(self.seed, G)).to(self.device)     # sequential recipe: host
        else:
            self.genome = iid_codes(self.seed, 1, 0, G, self.device)

    def lengths(self, a: int, b: int) -> torch.Tensor:
        """Lengths of reads a..b-1 (int64)."""
        if self.len_lo == self.len_hi:
            return torch.full((b - a,), min(self.len_lo, self.G), dtype=torch.int64, device=self.device)
        idx = torch.arange(a, b, dtype=torch.int64, device=self.device)
        lens = self.len_lo + umod(H(self.seed, 5, idx), self.len_hi - self.len_lo + 1)
        return torch.clamp(lens, max=self.G)

    def reads_ascii(self, a: int, b: int, lens: torch.Tensor | None = None) -> torch.Tensor:
        """Reads a..b-1 back to back as ASCII bytes (uint8 tensor on the recipe's device)."""
        idx = torch.arange(a, b, dtype=torch.int64, device=self.device)
        return self.reads_ascii_of(idx, self.lengths(a, b) if lens is None else lens)

    def lengths_of(self, idx: torch.Tensor) -> torch.Tensor:
        if self.len_lo == self.len_hi:
            return torch.full_like(idx, min(self.len_lo, self.G))
        return torch.clamp(self.len_lo + umod(H(self.seed, 5, idx), self.len_hi - self.len_lo + 1), max=self.G)

    def reads_ascii_of(self, idx: torch.Tensor, lens: torch.Tensor | None = None) -> torch.Tensor:
        """The reads with the given indices (int64 tensor, any order) back to back as ASCII bytes."""
        dev = self.device
        if lens is None:
            lens = self.lengths_of(idx)
        m = idx.numel()
        starts = umod(H(self.seed, 2, idx), self.G - lens + 1)
        strand = (H(self.seed, 3, idx) & 1) if self.both else torch.zeros_like(idx)
        off = torch.zeros(m + 1, dtype=torch.int64, device=dev)
        torch.cumsum(lens, 0, out=off[1:])
        tot = int(off[-1])
        if tot == 0:
            return torch.zeros(0, dtype=torch.uint8, device=dev)
        rid = torch.repeat_interleave(torch.arange(m, dtype=torch.int64, device=dev), lens, output_size=tot)
        k = torch.arange(tot, dtype=torch.int64, device=dev) - off[rid]
        st = strand[rid]
        gpos = torch.where(st == 0, starts[rid] + k, starts[rid] + lens[rid] - 1 - k)
        codes = self.genome[gpos]
        codes = torch.where(st == 0, codes, 3 - codes)
        if self.err_num:
            codes = substitute(codes, H(self.seed, 4, idx[rid] * 256 + k), self.err_num, self.err_den)
        lut = torch.tensor(list(b"ACGT"), dtype=torch.uint8, device=dev)
        return lut[codes.to(torch.int64)]


def read_chunks(recipe: ReadRecipe, chunk_reads: int):
    """The recipe's reads in chunks of at most `chunk_reads`: yields (a, b, lens int64[b - a], ascii uint8) on the recipe's
    device.  The whole ASCII form never exists at once (configs[4] is 100 GB of it)."""
    n = recipe.n_reads
    for a in range(0, n, chunk_reads):
        b = min(n, a + chunk_reads)
        lens = recipe.lengths(a, b)
        yield a, b, lens, recipe.reads_ascii(a, b, lens)


def offsets_of(recipe: ReadRecipe, step: int = 1 << 26) -> torch.Tensor:
    """read_offsets (int64[n_reads + 1]) of the recipe on its device."""
    n = recipe.n_reads
    off = torch.zeros(n + 1, dtype=torch.int64, device=recipe.device)
    run = 0
    for a in range(0, n, step):
        b = min(n, a + step)
        torch.cumsum(recipe.lengths(a, b), 0, out=off[a + 1:b + 1])
        off[a + 1:b + 1] += run
        run = int(off[b])
    return off
