"""Full-size runs of configs[3] (6.04e9 suffixes, several in-HBM batches, 64-bit ids) and configs[4] (1.01e11
suffixes, out-of-core: batches streamed to pinned host memory), generated chunk by chunk on the device.

A full plain oracle pass over these is 5-100 core-hours, so parity is checked on
  * oracle slices: for sampled base strings P, every suffix that begins with P is LISTED by a brute-force scan
    of the generated reads (torch ops, independent of the CUDA path), the number of suffixes below P is counted
    the same way, the owning reads are handed to oracle.bwt_of_listed, and the output slice must match byte
    for byte (a prefix range is a contiguous piece of B_R);
  * whole-output properties: symbol counts, and the first-n rule (the n end-marker suffixes sort first, by read
    index: PAPER.md:55).
Opt-in: CX_TEST_LARGE=1 (minutes of GPU time, tens of GB of host RAM).  Results of the last run: DESIGN.md section 12.
"""
import json
import os
import time

import numpy as np
import pytest
import torch

import oracle
from workloads import generate_torch as gt

pytestmark = [pytest.mark.gpu,
              pytest.mark.skipif(os.environ.get("CX_TEST_LARGE", "0") != "1", reason="set CX_TEST_LARGE=1")]

CODE = {ord("A"): 0, ord("C"): 1, ord("G"): 2, ord("T"): 3}


class PrefixProbe:
    """Brute-force listing of the suffixes that begin with the base string P, and the count of suffixes below P."""

    def __init__(self, text: str):
        self.text = text
        self.k = len(text)
        self.code = 0
        for ch in text.encode():
            self.code = self.code * 4 + CODE[ch]
        self.below = 0
        self.found = []       # (read, pos) tensors

    def scan(self, codes: torch.Tensor, rid: torch.Tensor, pos: torch.Tensor, rem: torch.Tensor, first_read: int, n_reads_chunk: int):
        """codes/rid/pos/rem: per base position of the chunk (code 0..3, read index inside the chunk, position in
        the read, bases left from here to the end of the read)."""
        k = self.k
        tot = codes.numel()
        win = torch.zeros(tot, dtype=torch.int64, device=codes.device)
        c64 = codes.to(torch.int64)
        for t in range(k):          # window code of the k symbols starting at every position, zero-padded past the chunk
            if t < tot:
                win[: tot - t] += c64[t:] << (2 * (k - 1 - t))
        full = rem >= k
        hit = full & (win == self.code)
        self.below += int((full & (win < self.code)).sum())
        # a suffix with r < k bases left is below P iff its r bases are <= the first r symbols of P ($ is the smallest symbol)
        short = ~full
        r = rem[short]
        self.below += int(((win[short] >> (2 * (k - r))) <= (torch.full_like(r, self.code) >> (2 * (k - r)))).sum())
        self.below += n_reads_chunk                       # the bare end-marker suffix of every read
        if bool(hit.any()):
            self.found.append(torch.stack([rid[hit] + first_read, pos[hit]], 1).cpu())

    def listed(self) -> np.ndarray:
        if not self.found:
            return np.zeros((0, 2), dtype=np.int64)
        lst = torch.cat(self.found).numpy()
        return lst[np.lexsort((lst[:, 1], lst[:, 0]))]


def generate_on_device(recipe: gt.ReadRecipe, probes, chunk_reads: int):
    """Packed reads + offsets on the device, produced chunk by chunk; the probes and the whole-output references
    (symbol counts, last base of every read) are accumulated from the same chunks."""
    import paper_1401_7457_b200 as cx
    dev = recipe.device
    n = recipe.n_reads
    lens_all = torch.empty(n, dtype=torch.int64, device=dev)
    for a in range(0, n, 1 << 26):
        b = min(n, a + (1 << 26))
        lens_all[a:b] = recipe.lengths(a, b)
    offsets = torch.zeros(n + 1, dtype=torch.int64, device=dev)
    torch.cumsum(lens_all, 0, out=offsets[1:])
    total = int(offsets[-1])
    packed = torch.zeros((total + 31) // 32 + 1, dtype=torch.int64, device=dev)
    last_base = torch.full((n,), ord("$"), dtype=torch.uint8, device=dev)
    counts = torch.zeros(256, dtype=torch.int64, device=dev)
    carry = torch.zeros(0, dtype=torch.uint8, device=dev)
    done_bases = 0                                   # bases already packed (a multiple of 32)
    for a in range(0, n, chunk_reads):
        b = min(n, a + chunk_reads)
        lens = lens_all[a:b]
        ascii_ = recipe.reads_ascii(a, b, lens)
        tot = ascii_.numel()
        counts += torch.bincount(ascii_.to(torch.int64), minlength=256)
        off = offsets[a:b + 1] - offsets[a]
        nz = lens > 0
        last_base[a:b][nz] = ascii_[(off[1:] - 1)[nz]]
        if probes and tot:
            rid = torch.repeat_interleave(torch.arange(b - a, dtype=torch.int64, device=dev), lens, output_size=tot)
            pos = torch.arange(tot, dtype=torch.int64, device=dev) - off[rid]
            rem = lens[rid] - pos
            codes = ((ascii_ >> 1) ^ (ascii_ >> 2)) & 3          # A,C,G,T -> 0,1,2,3 (ASCII trick, test side)
            for p in probes:
                p.scan(codes, rid, pos, rem, a, b - a)
            del rid, pos, rem, codes
        elif probes:
            for p in probes:
                p.below += b - a
        buf = torch.cat([carry, ascii_]) if carry.numel() else ascii_
        whole = buf.numel() // 32 * 32 if b < n else buf.numel()
        if whole:
            cx.cx_pack_reads(buf[:whole].contiguous(), packed[done_bases // 32: done_bases // 32 + (whole + 31) // 32])
        carry = buf[whole:].clone()
        done_bases += whole
        del ascii_, buf
    assert done_bases == total
    return packed, offsets, total, int(lens_all.max()), counts, last_base


def check_slices(recipe, probes, out, n_suffixes):
    """out: the BWT (device or host uint8 tensor).  Each probe's slice must equal the oracle on the listed suffixes."""
    report = []
    cpu = gt.ReadRecipe.__new__(gt.ReadRecipe)
    cpu.__dict__.update(recipe.__dict__)
    cpu.device = torch.device("cpu")
    cpu.genome = recipe.genome.cpu()
    for p in probes:
        lst = p.listed()
        assert lst.shape[0] > 0, f"probe {p.text} matched nothing; pick a shorter string"
        owners = np.unique(lst[:, 0])
        idx = torch.from_numpy(owners)
        lens = cpu.lengths_of(idx)
        sub_text = cpu.reads_ascii_of(idx, lens).numpy()
        sub_off = np.zeros(owners.size + 1, dtype=np.uint64)
        sub_off[1:] = np.cumsum(lens.numpy())
        remap = lst.copy()
        remap[:, 0] = np.searchsorted(owners, lst[:, 0])
        want, _ = oracle.bwt_of_listed(sub_text, sub_off, remap.astype(np.uint64))
        assert p.below + want.size <= n_suffixes
        got = out[p.below: p.below + want.size].cpu().numpy()
        assert np.array_equal(got, want), f"slice of prefix {p.text} differs from the oracle ({want.size} suffixes at {p.below})"
        report.append({"prefix": p.text, "offset": p.below, "suffixes": int(want.size)})
    return report


def run_config(index, probes_text, chunk_reads, workspace_bytes, host_out, scale=1.0):
    import paper_1401_7457_b200 as cx
    import gc
    dev = torch.device("cuda", 0)
    gc.collect()
    torch.cuda.empty_cache()                 # a previous config's workspace must not stay cached
    t0 = time.time()
    recipe = gt.ReadRecipe(index, scale, device=dev)
    probes = [PrefixProbe(t) for t in probes_text]
    packed, offsets, total, max_len, counts, last_base = generate_on_device(recipe, probes, chunk_reads)
    n = recipe.n_reads
    N = total + n
    torch.cuda.synchronize()
    t_gen = time.time() - t0
    torch.cuda.empty_cache()
    opts = dict(max_read_len=max_len, out_is_host_pinned=1 if host_out else 0, profile=1)
    plan = cx.Plan(n, total, workspace_bytes=workspace_bytes, **opts)
    out = torch.empty(N, dtype=torch.uint8, pin_memory=True) if host_out else torch.empty(N, dtype=torch.uint8, device=dev)
    torch.cuda.synchronize()
    t1 = time.time()
    plan.build(packed, offsets, n, out)
    torch.cuda.synchronize()
    t_build = time.time() - t1
    stats = plan.stats()
    kernel_ms = {k: round(v["ms"], 2) for k, v in plan.kernel_times().items() if v["launches"]}
    plan.free()
    del plan
    # whole-output properties
    got = torch.zeros(256, dtype=torch.int64, device=dev)
    for a in range(0, N, 1 << 30):
        got += torch.bincount(out[a:a + (1 << 30)].to(dev).to(torch.int64), minlength=256)
    counts[ord("$")] += n
    assert torch.equal(got, counts), "symbol counts of the output differ from the input's"
    assert torch.equal(out[:n].to(dev), last_base), "the first n symbols are not the last bases of the reads in read order"
    slices = check_slices(recipe, probes, out, N)
    res = {"config": index, "scale": scale, "n_reads": n, "total_bases": total, "n_suffixes": N, "generate_s": round(t_gen, 1),
           "build_s": round(t_build, 3), "suffixes_per_s": N / t_build, "gbases_per_hour": total / t_build * 3600 / 1e9,
           "stats": stats, "kernel_ms": kernel_ms, "slices": slices, "host_out": host_out}
    os.makedirs("gpurun_out", exist_ok=True)
    with open(f"gpurun_out/large_config{index}.json", "w") as f:
        json.dump(res, f)
    print(json.dumps(res))
    del out, packed, offsets, counts, last_base, got, recipe, probes
    gc.collect()
    torch.cuda.empty_cache()
    return res


def test_small_scale_of_the_large_path():
    # the same code path at a size the plain checks finish in seconds (ragged reads, several batches, host output)
    r = run_config(3, ["ACGTA", "TTG"], chunk_reads=7001, workspace_bytes=40 << 20, host_out=True, scale=0.0005)
    assert r["stats"]["n_batches"] > 1


def test_config4_full_size():
    r = run_config(3, ["ACGTACGTACG", "TTGACCATGC", "GGGGGGGG"], chunk_reads=2_000_000, workspace_bytes=130 << 30, host_out=False)
    assert r["n_suffixes"] > 6_000_000_000 and r["stats"]["id_bytes"] == 8 and r["stats"]["n_batches"] >= 2


def test_config5_full_size_out_of_core():
    r = run_config(4, ["ACGTACGTACGT", "TTGACCATGCA", "CCCCCCCCCC"], chunk_reads=2_500_000, workspace_bytes=110 << 30, host_out=True)
    assert r["n_suffixes"] == 101_000_000_000 and r["stats"]["n_batches"] >= 20
