"""Full-size parity of configs[2] (1.01e9 suffixes, one in-HBM batch), configs[3] (6.04e9 suffixes, several in-HBM batches,
64-bit ids) and configs[4] (1.01e11 suffixes, out-of-core: batches streamed to pinned host memory), in the launch
configuration bench.py times.  Inputs are generated chunk by chunk on the device (workloads/generate_torch.py, pinned to
the numpy recipes by tests/test_generators.py); nothing here comes from the CUDA path except the output under test.

A full plain oracle pass over these is 1-100 core-hours, so parity is checked on
  * oracle slices (bit-exact): for a seeded set of base strings P of equal length, every suffix that begins with P is
    LISTED by a brute-force scan of the generated reads (torch ops), the number of suffixes below P is counted the same
    way, the owning reads are handed to oracle.bwt_of_listed (the definition's comparator on the listed suffixes) and the
    output slice must match byte for byte (a prefix range is a contiguous piece of B_R);
  * whole-output properties, every position of the output looked at:
      - symbol counts, and the first-n rule (the n end-marker suffixes sort first, by read index: PAPER.md:55);
      - P6, partition by partition: the multiset of preceding symbols inside every l-prefix partition (l = 5; partitions
        are contiguous and ordered in B_R) equals what a linear scan of the reads counts for it;
      - LF-mapping inversion of a seeded sample of reads over the whole output (a rank table over blocks of 16 Ki symbols).
Gated on the box, not on an environment variable: a GPU with less free memory than the configuration needs (or a host
with less RAM than the pinned output of configs[4]) skips; a B200 with 180 GB runs all of them.
The sampled fraction per configuration is recorded in DESIGN.md section 12 and gpurun_out/large_config*.json.
"""
import concurrent.futures as cf
import gc
import json
import os
import time

import numpy as np
import pytest
import torch

import oracle
from workloads import generate as gen
from workloads import generate_torch as gt

pytestmark = pytest.mark.gpu

ELL = 5                       # partition prefix of the P6 check (test side; independent of the library's own l)
SYM_OF_BYTE = np.full(256, 7, dtype=np.int64)
for _i, _c in enumerate(b"$ACGT"):
    SYM_OF_BYTE[_c] = _i
RANK_BLOCK = 1 << 14


def _host_ram_gb() -> float:
    with open("/proc/meminfo") as f:
        for ln in f:
            if ln.startswith("MemAvailable:"):
                return int(ln.split()[1]) / (1 << 20)
    return 0.0


def _need(gpu_gb: float, host_gb: float):
    gc.collect()
    torch.cuda.empty_cache()                 # what earlier tests left in torch's cache is free memory too
    free = torch.cuda.mem_get_info(0)[0] / (1 << 30)
    if free < gpu_gb or _host_ram_gb() < host_gb:
        pytest.skip(f"needs {gpu_gb} GB of free GPU memory and {host_gb} GB of host RAM (have {free:.0f} GB, {_host_ram_gb():.0f} GB)")


def _code(text: str) -> int:
    c = 0
    for ch in text.encode():
        c = c * 4 + {65: 0, 67: 1, 71: 2, 84: 3}[ch]
    return c


class ProbeSet:
    """Brute-force listing of the suffixes that begin with each of several base strings of ONE length k, and the number of
    suffixes below each: one window code per base position, one binary search of it among the sorted probe codes."""

    def __init__(self, texts, device):
        assert len(set(len(t) for t in texts)) == 1 and len(set(texts)) == len(texts)
        self.k = len(texts[0])
        order = np.argsort([_code(t) for t in texts])
        self.texts = [texts[i] for i in order]
        self.codes = torch.tensor([_code(t) for t in self.texts], dtype=torch.int64, device=device)
        self.P = len(texts)
        self.below = torch.zeros(self.P, dtype=torch.int64, device=device)
        self.found = [[] for _ in range(self.P)]

    def scan(self, codes, rid, pos, rem, first_read, n_reads_chunk):
        """codes/rid/pos/rem: per base position of the chunk (code 0..3, read index inside the chunk, position in the
        read, bases left from here to the end of the read)."""
        k, P = self.k, self.P
        tot = codes.numel()
        win = torch.zeros(tot, dtype=torch.int64, device=codes.device)
        c64 = codes.to(torch.int64)
        for t in range(min(k, tot)):      # code of the k symbols starting at every position, zero-padded past the chunk
            win[: tot - t] += c64[t:] << (2 * (k - 1 - t))
        del c64
        full = rem >= k
        wf = win[full]
        # suffixes with >= k bases: below P iff their first k bases are; begin with P iff equal
        i = torch.bucketize(wf, self.codes, right=True)                     # probe codes <= mine
        self.below += torch.cumsum(torch.bincount(i, minlength=P + 1), 0)[:P]   # mine < code_p  <=>  i <= p
        hit = (i > 0) & (self.codes[(i - 1).clamp(min=0)] == wf)
        if bool(hit.any()):
            which = (i - 1)[hit]
            rp = torch.stack([rid[full][hit] + first_read, pos[full][hit]], 1)
            for p in torch.unique(which).tolist():
                self.found[p].append(rp[which == p].cpu())
        del wf, i, hit
        # a suffix with r < k bases left is below P iff its r bases are <= the first r symbols of P ($ is the smallest symbol)
        for r in range(1, k):
            sel = rem == r
            if not bool(sel.any()):
                continue
            v = win[sel] >> (2 * (k - r))
            tops = self.codes >> (2 * (k - r))                              # non-decreasing
            j = torch.bucketize(v, tops, right=False)                       # tops < mine;  mine <= tops[p]  <=>  j <= p
            self.below += torch.cumsum(torch.bincount(j, minlength=P + 1), 0)[:P]
        self.below += n_reads_chunk                                          # the bare end-marker suffix of every read

    def listed(self, p) -> np.ndarray:
        if not self.found[p]:
            return np.zeros((0, 2), dtype=np.int64)
        lst = torch.cat(self.found[p]).numpy()
        return lst[np.lexsort((lst[:, 1], lst[:, 0]))]


def generate_on_device(recipe: gt.ReadRecipe, probes: ProbeSet, chunk_reads: int):
    """Packed reads + offsets on the device, produced chunk by chunk; the probes and the whole-output references (symbol
    counts, last base of every read, preceding-symbol counts per l-prefix partition) are accumulated from the same chunks."""
    import paper_1401_7457_b200 as cx
    dev = recipe.device
    n = recipe.n_reads
    offsets = gt.offsets_of(recipe)
    total = int(offsets[-1])
    max_len = int((offsets[1:] - offsets[:-1]).max())
    packed = torch.zeros((total + 31) // 32 + 1, dtype=torch.int64, device=dev)
    last_base = torch.full((n,), ord("$"), dtype=torch.uint8, device=dev)
    counts = torch.zeros(256, dtype=torch.int64, device=dev)
    n_part = 4 ** ELL * (ELL + 1)
    part_syms = torch.zeros(n_part * 8, dtype=torch.int64, device=dev)    # [partition][symbol $ACGT] of the preceding symbols
    sym_lut = torch.from_numpy(SYM_OF_BYTE).to(dev)
    carry = torch.zeros(0, dtype=torch.uint8, device=dev)
    done = 0                                   # bases already packed (a multiple of 32)
    for a, b, lens, ascii_ in gt.read_chunks(recipe, chunk_reads):
        tot = ascii_.numel()
        counts += torch.bincount(ascii_.to(torch.int64), minlength=256)
        off = offsets[a:b + 1] - offsets[a]
        nz = lens > 0
        last_base[a:b][nz] = ascii_[(off[1:] - 1)[nz]]
        # the end-marker suffix of every read: partition 0 (no bases), preceded by the read's last base ('$' if empty)
        part_syms += torch.bincount(sym_lut[last_base[a:b].to(torch.int64)], minlength=n_part * 8)
        if tot:
            rid = torch.repeat_interleave(torch.arange(b - a, dtype=torch.int64, device=dev), lens, output_size=tot)
            pos = torch.arange(tot, dtype=torch.int64, device=dev) - off[rid]
            rem = lens[rid] - pos
            codes = ((ascii_ >> 1) ^ (ascii_ >> 2)) & 3          # A,C,G,T -> 0,1,2,3 (ASCII trick, test side)
            probes.scan(codes, rid, pos, rem, a, b - a)
            # partition of every suffix: (its first min(rem, l) bases, A-padded) * (l + 1) + min(rem, l); preceding symbol
            c64 = codes.to(torch.int64)
            kmer = torch.zeros(tot, dtype=torch.int64, device=dev)
            for t in range(ELL):
                inside = rem > t
                kmer[: tot - t] += torch.where(inside[: tot - t], c64[t:], torch.zeros_like(c64[t:])) << (2 * (ELL - 1 - t))
            part = kmer * (ELL + 1) + torch.clamp(rem, max=ELL)
            prev = torch.zeros(tot, dtype=torch.int64, device=dev)          # 0 = '$' (the suffix starts its read)
            prev[1:] = torch.where(pos[1:] > 0, c64[:-1] + 1, prev[1:])
            part_syms += torch.bincount(part * 8 + prev, minlength=n_part * 8)
            del rid, pos, rem, codes, c64, kmer, part, prev
        buf = torch.cat([carry, ascii_]) if carry.numel() else ascii_
        whole = buf.numel() // 32 * 32 if b < n else buf.numel()
        if whole:
            cx.cx_pack_reads(buf[:whole].contiguous(), packed[done // 32: done // 32 + (whole + 31) // 32])
        carry = buf[whole:].clone()
        done += whole
        del ascii_, buf
    assert done == total
    return packed, offsets, total, max_len, counts, last_base, part_syms.view(n_part, 8)


def check_slices(recipe, probes: ProbeSet, out, n_suffixes):
    """out: the BWT (device or pinned host uint8 tensor).  Every probe's slice must equal the oracle on the listed suffixes."""
    below = probes.below.cpu().numpy()
    jobs = []
    for p in range(probes.P):
        lst = probes.listed(p)
        assert lst.shape[0] > 0, f"probe {probes.texts[p]} matched nothing; pick a shorter string"
        owners = np.unique(lst[:, 0])
        idx = torch.from_numpy(owners).to(recipe.device)
        lens = recipe.lengths_of(idx)
        sub_text = recipe.reads_ascii_of(idx, lens).cpu().numpy()           # the owning reads, regenerated from the recipe
        sub_off = np.zeros(owners.size + 1, dtype=np.uint64)
        sub_off[1:] = np.cumsum(lens.cpu().numpy())
        remap = lst.copy()
        remap[:, 0] = np.searchsorted(owners, lst[:, 0])
        jobs.append((p, sub_text, sub_off, remap.astype(np.uint64)))
    oracle.build()
    with cf.ThreadPoolExecutor(max_workers=os.cpu_count() or 1) as pool:   # the C oracle runs outside the GIL
        wants = list(pool.map(lambda j: oracle.bwt_of_listed(j[1], j[2], j[3])[0], jobs))
    report = []
    for (p, _, _, _), want in zip(jobs, wants):
        at = int(below[p])
        assert at + want.size <= n_suffixes
        got = out[at: at + want.size].cpu().numpy()
        assert np.array_equal(got, want), f"slice of prefix {probes.texts[p]} differs from the oracle ({want.size} suffixes at {at})"
        report.append({"prefix": probes.texts[p], "offset": at, "suffixes": int(want.size)})
    return report


def whole_output_checks(out, N, n, counts, last_base, part_syms, dev):
    """One streaming pass over the whole output: symbol counts, P6 (preceding-symbol multiset of every partition) and the
    rank table (symbol counts per block of RANK_BLOCK positions) that LF inversion needs."""
    sym_lut = torch.from_numpy(SYM_OF_BYTE).to(dev)
    want_counts = counts.clone()
    want_counts[ord("$")] += n
    bounds = torch.cumsum(part_syms.sum(1), 0)                               # one past the last position of every partition
    assert int(bounds[-1]) == N
    n_part = part_syms.shape[0]
    got_part = torch.zeros(n_part * 8, dtype=torch.int64, device=dev)
    got_counts = torch.zeros(256, dtype=torch.int64, device=dev)
    n_blocks = (N + RANK_BLOCK - 1) // RANK_BLOCK
    block_syms = torch.zeros(n_blocks * 8, dtype=torch.int64, device=dev)
    step = 1 << 28
    for a in range(0, N, step):
        b = min(N, a + step)
        chunk = out[a:b].to(dev, non_blocking=True).to(torch.int64)
        got_counts += torch.bincount(chunk, minlength=256)
        sym = sym_lut[chunk]
        at = torch.arange(a, b, dtype=torch.int64, device=dev)
        got_part += torch.bincount(torch.bucketize(at, bounds, right=True) * 8 + sym, minlength=n_part * 8)
        block_syms += torch.bincount((at // RANK_BLOCK) * 8 + sym, minlength=n_blocks * 8)
        del chunk, sym, at
    assert torch.equal(got_counts, want_counts), "symbol counts of the output differ from the input's"
    assert torch.equal(out[:n].to(dev), last_base), "the first n symbols are not the last bases of the reads in read order"
    bad = (got_part.view(n_part, 8) != part_syms).any(1)
    assert not bool(bad.any()), f"preceding-symbol counts differ in {int(bad.sum())} of {n_part} l-prefix partitions (first: {int(bad.nonzero()[0])})"
    return block_syms.view(n_blocks, 8)[:, :5].cpu().numpy(), got_counts.cpu().numpy()


def lf_inversion(out, block_syms, sym_counts, recipe, read_ids):
    """Reconstruct the sampled reads from the output alone: start at row i (the $_i suffix), emit B[k],
    k = C[B[k]] + occ(B[k], k), until '$'; the emitted symbols reversed are read i."""
    out_np = out.numpy() if out.device.type == "cpu" else out.cpu().numpy()
    prefix = np.zeros((block_syms.shape[0] + 1, 5), dtype=np.int64)
    np.cumsum(block_syms, 0, out=prefix[1:])
    C = np.zeros(5, dtype=np.int64)
    C[1:] = np.cumsum([sym_counts[c] for c in b"$ACG"])
    idx = torch.from_numpy(np.asarray(read_ids, dtype=np.int64)).to(recipe.device)
    lens = recipe.lengths_of(idx).cpu().numpy()
    text = recipe.reads_ascii_of(idx).cpu().numpy()
    ends = np.cumsum(lens)
    for j, i in enumerate(read_ids):
        want = text[ends[j] - lens[j]: ends[j]].tobytes()
        got = bytearray()
        k = int(i)
        for _ in range(int(lens[j]) + 1):
            byte = int(out_np[k])
            if byte == ord("$"):
                break
            c = int(SYM_OF_BYTE[byte])
            blk = k // RANK_BLOCK
            occ = int(prefix[blk, c]) + int(np.count_nonzero(out_np[blk * RANK_BLOCK: k] == byte))
            got.append(byte)
            k = int(C[c]) + occ
        else:
            raise AssertionError(f"LF walk of read {i} did not reach '$' within its length")
        assert bytes(reversed(got)) == want, f"LF inversion of read {i} gave {bytes(reversed(got))!r}, want {want!r}"


def run_config(index, probe_texts, chunk_reads, workspace_bytes, host_out, lf_reads, scale=1.0):
    import paper_1401_7457_b200 as cx
    dev = torch.device("cuda", 0)
    gc.collect()
    torch.cuda.empty_cache()                 # a previous config's workspace must not stay cached
    t0 = time.time()
    recipe = gt.ReadRecipe(index, scale, device=dev)
    probes = ProbeSet(probe_texts, dev)
    packed, offsets, total, max_len, counts, last_base, part_syms = generate_on_device(recipe, probes, chunk_reads)
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
    del plan, packed
    torch.cuda.empty_cache()
    t2 = time.time()
    block_syms, sym_counts = whole_output_checks(out, N, n, counts, last_base, part_syms, dev)
    slices = check_slices(recipe, probes, out, N)
    rng = np.random.default_rng(7 + index)
    sample = np.sort(rng.choice(n, min(lf_reads, n), replace=False))
    lf_inversion(out, block_syms, sym_counts, recipe, sample)
    t_check = time.time() - t2
    sliced = sum(s["suffixes"] for s in slices)
    res = {"config": index, "scale": scale, "n_reads": n, "total_bases": total, "n_suffixes": N, "generate_s": round(t_gen, 1),
           "build_s": round(t_build, 3), "check_s": round(t_check, 1), "suffixes_per_s": N / t_build, "gbases_per_hour": total / t_build * 3600 / 1e9,
           "stats": stats, "kernel_ms": kernel_ms, "host_out": host_out,
           "checked": {"oracle_slices": len(slices), "oracle_slice_suffixes": sliced, "oracle_slice_fraction": sliced / N,
                       "whole_output": ["symbol counts", "first-n rule", f"P6 preceding-symbol multisets of all {part_syms.shape[0]} partitions (l = {ELL})"],
                       "lf_inverted_reads": int(sample.size)},
           "slices": slices}
    os.makedirs("gpurun_out", exist_ok=True)
    with open(f"gpurun_out/large_config{index}{'' if scale == 1.0 else '_scaled'}.json", "w") as f:
        json.dump(res, f)
    print(json.dumps({k: v for k, v in res.items() if k != "slices"}))
    del out, offsets, counts, last_base, part_syms, recipe, probes
    gc.collect()
    torch.cuda.empty_cache()
    return res


def _seeded_probes(seed: int, count: int, k: int, extra=()):
    """`count` distinct base strings of length k spread over the k-mer space (one per equal slice of it, seeded offset inside
    the slice), plus the given ones."""
    rng = np.random.default_rng(seed)
    space = 4 ** k
    codes = {int(s * space // count + rng.integers(0, max(1, space // count))) for s in range(count)}
    texts = {"".join("ACGT"[(c >> (2 * (k - 1 - t))) & 3] for t in range(k)) for c in codes}
    texts.update(extra)
    return sorted(texts)


def test_small_scale_of_the_large_path():
    # the same code path at a size the plain checks finish in seconds (ragged reads, several batches, host output)
    r = run_config(3, ["ACGTA", "TTGAC", "GGGGG", "CATCA"], chunk_reads=7001, workspace_bytes=40 << 20, host_out=True, lf_reads=300, scale=0.0005)
    assert r["stats"]["n_batches"] > 1
    r = run_config(2, _seeded_probes(1, 6, 4), chunk_reads=5003, workspace_bytes=None, host_out=False, lf_reads=200, scale=0.001)
    assert r["stats"]["n_batches"] == 1


def test_config3_full_size():
    # configs[2], 1.01e9 suffixes in one in-HBM batch: the bench workload
    _need(70, 24)
    r = run_config(2, _seeded_probes(2, 16, 5), chunk_reads=2_000_000, workspace_bytes=None, host_out=False, lf_reads=2000)
    assert r["n_suffixes"] == 1_010_000_000 and r["stats"]["n_batches"] == 1
    assert r["checked"]["oracle_slices"] >= 16 and r["checked"]["oracle_slice_suffixes"] >= 10_000_000


def test_config4_full_size():
    _need(150, 32)
    seed = gen.BASE_SEED + 3
    # prefixes inside repeat elements (their tie groups are the deep ones): 8 bases out of elements 0, 7 and 19 of the recipe
    inside = ["".join("ACGT"[c] for c in gen._iid_codes(seed, 7, e * 8192, 60)[20:28]) for e in (0, 7, 19)]
    r = run_config(3, _seeded_probes(3, 32, 8, extra=inside), chunk_reads=2_000_000, workspace_bytes=130 << 30, host_out=False, lf_reads=1000)
    assert r["n_suffixes"] > 6_000_000_000 and r["stats"]["id_bytes"] == 8 and r["stats"]["n_batches"] >= 2
    assert r["checked"]["oracle_slices"] >= 32


def test_config5_full_size_out_of_core():
    _need(170, 125)
    r = run_config(4, _seeded_probes(4, 64, 9), chunk_reads=2_500_000, workspace_bytes=136 << 30, host_out=True, lf_reads=1000)
    assert r["n_suffixes"] == 101_000_000_000 and r["stats"]["n_batches"] >= 10
    assert r["checked"]["oracle_slices"] >= 64 and r["checked"]["oracle_slice_suffixes"] >= 10_000_000
