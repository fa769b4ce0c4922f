#!/usr/bin/env python
"""bench.py -- one JSON line for BASELINE.json's metric: suffixes sorted/s (and Gbases/hour) of the
collection-BWT hot path on B200, with the dominant kernel's HBM roofline and the CPU oracle beside it.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config i] [--impl cx|reference]

A "step" is one pass of the whole hot path (rows a1-a8 of DESIGN.md: 2-bit pack, partition sizes,
batch plan, list + key build, onesweep sort, tie refinement, emit) over one synthetic collection.
At N=1 the workload is BASELINE.json configs[2] (10,000,000 reads x 100 bp, 30x over a seeded 33 Mbp
genome, both strands, 1 % substitutions -> 1.01e9 suffixes): the largest configuration that is sorted
as ONE in-HBM batch and whose host-resident end-to-end leg (1 GB in, 1 GB out) fits any box.  The two
larger configurations (configs[3]: 6.04e9 suffixes in two batches; configs[4]: 1.01e11 suffixes, the
paper's 1000M x 100 bp headline, streamed out of core) are measured in the same run as one-step records
under "other_configs" when the box has the memory for them (skip with --no-other-configs).
For N>1 (torchrun, one rank per GPU) every rank runs an independent replica with its own seed: the
north_star fixes the path to one GPU with no collectives.

`--impl reference` times the CPU oracle (oracle/, as it stands, one prefix range per process over all
host cores) on a bounded sample of the same recipe; nothing else in this file touches oracle/ except
the `cpu_baseline` leg.
"""
from __future__ import annotations

import argparse
import itertools
import json
import os
import statistics
import sys
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "suffixes_sorted_per_s"
UNIT = "suffixes/s"
DEFAULT_CONFIG = 2
WORKLOADS = {
    0: "configs[0]: 10,000 reads x 100 bp iid (1.01e6 suffixes)",
    1: "configs[1]: 1,000,000 reads x 100 bp at 100x over a seeded 1 Mbp genome (1.01e8 suffixes)",
    2: "configs[2]: 10,000,000 reads x 100 bp at 30x over 33 Mbp, both strands, 1% subst. (1.01e9 suffixes)",
    3: "configs[3]: 40,000,000 reads x 50-250 bp over a 50 Mbp repeat genome (~6.04e9 suffixes)",
    4: "configs[4]: 1,000,000,000 reads x 100 bp at 30x over 3.3 Gbp, both strands, 1% subst. (1.01e11 suffixes)",
}
# dram__bytes_read.sum + dram__bytes_write.sum per launch, from the committed `ncu --set full` captures of THIS round at the
# benched configuration (profiles/r02_ncu_full.md); keyed by (config, kernel class).  None until a capture exists.
NCU_TRAFFIC: dict = {(2, "finish"): 105_640_423_000, (2, "sort_pass"): 16_442_371_750, (2, "list"): 9_418_393_000, (2, "pack"): 1_195_345_000,
                     (2, "finish_block"): 316_000}
NCU_TRAFFIC_FILE = "profiles/r02_ncu_full.md"
FALLBACK_HBM_GBS = 6650.0     # /opt/skills/guides/B200_PROFILING.md, used only if MEASURED_PEAKS.json is absent
CPU_SAMPLE_SCALE = {0: 1.0, 1: 0.5, 2: 0.1, 3: 0.01, 4: 0.001}      # cpu_baseline: the recipe at this scale (coverage preserved), all cores
REF_SAMPLE_SCALE = {0: 1.0, 1: 0.25, 2: 0.04, 3: 0.004, 4: 0.0004}  # --impl reference: one step = the oracle on the recipe at this scale
KERNEL_NAMES = {"pack": "pack_kernel (a1)", "prep": "prep_kernel + tile_table_kernel", "hist": "bucket_hist_kernel (a2)",
                "list": "list_write_reads_kernel / list_write_kernel, or list_count + list_select per batch (a4+a5)", "sort_hist": "digit_hist_kernel (a6)",
                "sort_scan": "bin_scan_kernel (a6)", "sort_pass": "onesweep_pass_kernel (a6, one radix pass of the first sort)",
                "finish": "finish_warp_kernel (a7+a8: head flags, tie groups of <= 64 refined in registers, leftovers in dense queued windows, emit)",
                "finish_block": "finish_tile_kernel (a7+a8: tie groups of 65..256 refined in shared memory)",
                "refine_scan": "active_count + scan (a7, global path)",
                "refine_key": "refine_rekey_kernel (a7, global path)", "refine_write": "refine_writeback_kernel (a7+a8, global path)",
                "refine_sort": "onesweep_pass_kernel (a7, global path re-sort)", "fasta": "fasta_* kernels (NEXT-4 ingest)"}


def parse_args():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--config", type=int, default=DEFAULT_CONFIG, help="BASELINE.json configs index (0-based)")
    ap.add_argument("--scale", type=float, default=1.0, help="debug only: scale the workload down")
    ap.add_argument("--impl", default="cx", choices=["cx", "reference"])
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-other-configs", action="store_true", help="skip the one-step records of configs[3] and configs[4]")
    ap.add_argument("--all-configs", action="store_true", help="also add one-step records of configs[0] and configs[1] to other_configs")
    ap.add_argument("--key-bases", type=int, default=0, help="first-round key window w (0 = the library's default)")
    ap.add_argument("--shard", action="store_true", help="NEXT-2, with --gpus N > 1 under torchrun: ONE collection, rank k sorts the k-th of N contiguous "
                    "partition ranges (PAPER.md:103) and the pieces are exchanged (all-gather); strong scaling.  Default: independent replicas")
    ap.add_argument("--fasta", action="store_true", help="NEXT-4: the step starts from the collection's FASTA text (resident in HBM; pinned host for e2e): "
                    "cx_fasta_parse + pack + build")
    ap.add_argument("--shard-of", type=int, default=0, help="one GPU: time ONE shard of a W-way partition-range split (no exchange); with --shard-index")
    ap.add_argument("--shard-index", type=int, default=0)
    ap.add_argument("--table4", type=int, default=0, help="NEXT-3: the paper's read-length experiment instead of a config: read length 100/200/400, "
                    "1e10 x --scale bases (PAPER.md:184-189)")
    ap.add_argument("--max-batch", type=int, default=0, help="m1: most suffixes per batch (0 = as many as the workspace allows)")
    ap.add_argument("--out-bits", type=int, default=8, choices=[8, 4], help="NEXT-4: 4 = packed output, two symbols per byte")
    return ap.parse_args()


def hbm_peak():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    try:
        with open(path) as f:
            return float(json.load(f)["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs, torch copy read+write)"
    except Exception:
        return FALLBACK_HBM_GBS, "fallback (B200_PROFILING.md)"


class ClockSampler:
    """SM clock and throttle reasons sampled on a thread (NVML, every ~5 ms) while the timed region runs --
    the same fields as the profiling recipe's nvidia-smi clocks line, at a rate a 100 ms region can see."""

    def __init__(self, gpu_index: int):
        self.gpu = gpu_index
        self.sm, self.reasons, self.max_mhz, self.power = [], set(), None, []
        self._stop = False
        self._thread = None
        self._err = None

    def _run(self):
        try:
            import pynvml as nv
            nv.nvmlInit()
            # NVML indexes physical devices; honour CUDA_VISIBLE_DEVICES when it is a plain index list
            vis = os.environ.get("CUDA_VISIBLE_DEVICES", "")
            idx = self.gpu
            if vis and all(p.strip().isdigit() for p in vis.split(",")):
                idx = int(vis.split(",")[self.gpu])
            h = nv.nvmlDeviceGetHandleByIndex(idx)
            self.max_mhz = float(nv.nvmlDeviceGetMaxClockInfo(h, nv.NVML_CLOCK_SM))
            bits = {"hw_slowdown": nv.nvmlClocksThrottleReasonHwSlowdown,
                    "hw_thermal_slowdown": nv.nvmlClocksThrottleReasonHwThermalSlowdown,
                    "sw_thermal_slowdown": nv.nvmlClocksThrottleReasonSwThermalSlowdown,
                    "sw_power_cap": nv.nvmlClocksThrottleReasonSwPowerCap}
            while not self._stop:
                self.sm.append(float(nv.nvmlDeviceGetClockInfo(h, nv.NVML_CLOCK_SM)))
                r = nv.nvmlDeviceGetCurrentClocksThrottleReasons(h)
                for name, bit in bits.items():
                    if r & bit:
                        self.reasons.add(name)
                try:
                    self.power.append(nv.nvmlDeviceGetPowerUsage(h) / 1000.0)
                except Exception:
                    pass
                time.sleep(0.005)
        except Exception as e:  # pragma: no cover
            self._err = repr(e)

    def start(self):
        import threading
        self._thread = threading.Thread(target=self._run, daemon=True)
        self._thread.start()

    def stop(self) -> dict:
        self._stop = True
        if self._thread is not None:
            self._thread.join(timeout=5)
        if not self.sm:
            return {"sm_mhz": None, "sm_max_mhz": self.max_mhz, "samples": 0, "reasons": ["nvml unavailable: " + str(self._err)]}
        return {"sm_mhz": statistics.median(self.sm), "sm_min_mhz": min(self.sm), "sm_max_mhz": self.max_mhz, "samples": len(self.sm),
                "power_w_max": max(self.power) if self.power else None, "reasons": sorted(self.reasons)}


# --------------------------------------------------------------------------------------------------
# CPU oracle legs (the only code in this file that may touch oracle/)
# --------------------------------------------------------------------------------------------------
ORACLE_PREFIXES = [a + b for a in "ACGT" for b in "ACGT"]     # 16 ranges of the first two bases + the rest below


def _oracle_range(job):
    """One worker of the all-core leg: the plain oracle restricted to the suffixes that begin with `prefix`
    (a prefix range is a contiguous piece of B_R).  prefix '' = suffixes shorter than two bases and the
    end-marker suffixes: the full oracle on the collection of every read's last base (a tiny collection)."""
    import numpy as np
    path, prefix = job
    import oracle
    ascii_ = np.load(path + ".ascii.npy", mmap_mode="r")
    offsets = np.load(path + ".offsets.npy")
    t0 = time.perf_counter()
    _, piece = oracle.bwt_with_prefix(np.asarray(ascii_), offsets, prefix)
    return prefix, int(piece.size), time.perf_counter() - t0


def time_oracle_all_cores(coll, procs: int):
    """Wall time of the range-restricted oracle over all 16 two-base prefix ranges, `procs` processes (spawned: the
    parent may hold a CUDA context).  Returns (seconds, suffixes sorted)."""
    import multiprocessing as mp
    import tempfile

    import numpy as np
    import oracle
    oracle.build()
    with tempfile.TemporaryDirectory(dir="/dev/shm" if os.path.isdir("/dev/shm") else None) as td:
        path = os.path.join(td, "sample")
        np.save(path + ".ascii.npy", coll.ascii)
        np.save(path + ".offsets.npy", coll.offsets)
        ctx = mp.get_context("spawn")
        with ctx.Pool(procs) as pool:
            pool.map(_oracle_warm, range(procs))                   # start the workers (imports) outside the timed region
            t0 = time.perf_counter()
            res = pool.map(_oracle_range, [(path, p) for p in ORACLE_PREFIXES], chunksize=1)
            dt = time.perf_counter() - t0
    return dt, sum(r[1] for r in res)


def _oracle_warm(_):
    import numpy  # noqa: F401
    import oracle
    oracle.build()
    return 0


def oracle_sample(config: int, scale: float):
    from workloads import generate as gen
    coll = gen.config(config, scale)
    desc = (f"configs[{config}] recipe at scale {scale:g} (coverage preserved): {coll.n_reads:,} reads, {coll.n_suffixes:,} suffixes; "
            f"plain oracle (materialise, qsort with the definition's comparator, read off) restricted to each of the 16 two-base "
            f"prefix ranges, one range per process")
    return coll, desc


def cpu_baseline(config: int) -> dict:
    cores = os.cpu_count() or 1
    coll, desc = oracle_sample(config, CPU_SAMPLE_SCALE.get(config, 0.01))
    dt, sorted_n = time_oracle_all_cores(coll, cores)
    return {"value": sorted_n / dt, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": desc + f"; {sorted_n:,} suffixes sorted",
            "seconds": round(dt, 3), "host_cpus": cores}


def run_reference(args) -> None:
    """The reference arm of this tier = the oracle, timed as it stands on the host cores (rank 0 only)."""
    if int(os.environ.get("RANK", "0")) != 0:
        return
    cores = os.cpu_count() or 1
    coll, desc = oracle_sample(args.config, REF_SAMPLE_SCALE.get(args.config, 0.01) * args.scale)
    for _ in range(min(args.warmup, 1)):                 # a CPU program has nothing to warm but the page cache
        time_oracle_all_cores(coll, cores)
    runs = [time_oracle_all_cores(coll, cores) for _ in range(args.steps)]
    ms = 1e3 * sum(r[0] for r in runs) / len(runs)
    sorted_n = runs[0][1]
    value = sorted_n / (ms / 1e3)
    base_share = coll.total_bases * (sorted_n / coll.n_suffixes)
    line = {"impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": ms, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": "u8", "data": "synthetic", "config": {"workload": WORKLOADS[args.config], "sample": desc},
            "cpu_baseline": {"value": value, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": desc},
            "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gbases_per_hour": base_share / (ms / 1e3) * 3600 / 1e9, "gpu_launches": 0}
    print(json.dumps(line), flush=True)


# --------------------------------------------------------------------------------------------------
# multi-rank plumbing (replicas only: no data-path collective; covered on CPU by tests/test_bench_dist.py with gloo)
# --------------------------------------------------------------------------------------------------
def replica_seed(config: int, rank: int) -> int:
    """Every rank sorts its own collection of the same recipe: rank 0 uses the config's base seed."""
    from workloads import generate as gen
    return gen.BASE_SEED + config + 1000 * rank


def max_over_ranks(values, device) -> list:
    """Element-wise MAX of per-rank timings (the contract's 'max over ranks'); identity when not distributed."""
    import torch
    import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size() == 1:
        return [float(v) for v in values]
    t = torch.tensor(list(values), dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return [float(v) for v in t]


# --------------------------------------------------------------------------------------------------
# inputs
# --------------------------------------------------------------------------------------------------
def device_collection(index: int, scale: float, seed: int, dev, chunk_reads: int = 2_000_000, keep_ascii: bool = True):
    """configs[1..4] generated chunk by chunk on the device (workloads/generate_torch.py, pinned to the numpy recipes by
    tests/test_generators.py).  Returns (ascii uint8 | None, packed int64, offsets int64, n_reads, total_bases, max_len,
    symbol counts int64[256]).  With keep_ascii=False only the packed form is kept (configs[3], configs[4])."""
    import torch

    import paper_1401_7457_b200 as cx
    from workloads import generate_torch as gt
    recipe = gt.ReadRecipe(index, scale, seed=seed, device=dev)
    n = recipe.n_reads
    offsets = gt.offsets_of(recipe)
    total = int(offsets[-1])
    max_len = int((offsets[1:] - offsets[:-1]).max()) if n else 0
    packed = torch.zeros((total + 31) // 32 + 1, dtype=torch.int64, device=dev)
    ascii_all = torch.empty(total, dtype=torch.uint8, device=dev) if keep_ascii else None
    counts = torch.zeros(256, dtype=torch.int64, device=dev)
    carry = torch.zeros(0, dtype=torch.uint8, device=dev)
    done = 0                                  # bases packed so far (a multiple of 32)
    for a, b, lens, ascii_ in gt.read_chunks(recipe, chunk_reads):
        counts += torch.bincount(ascii_.to(torch.int64), minlength=256)
        if keep_ascii:
            o0 = int(offsets[a])
            ascii_all[o0:o0 + ascii_.numel()] = ascii_
        buf = torch.cat([carry, ascii_]) if carry.numel() else ascii_
        whole = buf.numel() // 32 * 32 if b < n else buf.numel()
        if whole:
            cx.cx_pack_reads(buf[:whole].contiguous(), packed[done // 32: done // 32 + (whole + 31) // 32])
        carry = buf[whole:].clone()
        done += whole
        del ascii_, buf
    assert done == total
    del recipe
    return ascii_all, packed, offsets, n, total, max_len, counts


def host_ram_gb() -> float:
    try:
        with open("/proc/meminfo") as f:
            for ln in f:
                if ln.startswith("MemAvailable:"):
                    return int(ln.split()[1]) / (1 << 20)
    except Exception:
        pass
    return 0.0


def one_step_record(index: int, dev, peak: float) -> dict:
    """configs[3] / configs[4] (and, with --all-configs, the small ones) as ONE timed build each: inputs generated on the
    device, packed reads resident in HBM, CUDA events around cx_bwt_build, per-class times from the same build (profile=1:
    events around every launch; the whole-build time of a run this long is not moved by them).  configs[4] streams its
    101 GB output to pinned host memory (a9)."""
    import gc

    import torch

    import paper_1401_7457_b200 as cx
    from workloads import generate as gen
    gc.collect()
    torch.cuda.empty_cache()
    free_gb = torch.cuda.mem_get_info(dev)[0] / (1 << 30)
    host_out = index == 4
    need_gpu, need_host = {0: 1, 1: 8, 2: 60, 3: 150, 4: 170}[index], {4: 115}.get(index, 4)
    if free_gb < need_gpu or host_ram_gb() < need_host:
        return {"workload": WORKLOADS[index], "skipped": f"needs {need_gpu} GB of HBM and {need_host} GB of host RAM; free: {free_gb:.0f} GB, {host_ram_gb():.0f} GB"}
    t0 = time.time()
    _, packed, offsets, n, total, max_len, counts = device_collection(index, 1.0, gen.BASE_SEED + index, dev, chunk_reads=2_500_000, keep_ascii=False) \
        if index >= 1 else _small_collection(index, dev)
    N = total + n
    torch.cuda.synchronize()
    gen_s = time.time() - t0
    torch.cuda.empty_cache()
    ws = {3: 130 << 30, 4: 136 << 30}.get(index)
    plan = cx.Plan(n, total, workspace_bytes=ws, max_read_len=max_len, out_is_host_pinned=1 if host_out else 0, profile=1, device=dev)
    out = torch.empty(N, dtype=torch.uint8, pin_memory=True) if host_out else torch.empty(N, dtype=torch.uint8, device=dev)
    stream = torch.cuda.current_stream()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    torch.cuda.synchronize()
    e0.record(stream)
    plan.build(packed, offsets, n, out)
    e1.record(stream)
    torch.cuda.synchronize()
    ms = e0.elapsed_time(e1)
    stats = plan.stats()
    times = plan.kernel_times()
    plan.free()
    del plan
    # whole-output invariant (the parity proper is tests/ -m gpu): symbol counts
    got = torch.zeros(256, dtype=torch.int64, device=dev)
    for a in range(0, N, 1 << 30):
        got += torch.bincount(out[a:a + (1 << 30)].to(dev).to(torch.int64), minlength=256)
    counts[ord("$")] += n
    ok = bool(torch.equal(got, counts))
    kernels = {k: {"ms": round(v["ms"], 2), "launches": v["launches"], "gb_s": round(v["bytes"] / (v["ms"] * 1e-3) / 1e9, 1) if v["ms"] > 0 else None,
                   "frac_of_peak": round(v["bytes"] / (v["ms"] * 1e-3) / 1e9 / peak, 4) if v["ms"] > 0 else None}
               for k, v in times.items() if v["launches"]}
    alg = sum(v["bytes"] for v in times.values())
    rec = {"workload": WORKLOADS[index], "n_reads": n, "total_bases": total, "n_suffixes": N, "steps": 1, "ms_per_step": ms,
           "value": N / (ms * 1e-3), "unit": UNIT, "gbases_per_hour": total / (ms * 1e-3) * 3600 / 1e9,
           "output": "pinned host memory, streamed batch by batch (a9); the D2H copies are inside the timed build" if host_out else "device",
           "n_batches": stats["n_batches"], "id_bytes": stats["id_bytes"], "sort_passes": stats["sort_passes"], "max_batch": stats["max_batch"],
           "refine_rounds": stats["refine_rounds"], "kernels": kernels,
           "pipeline": {"alg_bytes_per_suffix": round(alg / N, 1), "gb_s": round(alg / (ms * 1e-3) / 1e9, 1), "frac_of_peak": round(alg / (ms * 1e-3) / 1e9 / peak, 4)},
           "symbol_counts_ok": ok, "generate_s": round(gen_s, 1)}
    del out, packed, offsets, counts, got
    gc.collect()
    torch.cuda.empty_cache()
    if not ok:
        raise SystemExit(f"bench.py: configs[{index}]: output symbol counts differ from the input's")
    return rec


def _small_collection(index: int, dev):
    import numpy as np
    import torch

    import paper_1401_7457_b200 as cx
    from workloads import generate as gen
    c = gen.config(index)
    a = torch.from_numpy(c.ascii).to(dev)
    counts = torch.bincount(a.to(torch.int64), minlength=256)
    return a, cx.cx_pack_reads(a), torch.from_numpy(c.offsets.astype(np.int64)).to(dev), c.n_reads, c.total_bases, c.max_read_len, counts


# --------------------------------------------------------------------------------------------------
# the CUDA arm
# --------------------------------------------------------------------------------------------------
def run_cx(args) -> None:
    import numpy as np
    import torch
    import torch.distributed as dist

    import paper_1401_7457_b200 as cx
    from workloads import generate as gen

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device; the product path has no CPU fallback")
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    if world > 1:
        if args.shard:
            os.environ.setdefault("NCCL_DEBUG", "INFO")      # the communicator lines (ranks, transport) go to stderr beside the record
        dist.init_process_group("nccl", device_id=dev)
    cx.lib()
    if args.config >= 3 and not args.table4 and args.scale == 1.0:
        raise SystemExit("bench.py: configs[3] and configs[4] have no host-resident end-to-end leg; they are the one-step records under other_configs")

    # ---- synthetic input (seeded; replicas differ only in seed) -------------------------------------
    seed = replica_seed(args.config, 0 if args.shard else rank)
    if args.table4 or args.config == 0 or args.scale < 0.05:
        coll = gen.table4(args.table4, args.scale) if args.table4 else gen.config(args.config, args.scale, seed=seed)
        n_reads, total, max_len = coll.n_reads, coll.total_bases, coll.max_read_len
        h_ascii = torch.from_numpy(coll.ascii).pin_memory()
        h_off = torch.from_numpy(coll.offsets.astype(np.int64)).pin_memory()
        d_ascii, d_off = h_ascii.to(dev), h_off.to(dev)
        want_counts = torch.bincount(d_ascii.to(torch.int64), minlength=256)
        del coll
    else:
        d_ascii, _, d_off, n_reads, total, max_len, want_counts = device_collection(args.config, args.scale, seed, dev)
        h_ascii = torch.empty(total, dtype=torch.uint8).pin_memory()
        h_ascii.copy_(d_ascii)
        h_off = torch.empty(n_reads + 1, dtype=torch.int64).pin_memory()
        h_off.copy_(d_off)
    N = total + n_reads
    want_counts[ord("$")] += n_reads
    out_bytes = N if args.out_bits == 8 else (N + 1) // 2
    h_out = torch.empty(out_bytes, dtype=torch.uint8).pin_memory()
    d_packed = torch.empty((total + 31) // 32 + 1, dtype=torch.int64, device=dev)
    d_out = torch.empty(out_bytes, dtype=torch.uint8, device=dev)
    sharded = bool(args.shard) and world > 1
    one_shard = args.shard_of > 1 and not sharded
    plan_opts = dict(max_read_len=max_len, key_bases=args.key_bases or None, max_batch_suffixes=args.max_batch or None,
                     shard_index=rank if sharded else (args.shard_index if args.shard_of > 1 else None),
                     shard_count=world if sharded else (args.shard_of if args.shard_of > 1 else None), device=dev)
    if args.out_bits == 4:
        plan_opts["out_bits"] = 4
    plan = cx.Plan(n_reads, total, profile=0, **plan_opts)
    units = 1 if sharded else world      # collections sorted per step by the whole job
    flush = torch.empty(256 << 20, dtype=torch.uint8, device=dev)       # > 126 MB L2
    stream = torch.cuda.current_stream()

    fasta_ev = []
    if args.fasta:
        coll_f = gen.Collection(h_ascii.numpy(), h_off.numpy().astype(np.uint64))
        h_text = torch.from_numpy(np.frombuffer(gen.to_fasta(coll_f, line_width=0), dtype=np.uint8).copy()).pin_memory()
        d_text = h_text.to(dev)

    def ingest(timed=False):
        """ASCII bases + offsets of the step: resident already, or parsed from the FASTA text (NEXT-4)"""
        if not args.fasta:
            return d_ascii, d_off
        if timed:
            fasta_ev.append((torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)))
            fasta_ev[-1][0].record(stream)
        bases, offs = cx.cx_fasta_parse(d_text, max_reads=n_reads)
        if timed:
            fasta_ev[-1][1].record(stream)
        return bases, offs

    def build(p, offs=None):
        if sharded:
            cx.build_sharded(p, d_packed, d_off, n_reads, d_out)   # this rank's partition range, then the exchange of the pieces
        else:
            p.build(d_packed, d_off if offs is None else offs, n_reads, d_out)

    def step_device(p):
        a, o = ingest()
        cx.cx_pack_reads(a, d_packed, check=False)
        build(p, o if args.fasta else None)

    def step_e2e(p):
        """The call a user makes with HOST buffers: input from pinned host memory, result back in pinned host memory."""
        if args.fasta:
            d_text.copy_(h_text, non_blocking=True)
            a, o = ingest()
            cx.cx_pack_reads(a, d_packed, check=False)
            p.build(d_packed, o, n_reads, d_out)
        else:
            cx.pack_reads_from_host(h_ascii, d_ascii, d_packed, stream=stream)      # chunked H2D overlapped with the pack kernel
            d_off.copy_(h_off, non_blocking=True)
            build(p)
        h_out.copy_(d_out, non_blocking=True)
        stream.synchronize()

    def barrier():
        torch.cuda.synchronize()
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    warm = max(args.warmup, 3)
    for _ in range(warm):
        flush.fill_(1)
        step_device(plan)
    torch.cuda.synchronize()
    stats = plan.stats()
    # cheap whole-output invariants (the parity proper is tests/ -m gpu): |B| = N, n_reads '$', base counts
    if one_shard:
        N = stats["shard_suffixes"]          # the piece this run sorts; its parity is tests/test_shard.py
    elif args.out_bits == 8:
        got = torch.bincount(d_out.to(torch.int64), minlength=256)
        if not torch.equal(got, want_counts):
            raise SystemExit("bench.py: output symbol counts differ from the input's")

    # ---- device-resident timing (profile = 0: no events inside the library) ------------------------------------
    ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(args.steps)]
    sampler = ClockSampler(local)
    barrier()
    sampler.start()
    launches = 0
    for i in range(args.steps):
        flush.fill_(i)                       # L2 flush between timed iterations (outside the events)
        ev[i][0].record(stream)
        step_device(plan)
        ev[i][1].record(stream)
        stream.synchronize()
        launches += plan.stats()["kernel_launches"] + 1 + (10 if args.fasta else 0)
    barrier()
    clocks = sampler.stop()
    dev_ms = sum(a.elapsed_time(b) for a, b in ev) / args.steps

    # ---- end to end: pinned host in, pinned host out ----------------------------------------------------
    e2e_steps = max(3, min(args.steps, 10))

    def time_e2e(step):
        for _ in range(2):
            step()
        barrier()
        t0 = time.perf_counter()
        for _ in range(e2e_steps):
            step()
        torch.cuda.synchronize()
        ms = (time.perf_counter() - t0) * 1e3 / e2e_steps
        barrier()
        return ms

    e2e_variants = {"sequential": time_e2e(lambda: step_e2e(plan))}     # H2D, build into device memory, D2H: one after the other
    plan.free()
    del plan
    if not sharded and not one_shard and not args.fasta and args.out_bits == 8 and N >= 4_000_000:
        # the library's own pinned-host output path (a9): four batches, each batch's D2H copy on a side stream while the next
        # batch computes; and the same with the packed output (NEXT-4: half the bytes back over PCIe)
        def streamed(extra: dict, nbytes: int, check: bool) -> float:
            so = dict(plan_opts, out_is_host_pinned=1, max_batch_suffixes=N // 4 + N // 64, **extra)
            sp = cx.Plan(n_reads, total, profile=0, **so)
            h_res = h_out[:nbytes]

            def step():
                cx.pack_reads_from_host(h_ascii, d_ascii, d_packed, stream=stream)
                d_off.copy_(h_off, non_blocking=True)
                sp.build(d_packed, d_off, n_reads, h_res)       # returns when the last batch has been copied to the host
            ms = time_e2e(step)
            if check:                                            # the streamed result must be the same bytes
                got = torch.bincount(h_res.to(dev).to(torch.int64), minlength=256)
                if not torch.equal(got, want_counts):
                    raise SystemExit("bench.py: streamed output symbol counts differ from the input's")
            sp.free()
            return ms
        e2e_variants["streamed"] = streamed({}, N, True)
        e2e_variants["streamed_packed"] = streamed({"out_bits": 4}, (N + 1) // 2, False)

        def pipelined() -> float:
            """THROUGHPUT of back-to-back builds through cx.HostPipeline (two sets of buffers, three streams): while step i computes,
            step i + 1's reads are copied in and packed and step i - 1's output is copied out.  Every step's H2D and D2H is
            inside the timed region; ms per step = elapsed / steps.  Not the latency of one step: that is `sequential`."""
            pp = cx.Plan(n_reads, total, profile=0, **plan_opts)
            pipe = cx.HostPipeline(pp, n_reads, total)
            results = pipe.run(itertools.repeat((h_ascii, h_off, n_reads)))
            seen = []

            def step():
                seen.append(next(results))              # the result of the step before this one, complete in pinned host memory
            ms = time_e2e(step)
            for hout in seen[-2:]:                      # the last two results: one from each set of buffers
                got = torch.bincount(hout.to(dev).to(torch.int64), minlength=256)
                if not torch.equal(got, want_counts):
                    raise SystemExit("bench.py: pipelined output symbol counts differ from the input's")
            del results, pipe
            pp.free()
            return ms
        e2e_variants["pipelined"] = pipelined()
    e2e_name = min((k for k in e2e_variants if k != "streamed_packed"), key=lambda k: e2e_variants[k])
    e2e_ms = e2e_variants[e2e_name]

    # ---- per-class table: a separate pass with CUDA events around every launch (cx_bwt_kernel_time) --------------
    prof_steps = 3
    pplan = cx.Plan(n_reads, total, profile=1, **plan_opts)
    classes = {k: {"ms": 0.0, "launches": 0, "bytes": 0} for k in cx.KERNEL_CLASSES}
    pack_ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(prof_steps)]
    step_device(pplan)
    for i in range(prof_steps):
        flush.fill_(i)
        a, o = ingest(timed=True)
        pack_ev[i][0].record(stream)
        cx.cx_pack_reads(a, d_packed, check=False)
        pack_ev[i][1].record(stream)
        build(pplan, o if args.fasta else None)
        stream.synchronize()
        for k, v in pplan.kernel_times().items():
            for f in ("ms", "launches", "bytes"):
                classes[k][f] += v[f]
    pstats = pplan.stats()
    classes["pack"] = {"ms": sum(a.elapsed_time(b) for a, b in pack_ev), "launches": prof_steps, "bytes": prof_steps * (total + total // 4)}
    if args.fasta:      # two reads of the text, one write of the bases, 8 B per read (cx_fasta.cu)
        classes["fasta"] = {"ms": sum(a.elapsed_time(b) for a, b in fasta_ev), "launches": 10 * prof_steps,
                            "bytes": prof_steps * (2 * h_text.numel() + total + 8 * n_reads)}
    pplan.free()
    del pplan

    if world > 1:
        dev_ms, e2e_ms = max_over_ranks([dev_ms, e2e_ms], dev)
    if rank != 0:
        dist.destroy_process_group()
        return

    # ---- report --------------------------------------------------------------------------------------
    peak, peak_src = hbm_peak()
    kernels = {}
    for k, v in classes.items():
        if v["launches"] == 0:
            continue
        gbs = v["bytes"] / (v["ms"] * 1e-3) / 1e9 if v["ms"] > 0 else None
        kernels[k] = {"ms_per_step": round(v["ms"] / prof_steps, 4), "launches_per_step": v["launches"] / prof_steps,
                      "alg_bytes_per_step": v["bytes"] // prof_steps, "gb_s": round(gbs, 1) if gbs else None,
                      "frac_of_peak": round(gbs / peak, 4) if gbs else None}

    def roofline_of(cls: str) -> dict:
        c = classes[cls]
        per_launch_bytes = c["bytes"] / max(c["launches"], 1)
        per_launch_ms = c["ms"] / max(c["launches"], 1)
        ach = per_launch_bytes / (per_launch_ms * 1e-3) / 1e9 if per_launch_ms > 0 else 0.0
        key = (args.config, cls) if args.scale == 1.0 and not args.table4 and not args.fasta else None
        return {"kernel": KERNEL_NAMES.get(cls, cls), "class": cls, "bound": "hbm", "achieved": round(ach, 1), "peak": peak, "unit": "GB/s",
                "frac": round(ach / peak, 4), "traffic": NCU_TRAFFIC.get(key), "traffic_from": NCU_TRAFFIC_FILE if key in NCU_TRAFFIC else None,
                "peak_source": peak_src, "nominal_peak": 8000.0, "alg_bytes_per_launch": int(per_launch_bytes),
                "us_per_launch": round(per_launch_ms * 1e3, 2), "launches_per_step": c["launches"] / prof_steps,
                "share_of_kernel_time": round(c["ms"] / max(sum(x["ms"] for x in classes.values()), 1e-9), 4)}

    dominant = max((k for k in classes if classes[k]["launches"]), key=lambda k: classes[k]["ms"])
    total_alg = sum(v["bytes"] for v in classes.values()) / prof_steps
    kern_ms = sum(v["ms"] for v in classes.values()) / prof_steps
    wl = (f"Table 4 shape (PAPER.md:184-189): reads of {args.table4} bp, 30x, both strands, 1% subst." if args.table4
          else WORKLOADS.get(args.config, str(args.config))) + (f" x scale {args.scale:g}" if args.scale != 1 else "") \
        + (" [input: FASTA text, parsed on the device]" if args.fasta else "") + (" [output: 4 bits per symbol]" if args.out_bits == 4 else "")
    line = {
        "metric": METRIC, "value": units * N / (dev_ms * 1e-3), "unit": UNIT, "n_gpus": world, "steps": args.steps,
        "warmup": warm, "ms_per_step": dev_ms, "higher_is_better": True, "scaling": "strong" if sharded else "weak", "vs_baseline": None,
        "dtype": "u64", "data": "synthetic",
        "config": {"workload": wl, "n_reads": n_reads, "total_bases": total, "n_suffixes": N,
                   "parallelism": (f"{world} contiguous partition ranges (PAPER.md:103) + all-gather of the pieces" if sharded
                                   else "replicas only" if world > 1 else
                                   f"1 gpu, shard {args.shard_index} of {args.shard_of} only (its piece: {N} suffixes)" if one_shard else "1 gpu"),
                   "l2": "256 MiB L2-flush write between timed steps; working set >> L2", "prefix_len": 6,
                   "key_bases": "auto (15 bases in a 32-bit key up to 2^30 suffixes, else 19 bases in a 40-bit key)",
                   "timing": "value/ms_per_step: CUDA events around each step, library built with profile=0; kernels{}/roofline{}: a "
                             "separate pass of the same steps with CUDA events around every launch (profile=1)",
                   "id_bytes": stats["id_bytes"], "n_batches": stats["n_batches"], "sort_passes": stats["sort_passes"],
                   "refine_rounds": stats["refine_rounds"], "refine_elements": stats["refine_elements"],
                   "small_group_elems": stats["small_group_elems"]},
        "gbases_per_hour": units * total / (dev_ms * 1e-3) * 3600 / 1e9,
        "e2e": {"value": units * N / (e2e_ms * 1e-3), "unit": UNIT, "ms_per_step": e2e_ms, "steps": e2e_steps, "path": e2e_name,
                "h2d_bytes_per_step": int(h_text.numel()) if args.fasta else int(h_ascii.numel() + h_off.numel() * 8), "d2h_bytes_per_step": int(h_out.numel()),
                "variants_ms_per_step": {k: round(v, 3) for k, v in e2e_variants.items()},
                "selected": f"the fastest of the {sum(1 for k in e2e_variants if k != 'streamed_packed')} ASCII-output variants tried (all listed in variants_ms_per_step)",
                "kind": {"sequential": "latency of one step", "streamed": "latency of one step", "streamed_packed": "latency of one step",
                         "pipelined": "throughput of overlapped back-to-back steps (elapsed / steps)"}[e2e_name],
                "variants": "sequential: copy in, cx_bwt_build into device memory, copy out; streamed: cx_bwt_build with out_is_host_pinned in four "
                            "batches, each batch's copy overlapping the next batch's compute; pipelined: back-to-back builds, step i + 1's copy-in "
                            "and pack and step i - 1's copy-out on side streams while step i computes (two sets of buffers; every step's H2D and "
                            "D2H inside the timed region); streamed_packed: the same as streamed with out_bits = 4 "
                            "(half the bytes out; reported only here, e2e is the better of the two ASCII-output paths)"},
        "gpu_launches": int(launches),
        "clocks": clocks,
        # the kernel class with the largest share of the step, against the HBM roofline of its algorithmic bytes
        "roofline": roofline_of(dominant),
        # the metric also names the radix pass: first-sort launches only (the global path's small re-sorts are `refine_sort`)
        "roofline_sort_pass": roofline_of("sort_pass") if classes["sort_pass"]["launches"] else None,
        "finish_rank_compares_per_step": pstats["compare_ops"],     # diagnostic: 32-bit rank-key comparisons of the in-block refinement
        "pipeline": {"alg_bytes_per_step": int(total_alg), "alg_bytes_per_suffix": round(total_alg / N, 1),
                     "gb_s": round(total_alg / (dev_ms * 1e-3) / 1e9, 1), "frac_of_peak": round(total_alg / (dev_ms * 1e-3) / 1e9 / peak, 4),
                     "kernel_ms_per_step_profiled": round(kern_ms, 3)},
        "kernels": kernels,
        "paper_context": "CX1: 100 Gbases in 6,886 s on i7-3930K + GTX 680 (14.7 M suffixes/s, 52 Gbases/h; PAPER.md:141); BCR 46,899 s "
                         "(abstract: 'BRC ... 12 hours'); other hardware, context only",
    }
    # release everything of the main workload before the larger configurations
    del d_ascii, d_off, d_packed, d_out, h_ascii, h_off, h_out, flush, want_counts
    import gc
    gc.collect()
    torch.cuda.empty_cache()
    line["config"]["hbm_free_gb_before_other_configs"] = round(torch.cuda.mem_get_info(dev)[0] / (1 << 30), 1)
    if world == 1 and not args.no_other_configs and args.scale == 1.0 and not args.table4 and not one_shard:
        others = []
        for idx in ([0, 1] if args.all_configs else []) + [3, 4]:
            if idx == args.config:
                continue
            try:
                others.append(one_step_record(idx, dev, peak))
            except SystemExit:
                raise
            except Exception as e:  # a box too small for configs[4] must not cost the main measurement
                others.append({"workload": WORKLOADS[idx], "error": repr(e)[:300]})
        line["other_configs"] = others
    if world == 1 and not args.no_cpu_baseline:
        line["cpu_baseline"] = cpu_baseline(args.config)
    print(json.dumps(line), flush=True)
    if world > 1:
        dist.destroy_process_group()


def main():
    args = parse_args()
    if args.impl == "reference":
        run_reference(args)
    else:
        run_cx(args)


if __name__ == "__main__":
    main()
