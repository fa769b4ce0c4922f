#!/usr/bin/env python
"""bench.py -- one JSON line for BASELINE.json's metric: suffixes sorted/s (and Gbases/hour) of the
collection-BWT hot path on B200, with the dominant kernel's HBM roofline and the CPU oracle beside it.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config i] [--impl cx|reference]

A "step" is one pass of the whole hot path (rows a1-a8 of DESIGN.md: 2-bit pack, partition sizes,
batch plan, list + key build, onesweep sort, tie refinement, emit) over one synthetic collection.
At N=1 the workload is BASELINE.json configs[1] (1,000,000 reads x 100 bp, 100x coverage of a seeded
1 Mbp genome -> 1.01e8 suffixes), the case the paper's design is hardest on (deep shared substrings).
For N>1 (torchrun, one rank per GPU) every rank runs an independent replica with its own seed: the
north_star fixes the path to one GPU with no collectives.

`--impl reference` times the CPU oracle (oracle/, as it stands) on a bounded sample of the same
recipe; nothing else in this file touches oracle/ except the `cpu_baseline` leg.
"""
from __future__ import annotations

import argparse
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
WORKLOADS = {
    0: "configs[0]: 10,000 reads x 100 bp iid (1.01e6 suffixes)",
    1: "configs[1]: 1,000,000 reads x 100 bp at 100x over a seeded 1 Mbp genome (1.01e8 suffixes)",
    2: "configs[2]: 10,000,000 reads x 100 bp at 30x over 33 Mbp, both strands, 1% subst. (1.01e9 suffixes)",
    3: "configs[3]: 40,000,000 reads x 50-250 bp over a 50 Mbp repeat genome (~6.04e9 suffixes)",
    4: "configs[4]: 1,000,000,000 reads x 100 bp at 30x over 3.3 Gbp, both strands, 1% subst. (1.01e11 suffixes)",
}
# dram__bytes_read.sum + dram__bytes_write.sum per launch of the dominant kernel, from the committed
# `ncu --set full` capture named here (None until one exists for this workload).
NCU_TRAFFIC = {"file": "profiles/r01_ncu_full.md (onesweep_pass_kernel<u64 key|id word, keys-only>, configs[1])", "bytes_per_launch": 1_592_000_000}
FALLBACK_HBM_GBS = 6650.0     # /opt/skills/guides/B200_PROFILING.md, used only if MEASURED_PEAKS.json is absent
CPU_SAMPLE_SCALE = 0.1        # cpu_baseline leg: the workload's recipe at this scale (coverage preserved)
REF_SAMPLE_SCALE = 0.05       # --impl reference: one step = the oracle on the recipe at this scale


def parse_args():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--config", type=int, default=1, help="BASELINE.json configs index (0-based)")
    ap.add_argument("--scale", type=float, default=1.0, help="debug only: scale the workload down")
    ap.add_argument("--impl", default="cx", choices=["cx", "reference"])
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--key-bases", type=int, default=0, help="first-round key window w (0 = the library's default)")
    ap.add_argument("--shard", action="store_true", help="NEXT-2, with --gpus N > 1 under torchrun: ONE collection, rank k sorts the k-th of N contiguous "
                    "partition ranges (PAPER.md:103) and the pieces are exchanged (all-gather-v); strong scaling.  Default: independent replicas")
    ap.add_argument("--fasta", action="store_true", help="NEXT-4: the step starts from the collection's FASTA text (resident in HBM; pinned host for e2e): "
                    "cx_fasta_parse + pack + build")
    ap.add_argument("--shard-of", type=int, default=0, help="one GPU: time ONE shard of a W-way partition-range split (no exchange); with --shard-index")
    ap.add_argument("--shard-index", type=int, default=0)
    ap.add_argument("--table4", type=int, default=0, help="NEXT-3: the paper's read-length experiment instead of a config: read length 100/200/400, "
                    "1e10 x --scale bases (PAPER.md:184-189)")
    ap.add_argument("--max-batch", type=int, default=0, help="m1: most suffixes per batch (0 = as many as the workspace allows)")
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
def oracle_sample(config: int, scale: float):
    from workloads import generate as gen
    coll = gen.config(config, scale)
    desc = (f"configs[{config}] recipe at scale {scale:g} (coverage preserved): {coll.n_reads:,} reads, "
            f"{coll.n_suffixes:,} suffixes, full plain oracle (materialise, qsort with the definition's comparator, read off)")
    return coll, desc


def time_oracle(coll) -> float:
    import oracle
    t0 = time.perf_counter()
    oracle.bwt(coll.ascii, coll.offsets)
    return time.perf_counter() - t0


def cpu_baseline(config: int) -> dict:
    import oracle
    oracle.build()
    coll, desc = oracle_sample(config, CPU_SAMPLE_SCALE if config >= 1 else 1.0)
    dt = time_oracle(coll)
    return {"value": coll.n_suffixes / dt, "unit": UNIT, "cores": 1, "kind": "oracle", "sample": desc, "seconds": round(dt, 3),
            "host_cpus": os.cpu_count()}


def run_reference(args) -> None:
    """The reference arm of this tier = the oracle, timed as it stands on the host cores (rank 0 only)."""
    if int(os.environ.get("RANK", "0")) != 0:
        return
    import oracle
    oracle.build()
    coll, desc = oracle_sample(args.config, (REF_SAMPLE_SCALE if args.config >= 1 else 1.0) * args.scale)
    for _ in range(args.warmup):
        time_oracle(coll)
    times = [time_oracle(coll) for _ in range(args.steps)]
    ms = 1e3 * sum(times) / len(times)
    value = coll.n_suffixes / (ms / 1e3)
    line = {"impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": ms, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": "u64", "data": "synthetic", "config": {"workload": WORKLOADS[args.config], "sample": desc},
            "cpu_baseline": {"value": value, "unit": UNIT, "cores": 1, "kind": "oracle", "sample": desc},
            "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gbases_per_hour": coll.total_bases / (ms / 1e3) * 3600 / 1e9, "gpu_launches": 0}
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
        dist.init_process_group("nccl", device_id=dev)
    cx.lib()

    # ---- synthetic input (seeded; replicas differ only in seed) -------------------------------------
    if args.table4:
        coll = gen.table4(args.table4, args.scale)
    else:
        coll = gen.config(args.config, args.scale, seed=replica_seed(args.config, 0 if args.shard else rank))
    n_reads, total, N = coll.n_reads, coll.total_bases, coll.n_suffixes
    h_ascii = torch.from_numpy(coll.ascii).pin_memory()
    h_off = torch.from_numpy(coll.offsets.astype(np.int64)).pin_memory()
    h_out = torch.empty(N, dtype=torch.uint8).pin_memory()
    d_ascii = h_ascii.to(dev)
    d_off = h_off.to(dev)
    d_packed = torch.empty((total + 31) // 32 + 1, dtype=torch.int64, device=dev)
    d_out = torch.empty(N, dtype=torch.uint8, device=dev)
    sharded = bool(args.shard) and world > 1
    plan = cx.Plan(n_reads, total, max_read_len=coll.max_read_len, profile=1, key_bases=args.key_bases or None, max_batch_suffixes=args.max_batch or None,
                   shard_index=rank if sharded else (args.shard_index if args.shard_of > 1 else None),
                   shard_count=world if sharded else (args.shard_of if args.shard_of > 1 else None), device=dev)
    one_shard = args.shard_of > 1 and not sharded
    units = 1 if sharded else world      # collections sorted per step by the whole job
    flush = torch.empty(256 << 20, dtype=torch.uint8, device=dev)       # > 126 MB L2
    stream = torch.cuda.current_stream()

    fasta_ev = []
    if args.fasta:
        h_text = torch.from_numpy(np.frombuffer(gen.to_fasta(coll, line_width=0), dtype=np.uint8).copy()).pin_memory()
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

    def build():
        if sharded:
            cx.build_sharded(plan, d_packed, d_off, n_reads, d_out)   # this rank's partition range, then the exchange of the pieces
        else:
            plan.build(d_packed, d_off, n_reads, d_out)

    def step_device():
        a, o = ingest()
        cx.cx_pack_reads(a, d_packed, check=False)
        build() if not args.fasta else plan.build(d_packed, o, n_reads, d_out)

    def step_e2e():
        if args.fasta:
            d_text.copy_(h_text, non_blocking=True)
            a, o = ingest()
            cx.cx_pack_reads(a, d_packed, check=False)
            plan.build(d_packed, o, n_reads, d_out)
        else:
            d_ascii.copy_(h_ascii, non_blocking=True)
            d_off.copy_(h_off, non_blocking=True)
            cx.cx_pack_reads(d_ascii, d_packed, check=False)
            build()
        h_out.copy_(d_out, non_blocking=True)
        stream.synchronize()

    def barrier():
        torch.cuda.synchronize()
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    for _ in range(max(args.warmup, 3)):
        flush.fill_(1)
        step_device()
    torch.cuda.synchronize()
    stats = plan.stats()
    # cheap whole-output invariants (the parity proper is tests/ -m gpu): |B| = N, n_reads '$', base counts
    got = torch.bincount(d_out.to(torch.int64), minlength=128).cpu().numpy()
    want = np.bincount(coll.ascii, minlength=128)
    want[ord("$")] += n_reads
    if one_shard:
        N = stats["shard_suffixes"]          # the piece this run sorts; its parity is tests/test_shard.py
    elif not np.array_equal(got[:128], want[:128]):
        raise SystemExit("bench.py: output symbol counts differ from the input's")

    # ---- device-resident timing -----------------------------------------------------------------------
    classes = {k: {"ms": 0.0, "launches": 0, "bytes": 0} for k in cx.KERNEL_CLASSES}
    ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(args.steps)]
    pack_ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(args.steps)]
    sampler = ClockSampler(local)
    barrier()
    sampler.start()
    launches = 0
    for i in range(args.steps):
        flush.fill_(i)                       # L2 flush between timed iterations (outside the events)
        ev[i][0].record(stream)
        a, o = ingest(timed=True)
        pack_ev[i][0].record(stream)
        cx.cx_pack_reads(a, d_packed, check=False)
        pack_ev[i][1].record(stream)
        build() if not args.fasta else plan.build(d_packed, o, n_reads, d_out)
        ev[i][1].record(stream)
        stream.synchronize()
        for k, v in plan.kernel_times().items():
            for f in ("ms", "launches", "bytes"):
                classes[k][f] += v[f]
        launches += plan.stats()["kernel_launches"] + 1
    barrier()
    clocks = sampler.stop()
    dev_ms = sum(a.elapsed_time(b) for a, b in ev) / args.steps
    classes["pack"]["ms"] = sum(a.elapsed_time(b) for a, b in pack_ev)
    classes["pack"]["launches"] = args.steps
    classes["pack"]["bytes"] = args.steps * (total + total // 4)
    if args.fasta:      # two reads of the text, one write of the bases, 8 B per read (cx_fasta.cu)
        classes["fasta"] = {"ms": sum(a.elapsed_time(b) for a, b in fasta_ev), "launches": 10 * args.steps,
                            "bytes": args.steps * (2 * h_text.numel() + total + 8 * n_reads)}
        launches += 10 * args.steps

    # ---- end to end: pinned host in, pinned host out ----------------------------------------------------
    for _ in range(2):
        step_e2e()
    barrier()
    t0 = time.perf_counter()
    for _ in range(args.steps):
        step_e2e()
    torch.cuda.synchronize()
    e2e_ms = (time.perf_counter() - t0) * 1e3 / args.steps
    barrier()
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
        kernels[k] = {"ms_per_step": round(v["ms"] / args.steps, 4), "launches_per_step": v["launches"] / args.steps,
                      "alg_bytes_per_step": v["bytes"] // args.steps, "gb_s": round(gbs, 1) if gbs else None,
                      "frac_of_peak": round(gbs / peak, 4) if gbs else None}
    dom = classes["sort_pass"]
    bytes_per_launch = dom["bytes"] / max(dom["launches"], 1)
    ms_per_launch = dom["ms"] / max(dom["launches"], 1)
    achieved = bytes_per_launch / (ms_per_launch * 1e-3) / 1e9 if ms_per_launch > 0 else 0.0
    total_alg = sum(v["bytes"] for v in classes.values()) / args.steps
    kern_ms = sum(v["ms"] for v in classes.values()) / args.steps
    line = {
        "metric": METRIC, "value": units * N / (dev_ms * 1e-3), "unit": UNIT, "n_gpus": world, "steps": args.steps,
        "warmup": max(args.warmup, 3), "ms_per_step": dev_ms, "higher_is_better": True, "scaling": "strong" if sharded else "weak", "vs_baseline": None,
        "dtype": "u64", "data": "synthetic",
        "config": {"workload": (f"Table 4 shape (PAPER.md:184-189): reads of {args.table4} bp, 30x, both strands, 1% subst." if args.table4
                                else WORKLOADS.get(args.config, str(args.config))) + (f" x scale {args.scale:g}" if args.scale != 1 else "")
                               + (" [input: FASTA text, parsed on the device]" if args.fasta else ""),
                   "n_reads": n_reads, "total_bases": total, "n_suffixes": N, "parallelism": (f"{world} contiguous partition ranges (PAPER.md:103) + all-gather-v of the pieces" if sharded
                                                                                       else "replicas only" if world > 1 else
                                                                                       f"1 gpu, shard {args.shard_index} of {args.shard_of} only (its piece: {N} suffixes)" if one_shard else "1 gpu"),
                   "l2": "256 MiB L2-flush write between timed steps; working set >> L2", "prefix_len": 6, "key_bases": "auto (14 bases in a 32-bit key up to 2^30 suffixes, else ceil(log4 N)+1 bases in a 64-bit key)",
                   "id_bytes": stats["id_bytes"], "n_batches": stats["n_batches"], "sort_passes": stats["sort_passes"],
                   "refine_rounds": stats["refine_rounds"], "refine_elements": stats["refine_elements"],
                   "small_group_elems": stats["small_group_elems"]},
        "gbases_per_hour": units * total / (dev_ms * 1e-3) * 3600 / 1e9,
        "e2e": {"value": units * N / (e2e_ms * 1e-3), "unit": UNIT, "ms_per_step": e2e_ms,
                "h2d_bytes_per_step": int(h_text.numel()) if args.fasta else int(h_ascii.numel() + h_off.numel() * 8), "d2h_bytes_per_step": int(h_out.numel())},
        "gpu_launches": int(launches),
        "clocks": clocks,
        "roofline": {"kernel": "onesweep_pass_kernel (a6, one radix pass)", "bound": "hbm", "achieved": round(achieved, 1),
                     "peak": peak, "unit": "GB/s", "frac": round(achieved / peak, 4), "traffic": NCU_TRAFFIC["bytes_per_launch"] if args.config == 1 and args.scale == 1.0 else None,
                     "traffic_from": NCU_TRAFFIC["file"], "peak_source": peak_src, "nominal_peak": 8000.0,
                     "alg_bytes_per_launch": int(bytes_per_launch), "us_per_launch": round(ms_per_launch * 1e3, 2),
                     "launches_per_step": dom["launches"] / args.steps},
        # The in-block refinement (finish) is the largest share of the step and is bound by integer ALU issue, not HBM: its
        # algorithmic work is the number of 192-bit key comparisons its stable rank makes (counted by the kernel), nine
        # issue slots each (LDS.128 + LDS.64 + a seven-instruction borrow chain); peak = SMs x 128 lanes x SM clock / 9.
        "roofline_finish": finish_roofline(classes["finish"], stats, clocks, args.steps),
        "pipeline": {"alg_bytes_per_step": int(total_alg), "alg_bytes_per_suffix": round(total_alg / N, 1),
                     "gb_s": round(total_alg / (dev_ms * 1e-3) / 1e9, 1), "frac_of_peak": round(total_alg / (dev_ms * 1e-3) / 1e9 / peak, 4),
                     "kernel_ms_per_step": round(kern_ms, 3), "host_gap_ms_per_step": round(dev_ms - kern_ms, 3)},
        "kernels": kernels,
        "paper_context": "CX1: 100 Gbases in 6,886 s on i7-3930K + GTX 680 (14.7 M suffixes/s, 52 Gbases/h; PAPER.md:141); BCR 46,899 s "
                         "(abstract: 'BRC ... 12 hours'); other hardware, context only",
    }
    if world == 1 and not args.no_cpu_baseline:
        line["cpu_baseline"] = cpu_baseline(args.config)
    print(json.dumps(line), flush=True)
    if world > 1:
        dist.destroy_process_group()


def finish_roofline(cls: dict, stats: dict, clocks: dict, steps: int) -> dict:
    import torch
    n_sms = torch.cuda.get_device_properties(torch.cuda.current_device()).multi_processor_count
    mhz = clocks.get("sm_mhz") or clocks.get("sm_max_mhz") or 1965.0
    peak = n_sms * 128 * mhz * 1e6 / 9.0
    ms = cls["ms"] / max(steps, 1)
    achieved = stats["compare_ops"] / (ms * 1e-3) if ms > 0 else 0.0
    return {"kernel": "finish_tile_kernel (a7+a8)", "bound": "alu", "achieved": achieved, "peak": peak, "unit": "192-bit key comparisons/s",
            "frac": round(achieved / peak, 4), "compare_ops_per_step": stats["compare_ops"], "ms_per_step": round(ms, 4),
            "peak_derivation": f"{n_sms} SMs x 128 lanes x {mhz:.0f} MHz / 9 issue slots per comparison"}


def main():
    args = parse_args()
    if args.impl == "reference":
        run_reference(args)
    else:
        run_cx(args)


if __name__ == "__main__":
    main()
