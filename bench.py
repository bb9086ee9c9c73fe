#!/usr/bin/env python
"""Benchmark of the all-mode spMTTKRP hot path (BASELINE.json metric) on B200.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config C] [--impl ours|reference]

A "step" is one steady-state sweep of the whole hot path over the resident tensor: for every mode
d = 0..N-1 the remap into the mode-d layout (Alg. 3), the MTTKRP kernels (Alg. 2/4) and the split-row
fix-up, i.e. N remaps + N MTTKRPs (Alg. 5).  Workload: BASELINE.json configs[C]
(default C=1: 3-mode, 12,000 x 9,000 x 29,000, 77M nonzeros, Zipf 1.1, R=32), synthetic, seeded
(`workloads/`).  `--gpus N` runs N independent replicas (replicas only, no
collective on the data path).  One JSON line on stdout (rank 0).
"""
from __future__ import annotations

import argparse
import json
import os
import statistics
import subprocess
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "all-mode spMTTKRP GFLOP/s (nnz*N*R flops per mode, remap included)"
UNIT = "GFLOP/s"
FALLBACK_HBM_GBS = 6650.0          # /opt/skills/guides/B200_PROFILING.md fallback


def parse_args():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=50)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--config", type=int, default=1, help="index into BASELINE.json configs (0-based)")
    ap.add_argument("--rank", type=int, default=0, help="R (0 = the config's)")
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--nnz", type=int, default=0, help="override nnz (debug / scaled runs)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--cpu-sample-nnz", type=int, default=32_000_000)
    ap.add_argument("--partition-report", action="store_true",
                    help="also run the paper's Alg. 1 partitioner (kappa = 148) and report its load balance")
    return ap.parse_args()


def workload_name(spec, R):
    return f"configs[{spec.config_id - 1}] {spec.name} dims={'x'.join(str(d) for d in spec.dims)} nnz={spec.nnz} R={R}"


# ------------------------------------------------------------------------------------------------
# clocks sampling (B200_PROFILING.md "clocks DURING the timed region")
# ------------------------------------------------------------------------------------------------
class ClockSampler:
    QUERY = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
             "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
             "clocks_event_reasons.sw_power_cap")

    def __init__(self, gpu_index: int):
        self.samples = []
        self.proc = None
        self.gpu = gpu_index
        self.thread = None

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(self.gpu), f"--query-gpu={self.QUERY}",
                                          "--format=csv,noheader,nounits", "-lms", "100"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
        except OSError:
            self.proc = None
            return
        self.thread = threading.Thread(target=self._read, daemon=True)
        self.thread.start()

    def _read(self):
        for line in self.proc.stdout:
            self.samples.append((time.time(), line.strip()))

    def stop(self, t0: float, t1: float) -> dict:
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.15)
        self.proc.terminate()
        try:
            self.proc.wait(timeout=5)
        except subprocess.TimeoutExpired:
            self.proc.kill()
        rows = [s for (t, s) in self.samples if t0 - 0.05 <= t <= t1 + 0.15] or [s for (_, s) in self.samples]
        sm, smax, reasons = [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for r in rows:
            f = [x.strip() for x in r.split(",")]
            if len(f) < 7:
                continue
            try:
                sm.append(float(f[0]))
                smax.append(float(f[1]))
            except ValueError:
                continue
            for name, v in zip(names, f[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(name)
        return {"sm_mhz": statistics.median(sm) if sm else None, "sm_max_mhz": max(smax) if smax else None,
                "samples": len(sm), "reasons": sorted(reasons)}


# ------------------------------------------------------------------------------------------------
# the oracle legs (the only places bench.py may execute oracle/)
# ------------------------------------------------------------------------------------------------
def time_oracle_sample(spec, R, sample_nnz, tensor_cpu=None):
    """Times the fp64 oracle, as it stands, on the first `sample_nnz` nonzeros of the workload
    (all modes: stable sort by the output index + accumulation), all host cores.  GFLOP/s with the
    same flop convention."""
    import numpy as np
    import oracle
    import workloads as W
    if tensor_cpu is None:
        sub = spec.scaled(min(sample_nnz, spec.nnz))
        t = W.generate_tensor(sub)
        idx, vals = t.idx.numpy(), t.vals.numpy()
        what = f"{sub.nnz} nonzeros drawn from the workload's distribution (same dims and skew)"
    else:
        idx, vals = tensor_cpu
        idx = np.ascontiguousarray(idx[:, :sample_nnz])
        vals = np.ascontiguousarray(vals[:sample_nnz])
        what = f"first {vals.shape[0]} nonzeros of the workload's (shuffled) COO list"
    nnz = int(vals.shape[0])
    N = len(spec.dims)
    fac = [f.numpy() for f in W.generate_factors(spec, R)]
    threads = oracle.max_threads()
    oracle.build()
    t0 = time.perf_counter()
    for d in range(N):
        perm = oracle.sort_perm(spec.dims, idx, [d])
        oracle.mttkrp_mode(spec.dims, idx, vals, fac, d, perm=perm, threads=max(threads, 2))
    dt = time.perf_counter() - t0
    flops = float(nnz) * N * R * N
    return {"value": flops / dt / 1e9, "unit": UNIT, "cores": threads, "kind": "oracle",
            "sample": f"{what}, all {N} modes, stable sort + fp64 accumulation, {dt:.2f} s"}, dt, nnz


def run_reference(args):
    import workloads as W
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    spec = W.CONFIGS[args.config]
    if args.nnz:
        spec = spec.scaled(args.nnz)
    R = args.rank or spec.ranks[-1 if len(spec.ranks) == 1 else 2]
    N = len(spec.dims)
    sample = min(args.cpu_sample_nnz // 4, spec.nnz)
    times = []
    base = None
    tcpu = W.generate_tensor(spec.scaled(sample))
    tensor_cpu = (tcpu.idx.numpy(), tcpu.vals.numpy())
    for i in range(args.warmup + args.steps):
        base, dt, nnz = time_oracle_sample(spec, R, sample, tensor_cpu)
        if i >= args.warmup:
            times.append(dt)
    ms = 1e3 * sum(times) / len(times)
    value = float(nnz) * N * R * N / (ms / 1e3) / 1e9
    base["value"] = value
    line = {"impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": ms, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": "f64", "data": "synthetic", "config": {"workload": workload_name(spec, R), "sample_nnz": nnz},
            "cpu_baseline": base,
            "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line), flush=True)


# ------------------------------------------------------------------------------------------------
# the CUDA arm
# ------------------------------------------------------------------------------------------------
def run_ours(args):
    import torch
    import workloads as W
    import paper_2405_08470_b200 as P
    from paper_2405_08470_b200 import replicas

    P.load_library()                                   # fail loudly if the CUDA library is missing
    if not torch.cuda.is_available():
        raise RuntimeError("bench.py needs a CUDA device: the product path has no CPU fallback")
    _, _, local = replicas.env_ranks()
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    rank, world, local = replicas.init("nccl", dev)

    def barrier():
        replicas.barrier(dev)

    spec = W.CONFIGS[args.config]
    if args.nnz:
        spec = spec.scaled(args.nnz)
    R = args.rank or spec.ranks[-1 if len(spec.ranks) == 1 else 2]
    N = len(spec.dims)
    t_gen = time.perf_counter()
    t = W.generate_tensor(spec, dev)
    fac = W.generate_factors(spec, R, dev)
    U = W.distinct_per_mode(t)
    torch.cuda.synchronize()
    t_gen = time.perf_counter() - t_gen
    t_create = time.perf_counter()
    h = P.Mttkrp(spec.dims, t.idx, t.vals, max_rank=0 if args.no_e2e else R)
    torch.cuda.synchronize()
    t_create = time.perf_counter() - t_create
    checksums = t.checksums
    nnz = t.nnz
    sample_n = min(args.cpu_sample_nnz, nnz)
    tensor_cpu = None
    if rank == 0 and world == 1 and not args.no_cpu_baseline:
        tensor_cpu = (t.idx[:, :sample_n].cpu().numpy(), t.vals[:sample_n].cpu().numpy())
    del t
    torch.cuda.empty_cache()
    info = h.info()
    outs = [torch.empty((d, R), dtype=torch.float32, device=dev) for d in spec.dims]

    # launches of OUR kernels per sweep: remap + zero-fill (if any empty row) + mttkrp + fix-up (if any split row)
    launches_per_sweep = sum(2 + (1 if info["num_empty_rows"][d] else 0) + (1 if info["num_split_rows"][d] else 0)
                             for d in range(N)) if nnz else sum(1 for d in range(N))
    flops_per_sweep = float(nnz) * N * R * N
    rec = info["record_bytes"]
    bytes_mode = [nnz * rec + sum(U[m] for m in range(N) if m != d) * R * 4 + spec.dims[d] * R * 4 for d in range(N)]
    remap_bytes_mode = nnz * (2 * rec + 4)

    for _ in range(max(args.warmup, 3)):
        h.mttkrp_sweep(fac, outs)
    barrier()
    sampler = ClockSampler(local)
    sampler.start()
    time.sleep(0.25)
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    barrier()
    w0 = time.time()
    e0.record()
    for _ in range(args.steps):
        h.mttkrp_sweep(fac, outs)
    e1.record()
    barrier()
    w1 = time.time()
    ms_total = e0.elapsed_time(e1)
    clocks = sampler.stop(w0, w1)
    ms_total = replicas.max_over_ranks(ms_total, dev)
    ms_step = ms_total / args.steps
    value = world * flops_per_sweep / (ms_step * 1e-3) / 1e9

    # per-kernel-class device time (CUDA events on the launching stream, inside the library)
    h.timing_begin()
    for _ in range(args.steps):
        h.mttkrp_sweep(fac, outs)
    tm = h.timing_end()
    k_ms = tm["mttkrp_ms"] / max(1, tm["mttkrp_launches"])
    peaks_path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(peaks_path):
        peak, peak_src = float(json.load(open(peaks_path))["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
    else:
        peak, peak_src = FALLBACK_HBM_GBS, "fallback (B200_PROFILING.md)"
    alg_bytes_launch = sum(bytes_mode) / N
    achieved = alg_bytes_launch / (k_ms * 1e-3) / 1e9 if k_ms > 0 else 0.0
    traffic = l2_hit = l1_hit = None                   # ncu figures of that kernel, per launch (profiles/r1_traffic.csv)
    tpath = os.path.join(ROOT, "profiles", "r1_traffic.csv")
    if os.path.exists(tpath):
        import csv
        for row in csv.DictReader(open(tpath)):
            if row["config"] == str(args.config) and row["kernel"] == "k_mttkrp" and not args.nnz and not args.rank:
                traffic = float(row["dram_bytes_per_launch"])
                l2_hit, l1_hit = float(row["l2_hit_pct"]), float(row["l1_hit_pct"])
    total_k = tm["remap_ms"] + tm["zero_ms"] + tm["mttkrp_ms"] + tm["fixup_ms"]
    roofline = {"bound": "hbm", "kernel": "k_mttkrp", "achieved": achieved, "peak": peak, "unit": "GB/s",
                "frac": achieved / peak, "traffic": traffic, "peak_source": peak_src,
                "l2_hit_pct_ncu": l2_hit, "l1_hit_pct_ncu": l1_hit,
                "dram_GBs_ncu": (traffic / (k_ms * 1e-3) / 1e9) if (traffic and k_ms > 0) else None,
                "frac_of_nominal_8TBs": achieved / 8000.0,
                "algorithmic_bytes_per_launch": alg_bytes_launch, "avg_launch_ms": k_ms,
                "per_mode_algorithmic_bytes": bytes_mode}
    breakdown = {"remap_ms_per_sweep": tm["remap_ms"] / args.steps, "zero_ms_per_sweep": tm["zero_ms"] / args.steps,
                 "mttkrp_ms_per_sweep": tm["mttkrp_ms"] / args.steps, "fixup_ms_per_sweep": tm["fixup_ms"] / args.steps,
                 "remap_share": tm["remap_ms"] / total_k if total_k else None,
                 "remap_achieved_GBs": (N * remap_bytes_mode * args.steps) / (tm["remap_ms"] * 1e-3) / 1e9 if tm["remap_ms"] else None,
                 "mttkrp_only_GFLOPs": flops_per_sweep * args.steps / ((tm["mttkrp_ms"] + tm["zero_ms"] + tm["fixup_ms"]) * 1e-3) / 1e9
                 if tm["mttkrp_ms"] else None}

    # end to end through the host-buffer entry point (H2D of all factors + D2H of all Y_d every step)
    e2e = None
    if not args.no_e2e:
        fac_host = [f.cpu().pin_memory() for f in fac]
        out_host = [torch.empty((d, R), dtype=torch.float32).pin_memory() for d in spec.dims]
        for _ in range(2):
            h.mttkrp_sweep_host(fac_host, out_host)
        barrier()
        e0.record()
        for _ in range(args.steps):
            h.mttkrp_sweep_host(fac_host, out_host)
        e1.record()
        barrier()
        ms_e2e = e0.elapsed_time(e1)
        ms_e2e = replicas.max_over_ranks(ms_e2e, dev)
        io = sum(d * R * 4 for d in spec.dims)
        e2e = {"value": world * flops_per_sweep / (ms_e2e / args.steps * 1e-3) / 1e9, "unit": UNIT,
               "h2d_bytes_per_step": io, "d2h_bytes_per_step": io, "ms_per_step": ms_e2e / args.steps,
               "api": "mttkrp_sweep_host (pinned host factors in, pinned host Y_d out)"}

    partition = None
    if args.partition_report:
        # Alg. 1 with one partition per SM: whole rows, longest first.  Equal-nnz shards are
        # balanced by construction (max/mean = 1); this shows what indivisible rows cost on the same tensor.
        partition = {"kappa": 148, "max_over_mean": []}
        for d in range(N):
            _, loads = h.partition_rows(d, 148)
            partition["max_over_mean"].append(round(float(loads.max()) / (float(loads.sum()) / 148), 3))
        partition["note"] = "paper's Alg. 1 (whole rows, longest-first) on the same tensor; this library's equal-nnz shards: 1.0"

    cpu_baseline = None
    if rank == 0 and world == 1 and not args.no_cpu_baseline:
        cpu_baseline, _, _ = time_oracle_sample(spec, R, sample_n, tensor_cpu)

    if rank == 0:
        line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": max(args.warmup, 3),
                "ms_per_step": ms_step, "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f32",
                "data": "synthetic",
                "config": {"workload": workload_name(spec, R), "nmodes": N, "nnz": nnz, "R": R,
                           "step": f"one sweep = {N} remaps + {N} MTTKRPs", "l2": "inputs larger than L2 (2 tensor copies of "
                           f"{nnz * rec / 1e6:.0f} MB each alternate; L2 is 126 MB)", "replicas": world,
                           "checksums": checksums, "distinct_per_mode": U, "shard_nnz": info["shard_nnz"],
                           "num_shards": info["num_shards"], "split_rows": info["num_split_rows"],
                           "empty_rows": info["num_empty_rows"], "key_order": info["key_order"],
                           "remap_blocked": info["remap_blocked"],
                           "remap_avg_run": [round(x, 1) for x in info["remap_avg_run"]],
                           "bytes_held": info["bytes_held"], "bytes_paper_format": info["bytes_paper_format"],
                           "create_s": t_create, "generate_s": t_gen},
                "clocks": clocks, "e2e": e2e, "gpu_launches": launches_per_sweep * args.steps,
                "roofline": roofline, "breakdown": breakdown, "cpu_baseline": cpu_baseline, "partition": partition,
                "paper_context": "geomean speedups 1.5x / 2.0x / 21.7x over BLCO / MM-CSF / ParTI-GPU on RTX 3090 "
                                 "(PAPER.md:414); no absolute numbers published"}
        print(json.dumps(line), flush=True)
    h.destroy()
    replicas.finalize()


def main():
    args = parse_args()
    if args.impl == "reference":
        run_reference(args)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()
