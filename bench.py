#!/usr/bin/env python
"""bench.py -- pooled embedding lookups/s and achieved HBM GB/s of the fused multi-table lookup on B200.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--workload c5] [--impl ours|reference]
    python -m torch.distributed.run --nnodes=1 --nproc-per-node N ... bench.py --gpus N ...

A "step" is one pass of the whole hot path (plan build a1+a2, then the fused gather-and-pool a3) over one
batch of seeded synthetic input already resident in HBM; the timed loop rotates over R = 8 batches. The
default workload is BASELINE.json configs[4] (c5: 8 x 4e7 rows, D=64 fp32, B=65536, bags U{1..64}, uniform
indices) -- the configuration the north_star's bandwidth target is quoted on; it fits one GPU (82 GB).
Multi-GPU: the path shards by batch with no data-path collective (every rank holds all tables and its own
batch): weak scaling, value = bags of all ranks / max-over-ranks device time.

Prints ONE JSON line (rank 0). `--impl reference` times the CPU oracle (oracle/) on a bounded sample.
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

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

METRIC = "pooled embedding lookups/sec"
UNIT = "lookups/s"
R_BATCHES = 8


def parse_args():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=40)
    ap.add_argument("--warmup", type=int, default=5)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", default="c5")
    ap.add_argument("--quantum", type=int, default=0)
    ap.add_argument("--unroll", type=int, default=0)
    ap.add_argument("--block-threads", type=int, default=0)
    ap.add_argument("--blocks-per-sm", type=int, default=0)
    ap.add_argument("--mode", type=int, default=0)
    ap.add_argument("--row-l1-no-alloc", type=int, default=-1)
    ap.add_argument("--pdl", type=int, default=0)
    ap.add_argument("--e2e-steps", type=int, default=8)
    ap.add_argument("--cpu-seconds", type=float, default=12.0, help="target CPU time of the oracle baseline")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--rows-scale", type=float, default=1.0, help="debug: scale table heights (invalidates the run)")
    return ap.parse_args()


# ----------------------------------------------------------------------------------------------------
# helpers
# ----------------------------------------------------------------------------------------------------
def measured_peak():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    try:
        with open(path) as f:
            return float(json.load(f)["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs, copy)"
    except Exception:
        return 6650.0, "fallback (B200_PROFILING.md 6.65 TB/s)"


def ncu_traffic(workload: str):
    """dram bytes per lookup launch from the committed ncu --set full capture, if one exists for this workload."""
    try:
        with open(os.path.join(ROOT, "profiles", "ncu_traffic.json")) as f:
            return json.load(f).get(workload, {}).get("dram_bytes_per_launch")
    except Exception:
        return None


class ClockSampler:
    """Samples nvidia-smi clocks and throttle reasons during the timed region."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, gpu_index: int):
        self.idx = gpu_index
        self.samples = []
        self.proc = None

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(self.idx), f"--query-gpu={self.Q}",
                                          "--format=csv,noheader,nounits", "-lms", "100"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.thread = threading.Thread(target=self._read, daemon=True)
            self.thread.start()
        except Exception:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.samples.append((time.time(), line.strip()))

    def stop(self, t0: float, t1: float) -> dict:
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.15)
        self.proc.terminate()
        sm, mx, reasons = [], None, set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        rows = [s for s in self.samples if t0 - 0.05 <= s[0] <= t1 + 0.15] or self.samples
        for _, line in rows:
            p = [x.strip() for x in line.split(",")]
            try:
                sm.append(float(p[0]))
                mx = float(p[1])
                for n, v in zip(names, p[3:7]):
                    if v.lower().startswith("active"):
                        reasons.add(n)
            except Exception:
                continue
        return {"sm_mhz": statistics.median(sm) if sm else None, "sm_max_mhz": mx, "reasons": sorted(reasons),
                "samples": len(rows)}


def apply_options(plan, args, binding):
    if args.quantum:
        plan.set_quantum(args.quantum)
    plan.set_option(binding.OPT_UNROLL, args.unroll)
    plan.set_option(binding.OPT_BLOCK_THREADS, args.block_threads)
    plan.set_option(binding.OPT_BLOCKS_PER_SM, args.blocks_per_sm)
    plan.set_option(binding.OPT_MODE, args.mode)
    plan.set_option(binding.OPT_ROW_L1_NO_ALLOC, args.row_l1_no_alloc)
    plan.set_option(binding.OPT_PDL, args.pdl)


def workload_config(args):
    from paper_2606_21101_b200 import workloads as W
    cfg = W.CONFIGS[args.workload]
    rows = cfg.table_rows()
    if args.rows_scale != 1.0:
        rows = np.maximum(1, (rows * args.rows_scale).astype(np.int64))
    return cfg, rows


def describe(cfg, rows, extra=None):
    d = {"workload": f"{cfg.name} (BASELINE.json configs[{int(cfg.name[1]) - 1}])", "tables": cfg.T,
         "rows_total": int(rows.sum()), "D": cfg.D, "table_dtype": cfg.dtype, "batch": cfg.B,
         "bag_lengths": list(cfg.lengths), "indices": list(cfg.index_dist), "pooling": cfg.pooling,
         "rotating_batches": R_BATCHES,
         "l2": "inputs larger than L2 (no flush)" if cfg.name in ("c4", "c5") else "warm L2 (working set < L2)"}
    if extra:
        d.update(extra)
    return d


# ----------------------------------------------------------------------------------------------------
# CPU oracle legs
# ----------------------------------------------------------------------------------------------------
def oracle_sample(cfg, rows, n_samples):
    """A bounded sample of the workload: the first n_samples samples of batch 0, tables compacted to the rows
    they reference (the full tables do not fit on the host for c5)."""
    from paper_2606_21101_b200 import workloads as W
    batch = W.make_batch(cfg.scaled(B=n_samples), rows, cfg.seed)
    sub = W.compact_subproblem(cfg.scaled(B=n_samples), batch, np.arange(n_samples))
    return sub


def time_oracle(cfg, rows, target_seconds, steps=None, warmup=0):
    import oracle
    from paper_2606_21101_b200 import workloads as W
    oracle.build()
    n_samples = min(cfg.B, 1024)
    sub = oracle_sample(cfg, rows, n_samples)
    pooling = cfg.pooling_modes()
    K = 32

    def one_step():
        off, _, _ = oracle.plan(sub.lengths, K)
        oracle.lookup(sub.tables, W.DTYPE_CODE[cfg.dtype], n_samples, sub.indices, off, pooling)

    t = time.perf_counter()
    one_step()
    first = time.perf_counter() - t
    for _ in range(warmup):
        one_step()
    if steps is None:
        steps = max(1, int(target_seconds / max(first, 1e-4)))
    t = time.perf_counter()
    for _ in range(steps):
        one_step()
    dt = time.perf_counter() - t
    bags = n_samples * cfg.T * steps
    return {"value": bags / dt, "unit": UNIT, "cores": 1, "kind": "oracle",
            "sample": f"first {n_samples} samples of batch 0 ({n_samples * cfg.T} bags, {int(sub.indices.size)} rows), "
                      f"tables compacted to referenced rows; oracle plan + lookup, {steps} steps, {dt:.1f} s",
            "seconds": dt, "ms_per_step": dt / steps * 1e3, "steps": steps}


def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    cfg, rows = workload_config(args)
    r = time_oracle(cfg, rows, args.cpu_seconds, steps=None if args.steps == 40 else args.steps, warmup=min(args.warmup, 1))
    line = {"impl": "reference", "metric": METRIC, "value": r["value"], "unit": UNIT, "n_gpus": args.gpus,
            "steps": r["steps"], "warmup": min(args.warmup, 1), "ms_per_step": r["ms_per_step"],
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": describe(cfg, rows), "cpu_baseline": {k: r[k] for k in ("value", "unit", "cores", "kind", "sample")},
            "e2e": {"value": r["value"], "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line), flush=True)


# ----------------------------------------------------------------------------------------------------
# CUDA path
# ----------------------------------------------------------------------------------------------------
def run_ours(args):
    import torch
    from paper_2606_21101_b200 import binding, build, harness, workloads as W

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device; the DPI lookup has no CPU fallback")
    torch.cuda.set_device(local)
    dist = None
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    if rank == 0:
        build.build()
    if dist is not None:
        dist.barrier()
    binding.load_library()
    warmup = max(args.warmup, 3)
    steps = max(args.steps, 1)

    cfg, rows = workload_config(args)
    # every rank: all tables + its own rotating batches (batch-sharded replicas, no collective on the data path)
    dt = harness.make_device_tables(cfg, rows)
    batches = [harness.upload_batch(W.make_batch(cfg, rows, cfg.seed + 1000 * rank + r)) for r in range(R_BATCHES)]
    pooling = cfg.pooling_modes()
    plan = harness.make_plan(cfg, rows, harness.max_indices_bound(cfg))
    apply_options(plan, args, binding)
    out = harness.new_output(cfg)
    stream = torch.cuda.current_stream()

    def step(i):
        b = batches[i % R_BATCHES]
        plan.build(b.lengths, stream)
        plan.lookup(dt.ptrs, b.indices, out, pooling=pooling, stream=stream)

    def barrier():
        if dist is not None:
            dist.barrier()
        torch.cuda.synchronize()

    for i in range(warmup):
        step(i)
    barrier()

    # ---- timed region: K steps, CUDA events on the launching stream --------------------------------------
    sampler = ClockSampler(local)
    if rank == 0:
        sampler.start()
        time.sleep(0.25)
    ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(steps)]
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    launches0 = binding.launch_count()
    barrier()
    t0 = time.time()
    e0.record(stream)
    for i in range(steps):
        b = batches[i % R_BATCHES]
        plan.build(b.lengths, stream)
        ev[i][0].record(stream)
        plan.lookup(dt.ptrs, b.indices, out, pooling=pooling, stream=stream)
        ev[i][1].record(stream)
    e1.record(stream)
    barrier()
    t1 = time.time()
    launches = binding.launch_count() - launches0
    total_ms = e0.elapsed_time(e1)
    lookup_ms = [a.elapsed_time(b) for a, b in ev]
    clocks = sampler.stop(t0, t1) if rank == 0 else None

    if dist is not None:
        tt = torch.tensor([total_ms], device="cuda", dtype=torch.float64)
        dist.all_reduce(tt, op=dist.ReduceOp.MAX)
        total_ms = float(tt.item())

    # plan facts for the byte counts (after timing)
    Ns, Ss = [], []
    for b in batches:
        plan.build(b.lengths, stream)
        _, _, S, N = plan.export(stream)
        Ns.append(N)
        Ss.append(S)
    n_mean, s_mean = float(np.mean(Ns)), float(np.mean(Ss))
    bytes_step = W.algorithmic_bytes(cfg, cfg.G, n_mean, s_mean)

    # ---- end to end through the host-buffer entry point ----------------------------------------------------
    e2e = None
    if not args.no_e2e:
        hb = [(torch.from_numpy(b.host.lengths).pin_memory(), torch.from_numpy(np.ascontiguousarray(b.host.indices)).pin_memory())
              for b in batches[:2]]
        out_host = torch.empty((cfg.B, cfg.T * cfg.D), dtype=harness.TORCH_DTYPE[cfg.out]).pin_memory()
        for i in range(2):
            plan.forward_host(dt.ptrs, hb[i % 2][0], hb[i % 2][1], out_host, pooling=pooling, stream=stream)
        barrier()
        n_e2e = max(1, args.e2e_steps)
        a, b_ = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        a.record(stream)
        for i in range(n_e2e):
            plan.forward_host(dt.ptrs, hb[i % 2][0], hb[i % 2][1], out_host, pooling=pooling, stream=stream)
        b_.record(stream)
        barrier()
        e2e_ms = a.elapsed_time(b_)
        if dist is not None:
            tt = torch.tensor([e2e_ms], device="cuda", dtype=torch.float64)
            dist.all_reduce(tt, op=dist.ReduceOp.MAX)
            e2e_ms = float(tt.item())
        h2d = int(hb[0][0].numel() * 4 + hb[0][1].numel() * 4)
        d2h = int(out_host.numel() * out_host.element_size())
        e2e = {"value": cfg.G * n_e2e * world / (e2e_ms * 1e-3), "unit": UNIT, "h2d_bytes_per_step": h2d,
               "d2h_bytes_per_step": d2h, "ms_per_step": e2e_ms / n_e2e, "steps": n_e2e,
               "api": "dpi_forward_host (pinned host lengths/indices in, [B,T*D] block out, tables resident)"}

    if rank != 0:
        if dist is not None:
            dist.destroy_process_group()
        return

    peak, peak_src = measured_peak()
    lk_ms = statistics.mean(lookup_ms)
    achieved = bytes_step["lookup"] / (lk_ms * 1e-3) / 1e9
    roofline = {"bound": "hbm", "kernel": "lookup_kernel (a3 fused gather-and-pool)", "achieved": achieved,
                "peak": peak, "unit": "GB/s", "frac": achieved / peak, "peak_source": peak_src,
                "frac_of_nominal_8000": achieved / 8000.0, "traffic": ncu_traffic(cfg.name),
                "algorithmic_bytes_per_launch": bytes_step["lookup"], "kernel_ms_avg": lk_ms,
                "kernel_ms_min": min(lookup_ms), "kernel_ms_median": statistics.median(lookup_ms),
                "kernel_share_of_step": lk_ms * steps / total_ms}
    cpu = None
    if not args.no_cpu_baseline:
        r = time_oracle(cfg, rows, args.cpu_seconds)
        cpu = {k: r[k] for k in ("value", "unit", "cores", "kind", "sample")}
        cpu["host_cpus_visible"] = len(os.sched_getaffinity(0))

    line = {
        "metric": METRIC, "value": cfg.G * steps * world / (total_ms * 1e-3), "unit": UNIT, "n_gpus": world,
        "steps": steps, "warmup": warmup, "ms_per_step": total_ms / steps, "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None, "dtype": "f32", "data": "synthetic",
        "config": describe(cfg, rows, {"parallelism": f"batch-sharded replicas x{world}, no collective",
                                       "quantum_K": plan.info()["K"], "rows_gathered_per_step": n_mean,
                                       "segments_per_step": s_mean}),
        "row_gathers_per_s": n_mean * steps * world / (total_ms * 1e-3),
        "step_algorithmic_gbs": bytes_step["total"] * world / (total_ms / steps * 1e-3) / 1e9,
        "roofline": roofline, "cpu_baseline": cpu, "e2e": e2e, "gpu_launches": int(launches), "clocks": clocks,
        "device": torch.cuda.get_device_name(local),
    }
    print(json.dumps(line), flush=True)
    if dist is not None:
        dist.destroy_process_group()


def main():
    args = parse_args()
    if args.impl == "reference":
        run_reference(args)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()
