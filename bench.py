#!/usr/bin/env python
"""bench.py -- pooled embedding lookups/s and achieved HBM GB/s of the fused multi-table lookup on B200.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--workload c5] [--impl ours|reference]
    python -m torch.distributed.run --nnodes=1 --nproc-per-node N ... bench.py --gpus N ...

A "step" is one pass of the whole hot path (plan build a1+a2, then the fused gather-and-pool a3) over one
batch of seeded synthetic input already resident in HBM; the timed loop rotates over R = 8 batches. The
default workload is BASELINE.json configs[4] (c5: 8 x 4e7 rows, D=64 fp32, B=65536, bags U{1..64}, uniform
indices) -- the configuration the north_star's bandwidth target is quoted on; it fits one GPU (82 GB).
Multi-GPU: the path shards by batch with no data-path collective (every rank holds all tables and its own
batch): weak scaling, value = bags of all ranks / max-over-ranks device time. `--gpus N` without torchrun
(no WORLD_SIZE in the environment) starts the N ranks itself; the CUDA arm refuses if fewer than N devices are visible.

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
DTYPE_KEY = {"f32": "f32", "f16": "f16 tables, f32 accumulate", "bf16": "bf16 tables, f32 accumulate"}
UNIT = "lookups/s"
R_BATCHES = 8


def parse_args():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=None)
    ap.add_argument("--warmup", type=int, default=None)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", default="c5")
    ap.add_argument("--quantum", type=int, default=0)
    ap.add_argument("--unroll", type=int, default=0)
    ap.add_argument("--block-threads", type=int, default=0)
    ap.add_argument("--blocks-per-sm", type=int, default=0)
    ap.add_argument("--mode", type=int, default=0)
    ap.add_argument("--pdl", type=int, default=-1, help="-1: library default (on), 0 / 1: force")
    ap.add_argument("--host-chunks", type=int, default=0, help="dpi_forward_host: 0 auto, 1 unpipelined, n chunks")
    ap.add_argument("--host-direct-out", type=int, default=0,
                    help="dpi_forward_host: 0 auto (lookup stores straight into pinned out_host), 1 staged + D2H copy, 2 require direct")
    ap.add_argument("--kernel", default="output_first", choices=["output_first", "input_first"],
                    help="input_first = the paper's strawman mapping (ablation, PAPER.md:172-176)")
    ap.add_argument("--graph", type=int, default=-1, help="1: time a CUDA-graph replay of the K steps; 0: stream launches; -1: auto (graph for c1-c3)")
    ap.add_argument("--rotating-batches", type=int, default=R_BATCHES)
    ap.add_argument("--e2e-steps", type=int, default=8)
    ap.add_argument("--cpu-seconds", type=float, default=12.0, help="target CPU time of the oracle baseline")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--fused", type=int, default=-1, help="dpi_forward: -1 library default (auto), 0 auto, 1 fused whenever the layout allows, 2 always planner + lookup")
    ap.add_argument("--bag-hint", type=int, default=0, help="1: pass the recipe's longest bag as the OPTIONAL promise DPI_OPT_MAX_BAG_HINT "
                    "(the short-bag variant then runs as its own launch, chosen on the host); default 0 = no promise, the device picks")
    ap.add_argument("--vec-bytes", type=int, default=0, help="DPI_OPT_VEC_BYTES: 0 auto, 16 / 32 bytes of a row per lane and load")
    ap.add_argument("--shard", default="batch", choices=["batch", "tables"],
                    help="multi-GPU layout: batch-sharded replicas (default, DESIGN.md 9) or table-wise sharding with the all-to-all "
                         "fused into the lookup's store (NEXT-3, DESIGN.md 11.3)")
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


def csrc_hash() -> str:
    """sha256 (first 12 hex digits) over the CUDA sources and headers the library is built from: the key that ties an ncu
    capture in profiles/ncu_traffic.csv to the kernels it was taken on."""
    import hashlib
    h = hashlib.sha256()
    base = os.path.join(ROOT, "paper_2606_21101_b200", "csrc")
    for name in sorted(os.listdir(base)) + ["../../include/dpi.h"]:
        path = os.path.join(base, name)
        if os.path.isfile(path):
            h.update(name.encode())
            with open(path, "rb") as f:
                h.update(f.read())
    return h.hexdigest()[:12]


def ncu_traffic(workload: str, kernel: str):
    """dram__bytes_read.sum + dram__bytes_write.sum per launch of `kernel` on `workload` from the committed `ncu --set full`
    capture (profiles/ncu_traffic.csv, written from the .ncu-rep). Each row carries the csrc hash it was captured on: a
    capture of other sources is not reported (traffic = None) and the reason is returned beside it."""
    try:
        import csv
        with open(os.path.join(ROOT, "profiles", "ncu_traffic.csv")) as f:
            rows = [r for r in csv.DictReader(f) if r["workload"] == workload and r["kernel"] == kernel]
    except Exception:
        return None, "profiles/ncu_traffic.csv unreadable"
    if not rows:
        return None, f"no ncu capture of {kernel} on {workload} in profiles/ncu_traffic.csv"
    now = csrc_hash()
    for r in rows:
        if r.get("csrc_hash") == now:
            return float(r["dram_bytes_per_launch"]), None
    return None, (f"traffic_stale: the capture of {kernel} on {workload} ({rows[-1].get('source')}) was taken on csrc "
                  f"{rows[-1].get('csrc_hash')}, the library is now built from {now}")


class ClockSampler:
    """Samples SM clock and throttle reasons during the timed region: NVML in a thread (5 ms period), falling
    back to an `nvidia-smi -lms` subprocess when pynvml is unavailable."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")
    NAMES = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]

    def __init__(self, gpu_index: int):
        self.idx = gpu_index
        self.samples = []     # (time, sm_mhz, set(reasons), power_w)
        self.max_mhz = None
        self.proc = None
        self.nvml = None
        self._stop = threading.Event()
        self.thread = None

    def _physical_index(self):
        vis = os.environ.get("CUDA_VISIBLE_DEVICES")
        if vis:
            try:
                return int(vis.split(",")[self.idx])
            except Exception:
                pass
        return self.idx

    def start(self):
        try:
            import pynvml
            pynvml.nvmlInit()
            self.nvml = pynvml
            self.handle = pynvml.nvmlDeviceGetHandleByIndex(self._physical_index())
            self.max_mhz = float(pynvml.nvmlDeviceGetMaxClockInfo(self.handle, pynvml.NVML_CLOCK_SM))
            self.thread = threading.Thread(target=self._poll_nvml, daemon=True)
            self.thread.start()
            return
        except Exception:
            self.nvml = None
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(self._physical_index()), f"--query-gpu={self.Q}",
                                          "--format=csv,noheader,nounits", "-lms", "50"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.thread = threading.Thread(target=self._read_smi, daemon=True)
            self.thread.start()
        except Exception:
            self.proc = None

    def _poll_nvml(self):
        n = self.nvml
        bits = {"hw_slowdown": n.nvmlClocksEventReasonHwSlowdown if hasattr(n, "nvmlClocksEventReasonHwSlowdown") else 0x8,
                "hw_thermal_slowdown": 0x40, "sw_thermal_slowdown": 0x20, "sw_power_cap": 0x4}
        while not self._stop.is_set():
            try:
                mhz = float(n.nvmlDeviceGetClockInfo(self.handle, n.NVML_CLOCK_SM))
                try:
                    mask = int(n.nvmlDeviceGetCurrentClocksEventReasons(self.handle))
                except Exception:
                    mask = int(n.nvmlDeviceGetCurrentClocksThrottleReasons(self.handle))
                try:
                    pw = n.nvmlDeviceGetPowerUsage(self.handle) / 1000.0
                except Exception:
                    pw = None
                self.samples.append((time.time(), mhz, {k for k, b in bits.items() if mask & b}, pw))
            except Exception:
                pass
            time.sleep(0.005)

    def _read_smi(self):
        for line in self.proc.stdout:
            p = [x.strip() for x in line.split(",")]
            try:
                self.max_mhz = float(p[1])
                rs = {n for n, v in zip(self.NAMES, p[3:7]) if v.lower().startswith("active")}
                self.samples.append((time.time(), float(p[0]), rs, float(p[2])))
            except Exception:
                continue

    def stop(self, t0: float, t1: float) -> dict:
        if self.thread is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["clock sampling unavailable"]}
        time.sleep(0.06)
        self._stop.set()
        if self.proc is not None:
            self.proc.terminate()
        rows = [s for s in self.samples if t0 <= s[0] <= t1] or [s for s in self.samples if t0 - 0.1 <= s[0] <= t1 + 0.1]
        sm = [r[1] for r in rows]
        reasons = set().union(*[r[2] for r in rows]) if rows else set()
        pw = [r[3] for r in rows if r[3] is not None]
        return {"sm_mhz": statistics.median(sm) if sm else None, "sm_min_mhz": min(sm) if sm else None,
                "sm_max_mhz": self.max_mhz, "reasons": sorted(reasons), "samples": len(rows),
                "power_w_max": max(pw) if pw else None, "source": "nvml" if self.nvml else "nvidia-smi"}


def apply_options(plan, args, binding):
    if args.quantum:
        plan.set_quantum(args.quantum)
    plan.set_option(binding.OPT_UNROLL, args.unroll)
    plan.set_option(binding.OPT_BLOCK_THREADS, args.block_threads)
    plan.set_option(binding.OPT_BLOCKS_PER_SM, args.blocks_per_sm)
    plan.set_option(binding.OPT_MODE, args.mode)
    if args.pdl >= 0:
        plan.set_option(binding.OPT_PDL, args.pdl)
    plan.set_option(binding.OPT_HOST_CHUNKS, args.host_chunks)
    plan.set_option(binding.OPT_HOST_DIRECT_OUT, args.host_direct_out)
    plan.set_option(binding.OPT_VEC_BYTES, args.vec_bytes)


def workload_config(args):
    from paper_2606_21101_b200 import workloads as W
    cfg = W.CONFIGS[args.workload]
    rows = cfg.table_rows()
    if args.rows_scale != 1.0:
        rows = np.maximum(1, (rows * args.rows_scale).astype(np.int64))
    return cfg, rows


def describe(cfg, rows, extra=None, R=R_BATCHES):
    d = {"workload": f"{cfg.name} (BASELINE.json configs[{int(cfg.name[1]) - 1}])", "tables": cfg.T,
         "rows_total": int(rows.sum()), "D": cfg.D, "table_dtype": cfg.dtype, "batch": cfg.B,
         "bag_lengths": list(cfg.lengths), "indices": list(cfg.index_dist), "pooling": cfg.pooling,
         "rotating_batches": R,
         "l2": "inputs larger than L2 (no flush)" if cfg.name in ("c4", "c5") else "warm L2 (working set < L2)"}
    if extra:
        d.update(extra)
    return d


# ----------------------------------------------------------------------------------------------------
# CPU oracle legs
# ----------------------------------------------------------------------------------------------------
def synth_library():
    """libdpi_synth.so (seeded table generator on the device) by path, or None when it has not been built."""
    import ctypes
    path = os.path.join(os.path.dirname(os.path.abspath(__file__)), "paper_2606_21101_b200", "lib", "libdpi_synth.so")
    if not os.path.exists(path):
        return None
    lib = ctypes.CDLL(path)
    lib.dpi_synth_fill_table.restype = ctypes.c_int
    lib.dpi_synth_fill_table.argtypes = [ctypes.c_void_p, ctypes.c_uint64, ctypes.c_int, ctypes.c_uint64, ctypes.c_void_p]
    return lib


def host_mirror(cfg, rows, budget_bytes):
    """Host copy of the tables for the CPU legs: the full tables when they fit the budget (c1-c4), else
    a ROW-SCALED mirror -- the first rows_s[t] rows of every table, indices taken modulo rows_s[t] (c5: 82 GB do not fit a
    host). With a CUDA device the values are copied D2H from tables filled by the same device generator the GPU arm reads
    (bit-identical to the host generator, tests/test_gpu_parity.py::test_synth_fill_matches_host_generator); without one
    they are generated on the host under a smaller budget. Returns (tables, rows_s, scaled?)."""
    from paper_2606_21101_b200 import workloads as W
    total = int(rows.sum()) * cfg.row_bytes
    try:
        import torch
        cuda = torch.cuda.is_available()
    except Exception:
        cuda = False
    synth = synth_library() if cuda else None
    if synth is None:   # tables generated on the host: keep that bounded
        budget_bytes = min(budget_bytes, 1 << 30)
    scale = min(1.0, budget_bytes / max(total, 1))
    rows_s = np.maximum(1, np.floor(rows * scale)).astype(np.int64) if scale < 1.0 else rows.copy()
    tables = []
    if synth is not None:
        # the seeded generator's device restatement (libdpi_synth.so: no method arithmetic), loaded directly -- this leg touches
        # neither the product's binding nor libdpi.so; if the helper library has not been built the host generator is used
        import torch
        tdt = {"f32": torch.float32, "f16": torch.float16, "bf16": torch.bfloat16}[cfg.dtype]
        for t in range(cfg.T):
            buf = torch.empty((int(rows_s[t]), cfg.D), dtype=tdt, device="cuda")
            rc = synth.dpi_synth_fill_table(buf.data_ptr(), buf.numel(), W.DTYPE_CODE[cfg.dtype], W.value_key(cfg.seed, t),
                                            torch.cuda.current_stream().cuda_stream)
            if rc != 0:
                raise SystemExit(f"bench.py: dpi_synth_fill_table failed with cudaError {rc}")
            h = buf.cpu()
            tables.append(h.view(torch.int16).numpy().view(np.uint16) if cfg.dtype == "bf16" else h.numpy())
            del buf
        torch.cuda.empty_cache()
    else:
        tables = [W.full_table_storage(cfg, t, int(rows_s[t])) for t in range(cfg.T)]
    return tables, rows_s, scale < 1.0


def time_oracle(cfg, rows, target_seconds, steps=None, warmup=0):
    """The oracle as it stands on the host cores: plan (a1 + a2) + lookup (a3) on a bounded sample of batch 0 -- the first
    n samples, n chosen so that the two legs together take about target_seconds -- against a host mirror of the tables
    (row-scaled when the tables do not fit: c5). Two legs on the same sample: one thread (oracle_lookup) and all visible cores
    (oracle_lookup_par, OpenMP over samples), asserted bit-identical."""
    import oracle
    from paper_2606_21101_b200 import workloads as W
    oracle.build()
    try:
        avail = int(next(l for l in open("/proc/meminfo") if l.startswith("MemAvailable")).split()[1]) * 1024
    except Exception:
        avail = 8 << 30
    tables, rows_s, scaled = host_mirror(cfg, rows, min(avail // 4, 16 << 30))
    pooling = cfg.pooling_modes()
    K = 32
    code = W.DTYPE_CODE[cfg.dtype]

    def sample(n):
        sub_cfg = cfg.scaled(B=n)
        b = W.make_batch(sub_cfg, rows, cfg.seed)      # the first n samples of batch 0 (counter-based draws)
        idx = b.indices
        if scaled:
            tab = (np.repeat(np.arange(sub_cfg.G, dtype=np.int64), b.lengths) % cfg.T)
            idx = (idx.astype(np.int64) % rows_s[tab]).astype(np.int32)
        return b.lengths, idx

    def one_step(n, ln, idx, par, out=None):
        off, _, _ = oracle.plan(ln, K)
        if par:
            return oracle.lookup_par(tables, code, n, idx, off, pooling, out=out)
        return oracle.lookup(tables, code, n, idx, off, pooling, out=out), 1

    # probe on 256 samples, then size the sample for ~ target_seconds / 4 per single-thread step
    n0 = min(cfg.B, 256)
    ln, idx = sample(n0)
    t = time.perf_counter()
    one_step(n0, ln, idx, False)
    per_sample = max((time.perf_counter() - t) / n0, 1e-7)
    n = int(min(cfg.B, max(n0, (target_seconds / 4) / per_sample)))
    ln, idx = sample(n)
    ref1, _ = one_step(n, ln, idx, False)
    refp, team = one_step(n, ln, idx, True)
    assert np.array_equal(ref1.view(np.uint64), refp.view(np.uint64)), "all-cores oracle leg differs from the single-thread oracle"
    del refp
    block = ref1   # the timed steps write into one already-touched block (first-touch page faults are not the oracle)
    legs = {}
    for name, par in (("single_thread", False), ("all_cores", True)):
        for _ in range(warmup):
            one_step(n, ln, idx, par, block)
        t = time.perf_counter()
        one_step(n, ln, idx, par, block)
        first = time.perf_counter() - t
        k = steps if steps is not None else max(1, int((target_seconds / 2) / max(first, 1e-4)))
        t = time.perf_counter()
        for _ in range(k):
            one_step(n, ln, idx, par, block)
        dt = time.perf_counter() - t
        legs[name] = {"value": n * cfg.T * k / dt, "unit": UNIT, "cores": team if par else 1, "seconds": dt, "steps": k,
                      "ms_per_step": dt / k * 1e3}
    mirror = (f"row-scaled host mirror ({int(rows_s.sum())} of {int(rows.sum())} rows, indices modulo the reduced heights)" if scaled
              else "full host mirror of the tables")
    what = (f"first {n} of {cfg.B} samples of batch 0 ({n * cfg.T} bags, {int(idx.size)} rows gathered), {mirror}; "
            f"oracle plan + lookup per step")
    main = legs["all_cores"]
    return {"value": main["value"], "unit": UNIT, "cores": main["cores"], "kind": "oracle",
            "sample": f"{what}; all-cores leg (OpenMP over samples, bit-identical to the single-thread oracle): {main['steps']} steps, {main['seconds']:.1f} s",
            "single_thread": {"value": legs["single_thread"]["value"], "unit": UNIT, "cores": 1,
                              "steps": legs["single_thread"]["steps"], "seconds": legs["single_thread"]["seconds"]},
            "host_cpus_visible": len(os.sched_getaffinity(0)), "tables_row_scaled": scaled,
            "seconds": main["seconds"], "ms_per_step": main["ms_per_step"], "steps": main["steps"]}


def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    cfg, rows = workload_config(args)
    r = time_oracle(cfg, rows, args.cpu_seconds, steps=args.steps, warmup=min(args.warmup or 0, 1))
    line = {"impl": "reference", "metric": METRIC, "value": r["value"], "unit": UNIT, "n_gpus": args.gpus,
            "steps": r["steps"], "warmup": min(args.warmup or 0, 1), "ms_per_step": r["ms_per_step"],
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": describe(cfg, rows),
            "cpu_baseline": {k: r[k] for k in ("value", "unit", "cores", "kind", "sample", "single_thread", "host_cpus_visible", "tables_row_scaled")},
            "e2e": {"value": r["value"], "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line), flush=True)


# ----------------------------------------------------------------------------------------------------
# CUDA path
# ----------------------------------------------------------------------------------------------------
def link_floor(h2d_bytes: int, d2h_bytes: int, device: str, reps: int = 5) -> dict:
    """Host-link ceiling for one e2e step, measured in this run: pinned-memory cudaMemcpyAsync of exactly the step's byte
    counts -- H2D alone, D2H alone, and both at once on two streams (one copy per direction). The floor of an e2e step is
    the concurrent figure: no schedule can beat both directions streaming flat out."""
    import torch
    hi = torch.empty(max(h2d_bytes, 1), dtype=torch.uint8).pin_memory()
    ho = torch.empty(max(d2h_bytes, 1), dtype=torch.uint8).pin_memory()
    di = torch.empty(max(h2d_bytes, 1), dtype=torch.uint8, device=device)
    do = torch.empty(max(d2h_bytes, 1), dtype=torch.uint8, device=device)
    s1, s2 = torch.cuda.Stream(), torch.cuda.Stream()

    def run(h2d, d2h):
        best = None
        for _ in range(reps + 1):
            torch.cuda.synchronize()
            a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            j = torch.cuda.Event()
            a.record(s1)
            s2.wait_event(a)
            if h2d:
                with torch.cuda.stream(s1):
                    di.copy_(hi, non_blocking=True)
            if d2h:
                with torch.cuda.stream(s2):
                    ho.copy_(do, non_blocking=True)
            j.record(s2)
            s1.wait_event(j)
            b.record(s1)
            torch.cuda.synchronize()
            t = a.elapsed_time(b)
            best = t if best is None else min(best, t)
        return best

    h, d, both = run(True, False), run(False, True), run(True, True)
    return {"h2d_ms": h, "d2h_ms": d, "both_ms": both, "h2d_gbs": h2d_bytes / h / 1e6, "d2h_gbs": d2h_bytes / d / 1e6,
            "both_gbs": (h2d_bytes + d2h_bytes) / both / 1e6}


def unique_rows(batch, T):
    """Distinct (table, row) pairs one batch gathers: the entries of table t are those of bags g = b*T + t (sample-major)."""
    lengths = np.asarray(batch.lengths, dtype=np.int64)
    table_of_entry = np.repeat(np.tile(np.arange(T, dtype=np.int64), lengths.size // T), lengths)
    idx = np.asarray(batch.indices, dtype=np.int64)
    return int(np.unique(table_of_entry * (1 << 32) + idx).size) if idx.size else 0


def spawn_ranks(args):
    """`python bench.py --gpus N` without torchrun: start the N ranks ourselves (one process per GPU, rendezvous on 127.0.0.1)
    and pass their output through; rank 0 prints the one JSON line."""
    import socket
    import subprocess
    if args.impl != "reference":
        import torch
        have = torch.cuda.device_count() if torch.cuda.is_available() else 0
        if have < args.gpus:
            raise SystemExit(f"bench.py: --gpus {args.gpus} but only {have} CUDA device(s) visible; refusing to report n_gpus={args.gpus}")
    with socket.socket() as sk:
        sk.bind(("127.0.0.1", 0))
        port = sk.getsockname()[1]
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", f"--nproc-per-node={args.gpus}", "--master-addr", "127.0.0.1",
           "--master-port", str(port), os.path.abspath(__file__)] + sys.argv[1:]
    raise SystemExit(subprocess.call(cmd))


def run_ours(args):
    import torch
    from paper_2606_21101_b200 import binding, build, harness, sharding, workloads as W

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
    device = f"cuda:{local}"

    cfg, rows = workload_config(args)
    small = cfg.name in ("c1", "c2", "c3")
    warmup = max(args.warmup if args.warmup is not None else 5, 3)
    steps = max(args.steps if args.steps is not None else (2000 if small else 200), 1)
    use_graph = small if args.graph < 0 else bool(args.graph)
    R = max(1, args.rotating_batches)

    # every rank: all tables + its own shard of each global batch of world*B samples (batch-sharded replicas,
    # no collective on the data path)
    dt = harness.make_device_tables(cfg, rows, device=device)
    batches = [harness.upload_batch(sharding.make_batch_shard(cfg, rows, cfg.seed + r, rank, world), device=device)
               for r in range(R)]
    pooling = cfg.pooling_modes()
    plan = harness.make_plan(cfg, rows, harness.max_indices_bound(cfg), bag_hint=bool(args.bag_hint))   # default: no promise, the device picks
    apply_options(plan, args, binding)
    if args.fused >= 0:
        plan.set_option(binding.OPT_FUSED, args.fused)
    out = harness.new_output(cfg, device=device)
    stream = torch.cuda.Stream()  # a non-default stream: every launch and every event of the timed region is on it

    ablation = args.kernel == "input_first"

    def step(i, s):
        b = batches[i % R]
        if ablation:
            plan.build(b.lengths, s)
            plan.lookup_input_first(dt.ptrs, b.indices, out, pooling=pooling, stream=s)
        else:   # the public one-call path: ONE fused launch (a1+a2+a3) when eligible, else planner + lookup
            plan.forward(b.lengths, dt.ptrs, b.indices, out, pooling=pooling, stream=s)

    def barrier():
        if dist is not None:
            dist.barrier()
        torch.cuda.synchronize()

    def max_ms(ms):
        return sharding.max_over_ranks(ms, dist, device=device)

    with torch.cuda.stream(stream):
        n0 = binding.launch_count()
        step(0, stream)
        launches_per_step = binding.launch_count() - n0
        for i in range(1, warmup):
            step(i, stream)
    barrier()
    fused = (not ablation) and launches_per_step == 1

    graph = None
    if use_graph:  # capture the K steps once; the timed region replays them with no host work in between
        graph = torch.cuda.CUDAGraph()
        with torch.cuda.graph(graph, stream=stream):
            for i in range(steps):
                step(i, torch.cuda.current_stream())
        graph.replay()  # one untimed replay (instantiation / upload)
        barrier()

    # ---- timed region: K steps, CUDA events on the launching stream --------------------------------------
    sampler = ClockSampler(local)
    if rank == 0:
        sampler.start()
        time.sleep(0.05)
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    launches0 = binding.launch_count()
    barrier()
    t0 = time.time()
    with torch.cuda.stream(stream):
        e0.record(stream)
        if graph is not None:
            graph.replay()
        else:
            for i in range(steps):
                step(i, stream)
        e1.record(stream)
    barrier()
    t1 = time.time()
    launches = launches_per_step * steps if graph is not None else binding.launch_count() - launches0
    total_ms = max_ms(e0.elapsed_time(e1))
    clocks = sampler.stop(t0, t1) if rank == 0 else None

    # ---- the dominant kernel alone: per-launch CUDA events, same stream, same batches ---------------------
    # (plain launches here: with programmatic dependent launch the kernel's prologue may start under the previous kernel's
    #  tail, and an event pair would then time more than the kernel itself; the timed steps above keep the library default).
    # Fused path: the ONE kernel of the step (a1+a2+a3). Otherwise: the lookup kernel (a3) behind an untimed planner launch.
    n_k = min(steps, 200)
    ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(n_k)]
    pdl_was = plan.get_option(binding.OPT_PDL)
    plan.set_option(binding.OPT_PDL, 0)
    with torch.cuda.stream(stream):
        for i in range(n_k):
            b = batches[i % R]
            if fused:
                ev[i][0].record(stream)
                plan.forward(b.lengths, dt.ptrs, b.indices, out, pooling=pooling, stream=stream)
                ev[i][1].record(stream)
            else:
                plan.build(b.lengths, stream)
                ev[i][0].record(stream)
                if ablation:
                    plan.lookup_input_first(dt.ptrs, b.indices, out, pooling=pooling, stream=stream)
                else:
                    plan.lookup(dt.ptrs, b.indices, out, pooling=pooling, stream=stream)
                ev[i][1].record(stream)
    barrier()
    kernel_ms = [a.elapsed_time(b) for a, b in ev]
    kernel_ms_source = "CUDA-event pair around each of %d plain stream launches" % n_k
    plain_graph_ms = None
    if graph is not None:
        # A microsecond-scale kernel cannot be timed by an event pair around ONE stream launch: the pair measures launch
        # latency (round 2 printed kernel times longer than the graph-replayed step that contains the kernel). For the
        # graph-launched configs the kernel time is taken from graph replays instead: the step itself when it is ONE launch,
        # else the step minus a graph of the planner launches alone. A graph of back-to-back PLAIN launches (PDL off, no overlap
        # between consecutive kernels) is reported beside it.
        def graph_ms(body):
            g = torch.cuda.CUDAGraph()
            with torch.cuda.graph(g, stream=stream):
                for i in range(n_k):
                    body(batches[i % R], torch.cuda.current_stream())
            g.replay()
            barrier()
            best = None
            for _ in range(3):
                a_, b2 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                with torch.cuda.stream(stream):
                    a_.record(stream)
                    g.replay()
                    b2.record(stream)
                barrier()
                t = a_.elapsed_time(b2) / n_k
                best = t if best is None else min(best, t)
            return best

        def whole(b, s_):
            if ablation:
                plan.build(b.lengths, s_)
                plan.lookup_input_first(dt.ptrs, b.indices, out, pooling=pooling, stream=s_)
            else:
                plan.forward(b.lengths, dt.ptrs, b.indices, out, pooling=pooling, stream=s_)

        plain_graph_ms = graph_ms(whole)          # PDL off: consecutive kernels do not overlap
        plan.set_option(binding.OPT_PDL, pdl_was)
        step_graph_ms = total_ms / steps
        if fused:
            # one launch per step: the kernel IS the graph-replayed step (with PDL on, as timed, consecutive launches overlap by
            # their prologue, so the step can be a little shorter than a plain back-to-back launch)
            kernel_ms = [step_graph_ms]
            kernel_ms_source = "the graph-replayed step itself (one launch per step, library-default PDL)"
        else:
            kernel_ms = [step_graph_ms - graph_ms(lambda b, s_: plan.build(b.lengths, s_))]
            kernel_ms_source = ("graph-replayed step minus a graph of %d planner launches alone (best of 3 replays, / %d), "
                                "library-default PDL" % (n_k, n_k))
    plan.set_option(binding.OPT_PDL, pdl_was)
    # and the stream-launched step (no graph), for the graph-vs-stream comparison
    s0, s1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    with torch.cuda.stream(stream):
        s0.record(stream)
        for i in range(n_k):
            step(i, stream)
        s1.record(stream)
    barrier()
    stream_step_ms = s0.elapsed_time(s1) / n_k

    # plan facts for the byte counts (after timing)
    Ns, Ss, max_lens = [], [], []
    for b in batches:
        plan.build(b.lengths, stream)
        _, _, S, N = plan.export(stream)
        Ns.append(N)
        Ss.append(S)
        max_lens.append(plan.stats(stream)[1])
    n_mean, s_mean = float(np.mean(Ns)), float(np.mean(Ss))
    bytes_step = W.algorithmic_bytes(cfg, cfg.G, n_mean, s_mean)
    # north_star: "also shown with unique-row bytes" -- distinct (table, row) pairs a batch touches (np.unique per table on the
    # host, after timing, mean over the rotating batches): the row bytes a perfect cache would fetch from HBM
    uniq_rows = float(np.mean([unique_rows(b.host, cfg.T) for b in batches]))

    # ---- end to end through the host-buffer entry point ----------------------------------------------------
    e2e = None
    if not args.no_e2e:
        hb = [(torch.from_numpy(b.host.lengths).pin_memory(), torch.from_numpy(np.ascontiguousarray(b.host.indices)).pin_memory())
              for b in batches[:2]]
        out_host = torch.empty((cfg.B, cfg.T * cfg.D), dtype=harness.TORCH_DTYPE[cfg.out]).pin_memory()
        nb = len(hb)
        for i in range(3):
            plan.forward_host(dt.ptrs, hb[i % nb][0], hb[i % nb][1], out_host, pooling=pooling, stream=stream)
        barrier()
        n_e2e = max(1, args.e2e_steps)
        a, b_ = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        a.record(stream)
        for i in range(n_e2e):
            plan.forward_host(dt.ptrs, hb[i % nb][0], hb[i % nb][1], out_host, pooling=pooling, stream=stream)
        b_.record(stream)
        barrier()
        e2e_ms = max_ms(a.elapsed_time(b_))
        h2d = int(hb[0][0].numel() * 4 + hb[0][1].numel() * 4)
        d2h = int(out_host.numel() * out_host.element_size())
        e2e = {"value": sharding.job_throughput(cfg.G, n_e2e, world, e2e_ms), "unit": UNIT, "h2d_bytes_per_step": h2d,
               "d2h_bytes_per_step": d2h, "ms_per_step": e2e_ms / n_e2e, "steps": n_e2e,
               "api": "dpi_forward_host (pinned host lengths/indices in, [B,T*D] block out, tables resident)",
               "d2h": ("staged device block + cudaMemcpyAsync" if args.host_direct_out == 1 else
                       "fused into the lookup's store: the kernel writes the block straight into the pinned host buffer over PCIe")}
        if rank == 0:   # the host link's own ceiling for exactly these byte counts, measured in this run
            lf = link_floor(h2d, d2h, device)
            e2e["link"] = lf
            e2e["link_floor_ms"] = lf["both_ms"]
            e2e["frac_of_link"] = lf["both_ms"] / (e2e_ms / n_e2e)

    if rank != 0:
        if dist is not None:
            dist.destroy_process_group()
        return

    peak, peak_src = measured_peak()
    k_ms = statistics.mean(kernel_ms)
    if ablation:
        kname, ncu_name, variant = "input_first_kernel (ablation)", "input_first_kernel", "input-first ablation"
    elif fused:
        kname, ncu_name = "fused_forward_kernel (a1 + a2 + a3 in one launch)", "fused_forward_kernel"
        variant = "fused single launch (dpi_forward): chained scan + lane-group-per-bag pooling"
    else:
        short = harness.short_bag_rule(int(max(max_lens)), cfg.G) and args.mode == 0
        kname = "lookup_kernel (a3 fused gather-and-pool" + (", short-bag body picked on the device from a1's max_len)" if short else ")")
        ncu_name = "lookup_kernel"
        variant = "planner + " + ("short-bag body of lookup_kernel (device-picked)" if short else "balanced segments")
        if args.bag_hint and harness.lookup_variant(cfg, args.mode).startswith("short-bag"):
            kname, ncu_name = "direct_kernel (a3, short-bag variant as its own launch, chosen on the host from the promise)", "direct_kernel"
            variant = "planner + direct_kernel (DPI_OPT_MAX_BAG_HINT promise)"
    k_bytes = bytes_step["total"] if fused else bytes_step["lookup"]
    achieved = k_bytes / (k_ms * 1e-3) / 1e9
    # the same launch counted with every distinct row once: algorithmic bytes minus the repeated row reads
    uniq_bytes = k_bytes - (n_mean - uniq_rows) * cfg.row_bytes
    step_ms = total_ms / steps
    if graph is None and k_ms > step_ms:
        # stream-launched microsecond-scale steps (--graph 0 on c1-c3, as the ncu captures run them): an event pair around ONE
        # launch times launch latency; the step, which contains the kernel, is the tighter bound
        kernel_ms_source += "; capped at the stream-launched step (the event pairs read %.2f us: launch latency)" % (k_ms * 1e3)
        k_ms = step_ms
    if k_ms > step_ms * 1.02:
        raise SystemExit(f"bench.py: kernel time {k_ms:.5f} ms exceeds the step it is part of ({step_ms:.5f} ms): the kernel timing is broken")
    traffic, traffic_note = ncu_traffic(cfg.name, ncu_name)
    roofline = {"bound": "hbm", "kernel": kname, "achieved": achieved,
                "peak": peak, "unit": "GB/s", "frac": achieved / peak, "peak_source": peak_src,
                "frac_of_nominal_8000": achieved / 8000.0, "traffic": traffic,
                "algorithmic_bytes_per_launch": k_bytes, "kernel_ms_avg": k_ms,
                "kernel_ms_min": min(kernel_ms), "kernel_ms_median": statistics.median(kernel_ms),
                "kernel_launches_timed": n_k, "kernel_ms_source": kernel_ms_source,
                "kernel_ms_plain_launch_graph": plain_graph_ms,   # graph of back-to-back plain (PDL-off) launches of the step, / launches
                "kernel_share_of_step": k_ms / (step_ms if graph is not None else stream_step_ms),
                "unique_rows_per_launch": uniq_rows, "unique_row_bytes": uniq_bytes,
                "unique_row_gbs": uniq_bytes / (k_ms * 1e-3) / 1e9, "unique_row_frac": uniq_bytes / (k_ms * 1e-3) / 1e9 / peak}
    if traffic_note:
        roofline["traffic_note"] = traffic_note
    cpu = None
    if not args.no_cpu_baseline:
        r = time_oracle(cfg, rows, args.cpu_seconds)
        cpu = {k: r[k] for k in ("value", "unit", "cores", "kind", "sample", "single_thread", "host_cpus_visible", "tables_row_scaled")}

    line = {
        "metric": METRIC, "value": sharding.job_throughput(cfg.G, steps, world, total_ms), "unit": UNIT, "n_gpus": world,
        "steps": steps, "warmup": warmup, "ms_per_step": total_ms / steps, "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None, "dtype": DTYPE_KEY[cfg.dtype], "data": "synthetic",
        "config": describe(cfg, rows, {"parallelism": f"batch-sharded replicas x{world}, no collective",
                                       "launch": "CUDA graph replay of the K steps" if graph is not None else "stream launches",
                                       "api": "dpi_forward" if not ablation else "dpi_plan_build + dpi_lookup_input_first",
                                       "launches_per_step": launches_per_step,
                                       "quantum_K": plan.info()["K"], "max_bag_hint": harness.max_bag_length(cfg) if args.bag_hint else 0,
                                       "max_len_measured_by_a1": int(max(max_lens)),
                                       "lookup_variant": variant, "rows_gathered_per_step": n_mean,
                                       "segments_per_step": s_mean}, R),
        "row_gathers_per_s": n_mean * steps * world / (total_ms * 1e-3),
        "step_algorithmic_gbs": bytes_step["total"] * world / (total_ms / steps * 1e-3) / 1e9,
        "stream_launched_ms_per_step": stream_step_ms,
        "roofline": roofline, "cpu_baseline": cpu, "e2e": e2e, "gpu_launches": int(launches), "clocks": clocks,
        "device": torch.cuda.get_device_name(local), "csrc_hash": csrc_hash(),
    }
    print(json.dumps(line), flush=True)
    if dist is not None:
        dist.destroy_process_group()


def run_table_sharded(args):
    """NEXT-3: every rank holds a SUBSET of the tables and the bags of those tables for the
    whole global batch of cfg.B samples; its fused lookup stores each pooled vector straight into the batch shard of the rank
    that owns the sample (dpi_lookup_ex out_peers_dev over CUDA IPC / NVLink). Strong scaling: the global batch is fixed.
    A step = planner + lookup on every rank + the barrier that makes all shards complete. Ranks may share a device (the
    control plane is then gloo): that exercises the glue, not NVLink."""
    import torch
    import torch.distributed as dist
    from paper_2606_21101_b200 import binding, build, harness, sharding, workloads as W

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    n_dev = torch.cuda.device_count()
    if n_dev == 0:
        raise SystemExit("bench.py: no CUDA device; the DPI lookup has no CPU fallback")
    local = int(os.environ.get("LOCAL_RANK", "0")) % n_dev
    torch.cuda.set_device(local)
    device = f"cuda:{local}"
    shared_device = world > n_dev
    if world > 1:
        if shared_device:
            dist.init_process_group("gloo")
        else:
            dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    if rank == 0:
        build.build()
    if world > 1:
        dist.barrier()
    binding.load_library()
    cfg, rows = workload_config(args)
    warmup = max(args.warmup if args.warmup is not None else 5, 3)
    steps = max(args.steps if args.steps is not None else 50, 1)
    R = max(1, min(args.rotating_batches, 4))
    dims = [cfg.D] * cfg.T
    mean_len = {"const": lambda l: l[1], "uniform": lambda l: (l[1] + l[2]) / 2, "poisson": lambda l: l[1]}[cfg.lengths[0]](cfg.lengths)
    tw = sharding.TableWiseLookup(dims, rows, W.DTYPE_CODE[cfg.dtype], harness.TORCH_DTYPE[cfg.out], cfg.B,
                                  harness.max_indices_bound(cfg), device, cost=[mean_len * cfg.row_bytes] * cfg.T,
                                  out_dtype_code=W.DTYPE_CODE[cfg.out] if cfg.out != cfg.dtype else None)
    mine = tw.mine
    tables = []
    for t in mine:   # this rank's tables only, filled in place with the seeded recipe
        buf = torch.empty((int(rows[t]), cfg.D), dtype=harness.TORCH_DTYPE[cfg.dtype], device=device)
        binding.synth_fill_table(buf, buf.numel(), W.DTYPE_CODE[cfg.dtype], W.value_key(cfg.seed, t))
        tables.append(buf)
    ptrs = torch.tensor([t.data_ptr() for t in tables] or [0], dtype=torch.int64, device=device)
    pooling = cfg.pooling_modes()[mine] if mine else None
    batches = []
    for r in range(R):
        local_b = sharding.table_shard_batch(W.make_batch(cfg, rows, cfg.seed + r), cfg.T, mine)
        batches.append(harness.upload_batch(local_b, device=device))
    stream = torch.cuda.Stream()

    def step(i):
        b = batches[i % R]
        with torch.cuda.stream(stream):
            tw.forward(b.lengths, b.indices, ptrs, pooling=pooling, stream=stream)

    for i in range(warmup):
        step(i)
    sampler = ClockSampler(local)
    if rank == 0:
        sampler.start()
        time.sleep(0.05)
    tw.out.barrier()
    launches0 = binding.launch_count()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    t0 = time.time()
    e0.record(stream)
    for i in range(steps):
        step(i)
    e1.record(stream)
    tw.out.barrier()
    t1 = time.time()
    launches = binding.launch_count() - launches0
    ms = e0.elapsed_time(e1)
    if world > 1:
        allms = [None] * world
        dist.all_gather_object(allms, ms)
        ms = max(allms)
    clocks = sampler.stop(t0, t1) if rank == 0 else None
    n_local = float(np.mean([b.N for b in batches]))
    if rank == 0:
        line = {"metric": METRIC, "value": cfg.G * steps / (ms * 1e-3), "unit": UNIT, "n_gpus": world, "steps": steps, "warmup": warmup,
                "ms_per_step": ms / steps, "higher_is_better": True, "scaling": "strong", "vs_baseline": None,
                "dtype": DTYPE_KEY[cfg.dtype], "data": "synthetic",
                "config": describe(cfg, rows, {"parallelism": f"table-wise sharding x{world}: rank r pools its tables for the whole batch and "
                                               "stores into the batch shard of the sample's owner",
                                               "comm": "peer stores (CUDA IPC mapped blocks), no NCCL on the data path; one control-plane "
                                                       "barrier per step",
                                               "ranks_share_a_device": shared_device, "tables_of_rank0": mine,
                                               "rows_gathered_per_step_rank0": n_local, "launch": "stream launches"}, R),
                "gpu_launches": int(launches), "clocks": clocks, "device": torch.cuda.get_device_name(local),
                "roofline": None, "cpu_baseline": None, "e2e": None,
                "note": "NEXT-3 demonstration mode; the headline bench is the default --shard batch"}
        print(json.dumps(line), flush=True)
    tw.close()
    if world > 1:
        dist.destroy_process_group()


def main():
    args = parse_args()
    if args.gpus > 1 and "WORLD_SIZE" not in os.environ:
        spawn_ranks(args)   # does not return
    if "WORLD_SIZE" in os.environ and int(os.environ["WORLD_SIZE"]) != args.gpus and args.shard != "tables":
        raise SystemExit(f"bench.py: --gpus {args.gpus} disagrees with WORLD_SIZE={os.environ['WORLD_SIZE']}")
    if args.impl == "reference":
        run_reference(args)
    elif args.shard == "tables":
        run_table_sharded(args)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()
