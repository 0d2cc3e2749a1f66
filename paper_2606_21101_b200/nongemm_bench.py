"""Measurements for SURVEY.md 8(f) NEXT-4, one B200:

    python -m paper_2606_21101_b200.nongemm_bench [--out gpurun_out/next4.md]

  1. the fused non-GEMM operators against the HBM roofline: algorithmic bytes / CUDA-event time, inputs rotated over
     buffers that together exceed the 126 MB L2 (so every launch streams from HBM), and once more with a warm L2;
  2. Algorithm 2 (evaluation in V-G/V-H): a DeepFM-shaped pair of modules on an
     X_embed block of c2's shape -- explicit = [FM], implicit = [GEMM, bias+relu] x 3 + [GEMM, bias+sigmoid] -- run
     through dpi_launcher_run with one stream and with two, both as plain stream launches and as CUDA-graph replays.
     The GEMMs are torch.matmul (cuBLAS: plain library GEMMs); everything else is this repo's kernels.
Synthetic seeded inputs only. Prints markdown tables; nothing here is part of bench.py's contract."""
from __future__ import annotations

import argparse
import json
import os
import sys

import numpy as np
import torch

from . import harness, nongemm
from . import workloads as W

TORCH = {"f32": torch.float32, "f16": torch.float16, "bf16": torch.bfloat16}
ELT = {"f32": 4, "f16": 2, "bf16": 2}


def peak_gbs():
    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    try:
        with open(os.path.join(root, "MEASURED_PEAKS.json")) as f:
            return float(json.load(f)["hbm_gbs"]), "MEASURED_PEAKS.json hbm_gbs"
    except Exception:
        return 6650.0, "fallback 6.65 TB/s (B200_PROFILING.md)"


def dense(seed, sub, shape, dtype, scale=0.25):
    x = torch.from_numpy(W.dense_values_f32(seed, sub, shape, scale)).cuda()
    return x.to(TORCH[dtype])


def time_rotating(make_call, n_buffers, launches=24, replays=20, warmup=3):
    """us per launch: `launches` calls (rotating over the buffer sets) are captured into ONE CUDA graph and the graph
    is replayed, so the figure is GPU time per launch -- the Python/ctypes cost of a call (~10 us) would otherwise
    hide every kernel shorter than that. Median and min over `replays` replays."""
    st = torch.cuda.Stream()
    with torch.cuda.stream(st):
        for i in range(warmup):
            make_call(i % n_buffers, st.cuda_stream)
        st.synchronize()
        g = torch.cuda.CUDAGraph()
        with torch.cuda.graph(g, stream=st):
            for i in range(launches):
                make_call(i % n_buffers, st.cuda_stream)
        g.replay()
        st.synchronize()
        evs = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(replays)]
        for a, b in evs:
            a.record(st)
            g.replay()
            b.record(st)
        st.synchronize()
    t = sorted(a.elapsed_time(b) * 1e3 / launches for a, b in evs)
    return t[len(t) // 2], t[0]


def n_rot(bytes_per_set):
    return max(2, int(np.ceil(400e6 / max(bytes_per_set, 1))))  # > 3 x L2 in flight across the rotation


def bench_operators(lines):
    peak, src = peak_gbs()
    lines += ["## 1. Fused non-GEMM operators vs the HBM roofline", "",
              f"Peak = {peak:.1f} GB/s ({src}). `cold` rotates over enough buffers to exceed L2 (every launch streams from HBM); "
              "`warm` re-runs one buffer set (L2-resident when it fits in 126 MB). us = GPU time per launch (24 launches per CUDA graph replay). Algorithmic bytes: FM `B*T*D*elt + 4B`; "
              "cross `4*B*F*elt + 4F`; bias_act `2*B*F*elt + 4F`.", "",
              "| operator | shape | dtype | bytes/launch (MB) | cold us (median) | cold GB/s | frac of peak | warm us | warm GB/s |",
              "|---|---|---|---|---|---|---|---|---|"]
    fm_shapes = [("c2 block", 4096, 26, 16, "f32"), ("c3 block", 16384, 22, 32, "f16"), ("c4 block (f32 out)", 8192, 100, 64, "f32"),
                 ("c5 block", 65536, 8, 64, "f32"), ("4 x c5 block", 262144, 8, 64, "f32")]
    for name, B, T, D, dt in fm_shapes:
        nbytes = B * T * D * ELT[dt] + 4 * B
        R = min(n_rot(nbytes), 64)
        xs = [dense(1, r, (B, T * D), dt) for r in range(R)]
        y = torch.empty((B,), device="cuda")
        call = lambda r, st: nongemm.fm_interaction(xs[r], W.DTYPE_CODE[dt], B, T, D, y=y, stream=st)
        cold, _ = time_rotating(call, R)
        warm, _ = time_rotating(call, 1)
        lines.append(f"| fm_interaction | {name} [{B}, {T}x{D}] | {dt} | {nbytes / 1e6:.2f} | {cold:.2f} | {nbytes / cold / 1e3:.0f} | "
                     f"{nbytes / cold / 1e3 / peak:.3f} | {warm:.2f} | {nbytes / warm / 1e3:.0f} |")
        del xs
    ew_shapes = [(4096, 416, "f32"), (65536, 416, "f32"), (65536, 512, "f32"), (65536, 1024, "bf16"), (262144, 512, "f32")]
    for B, F, dt in ew_shapes:
        per = B * F * ELT[dt]
        R = min(n_rot(4 * per), 32)
        x0 = [dense(2, r, (B, F), dt) for r in range(R)]
        xl = [dense(3, r, (B, F), dt) for r in range(R)]
        u = [dense(4, r, (B, F), dt, 2.0) for r in range(R)]
        out = [torch.empty((B, F), dtype=TORCH[dt], device="cuda") for r in range(R)]
        bias = torch.from_numpy(W.dense_values_f32(5, 0, (F,), 1.0)).cuda()
        nbytes = 4 * per + 4 * F
        call = lambda r, st: nongemm.cross_combine(x0[r], xl[r], u[r], bias, out[r], W.DTYPE_CODE[dt], B, F, stream=st)
        cold, _ = time_rotating(call, R)
        warm, _ = time_rotating(call, 1)
        lines.append(f"| cross_combine | [{B}, {F}] | {dt} | {nbytes / 1e6:.2f} | {cold:.2f} | {nbytes / cold / 1e3:.0f} | "
                     f"{nbytes / cold / 1e3 / peak:.3f} | {warm:.2f} | {nbytes / warm / 1e3:.0f} |")
        nbytes = 2 * per + 4 * F
        for act, an in ((nongemm.ACT_RELU, "relu"), (nongemm.ACT_SIGMOID, "sigmoid")):
            call = lambda r, st, act=act: nongemm.bias_act(u[r], bias, out[r], W.DTYPE_CODE[dt], B, F, act, stream=st)
            cold, _ = time_rotating(call, R)
            warm, _ = time_rotating(call, 1)
            lines.append(f"| bias_act {an} | [{B}, {F}] | {dt} | {nbytes / 1e6:.2f} | {cold:.2f} | {nbytes / cold / 1e3:.0f} | "
                         f"{nbytes / cold / 1e3 / peak:.3f} | {warm:.2f} | {nbytes / warm / 1e3:.0f} |")
        del x0, xl, u, out
    lines.append("")


class TwoModuleModel:
    """Synthetic two-module forward on an X_embed block [B, T*D] (random-init weights):
      deepfm  explicit = [FM over the block];                              implicit = MLP
      dcnv2   explicit = n_cross x [GEMM F->F, cross_combine] (F = T*D);  implicit = MLP
    MLP = [GEMM, bias+relu] per hidden layer + [GEMM -> 8, bias+sigmoid] (8 outputs keep rows 16-byte aligned)."""

    def __init__(self, kind, B, T=26, D=16, hidden=(1024, 512, 256), dtype="f32", n_cross=3):
        td, code, F = TORCH[dtype], W.DTYPE_CODE[dtype], T * D
        self.x = dense(7, 0, (B, F), dtype)
        dims = [F, *hidden, 8]
        self.w = [dense(8, i, (dims[i], dims[i + 1]), dtype, 1.0 / np.sqrt(dims[i])) for i in range(len(dims) - 1)]
        self.b = [torch.from_numpy(W.dense_values_f32(9, i, (dims[i + 1],), 0.1)).cuda() for i in range(len(dims) - 1)]
        self.h = [torch.empty((B, dims[i + 1]), dtype=td, device="cuda") for i in range(len(dims) - 1)]

        def gemm(src, w, dst):
            def launch(s):
                with torch.cuda.stream(torch.cuda.ExternalStream(s)):
                    torch.matmul(src, w, out=dst)
            return launch

        self.implicit = []
        for i in range(len(self.w)):
            a = nongemm.ACT_SIGMOID if i == len(self.w) - 1 else nongemm.ACT_RELU
            self.implicit.append(gemm(self.x if i == 0 else self.h[i - 1], self.w[i], self.h[i]))
            self.implicit.append(lambda s, i=i, a=a: nongemm.bias_act(self.h[i], self.b[i], self.h[i], code, B, dims[i + 1], a, stream=s))
        if kind == "deepfm":
            self.y_fm = torch.empty((B,), device="cuda")
            self.explicit = [lambda s: nongemm.fm_interaction(self.x, code, B, T, D, y=self.y_fm, stream=s)]
        else:
            self.cw = [dense(10, i, (F, F), dtype, 1.0 / np.sqrt(F)) for i in range(n_cross)]
            self.cb = [torch.from_numpy(W.dense_values_f32(11, i, (F,), 0.1)).cuda() for i in range(n_cross)]
            self.u = torch.empty((B, F), dtype=td, device="cuda")
            self.xl = [torch.empty((B, F), dtype=td, device="cuda") for _ in range(2)]
            self.explicit = []
            for i in range(n_cross):
                src = self.x if i == 0 else self.xl[(i - 1) % 2]
                self.explicit.append(gemm(src, self.cw[i], self.u))
                self.explicit.append(lambda s, i=i, src=src: nongemm.cross_combine(self.x, src, self.u, self.cb[i], self.xl[i % 2],
                                                                                    code, B, F, stream=s))


def time_forward(run, main, n=200):
    t = []
    for _ in range(n):
        a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        a.record(main)
        run()
        b.record(main)
        t.append((a, b))
    main.synchronize()
    return sorted(x.elapsed_time(y) * 1e3 for x, y in t)[n // 2]


def bench_launcher(lines):
    lines += ["## 2. Algorithm 2: one stream vs two streams (two-module forwards on a c2-shaped block, T = 26, D = 16)", "",
              "deepfm: explicit = [fm_interaction], implicit = MLP 416-1024-512-256-8 as [GEMM, bias+relu] x 3 + [GEMM, bias+sigmoid]. "
              "dcnv2: explicit = 3 x [GEMM 416->416, cross_combine], same MLP. GEMMs = torch.matmul (cuBLAS); non-GEMM operators = "
              "this repo. Launch order from `dpi_bfs_schedule` (the module with more operators first, PAPER.md:247). us per forward "
              "of the two modules, median of 200. `stream` = `dpi_launcher_run` launching live (each operator is a Python callback "
              "here, so small batches measure the host); `graph` = the same call captured once into a CUDA graph and replayed.", "",
              "| model | dtype | batch | stream, 1 stream | stream, 2 streams | graph, 1 stream | graph, 2 streams | 2-stream speed-up (graph) |",
              "|---|---|---|---|---|---|---|---|"]
    L = nongemm.Launcher()
    main = torch.cuda.Stream()
    for kind, dtype in (("deepfm", "f32"), ("deepfm", "bf16"), ("dcnv2", "f32"), ("dcnv2", "bf16")):
        for B in (512, 4096, 16384, 65536):
            m = TwoModuleModel(kind, B, dtype=dtype)
            res = {}
            with torch.cuda.stream(main):
                for ns in (1, 2):
                    run = lambda: L.run(m.explicit, m.implicit, n_streams=ns, stream=main)
                    for _ in range(5):
                        run()
                    main.synchronize()
                    res[("stream", ns)] = time_forward(run, main)
                    g = torch.cuda.CUDAGraph()
                    with torch.cuda.graph(g, stream=main):
                        run()
                    for _ in range(5):
                        g.replay()
                    main.synchronize()
                    res[("graph", ns)] = time_forward(g.replay, main)
                    del g
            lines.append(f"| {kind} | {dtype} | {B} | {res[('stream', 1)]:.1f} | {res[('stream', 2)]:.1f} | {res[('graph', 1)]:.1f} | "
                         f"{res[('graph', 2)]:.1f} | {res[('graph', 1)] / res[('graph', 2)]:.2f}x |")
            del m
    L.destroy()
    lines.append("")


def bench_forward_fm(lines):
    """dpi_forward_fm (lookup + FM term, ONE launch on the small configs) against the chain dpi_forward -> dpi_fm_interaction
    (two launches) and planner + lookup + FM (three): GPU time per step from graph replays over rotating batches."""
    from . import binding
    lines += ["## dpi_forward_fm: the lookup and its first non-GEMM consumer as one operator (PAPER.md:188)", "",
              "GPU time per step (us), CUDA-graph replays of 24 steps over 8 rotating batches, median (min).", "",
              "| workload | forward_fm (1 launch) | forward + fm (2 launches) | plan + lookup + fm (3 launches) |", "|---|---|---|---|"]
    for name in ("c1", "c2", "c3"):
        cfg = W.CONFIGS[name]
        rows = cfg.table_rows()
        dt = harness.make_device_tables(cfg, rows)
        batches = [harness.upload_batch(W.make_batch(cfg, rows, cfg.seed + r)) for r in range(8)]
        pooling = cfg.pooling_modes()
        plan = harness.make_plan(cfg, rows, harness.max_indices_bound(cfg))
        out = harness.new_output(cfg)
        y = torch.zeros(cfg.B, device="cuda")
        code = W.DTYPE_CODE[cfg.out]

        def one(i, s):
            b = batches[i]
            nongemm.forward_fm(plan, b.lengths, dt.ptrs, b.indices, out, y=y, pooling=pooling, stream=s)

        def two(i, s):
            b = batches[i]
            plan.forward(b.lengths, dt.ptrs, b.indices, out, pooling=pooling, stream=s)
            nongemm.fm_interaction(out, code, cfg.B, cfg.T, cfg.D, y=y, stream=s)

        def three(i, s):
            b = batches[i]
            plan.build(b.lengths, s)
            plan.lookup(dt.ptrs, b.indices, out, pooling=pooling, stream=s)
            nongemm.fm_interaction(out, code, cfg.B, cfg.T, cfg.D, y=y, stream=s)

        res = [time_rotating(f, 8) for f in (one, two, three)]
        lines.append(f"| {name} | " + " | ".join(f"{m:.2f} ({lo:.2f})" for m, lo in res) + " |")
        plan.destroy()
        del dt, batches
        torch.cuda.empty_cache()
    lines.append("")


def profile_pass():
    """Three plain launches of each operator at a 65 536-row shape (no graphs, no timing): the target of an
    `ncu --set full -k regex:"fm_kernel|cross_combine|bias_act"` capture."""
    B, T, D, F = 65536, 8, 64, 512
    x = [dense(1, r, (B, T * D), "f32") for r in range(3)]
    y = torch.empty((B,), device="cuda")
    x0, xl, u = (dense(2 + i, 0, (B, F), "f32") for i in range(3))
    out = torch.empty((B, F), device="cuda")
    bias = torch.from_numpy(W.dense_values_f32(5, 0, (F,), 1.0)).cuda()
    for r in range(3):
        nongemm.fm_interaction(x[r], 0, B, T, D, y=y)
    for r in range(3):
        nongemm.cross_combine(x0, xl, u, bias, out, 0, B, F)
    for r in range(3):
        nongemm.bias_act(u, bias, out, 0, B, F, nongemm.ACT_RELU)
    for r in range(3):
        nongemm.bias_act(u, bias, out, 0, B, F, nongemm.ACT_SIGMOID)
    torch.cuda.synchronize()
    print("profile pass done: 3 launches each of fm_kernel, cross_combine_kernel, bias_act_kernel (relu, sigmoid)")


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--out", default="")
    ap.add_argument("--skip-launcher", action="store_true")
    ap.add_argument("--profile", action="store_true", help="only launch each operator three times (for ncu)")
    ap.add_argument("--forward-fm", action="store_true", help="only the dpi_forward_fm comparison")
    args = ap.parse_args()
    harness.require_cuda()
    torch.cuda.set_device(0)
    if args.profile:
        return profile_pass()
    lines = ["# NEXT-4 measurements (python -m paper_2606_21101_b200.nongemm_bench)", "",
             f"Device: {torch.cuda.get_device_name(0)}. CUDA events on the launching stream, after warm-up. Synthetic seeded inputs.", ""]
    if args.forward_fm:
        bench_forward_fm(lines)
    else:
        bench_operators(lines)
        bench_forward_fm(lines)
        if not args.skip_launcher:
            bench_launcher(lines)
    text = "\n".join(lines)
    print(text)
    if args.out:
        os.makedirs(os.path.dirname(os.path.abspath(args.out)), exist_ok=True)
        with open(args.out, "w") as f:
            f.write(text + "\n")


if __name__ == "__main__":
    sys.exit(main())
