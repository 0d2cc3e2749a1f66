"""Scenario sweeps of the paper's Fig. 10 / Fig. 11 on synthetic Criteo-shaped one-hot input.

    python -m paper_2606_21101_b200.sweeps [--only fig10_batch,fig11_dim] [--out gpurun_out/sweeps.md]
    python -m paper_2606_21101_b200.sweeps --only forward_crossover [--out ...]   # one launch vs two, over batch size

The paper varies four things around the embedding stage (§V-F): batch size (D = 32),
embedding dimension (B = 2048), number of feature fields (B = 2048, D = 32, 5e5 features per field) and
number of features per field (B = 2048, D = 32, 50 fields), and in Fig. 11 compares its
output-first workload allocation with the input-first strawman over batch size and embedding dimension
("when the batch size is 65,536 and when the embedding dimension is 60 ... 10.3x and 9.2x").
The paper runs them on Criteo through its comparison frameworks; here every point is a seeded synthetic
one-hot workload with c2's recipe (26 fields, heights log-uniform in [10, 1e6], Zipf 1.05, fp32) unless
the sweep fixes the shape itself. Three timings per point, CUDA events on one stream, after warm-up:

* ``output_first``  dpi_lookup (the product kernel), per launch, and plan + lookup as a replayed CUDA graph
* ``alg1_direct``   dpi_lookup_onehot: Algorithm 1 as one plan-free launch (the workload is one-hot, so the plan is pure
                    arithmetic), per launch and as a replayed CUDA graph
* ``input_first``   dpi_lookup_input_first (the ablation kernel, same plan, same results bit for bit)
* ``per_table``     context only: one ``torch.nn.functional.embedding`` launch per table and a ``torch.cat``
                    -- the k-serial-lookups-plus-concat structure the paper starts from,
                    NOT one of the paper's comparison systems and not a target.

Plumbing only: no arithmetic of the method lives here.
"""
from __future__ import annotations

import argparse
import json
import os
import statistics
import sys
from typing import Dict, List

import numpy as np


def _time_calls(fn, stream, n: int, warmup: int = 5) -> Dict[str, float]:
    """Per-call device time of fn() on `stream` (CUDA events around every call)."""
    import torch
    with torch.cuda.stream(stream):
        for _ in range(warmup):
            fn()
    torch.cuda.synchronize()
    ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(n)]
    with torch.cuda.stream(stream):
        for a, b in ev:
            a.record(stream)
            fn()
            b.record(stream)
    torch.cuda.synchronize()
    ms = [a.elapsed_time(b) for a, b in ev]
    return {"avg_us": 1e3 * statistics.mean(ms), "min_us": 1e3 * min(ms), "med_us": 1e3 * statistics.median(ms)}


def _time_graph(step, stream, n: int) -> float:
    """us per step of n steps captured once in a CUDA graph and replayed."""
    import torch
    g = torch.cuda.CUDAGraph()
    with torch.cuda.graph(g, stream=stream):
        for i in range(n):
            step(i, torch.cuda.current_stream())
    g.replay()
    torch.cuda.synchronize()
    a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    with torch.cuda.stream(stream):
        a.record(stream)
        g.replay()
        b.record(stream)
    torch.cuda.synchronize()
    return 1e3 * a.elapsed_time(b) / n


def run_point(cfg, n_iter: int = 200, rotating: int = 4, with_torch: bool = True) -> dict:
    import torch
    import torch.nn.functional as F
    from . import harness, workloads as W

    rows = cfg.table_rows()
    dt = harness.make_device_tables(cfg, rows)
    batches = [harness.upload_batch(W.make_batch(cfg, rows, cfg.seed + r)) for r in range(rotating)]
    plan = harness.make_plan(cfg, rows, harness.max_indices_bound(cfg))
    out = harness.new_output(cfg)
    pooling = cfg.pooling_modes()
    stream = torch.cuda.Stream()
    k = [0]

    def nxt():
        k[0] += 1
        return batches[k[0] % rotating]

    plan.build(batches[0].lengths, stream)
    res = {"T": cfg.T, "B": cfg.B, "D": cfg.D, "rows_total": int(rows.sum()), "K": plan.info()["K"]}
    res["output_first"] = _time_calls(lambda: plan.lookup(dt.ptrs, nxt().indices, out, pooling=pooling, stream=stream), stream, n_iter)
    res["input_first"] = _time_calls(lambda: plan.lookup_input_first(dt.ptrs, nxt().indices, out, pooling=pooling, stream=stream),
                                     stream, max(20, n_iter // 4))

    res["alg1_direct"] = _time_calls(lambda: plan.lookup_onehot(dt.ptrs, nxt().indices, out, stream=stream), stream, n_iter)
    res["alg1_direct_graph_us"] = _time_graph(lambda i, s: plan.lookup_onehot(dt.ptrs, batches[i % rotating].indices, out, stream=s),
                                              stream, n_iter)
    res["lookup_graph_us"] = _time_graph(lambda i, s: plan.lookup(dt.ptrs, batches[i % rotating].indices, out, pooling=pooling, stream=s),
                                         stream, n_iter)

    def step(i, s):
        b = batches[i % rotating]
        plan.build(b.lengths, s)
        plan.lookup(dt.ptrs, b.indices, out, pooling=pooling, stream=s)

    res["plan_plus_lookup_graph_us"] = _time_graph(step, stream, n_iter)

    def stream_step():
        k[0] += 1
        step(k[0], stream)

    res["plan_plus_lookup_stream"] = _time_calls(stream_step, stream, n_iter)

    if with_torch:
        # context: k serial per-table lookups + concat, ids as the int64 [B, T] matrix frameworks feed
        ids = [torch.from_numpy(b.host.indices.reshape(cfg.B, cfg.T).astype(np.int64)).cuda() for b in batches]

        def per_table():
            x = ids[k[0] % rotating]
            k[0] += 1
            return torch.cat([F.embedding(x[:, t], dt.tables[t]) for t in range(cfg.T)], dim=1)

        res["per_table"] = _time_calls(per_table, stream, max(20, n_iter // 4))
        with torch.cuda.stream(stream):
            ref = torch.cat([F.embedding(ids[0][:, t], dt.tables[t]) for t in range(cfg.T)], dim=1)
            plan.build(batches[0].lengths, stream)
            plan.lookup(dt.ptrs, batches[0].indices, out, pooling=pooling, stream=stream)
        torch.cuda.synchronize()
        res["equals_per_table_result"] = bool(torch.equal(ref, out))
    bytes_lookup = W.algorithmic_bytes(cfg, cfg.G, cfg.G)["lookup"]
    res["algorithmic_MB"] = bytes_lookup / 1e6
    res["output_first_GBs"] = bytes_lookup / (res["output_first"]["avg_us"] * 1e-6) / 1e9
    res["input_first_GBs"] = bytes_lookup / (res["input_first"]["avg_us"] * 1e-6) / 1e9
    plan.destroy()
    del dt, batches, out
    torch.cuda.empty_cache()
    return res


def run_forward_crossover(n_iter: int = 200, rotating: int = 8) -> str:
    """Where does ONE launch (dpi_forward's fused kernel) stop paying off? Graph-replayed us per step over batch size for a
    one-hot shape (c2's recipe, D = 16) and a 1-3-entries shape (c3's recipe, fp16 D = 32, mean): fused forced on
    (DPI_OPT_FUSED = 1; '-' where a chunk would exceed the kernel's 2048 bags), two launches without a promise (device-picked
    variant), two launches with the bag-length promise. The auto rule's ceiling (DPI_OPT_FUSED_MAX_BAGS) is read off this table."""
    import torch
    from . import binding, harness, workloads as W
    lines = ["## forward_crossover", "",
             "Graph-replayed us per step (plan + lookup work of one batch), 8 rotating batches. fused = `dpi_forward` with `DPI_OPT_FUSED = 1`; two launches ="
             " `DPI_OPT_FUSED = 2`, without / with `DPI_OPT_MAX_BAG_HINT`.", "",
             "| shape | B | bags G | fused (1 launch) | two launches, no promise | two launches, promise | fused / no promise | fused / promise |",
             "|---|---|---|---|---|---|---|---|"]
    shapes = [("one id per bag (c2 recipe)", W.C2, (512, 2048, 4096, 8192, 16384, 32768, 65536)),
              ("1-3 ids per bag (c3 recipe)", W.C3, (512, 2048, 8192, 16384, 32768, 65536, 98304))]
    for label, base, sizes in shapes:
        for B in sizes:
            cfg = base.scaled(name=f"{base.name}-B{B}", B=B)
            rows = cfg.table_rows()
            dt = harness.make_device_tables(cfg, rows)
            batches = [harness.upload_batch(W.make_batch(cfg, rows, cfg.seed + r)) for r in range(rotating)]
            out = harness.new_output(cfg)
            pooling = cfg.pooling_modes()
            stream = torch.cuda.Stream()
            res = []
            for fused, hint in ((1, False), (2, False), (2, True)):
                plan = harness.make_plan(cfg, rows, harness.max_indices_bound(cfg), bag_hint=hint)
                plan.set_option(binding.OPT_FUSED, fused)

                def step(i, st, plan=plan):
                    b = batches[i % rotating]
                    plan.forward(b.lengths, dt.ptrs, b.indices, out, pooling=pooling, stream=st)

                with torch.cuda.stream(stream):
                    n0 = binding.launch_count()
                    step(0, stream)
                    launches = binding.launch_count() - n0
                    for i in range(1, 4):
                        step(i, stream)
                torch.cuda.synchronize()
                us = _time_graph(step, stream, n_iter)
                res.append(None if (fused == 1 and launches != 1) else us)
                plan.destroy()
            f, n, h = res
            fmt = lambda x: "-" if x is None else f"{x:.2f}"
            lines.append(f"| {label} | {B} | {cfg.G} | {fmt(f)} | {fmt(n)} | {fmt(h)} | " +
                         ("-" if f is None else f"{f / n:.2f}") + " | " + ("-" if f is None else f"{f / h:.2f}") + " |")
            print(lines[-1], flush=True)
            del dt, batches, out
            torch.cuda.empty_cache()
    lines.append("")
    return "\n".join(lines)


def sweep_points() -> Dict[str, List]:
    from . import workloads as W
    base = W.C2  # 26 one-hot fields, heights log-uniform [10, 1e6], Zipf 1.05, fp32, sum
    batches = [512, 1024, 2048, 4096, 8192, 16384, 32768, 65536]
    return {
        "fig10_batch": [("B", b, base.scaled(name=f"B{b}", D=32, B=b)) for b in batches],
        "fig10_dim": [("D", d, base.scaled(name=f"D{d}", D=d, B=2048)) for d in (4, 8, 16, 32, 64, 128)],
        "fig10_fields": [("T", t, base.scaled(name=f"T{t}", T=t, rows=(500_000,) * t, D=32, B=2048)) for t in (5, 10, 20, 50, 100)],
        "fig10_features": [("rows", n, base.scaled(name=f"n{n}", T=50, rows=(n,) * 50, D=32, B=2048))
                           for n in (1_000, 10_000, 100_000, 1_000_000, 10_000_000)],
        # Fig. 11's batch sweep is fig10_batch (every point times both kernels); its dimension sweep at B = 65536:
        "fig11_dim": [("D", d, base.scaled(name=f"D{d}", D=d, B=65536)) for d in (4, 12, 20, 28, 36, 44, 52, 60)],
    }


def to_markdown(results: Dict[str, List[dict]]) -> str:
    lines = []
    for name, pts in results.items():
        lines += [f"## {name}", "",
                  "| " + pts[0]["axis"] + " | T | B | D | alg. MB | output-first us (avg / min) | GB/s | input-first us | GB/s | "
                  "input/output | plan+lookup graph us | stream us | per-table torch us | per-table/ours(stream) | "
                  "lookup only, graph us | alg1 direct us (avg / min) | alg1 direct, graph us |",
                  "|---|---|---|---|---|---|---|---|---|---|---|---|---|---|---|---|---|"]
        for p in pts:
            of, inf = p["output_first"], p["input_first"]
            pt = p.get("per_table", {}).get("avg_us")
            st = p["plan_plus_lookup_stream"]["avg_us"]
            lines.append(f"| {p['axis_value']} | {p['T']} | {p['B']} | {p['D']} | {p['algorithmic_MB']:.2f} | "
                         f"{of['avg_us']:.1f} / {of['min_us']:.1f} | {p['output_first_GBs']:.0f} | {inf['avg_us']:.1f} | "
                         f"{p['input_first_GBs']:.0f} | {inf['avg_us'] / of['avg_us']:.2f}x | {p['plan_plus_lookup_graph_us']:.1f} | "
                         f"{st:.1f} | " + (f"{pt:.1f} | {pt / st:.1f}x |" if pt else "- | - |") +
                         (f" {p['lookup_graph_us']:.1f} | {p['alg1_direct']['avg_us']:.1f} / {p['alg1_direct']['min_us']:.1f} | "
                          f"{p['alg1_direct_graph_us']:.1f} |" if "alg1_direct" in p else " - | - | - |"))
        lines.append("")
    return "\n".join(lines)


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--only", default="")
    ap.add_argument("--iters", type=int, default=200)
    ap.add_argument("--out", default="gpurun_out/sweeps_fig10_fig11.md")
    ap.add_argument("--no-torch", action="store_true")
    args = ap.parse_args()
    from . import binding, build, harness
    harness.require_cuda()
    build.build()
    binding.load_library()
    sweeps = sweep_points()
    only = [s for s in args.only.split(",") if s]
    if only == ["forward_crossover"]:
        text = run_forward_crossover(n_iter=args.iters)
        os.makedirs(os.path.dirname(os.path.abspath(args.out)) or ".", exist_ok=True)
        with open(args.out, "w") as f:
            f.write(text)
        print("wrote", args.out)
        return
    results = {}
    for name, pts in sweeps.items():
        if only and name not in only:
            continue
        results[name] = []
        for axis, val, cfg in pts:
            r = run_point(cfg, n_iter=args.iters, with_torch=not args.no_torch)
            r.update({"axis": axis, "axis_value": val})
            results[name].append(r)
            print(json.dumps({"sweep": name, **r}), flush=True)
    os.makedirs(os.path.dirname(os.path.abspath(args.out)) or ".", exist_ok=True)
    with open(args.out, "w") as f:
        f.write(to_markdown(results))
    with open(os.path.splitext(args.out)[0] + ".json", "w") as f:
        json.dump(results, f, indent=1)
    print("wrote", args.out)


if __name__ == "__main__":
    sys.exit(main())
