"""Bench context (SURVEY.md 8(d) "random-access ceiling"): what one B200 sustains for independent whole-row reads with
no indices, no pooling and no output -- the number the fused lookup's row stream can be held against.

    python -m paper_2606_21101_b200.ceiling [--out gpurun_out/ceiling.md]

For row sizes 64 / 128 / 256 / 512 B and spans 1 / 8 / 80 GB: random rows (counter hash) and consecutive rows, reading
4.3 GB per launch (c5's gathered bytes). Helper kernel in libdpi_synth.so; not part of the method.

    python -m paper_2606_21101_b200.ceiling --probe pcie [--out gpurun_out/pcie.md]

The host link's ceiling for the end-to-end number (dpi_forward_host): one pinned-memory cudaMemcpyAsync per direction,
H2D alone, D2H alone and both at once on two streams, 16 ... 256 MB (torch only issues the copies)."""
from __future__ import annotations

import argparse
import os

import torch

from . import binding, harness
from .nongemm_bench import peak_gbs


def pcie_probe() -> str:
    sizes = [16, 32, 64, 128, 256]
    big = max(sizes) << 20
    hi, ho = torch.empty(big, dtype=torch.uint8).pin_memory(), torch.empty(big, dtype=torch.uint8).pin_memory()
    di, do = torch.empty(big, dtype=torch.uint8, device="cuda"), torch.empty(big, dtype=torch.uint8, device="cuda")
    s1, s2 = torch.cuda.Stream(), torch.cuda.Stream()

    def run(n, h2d, d2h):
        ts = []
        for it in range(7):
            torch.cuda.synchronize()
            a, b, j = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True), torch.cuda.Event()
            a.record(s1)
            s2.wait_event(a)
            if h2d:
                with torch.cuda.stream(s1):
                    di[:n].copy_(hi[:n], non_blocking=True)
            if d2h:
                with torch.cuda.stream(s2):
                    ho[:n].copy_(do[:n], non_blocking=True)
            j.record(s2)
            s1.wait_event(j)
            b.record(s1)
            torch.cuda.synchronize()
            if it >= 2:
                ts.append(a.elapsed_time(b))
        return min(ts)

    lines = ["# Host-link ceiling probe (python -m paper_2606_21101_b200.ceiling --probe pcie)", "",
             f"Device {torch.cuda.get_device_name(0)}; pinned host buffers, ONE cudaMemcpyAsync per direction and measurement, CUDA "
             "events, best of 5 after 2 warm-ups. 'both' = H2D and D2H of the same size at once on two streams; its GB/s counts "
             "both directions.", "",
             "| MB per direction | H2D ms | H2D GB/s | D2H ms | D2H GB/s | both ms | both GB/s (sum) |", "|---|---|---|---|---|---|---|"]
    for mb in sizes:
        n = mb << 20
        h, d, both = run(n, True, False), run(n, False, True), run(n, True, True)
        lines.append(f"| {mb} | {h:.3f} | {n / h / 1e6:.1f} | {d:.3f} | {n / d / 1e6:.1f} | {both:.3f} | {2 * n / both / 1e6:.1f} |")
    return "\n".join(lines)


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--out", default="")
    ap.add_argument("--probe", default="rows", choices=["rows", "pcie"])
    args = ap.parse_args()
    harness.require_cuda()
    torch.cuda.set_device(0)
    if args.probe == "pcie":
        text = pcie_probe()
        print(text)
        if args.out:
            os.makedirs(os.path.dirname(os.path.abspath(args.out)), exist_ok=True)
            with open(args.out, "w") as f:
                f.write(text + "\n")
        return
    peak, src = peak_gbs()
    buf = torch.empty(80 * (1 << 30), dtype=torch.uint8, device="cuda")
    buf.zero_()
    sink = torch.zeros(4, dtype=torch.int32, device="cuda")
    read_bytes = 4_300_000_000
    lines = ["# Row-read ceiling probe (python -m paper_2606_21101_b200.ceiling)", "",
             f"Device {torch.cuda.get_device_name(0)}; {read_bytes / 1e9:.1f} GB read per launch; CUDA events, best of 5 after 2 warm-ups; "
             f"copy peak {peak:.1f} GB/s ({src}). No indices, no accumulation, no output: an upper bound for the lookup's row stream.", "",
             "| row bytes | span | order | unroll | CTAs/SM | GB/s | frac of copy peak |", "|---|---|---|---|---|---|---|"]
    st = torch.cuda.current_stream()
    for row_bytes in (64, 128, 256, 512):
        for span_gb in (1, 8, 80):
            span_rows = span_gb * (1 << 30) // row_bytes
            n_rows = read_bytes // row_bytes
            for random in (1, 0):
                best = None
                for unroll, cps in ((4, 8), (8, 4), (2, 8)):
                    ts = []
                    for it in range(7):
                        a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                        a.record(st)
                        binding.synth_row_read_probe(buf, span_rows, row_bytes, n_rows, 1234 + it, random, unroll, cps, sink)
                        b.record(st)
                        torch.cuda.synchronize()
                        if it >= 2:
                            ts.append(a.elapsed_time(b))
                    gbs = n_rows * row_bytes / min(ts) / 1e6
                    if best is None or gbs > best[0]:
                        best = (gbs, unroll, cps)
                lines.append(f"| {row_bytes} | {span_gb} GB | {'random' if random else 'consecutive'} | {best[1]} | {best[2]} | "
                             f"{best[0]:.0f} | {best[0] / peak:.3f} |")
    text = "\n".join(lines)
    print(text)
    if args.out:
        os.makedirs(os.path.dirname(os.path.abspath(args.out)), exist_ok=True)
        with open(args.out, "w") as f:
            f.write(text + "\n")


if __name__ == "__main__":
    main()
