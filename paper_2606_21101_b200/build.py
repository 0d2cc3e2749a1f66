"""Builds the in-tree CUDA libraries with nvcc for sm_100a (cross-compiles without a GPU).

    python -m paper_2606_21101_b200.build [--force]

Outputs (git-ignored, shipped to the GPU box by gpurun):
    paper_2606_21101_b200/lib/libdpi.so        the product: planner + fused lookup behind include/dpi.h
    paper_2606_21101_b200/lib/libdpi_synth.so  bench/test helper: device-side synthetic table fill
"""
from __future__ import annotations

import concurrent.futures as cf
import os
import shutil
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
LIBDIR = os.path.join(HERE, "lib")
OBJDIR = os.path.join(HERE, "build")
INCLUDE = os.path.join(os.path.dirname(HERE), "include")

ARCH = ["-gencode", "arch=compute_100a,code=sm_100a"]
NVCC_FLAGS = ["-O3", "-std=c++17", "-lineinfo", "-Xcompiler", "-fPIC", "-Xptxas", "-v"]

LIBS = {
    "libdpi.so": ["dpi_api.cu", "plan_kernels.cu", "plan64_kernels.cu", "lookup_f32.cu", "lookup_f16.cu", "lookup_bf16.cu",
                  "ablation_input_first.cu", "lookup_onehot.cu", "lookup_direct.cu", "forward_fused.cu", "forward_noalloc.cu", "nongemm_kernels.cu", "nongemm_api.cu", "peer_api.cu"],
    "libdpi_synth.so": ["synth_fill.cu"],
}
HEADERS = ["dpi_internal.cuh", "lookup_kernels.cuh", "lookup_dispatch.inc", os.path.join(INCLUDE, "dpi.h"),
           os.path.join(INCLUDE, "dpi_nongemm.h")]


def _nvcc() -> str:
    exe = shutil.which("nvcc") or "/usr/local/cuda/bin/nvcc"
    if not os.path.exists(exe):
        raise RuntimeError("nvcc not found: libdpi has no prebuilt or CPU fallback")
    return exe


def _newest_header() -> float:
    return max(os.path.getmtime(h if os.path.isabs(h) else os.path.join(CSRC, h)) for h in HEADERS)


def _compile(src: str, force: bool) -> str:
    obj = os.path.join(OBJDIR, src.replace(".cu", ".o"))
    path = os.path.join(CSRC, src)
    stamp = max(os.path.getmtime(path), _newest_header(), os.path.getmtime(__file__))
    if not force and os.path.exists(obj) and os.path.getmtime(obj) >= stamp:
        return obj
    cmd = [_nvcc(), *ARCH, *NVCC_FLAGS, "-I", INCLUDE, "-c", path, "-o", obj]
    r = subprocess.run(cmd, capture_output=True, text=True)
    with open(obj + ".log", "w") as f:
        f.write(" ".join(cmd) + "\n" + r.stdout + r.stderr)
    if r.returncode != 0:
        raise RuntimeError(f"nvcc failed for {src}:\n{r.stdout}\n{r.stderr}")
    return obj


def build(force: bool = False, verbose: bool = False) -> dict:
    os.makedirs(LIBDIR, exist_ok=True)
    os.makedirs(OBJDIR, exist_ok=True)
    srcs = sorted({s for v in LIBS.values() for s in v})
    with cf.ThreadPoolExecutor(max_workers=min(8, len(srcs))) as ex:
        objs = dict(zip(srcs, ex.map(lambda s: _compile(s, force), srcs)))
    out = {}
    for lib, members in LIBS.items():
        target = os.path.join(LIBDIR, lib)
        members_o = [objs[m] for m in members]
        if force or not os.path.exists(target) or os.path.getmtime(target) < max(os.path.getmtime(o) for o in members_o):
            tmp = target + f".tmp{os.getpid()}"
            cmd = [_nvcc(), *ARCH, "-shared", "-o", tmp, *members_o, "-lcudart"]
            r = subprocess.run(cmd, capture_output=True, text=True)
            if r.returncode != 0:
                raise RuntimeError(f"link failed for {lib}:\n{r.stdout}\n{r.stderr}")
            os.replace(tmp, target)
        out[lib] = target
        if verbose:
            print("built", target)
    return out


def lib_path(name: str = "libdpi.so") -> str:
    return os.path.join(LIBDIR, name)


if __name__ == "__main__":
    build(force="--force" in sys.argv, verbose=True)
