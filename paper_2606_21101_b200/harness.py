"""Device-side set-up of a synthetic workload for tests, smoke and bench (plumbing only).

PyTorch owns the device memory and the stream; tables are filled in place by ``libdpi_synth.so`` (the
device restatement of the generator in ``workloads``), sparse inputs are generated on the host with
``workloads`` and copied over. No arithmetic of the method lives here.
"""
from __future__ import annotations

from dataclasses import dataclass
from typing import List, Optional

import numpy as np
import torch

from . import binding, workloads as W

TORCH_DTYPE = {"f32": torch.float32, "f16": torch.float16, "bf16": torch.bfloat16}


def require_cuda():
    if not torch.cuda.is_available():
        raise RuntimeError("no CUDA device: the DPI lookup has no CPU fallback")


@dataclass
class DeviceTables:
    cfg: W.Config
    rows: np.ndarray            # int64[T]
    tables: List[torch.Tensor]  # T device tensors [rows_t, D]
    ptrs: torch.Tensor          # int64[T] device array of table base pointers

    def nbytes(self) -> int:
        return int(sum(t.numel() * t.element_size() for t in self.tables))


def make_device_tables(cfg: W.Config, rows: Optional[np.ndarray] = None, device="cuda:0") -> DeviceTables:
    """Allocate and fill all tables on the device with the seeded value recipe."""
    require_cuda()
    rows = cfg.table_rows() if rows is None else np.asarray(rows, dtype=np.int64)
    tables = []
    for t in range(cfg.T):
        buf = torch.empty((int(rows[t]), cfg.D), dtype=TORCH_DTYPE[cfg.dtype], device=device)
        binding.synth_fill_table(buf, buf.numel(), W.DTYPE_CODE[cfg.dtype], W.value_key(cfg.seed, t))
        tables.append(buf)
    ptrs = torch.tensor([t.data_ptr() for t in tables], dtype=torch.int64, device=device)
    return DeviceTables(cfg, rows, tables, ptrs)


def tables_from_host(cfg: W.Config, host_tables: List[np.ndarray], device="cuda:0") -> DeviceTables:
    """Upload explicit host tables (storage format: float32 / float16 / uint16-bf16-bits)."""
    require_cuda()
    tables = []
    for a in host_tables:
        a = np.ascontiguousarray(a)
        if cfg.dtype == "bf16":
            t = torch.from_numpy(a.view(np.int16)).to(device).view(torch.bfloat16)
        else:
            t = torch.from_numpy(a).to(device)
        assert t.dtype == TORCH_DTYPE[cfg.dtype] and t.shape[1] == cfg.D
        tables.append(t.contiguous())
    ptrs = torch.tensor([t.data_ptr() for t in tables], dtype=torch.int64, device=device)
    rows = np.asarray([t.shape[0] for t in tables], dtype=np.int64)
    return DeviceTables(cfg, rows, tables, ptrs)


def tables_from_host_mixed(host_tables: List[np.ndarray], dtype: str, device="cuda:0"):
    """Upload host tables of possibly different widths; returns (device tensors, device pointer array)."""
    require_cuda()
    tables = []
    for a in host_tables:
        a = np.ascontiguousarray(a)
        t = torch.from_numpy(a.view(np.int16)).to(device).view(torch.bfloat16) if dtype == "bf16" else torch.from_numpy(a).to(device)
        assert t.dtype == TORCH_DTYPE[dtype]
        tables.append(t.contiguous())
    return tables, torch.tensor([t.data_ptr() for t in tables], dtype=torch.int64, device=device)


@dataclass
class DeviceBatch:
    lengths: torch.Tensor  # int32[G] device
    indices: torch.Tensor  # int32[N] device (never empty: one pad element keeps data_ptr valid)
    N: int
    host: W.Batch


def upload_batch(batch: W.Batch, device="cuda:0") -> DeviceBatch:
    ln = torch.from_numpy(np.ascontiguousarray(batch.lengths, dtype=np.int32)).to(device)
    idx_host = np.ascontiguousarray(batch.indices, dtype=np.int32)
    if idx_host.size == 0:
        idx_host = np.zeros(1, dtype=np.int32)
    return DeviceBatch(ln, torch.from_numpy(idx_host).to(device), batch.N, batch)


def new_output(cfg: W.Config, device="cuda:0", fill_nan: bool = False) -> torch.Tensor:
    out = torch.empty((cfg.B, cfg.T * cfg.D), dtype=TORCH_DTYPE[cfg.out], device=device)
    if fill_nan:
        out.fill_(float("nan"))  # a bag the kernel forgets to write shows up as NaN in the parity check
    return out


def out_to_f64(out: torch.Tensor) -> np.ndarray:
    """Device output block -> host float64 (exact widening)."""
    return out.detach().to("cpu").to(torch.float64).numpy()


def max_bag_length(cfg: W.Config) -> int:
    """Longest bag the config's length recipe can draw (a schema fact, known before any batch exists)."""
    kind = cfg.lengths[0]
    return int(cfg.lengths[1]) if kind == "const" else int(cfg.lengths[2])


def short_bag_rule(max_len: int, G: int) -> bool:
    """Reporting mirror of short_bag_rule in csrc/dpi_internal.cuh (the device applies it to a1's max_len)."""
    return max_len <= 8 if max_len >= 2 else G <= 500000


def lookup_variant(cfg: W.Config, mode: int = 0) -> str:
    """Which a3 body dpi_lookup ends up in for this config (reporting only)."""
    short = short_bag_rule(max_bag_length(cfg), cfg.G)
    return "short-bag (lane group per bag)" if (mode == 6 or (mode == 0 and short)) else "balanced segments"


def make_plan(cfg: W.Config, rows: np.ndarray, max_indices: int, bag_hint: bool = False) -> binding.Plan:
    """bag_hint: pass the recipe's longest bag as the OPTIONAL promise DPI_OPT_MAX_BAG_HINT (the short-bag variant then runs as
    its own launch, chosen on the host). Default: no hint -- the device picks from a1's max_len."""
    plan = binding.Plan(rows, cfg.D, W.DTYPE_CODE[cfg.dtype], cfg.B, max_indices)
    if cfg.out != cfg.dtype:
        plan.set_out_dtype(W.DTYPE_CODE[cfg.out])
    if bag_hint:
        plan.set_option(binding.OPT_MAX_BAG_HINT, max(max_bag_length(cfg), 0))
    return plan


def max_indices_bound(cfg: W.Config) -> int:
    """Upper bound on N for any batch of this config (capacity of the plan)."""
    kind = cfg.lengths[0]
    if kind == "const":
        per = int(cfg.lengths[1])
    elif kind == "uniform":
        per = int(cfg.lengths[2])
    else:
        per = int(cfg.lengths[2])
    return cfg.G * per
