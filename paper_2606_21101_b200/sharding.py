"""Multi-GPU layout of the path: batch-sharded replicas, no data-path collective.

Bags are independent units ("do not query the same embedding table"; Alg. 1 has no cross-sample
term), so the path shards by SAMPLE: every rank holds all tables and a contiguous slice of the global batch,
builds its own plan and runs its own fused lookup; rank r's output block is rows [b_lo, b_hi) of the global
``[B_global, T*D]`` matrix. Nothing is exchanged on the data path -- the only collective is the
max-over-ranks of the device time, for reporting. This module is host-side layout only (no arithmetic of
the method): which samples a rank owns, how to cut or draw its slice of a global batch, and the timing
reduction. tests/test_sharding_gloo.py runs it with world_size 2 on the gloo backend.
"""
from __future__ import annotations

from typing import Optional, Tuple

import numpy as np

from . import workloads as W


def shard_range(B_global: int, rank: int, world: int) -> Tuple[int, int]:
    """Contiguous, balanced sample range [b_lo, b_hi) of rank `rank`: the first B_global % world ranks get one
    extra sample. Ranges tile [0, B_global) in rank order."""
    if not (0 <= rank < world) or B_global < 0:
        raise ValueError("bad rank/world/B_global")
    q, r = divmod(B_global, world)
    lo = rank * q + min(rank, r)
    return lo, lo + q + (1 if rank < r else 0)


def shard_batch(batch: W.Batch, T: int, rank: int, world: int) -> Tuple[W.Batch, int, int]:
    """Cut rank `rank`'s slice out of a global host batch (sample-major bags, bag-contiguous indices).
    Returns (local batch, b_lo, b_hi). Pure slicing: the entry range of a bag range is found by summing
    lengths (layout only)."""
    G = batch.lengths.shape[0]
    if G % T:
        raise ValueError("len(lengths) is not a multiple of T")
    b_lo, b_hi = shard_range(G // T, rank, world)
    ln = batch.lengths.astype(np.int64)
    e_lo = int(ln[: b_lo * T].sum())
    e_hi = e_lo + int(ln[b_lo * T: b_hi * T].sum())
    return W.Batch(batch.lengths[b_lo * T: b_hi * T].copy(), batch.indices[e_lo:e_hi].copy()), b_lo, b_hi


def make_batch_shard(cfg: W.Config, rows: np.ndarray, batch_seed: int, rank: int, world: int) -> W.Batch:
    """Rank `rank`'s shard of the global batch of world*cfg.B samples (weak scaling: cfg.B samples per rank),
    drawn directly from the counter-based generator: equal to
    ``shard_batch(make_batch(cfg.scaled(B=world*cfg.B), rows, batch_seed), cfg.T, rank, world)`` without
    drawing the other ranks' indices (only their bag lengths, to find this shard's first entry)."""
    G = cfg.G
    entry_base = 0
    for r in range(rank):
        entry_base += int(W.make_lengths(cfg, batch_seed, bag_base=r * G).astype(np.int64).sum())
    ln = W.make_lengths(cfg, batch_seed, bag_base=rank * G)
    return W.Batch(ln, W.make_indices(cfg, rows, ln, batch_seed, entry_base=entry_base))


def max_over_ranks(value: float, dist=None, device: Optional[str] = None) -> float:
    """Reporting reduction: the slowest rank's device time (all ranks receive it). `dist` is
    torch.distributed (initialised) or None for a single process."""
    if dist is None or not dist.is_initialized() or dist.get_world_size() == 1:
        return float(value)
    import torch
    t = torch.tensor([float(value)], dtype=torch.float64, device=device or "cpu")
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def job_throughput(units_per_rank_step: int, steps: int, world: int, max_ms: float) -> float:
    """Whole-job metric: units all ranks processed / slowest rank's time."""
    return units_per_rank_step * steps * world / (max_ms * 1e-3)


# ----------------------------------------------------------------------------------------------------
# Table-wise sharding with a fused all-to-all
# ----------------------------------------------------------------------------------------------------
# When the tables do not fit (or should not be replicated on) one GPU, rank r holds a SUBSET of the tables, sees
# the sparse inputs of the WHOLE global batch for those tables, and its fused lookup stores every pooled vector
# straight into the batch shard of the rank that owns the sample (dpi_lookup_ex out_peers_dev: peer-mapped memory
# over NVLink) at the table's GLOBAL column. The classic formulation -- local [B_global, T_local*D] block, then an
# all-to-all -- collapses into the lookup kernel's store; what remains on the stream is a barrier. Host-side
# layout only: which tables a rank owns, which bags it receives, where its columns go.


def partition_tables(cost, world: int):
    """Longest-processing-time greedy split of tables over ranks, balanced by `cost[t]` (expected gathered bytes of
    table t: mean bag length x row bytes). Returns a list of `world` ascending table-id lists; every table appears
    exactly once. Deterministic: ties go to the lower table id, then to the lower rank."""
    cost = np.asarray(cost, dtype=np.float64)
    if world < 1 or cost.ndim != 1:
        raise ValueError("bad world / cost")
    load = np.zeros(world)
    owned = [[] for _ in range(world)]
    for t in sorted(range(cost.shape[0]), key=lambda i: (-cost[i], i)):
        r = int(np.argmin(load))  # first minimum = lowest rank
        owned[r].append(t)
        load[r] += cost[t]
    return [sorted(o) for o in owned]


def table_columns(dims) -> np.ndarray:
    """Global first column (in elements) of every table in the concatenated row: prefix sum of dims."""
    dims = np.asarray(dims, dtype=np.int64)
    return np.concatenate(([0], np.cumsum(dims)))[:-1]


def table_shard_batch(batch: W.Batch, T: int, tables) -> W.Batch:
    """The sparse inputs rank r receives under table-wise sharding: every sample of the global batch, only the
    bags of `tables` (ascending global ids), still sample-major with T_local = len(tables) bags per sample and
    bag-contiguous indices. Pure selection (the entry position of a bag is found by summing lengths: layout only)."""
    tables = np.asarray(tables, dtype=np.int64)
    G = batch.lengths.shape[0]
    if G % T:
        raise ValueError("len(lengths) is not a multiple of T")
    B = G // T
    ln = batch.lengths.astype(np.int64)
    starts = np.concatenate(([0], np.cumsum(ln)))
    bags = (np.arange(B, dtype=np.int64)[:, None] * T + tables[None, :]).reshape(-1)
    sel_ln = ln[bags]
    n = int(sel_ln.sum())
    src = np.repeat(starts[bags], sel_ln) + (np.arange(n) - np.repeat(np.cumsum(sel_ln) - sel_ln, sel_ln))
    return W.Batch(sel_ln.astype(np.int32), np.ascontiguousarray(batch.indices[src]))


def peer_output_buffers(rows_per_rank: int, width: int, torch_dtype, device, group=None):
    """Allocate this rank's [rows_per_rank, width] batch shard where the other ranks' kernels can store into it and
    return (local tensor, int64 device tensor with every rank's base pointer, barrier callable).
    world 1 (or no process group): an ordinary tensor and its own pointer. world > 1: torch symmetric memory
    (CUDA IPC / multicast-capable allocations exchanged at rendezvous), pointers from the handle."""
    import torch
    import torch.distributed as dist
    world = dist.get_world_size(group) if (dist.is_available() and dist.is_initialized()) else 1
    if world == 1:
        out = torch.empty((rows_per_rank, width), dtype=torch_dtype, device=device)
        ptrs = torch.tensor([out.data_ptr()], dtype=torch.int64, device=device)
        return out, ptrs, (lambda: None)
    import torch.distributed._symmetric_memory as symm_mem
    out = symm_mem.empty((rows_per_rank, width), dtype=torch_dtype, device=device)
    hdl = symm_mem.rendezvous(out, group=group if group is not None else dist.group.WORLD)
    ptrs = torch.tensor([int(p) for p in hdl.buffer_ptrs], dtype=torch.int64, device=device)
    return out, ptrs, (lambda: hdl.barrier(channel=0))  # device-side barrier on the current stream
