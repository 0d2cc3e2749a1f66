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
