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


class _DeviceBlock:
    """A raw device allocation presented to torch through __cuda_array_interface__ (no copy, no ownership)."""

    def __init__(self, ptr: int, shape, typestr: str):
        self.__cuda_array_interface__ = {"shape": tuple(shape), "typestr": typestr, "data": (ptr, False), "version": 2}


_TYPESTR = {"torch.float32": "<f4", "torch.float16": "<f2", "torch.bfloat16": "<u2"}


class PeerOutput:
    """This rank's [rows_per_rank, width] batch shard, allocated where the other ranks' lookup kernels can store into it
    (dpi_peer_alloc: one dedicated allocation + CUDA IPC handle), plus every rank's base pointer as the device array
    dpi_lookup_ex(out_peers_dev) takes. Works for ranks on different GPUs (stores cross NVLink) and for ranks sharing one
    device (the one-GPU test of the multi-process glue). world 1 / no process group: a plain local block.

    `local` is a torch view of this rank's block; `ptrs` the int64 device tensor [world]; `barrier()` orders consumers
    after ALL ranks' kernels (synchronise the current device, then a control-plane barrier); `close()` unmaps and frees."""

    def __init__(self, rows_per_rank: int, width: int, torch_dtype, device, group=None):
        import torch
        import torch.distributed as dist
        from . import binding
        self._dist = dist if (dist.is_available() and dist.is_initialized()) else None
        self._group = group
        self.world = self._dist.get_world_size(group) if self._dist else 1
        self.rank = self._dist.get_rank(group) if self._dist else 0
        elt = torch.empty((), dtype=torch_dtype).element_size()
        nbytes = max(1, rows_per_rank * width * elt)
        with torch.cuda.device(device):
            self._own, handle = binding.peer_alloc(nbytes)
            handles = [handle]
            if self.world > 1:
                handles = [None] * self.world
                self._dist.all_gather_object(handles, handle, group=group)
            self._opened = []
            base = []
            for r, h in enumerate(handles):
                if r == self.rank:
                    base.append(self._own)
                else:
                    p = binding.peer_open(h)
                    self._opened.append(p)
                    base.append(p)
        block = _DeviceBlock(self._own, (rows_per_rank, width), _TYPESTR[str(torch_dtype)])
        local = torch.as_tensor(block, device=device)
        self.local = local.view(torch.bfloat16) if torch_dtype == torch.bfloat16 else local
        self.ptrs = torch.tensor(base, dtype=torch.int64, device=device)
        self._device = device

    def barrier(self):
        import torch
        torch.cuda.synchronize(self._device)
        if self._dist and self.world > 1:
            self._dist.barrier(group=self._group)

    def close(self):
        from . import binding
        import torch
        if self._own is None:
            return
        torch.cuda.synchronize(self._device)
        for p in self._opened:
            binding.peer_close(p)
        self._opened = []
        if self._dist and self.world > 1:
            self._dist.barrier(group=self._group)   # nobody still maps the block when it is freed
        binding.peer_free(self._own)
        self._own = None
        self.local = None


def peer_output_buffers(rows_per_rank: int, width: int, torch_dtype, device, group=None):
    """(local tensor, device pointer array of every rank's block, barrier callable) -- see PeerOutput."""
    po = PeerOutput(rows_per_rank, width, torch_dtype, device, group)
    return po.local, po.ptrs, po.barrier


class TableWiseLookup:
    """Table-wise sharded lookup with the all-to-all fused into the store:
    the single entry point that wires partition_tables -> table_shard_batch -> PeerOutput -> dpi_lookup_ex(out_peers_dev)
    -> barrier. Rank r holds `tables_r` (all rows of each) and, per call, receives the bags of its tables for EVERY sample of
    the global batch; its kernel stores each pooled vector into the batch shard of the rank that owns the sample, at the
    table's global column. After `forward` returns, `out.local` holds this rank's rows [rank * rows_per_rank, ...) of the
    global [B, sum dims] block, complete. Comm on the data path: peer stores only, no NCCL.

    The output shard is DOUBLE-BUFFERED: step k stores into block k % 2 of every rank. There is one barrier per step, after
    the stores; a rank that leaves it may start step k+1 at once, and its kernel then stores into the OTHER block of its
    peers, which may still be reading step k's result. Block k % 2 is written again only in step k+2, which a peer reaches
    after the barrier of step k+1 -- and every rank enters that barrier through a device synchronise, i.e. after whatever it
    had enqueued on step k's result. Hence the contract: the tensor `forward` returns stays valid until the second-next
    `forward` call on this object; enqueue its consumers before calling `forward` again (any stream of this device)."""

    def __init__(self, dims, table_rows, dtype_code: int, torch_dtype, B_global: int, max_indices: int, device, cost=None,
                 group=None, out_dtype_code=None):
        import torch.distributed as dist
        from . import binding
        on = dist.is_available() and dist.is_initialized()
        self.world = dist.get_world_size(group) if on else 1
        self.rank = dist.get_rank(group) if on else 0
        dims = np.asarray(dims, dtype=np.int64)
        table_rows = np.asarray(table_rows, dtype=np.int64)
        self.T = int(dims.shape[0])
        self.B = int(B_global)
        self.parts = partition_tables(dims if cost is None else cost, self.world)
        self.mine = self.parts[self.rank]
        self.columns = table_columns(dims)
        self.width = int(dims.sum())
        self.rows_per_rank = -(-self.B // self.world)
        self.device = device
        self.plan = None
        if self.mine:
            self.plan = binding.Plan(table_rows[self.mine], np.asarray(dims[self.mine], np.int32), dtype_code, self.B, max_indices)
            if out_dtype_code is not None:
                self.plan.set_out_dtype(out_dtype_code)
            self.plan.set_columns([int(self.columns[t]) for t in self.mine])
        self.outs = [PeerOutput(self.rows_per_rank, self.width, torch_dtype, device, group) for _ in range(2)]
        self._step = 0

    @property
    def out(self) -> "PeerOutput":
        """The block the most recent `forward` filled (block 0 before the first call)."""
        return self.outs[(self._step - 1) % 2] if self._step else self.outs[0]

    def fill(self, value: float):
        """Fill both local blocks (tests: NaN sentinel) and wait until every rank has done so."""
        for o in self.outs:
            o.local.fill_(value)
        self.outs[0].barrier()

    def forward(self, lengths_dev, indices_dev, table_ptrs_dev, pooling=None, stream=None):
        """lengths / indices: this rank's table shard of the global batch (table_shard_batch), on the device; table_ptrs_dev:
        device pointer array of this rank's tables (ascending global id). Returns this rank's complete batch shard."""
        buf = self.outs[self._step % 2]
        if self.plan is not None:
            self.plan.build(lengths_dev, stream)
            self.plan.lookup_ex(table_ptrs_dev, indices_dev, None, pooling=pooling, out_ld=self.width,
                                out_peers_dev=buf.ptrs, n_peers=self.world, rows_per_peer=self.rows_per_rank, stream=stream)
        buf.barrier()
        self._step += 1
        return buf.local

    def close(self):
        if self.plan is not None:
            self.plan.destroy()
            self.plan = None
        for o in self.outs:
            o.close()


def table_wise_forward(tw: "TableWiseLookup", lengths_dev, indices_dev, table_ptrs_dev, pooling=None, stream=None):
    """Functional spelling of TableWiseLookup.forward."""
    return tw.forward(lengths_dev, indices_dev, table_ptrs_dev, pooling=pooling, stream=stream)
