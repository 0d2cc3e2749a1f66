"""N > 1 path on CPU: batch-sharded replicas with no data-path collective, world_size 2 on the
gloo backend. Each rank cuts/draws its shard, evaluates it with the oracle (test infrastructure), and the
gathered row blocks must equal the oracle on the global batch; the reporting reduction is max over ranks."""
import os
import socket

import numpy as np
import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

import oracle
from paper_2606_21101_b200 import sharding, workloads as W
from tests.parity import host_offsets

CFG = W.Config("sh", 3, (50, 7, 400), 16, "f32", 37, ("uniform", 0, 5), ("zipf", 1.1), "half", seed=21)


def test_shard_ranges_tile_the_batch():
    for B in (0, 1, 7, 64, 65537):
        for world in (1, 2, 3, 8):
            r = [sharding.shard_range(B, k, world) for k in range(world)]
            assert r[0][0] == 0 and r[-1][1] == B
            assert all(r[i][1] == r[i + 1][0] for i in range(world - 1))
            sizes = [b - a for a, b in r]
            assert max(sizes) - min(sizes) <= 1 and sizes == sorted(sizes, reverse=True)
    with pytest.raises(ValueError):
        sharding.shard_range(4, 2, 2)


@pytest.mark.parametrize("world", [1, 2, 4])
def test_direct_shard_draw_equals_slicing_the_global_batch(world):
    rows = CFG.table_rows()
    glob = W.make_batch(CFG.scaled(B=world * CFG.B), rows, 5)
    for rank in range(world):
        cut, b_lo, b_hi = sharding.shard_batch(glob, CFG.T, rank, world)
        drawn = sharding.make_batch_shard(CFG, rows, 5, rank, world)
        assert (b_lo, b_hi) == (rank * CFG.B, (rank + 1) * CFG.B)
        assert np.array_equal(cut.lengths, drawn.lengths) and np.array_equal(cut.indices, drawn.indices)


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    p = s.getsockname()[1]
    s.close()
    return p


def _worker(rank, world, port, B_global, q):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        cfg = CFG.scaled(B=B_global)
        rows = cfg.table_rows()
        tables = [W.full_table_storage(cfg, t, int(rows[t])) for t in range(cfg.T)]
        glob = W.make_batch(cfg, rows, 9)
        mine, b_lo, b_hi = sharding.shard_batch(glob, cfg.T, rank, world)
        pooling = cfg.pooling_modes()
        local = oracle.lookup(tables, oracle.F32, b_hi - b_lo, mine.indices, host_offsets(mine.lengths), pooling)
        # reporting only: gather the row blocks (uneven shards -> gather objects) and the max-over-ranks time
        blocks = [None] * world
        dist.all_gather_object(blocks, (b_lo, b_hi, local))
        t_max = sharding.max_over_ranks(10.0 + rank, dist)
        if rank == 0:
            full = np.empty((B_global, cfg.T * cfg.D))
            for lo, hi, blk in blocks:
                full[lo:hi] = blk
            ref = oracle.lookup(tables, oracle.F32, B_global, glob.indices, host_offsets(glob.lengths), pooling)
            q.put((bool(np.array_equal(full, ref)), t_max, [(lo, hi) for lo, hi, _ in blocks]))
    finally:
        dist.destroy_process_group()


@pytest.mark.parametrize("B_global", [37, 64])
def test_world2_gloo_batch_sharded_replicas(B_global):
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, 2, port, B_global, q)) for r in range(2)]
    for p in procs:
        p.start()
    for p in procs:
        p.join(120)
        assert p.exitcode == 0
    same, t_max, ranges = q.get(timeout=10)
    assert same
    assert t_max == 11.0                       # the slower rank's time, seen by every rank
    assert ranges == [sharding.shard_range(B_global, r, 2) for r in range(2)]
    assert sharding.job_throughput(100, 4, 2, 8.0) == 100 * 4 * 2 / 8e-3


# --------------------------------------------------------------------------------------------------
# table-wise sharding + fused all-to-all: host logic
# --------------------------------------------------------------------------------------------------
def test_partition_tables_is_a_balanced_partition():
    rng = np.random.default_rng(0)
    for T, world in ((1, 1), (5, 2), (26, 4), (100, 8), (3, 8)):
        cost = rng.uniform(1, 100, size=T)
        parts = sharding.partition_tables(cost, world)
        assert len(parts) == world and sorted(sum(parts, [])) == list(range(T))
        assert all(p == sorted(p) for p in parts)
        loads = np.array([cost[p].sum() for p in parts])
        assert loads.max() - loads.min() <= cost.max() + 1e-9   # LPT: no rank exceeds another by more than one table
    assert sharding.partition_tables([5, 1, 1, 1, 4, 3], 2) == [[0, 1, 2, 3], [4, 5]]
    assert list(sharding.table_columns([4, 8, 16])) == [0, 4, 12]


def test_table_shard_batch_selects_whole_bags_in_order():
    cfg = CFG.scaled(B=11)
    rows = cfg.table_rows()
    glob = W.make_batch(cfg, rows, 3)
    off = host_offsets(glob.lengths)
    for tabs in ([0], [1, 2], [0, 2], [0, 1, 2]):
        sub = sharding.table_shard_batch(glob, cfg.T, tabs)
        want_len, want_idx = [], []
        for b in range(cfg.B):
            for t in tabs:
                g = b * cfg.T + t
                want_len.append(glob.lengths[g])
                want_idx.extend(glob.indices[off[g]:off[g + 1]])
        assert np.array_equal(sub.lengths, np.array(want_len, np.int32))
        assert np.array_equal(sub.indices, np.array(want_idx, np.int32).reshape(-1))


def _table_worker(rank, world, port, B_global, q):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        dims = [16, 8, 32, 8, 16]
        T = len(dims)
        cfg = W.Config("tw", T, (50, 7, 400, 90, 3), 32, "f32", B_global, ("uniform", 0, 5), ("zipf", 1.1), "sum", seed=4)
        rows = cfg.table_rows()
        tables = W.mixed_dim_tables(cfg.seed, dims, rows, "f32")
        glob = W.make_batch(cfg, rows, 9)
        pooling = np.array([0, 1, 0, 1, 0], np.uint8)
        mine = sharding.partition_tables(np.asarray(dims) * 2.5, world)[rank]
        cols = sharding.table_columns(dims)
        local = sharding.table_shard_batch(glob, T, mine)
        # this rank's column blocks for EVERY sample of the global batch (the oracle stands in for the kernel)
        blk = oracle.lookup_general([tables[t] for t in mine], oracle.F32, B_global, local.indices,
                                    host_offsets(local.lengths).astype(np.int64), pooling[mine])
        # the exchange the fused kernel performs by storing to peer memory: sample b -> rank b // rows_per_rank at the
        # tables' global columns. Here: gather everybody's blocks and let each rank assemble its own batch shard.
        rows_per_rank = -(-B_global // world)
        got = [None] * world
        dist.all_gather_object(got, (mine, blk))
        lo, hi = rank * rows_per_rank, min(B_global, (rank + 1) * rows_per_rank)
        shard = np.full((hi - lo, sum(dims)), np.nan)
        for tabs, b in got:
            c = 0
            for t in tabs:
                shard[:, cols[t]:cols[t] + dims[t]] = b[lo:hi, c:c + dims[t]]
                c += dims[t]
        ref = oracle.lookup_general(tables, oracle.F32, B_global, glob.indices, host_offsets(glob.lengths).astype(np.int64), pooling)
        ok = bool(np.array_equal(shard, ref[lo:hi]))
        oks = [None] * world
        dist.all_gather_object(oks, ok)
        if rank == 0:
            q.put(all(oks))
    finally:
        dist.destroy_process_group()


@pytest.mark.parametrize("B_global", [37, 64])
def test_world2_gloo_table_wise_sharding_assembles_the_global_block(B_global):
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_table_worker, args=(r, 2, port, B_global, q)) for r in range(2)]
    for p in procs:
        p.start()
    for p in procs:
        p.join(120)
        assert p.exitcode == 0
    assert q.get(timeout=10)
