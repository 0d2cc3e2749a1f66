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
