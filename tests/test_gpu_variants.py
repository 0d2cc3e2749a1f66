"""GPU parity of the interface variants through dpi_lookup_ex: mixed per-table dims,
int64 ids, per-entry weights, table-major bags, output row pitch -- against oracle.lookup_general on the same
seeded inputs, with the tolerances of tests/parity.py."""
import numpy as np
import pytest
import torch

import oracle
from paper_2606_21101_b200 import binding, harness, workloads as W
from tests.parity import assert_outputs_match_general, host_offsets

pytestmark = pytest.mark.gpu

TORCH_OUT = {"f32": torch.float32, "f16": torch.float16, "bf16": torch.bfloat16}


@pytest.fixture(scope="module", autouse=True)
def _lib():
    from paper_2606_21101_b200 import build
    build.build()
    binding.load_library()
    harness.require_cuda()


def _problem(seed, dims, rows, B, lengths_spec, index_dist=("uniform",)):
    """Sample-major batch over tables of the given dims: lengths, indices (workloads' draws) and host tables."""
    T = len(dims)
    cfg = W.Config("var", T, tuple(int(r) for r in rows), int(max(dims)), "f32", B, lengths_spec, index_dist, "sum", seed)
    batch = W.make_batch(cfg, np.asarray(rows, dtype=np.int64), seed)
    return batch.lengths, batch.indices


def _run(dims, rows, B, dtype, lengths_spec, *, seed=3, out_dtype=None, table_major=False, idx64=False, weighted=False,
         pooling=None, out_ld=0, K=0, force_general=False, mode=0, off64=False, explicit_offsets=False):
    T = len(dims)
    out_dtype = out_dtype or dtype
    lengths, indices = _problem(seed, dims, rows, B, lengths_spec)
    weights = W.make_weights(seed, indices.shape[0]) if weighted else None
    host_tables = W.mixed_dim_tables(seed, dims, rows, dtype)
    pooling = np.zeros(T, np.uint8) if pooling is None else np.asarray(pooling, np.uint8)
    L_bt = lengths.reshape(B, T).copy()

    ln, idx, wgt = lengths, indices, weights
    if table_major:
        if weighted:
            ln, idx, wgt = W.to_table_major(T, B, lengths, indices, weights)
        else:
            ln, idx = W.to_table_major(T, B, lengths, indices)
    ref = oracle.lookup_general(host_tables, W.DTYPE_CODE[dtype], B, idx, host_offsets(ln).astype(np.int64), pooling,
                                weights=wgt, bag_order=oracle.TABLE_MAJOR if table_major else oracle.SAMPLE_MAJOR)

    tables, ptrs = harness.tables_from_host_mixed(host_tables, dtype)
    plan = binding.Plan(rows, np.asarray(dims, np.int32), W.DTYPE_CODE[dtype], B, max(int(idx.shape[0]), 1))
    if out_dtype != dtype:
        plan.set_out_dtype(W.DTYPE_CODE[out_dtype])
    plan.set_layout(binding.BAGS_TABLE_MAJOR if table_major else binding.BAGS_SAMPLE_MAJOR,
                    binding.IDX_I64 if idx64 else binding.IDX_I32)
    if off64:
        plan.set_offset_type(binding.OFF_I64)
    if K:
        plan.set_quantum(K)
    plan.set_option(binding.OPT_MODE, mode)
    ln_dev = torch.from_numpy(np.ascontiguousarray(ln, dtype=np.int32)).cuda()
    idx_host = np.ascontiguousarray(idx, dtype=np.int64 if idx64 else np.int32)
    if idx_host.size == 0:
        idx_host = np.zeros(1, idx_host.dtype)
    idx_dev = torch.from_numpy(idx_host).cuda()
    wgt_dev = torch.from_numpy(wgt).cuda() if weighted and wgt.size else (torch.zeros(1, device="cuda") if weighted else None)
    plan.build(ln_dev)
    assert plan.check_indices(idx_dev) == 0
    off_dev = None
    if off64:   # the plan itself: bit-exact against the 64-bit oracle plan
        off, seg, S, N, seg_off = plan.export64()
        o_off, o_seg, o_S, o_seg_off = oracle.plan64(ln, plan.info()["K"])
        assert N == int(np.asarray(ln, np.int64).sum()) and S == o_S
        assert np.array_equal(off, o_off) and np.array_equal(seg, o_seg) and np.array_equal(seg_off, o_seg_off)
        assert plan.stats() == oracle.plan_stats(ln)
        with pytest.raises(binding.DpiError):
            plan.export()
        if explicit_offsets:
            off_dev = torch.from_numpy(o_off).cuda()
    width = int(np.sum(dims))
    assert plan.plan_out_width() == width
    ld = out_ld or width
    out = torch.full((B, ld), float("nan"), dtype=TORCH_OUT[out_dtype], device="cuda")
    plan.lookup_ex(ptrs, idx_dev, out, pooling=pooling, weights_dev=wgt_dev, out_ld=out_ld, offsets_dev=off_dev,
                   flags=binding.LOOKUP_FORCE_GENERAL if force_general else 0)
    torch.cuda.synchronize()
    got_full = harness.out_to_f64(out)
    if ld > width:
        assert np.isnan(got_full[:, width:]).all(), "columns beyond this call's block must stay untouched"
    got = got_full[:, :width]
    plan.destroy()
    del tables
    return assert_outputs_match_general(got, ref, L_bt, dims, dtype, out_dtype, weighted=weighted)


LENGTHS = [("const", 1), ("uniform", 0, 5), ("poisson", 20.0, 100, 0.05)]


@pytest.mark.parametrize("lengths", LENGTHS)
@pytest.mark.parametrize("dtype,out", [("f32", None), ("f16", None), ("bf16", "f32")])
def test_general_kernel_equals_oracle_on_the_plain_layout(dtype, out, lengths):
    """Nothing generalised, general instantiation forced: same results as the dense kernel's contract."""
    D = 16 if dtype == "f32" else 32
    _run([D] * 7, [1000, 50, 7, 3000, 1, 640, 99], 333, dtype, lengths, out_dtype=out, force_general=True)


@pytest.mark.parametrize("lengths", LENGTHS)
@pytest.mark.parametrize("dtype,out", [("f32", None), ("f16", None), ("f16", "f32"), ("bf16", "f32"), ("bf16", None)])
def test_mixed_dims(dtype, out, lengths):
    dims = [4, 16, 8, 64, 4, 12, 32] if dtype == "f32" else [8, 16, 64, 128, 8, 24, 32]
    _run(dims, [1000, 50, 7, 3000, 1, 640, 99], 257, dtype, lengths, out_dtype=out)


@pytest.mark.parametrize("lengths", LENGTHS)
def test_int64_indices(lengths):
    _run([16] * 5, [1000, 50, 7, 3000, 640], 300, "f32", lengths, idx64=True)
    _run([32] * 5, [1000, 50, 7, 3000, 640], 300, "f16", lengths, idx64=True, pooling=[1, 0, 1, 0, 1])


@pytest.mark.parametrize("lengths", LENGTHS)
@pytest.mark.parametrize("dtype,out", [("f32", None), ("bf16", "f32"), ("f16", None)])
def test_per_entry_weights(dtype, out, lengths):
    D = 16 if dtype == "f32" else 64
    _run([D] * 6, [1000, 50, 7, 3000, 640, 2], 280, dtype, lengths, out_dtype=out, weighted=True)


@pytest.mark.parametrize("lengths", LENGTHS)
@pytest.mark.parametrize("dtype,out", [("f32", None), ("bf16", "f32")])
def test_table_major_bags(dtype, out, lengths):
    D = 16 if dtype == "f32" else 64
    _run([D] * 6, [1000, 50, 7, 3000, 640, 2], 280, dtype, lengths, out_dtype=out, table_major=True, pooling=[0, 1, 0, 1, 1, 0])


@pytest.mark.parametrize("K", [1, 7, 64, 100000])
@pytest.mark.parametrize("mode", [0, 1, 2, 3])
def test_everything_at_once_any_quantum_any_mode(K, mode):
    _run([4, 16, 8, 64, 4, 12, 32], [1000, 50, 7, 3000, 1, 640, 99], 129, "f32", ("poisson", 6.0, 40, 0.1),
         table_major=True, idx64=True, weighted=True, out_ld=4 + 16 + 8 + 64 + 4 + 12 + 32 + 20, K=K, mode=mode)


def test_output_row_pitch_writes_only_its_own_block():
    _run([16] * 4, [100, 50, 7, 300], 64, "f32", ("uniform", 0, 3), out_ld=64 + 8)
    _run([32] * 4, [100, 50, 7, 300], 64, "bf16", ("uniform", 0, 3), out_dtype="f32", out_ld=128 + 16)


def test_unit_weights_are_bit_identical_to_the_unweighted_lookup():
    rows, dims, B = [500, 20, 3000], [16, 16, 16], 500
    lengths, indices = _problem(5, dims, rows, B, ("uniform", 0, 9))
    host_tables = W.mixed_dim_tables(5, dims, rows, "f32")
    tables, ptrs = harness.tables_from_host_mixed(host_tables, "f32")
    plan = binding.Plan(rows, np.asarray(dims, np.int32), 0, B, int(indices.shape[0]))
    plan.build(torch.from_numpy(lengths).cuda())
    idx = torch.from_numpy(indices).cuda()
    a = torch.empty((B, 48), device="cuda")
    b = torch.empty((B, 48), device="cuda")
    plan.lookup(ptrs, idx, a)
    plan.lookup_ex(ptrs, idx, b, weights_dev=torch.ones(indices.shape[0], device="cuda"))
    torch.cuda.synchronize()
    assert torch.equal(a, b)
    plan.destroy()


def test_variant_argument_validation():
    rows, dims = [10, 10], [16, 16]
    plan = binding.Plan(rows, np.asarray(dims, np.int32), 0, 4, 8)
    ln = torch.ones(8, dtype=torch.int32, device="cuda")
    plan.build(ln)
    idx = torch.zeros(8, dtype=torch.int32, device="cuda")
    out = torch.empty((4, 40), device="cuda")
    tabs = [torch.zeros((10, 16), device="cuda") for _ in range(2)]
    ptrs = torch.tensor([t.data_ptr() for t in tabs], dtype=torch.int64, device="cuda")
    with pytest.raises(binding.DpiError) as e:   # weights + mean pooling
        plan.lookup_ex(ptrs, idx, out, pooling=[1, 0], weights_dev=torch.ones(8, device="cuda"))
    assert e.value.status == 2
    with pytest.raises(binding.DpiError) as e:   # pitch smaller than the row
        plan.lookup_ex(ptrs, idx, out, out_ld=16)
    assert e.value.status == 1
    with pytest.raises(binding.DpiError) as e:   # pitch that breaks 16-byte row alignment
        plan.lookup_ex(ptrs, idx, out, out_ld=33)
    assert e.value.status == 1
    with pytest.raises(binding.DpiError):
        plan.set_layout(2, 0)
    with pytest.raises(binding.DpiError):
        plan.set_layout(0, 5)
    plan.set_layout(binding.BAGS_TABLE_MAJOR, binding.IDX_I32)
    with pytest.raises(binding.DpiError) as e:   # the ablation kernel knows only the plain layout
        plan.lookup_input_first(ptrs, idx, out)
    assert e.value.status == 2
    plan.destroy()


# --------------------------------------------------------------------------------------------------
# NEXT-3: table-wise sharding with the all-to-all fused into the lookup's store (dpi_lookup_ex out_peers_dev)
# --------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("world", [1, 2, 3])
@pytest.mark.parametrize("dtype,out", [("f32", None), ("bf16", "f32"), ("f16", None)])
def test_table_wise_shards_scatter_into_peer_batch_shards(world, dtype, out):
    """`world` table shards take turns on this one GPU (no kernel waits on another: each is an ordinary launch); the
    "peers" are `world` separate device buffers, one batch shard each. Every shard's kernel stores its tables' column
    blocks into the buffer that owns the sample; afterwards the stacked buffers must be the oracle's global block."""
    from paper_2606_21101_b200 import sharding
    out = out or dtype
    dims = [16, 8, 32, 8, 16, 64, 8] if dtype == "f32" else [16, 8, 32, 8, 16, 64, 24]
    T, B = len(dims), 203
    rows = [50, 7, 400, 90, 3, 1000, 12]
    cfg = W.Config("tw", T, tuple(rows), max(dims), dtype, B, ("poisson", 5.0, 30, 0.1), ("zipf", 1.1), "sum", seed=6)
    glob = W.make_batch(cfg, np.asarray(rows, np.int64), 9)
    host_tables = W.mixed_dim_tables(cfg.seed, dims, rows, dtype)
    pooling = np.array([0, 1, 0, 1, 0, 1, 0], np.uint8)
    ref = oracle.lookup_general(host_tables, W.DTYPE_CODE[dtype], B, glob.indices, host_offsets(glob.lengths).astype(np.int64), pooling)

    width = int(sum(dims))
    rows_per_rank = -(-B // world)
    shards = [torch.full((rows_per_rank, width), float("nan"), dtype=TORCH_OUT[out], device="cuda") for _ in range(world)]
    peers = torch.tensor([s.data_ptr() for s in shards], dtype=torch.int64, device="cuda")
    cols = sharding.table_columns(dims)
    parts = sharding.partition_tables(np.asarray(dims, float), world)
    keep = []
    for mine in parts:
        if not mine:
            continue
        local = sharding.table_shard_batch(glob, T, mine)
        tables, ptrs = harness.tables_from_host_mixed([host_tables[t] for t in mine], dtype)
        plan = binding.Plan([rows[t] for t in mine], np.asarray([dims[t] for t in mine], np.int32), W.DTYPE_CODE[dtype], B,
                            max(local.N, 1))
        if out != dtype:
            plan.set_out_dtype(W.DTYPE_CODE[out])
        plan.set_columns(cols[mine])
        ln = torch.from_numpy(local.lengths).cuda()
        idx = torch.from_numpy(local.indices if local.N else np.zeros(1, np.int32)).cuda()
        plan.build(ln)
        plan.lookup_ex(ptrs, idx, None, pooling=pooling[mine], out_ld=width, out_peers_dev=peers, n_peers=world,
                       rows_per_peer=rows_per_rank)
        keep.append((plan, tables, ln, idx))
    torch.cuda.synchronize()
    got = torch.cat(shards, dim=0)[:B]
    L_bt = glob.lengths.reshape(B, T)
    assert_outputs_match_general(harness.out_to_f64(got), ref, L_bt, dims, dtype, out)
    for plan, *_ in keep:
        plan.destroy()


def test_set_columns_validation_and_reset():
    plan = binding.Plan([10, 10], np.asarray([16, 8], np.int32), 0, 4, 8)
    assert plan.plan_out_width() == 24
    plan.set_columns([32, 0])
    assert plan.plan_out_width() == 48
    with pytest.raises(binding.DpiError):
        plan.set_columns([2, 0])       # 8-byte aligned column
    with pytest.raises(binding.DpiError):
        plan.set_columns([-4, 0])
    plan.set_columns(None)
    assert plan.plan_out_width() == 24
    plan.destroy()


def test_general_kernel_at_the_maximum_table_count():
    """T = DPI_MAX_TABLES with mixed dims, weights and int64 ids: 32 KB of per-table records + the per-warp staging
    exceed the default 48 KB of dynamic shared memory, so this also covers the opt-in path of the launch."""
    T = 2048
    dims = [8 if t % 3 else 16 for t in range(T)]
    rows = [int(t * 5 % 11 + 1) for t in range(T)]
    _run(dims, rows, 3, "bf16", ("uniform", 0, 3), out_dtype="f32", idx64=True, weighted=True, K=64)
    _run([d // 2 for d in dims], rows, 2, "f32", ("const", 1), table_major=True, pooling=[t & 1 for t in range(T)])


@pytest.mark.parametrize("lengths", [("const", 1), ("uniform", 0, 3), ("poisson", 20.0, 100, 0.05)])
@pytest.mark.parametrize("dtype,out", [("f32", None), ("bf16", "f32"), ("f16", None)])
def test_int64_ids_through_the_short_bag_variant(dtype, out, lengths):
    """DPI_OPT_MODE = 6 with int64 ids: the short-bag variant reads the low words itself instead of falling back to the
    general kernel; equal dims (the variant's precondition)."""
    D = 16 if dtype == "f32" else 32
    _run([D] * 7, [1000, 50, 7, 3000, 1, 640, 99], 333, dtype, lengths, out_dtype=out, idx64=True, mode=6,
         pooling=[0, 1, 0, 1, 1, 0, 1])


# --------------------------------------------------------------------------------------------------
# NEXT-2 completion: 64-bit offsets (dpi_plan_set_offset_type; DESIGN.md 11.2 V6)
# --------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("lengths", LENGTHS + [("uniform", 0, 300)])
@pytest.mark.parametrize("dtype,out", [("f32", None), ("f16", None), ("bf16", "f32")])
@pytest.mark.parametrize("K", [0, 7, 1000])
def test_64bit_offsets_plan_and_lookup_match_the_oracle(dtype, out, lengths, K):
    """Same inputs as the 32-bit tests, the plan kept in int64: offsets / seg_off / S bit-exact against oracle.plan64, the block
    against the oracle; staged tasks, tasks too large for the staging buffers (U{0..300} bags at K = 1000) and K = 7."""
    D = 16 if dtype == "f32" else 32
    _run([D] * 5, [1000, 17, 4000, 1, 250], 333, dtype, lengths, out_dtype=out, off64=True, K=K, pooling=[0, 1, 0, 1, 1])


def test_64bit_offsets_with_every_other_variant_and_through_dpi_forward():
    dims, rows = [16, 8, 32, 8, 24], [50, 7, 400, 90, 3]
    _run(dims, rows, 257, "f32", ("uniform", 0, 9), off64=True, idx64=True, weighted=True, explicit_offsets=True)
    _run(dims, rows, 129, "bf16", ("poisson", 20.0, 100, 0.05), out_dtype="f32", off64=True, table_major=True, out_ld=128,
         pooling=[1, 0, 1, 0, 1])
    _run([32] * 4, rows[:4], 64, "f16", ("const", 0), off64=True)          # all bags empty
    _run([16], [9], 1, "f32", ("const", 5000), off64=True, K=32)            # one long bag across many quanta
    # dpi_forward on a 64-bit plan = 64-bit planner (two launches) + general lookup; dpi_forward_host refuses
    cfg = W.Config("f64", 3, (100, 20, 7), 16, "f32", 50, ("uniform", 0, 6), ("uniform",), "half", 5)
    rows3 = cfg.table_rows()
    host_tables = [W.full_table_storage(cfg, t, int(rows3[t])) for t in range(cfg.T)]
    dt = harness.tables_from_host(cfg, host_tables)
    batch = W.make_batch(cfg, rows3, None)
    db = harness.upload_batch(batch)
    plan = harness.make_plan(cfg, rows3, max(batch.N, 1))
    plan.set_offset_type(binding.OFF_I64, 1 << 33)
    out = harness.new_output(cfg, fill_nan=True)
    before = binding.launch_count()
    plan.forward(db.lengths, dt.ptrs, db.indices, out, pooling=cfg.pooling_modes())
    assert binding.launch_count() - before == 3
    torch.cuda.synchronize()
    ref = oracle.lookup_general(host_tables, oracle.F32, cfg.B, batch.indices, host_offsets(batch.lengths).astype(np.int64),
                                cfg.pooling_modes())
    assert_outputs_match_general(harness.out_to_f64(out), ref, batch.lengths.reshape(cfg.B, cfg.T), [cfg.D] * cfg.T, "f32", "f32")
    with pytest.raises(binding.DpiError) as e:
        plan.forward_host(dt.ptrs, torch.from_numpy(batch.lengths), torch.from_numpy(batch.indices),
                          torch.empty((cfg.B, cfg.T * cfg.D)))
    assert e.value.status == 2
    plan.set_offset_type(binding.OFF_I32, max(batch.N, 1))   # and back: the 32-bit single-launch planner again
    plan.build(db.lengths)
    assert plan.export()[3] == batch.N
    plan.destroy()


def test_64bit_offsets_with_more_than_2_pow_31_index_entries():
    """N = 2^31 + 2^18 entries in one batch (int32 ids: 8.6 GB on the device): 8192 bags of 262 176 entries over two tiny
    tables of 16-byte rows. Offsets beyond 2^31 must be exact (plan vs closed form and vs oracle.plan64) and the pooled
    block must match the oracle, which walks all 2.1e9 entries once."""
    free, _ = torch.cuda.mem_get_info()
    if free < 24 << 30:
        pytest.skip("needs 24 GB of free device memory")
    B, T, L = 4096, 2, 262176
    G = B * T
    N = G * L
    assert N > (1 << 31)
    rows = [1000, 37]
    rng = np.random.default_rng(7)
    lengths = np.full(G, L, np.int32)
    lengths[5] -= 3; lengths[6] += 3; lengths[G - 1] -= 1; lengths[0] += 1           # not all equal
    block = rng.integers(0, 37, size=1 << 20).astype(np.int32)                        # valid for either table
    idx = np.tile(block, N // block.size + 1)[:N]
    tables = [(rng.integers(-8, 9, size=(r, 4)) / 64.0).astype(np.float32) for r in rows]   # sums stay exact in fp32
    off = np.concatenate(([0], np.cumsum(lengths.astype(np.int64))))
    plan = binding.Plan(rows, np.asarray([4, 4], np.int32), 0, B, 1)
    plan.set_offset_type(binding.OFF_I64, N)
    dev_tables, ptrs = harness.tables_from_host_mixed(tables, "f32")
    ln_dev = torch.from_numpy(lengths).cuda()
    idx_dev = torch.from_numpy(idx).cuda()
    plan.build(ln_dev)
    g_off, g_seg, S, g_N, g_seg_off = plan.export64()
    assert g_N == N and np.array_equal(g_off, off)
    o_off, o_seg, o_S, o_seg_off = oracle.plan64(lengths, plan.info()["K"])
    assert S == o_S and np.array_equal(g_seg, o_seg) and np.array_equal(g_seg_off, o_seg_off)
    assert plan.check_indices(idx_dev) == 0
    out = torch.full((B, 8), float("nan"), dtype=torch.float32, device="cuda")
    pooling = np.array([0, 1], np.uint8)
    plan.lookup_ex(ptrs, idx_dev, out, pooling=pooling)
    torch.cuda.synchronize()
    got = harness.out_to_f64(out)
    del idx_dev
    ref = oracle.lookup_general(tables, oracle.F32, B, idx, off, pooling)
    # multiples of 1/64 with |sum| < 2^18 * 1/8: every partial sum is exactly representable in fp32 -> sum pooling exact
    assert np.array_equal(got[:, :4], ref[:, :4])
    assert np.allclose(got[:, 4:], ref[:, 4:], rtol=1e-6, atol=1e-7)
    plan.destroy()
