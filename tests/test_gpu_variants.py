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
         pooling=None, out_ld=0, K=0, force_general=False, mode=0):
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
    width = int(np.sum(dims))
    assert plan.plan_out_width() == width
    ld = out_ld or width
    out = torch.full((B, ld), float("nan"), dtype=TORCH_OUT[out_dtype], device="cuda")
    plan.lookup_ex(ptrs, idx_dev, out, pooling=pooling, weights_dev=wgt_dev, out_ld=out_ld,
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
