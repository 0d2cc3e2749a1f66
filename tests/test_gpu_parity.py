"""GPU parity tests proper (`-m gpu`): the CUDA path, called through the C ABI, against the CPU oracle on the
same seeded inputs. Plan: bit-exact. Outputs: north_star tolerances (tests/parity.py)."""
import numpy as np
import pytest
import torch

import oracle
from paper_2606_21101_b200 import binding, harness, workloads as W
from tests.parity import assert_outputs_match, host_offsets, oracle_reference

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module", autouse=True)
def _lib():
    from paper_2606_21101_b200 import build
    build.build()
    binding.load_library()
    harness.require_cuda()


# --------------------------------------------------------------------------------------------------
# generator: host and device implementations of the same counter-based recipe agree bit for bit
# --------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("dtype", ["f32", "f16", "bf16"])
def test_synth_fill_matches_host_generator(dtype):
    cfg = W.Config("g", 2, (3001, 517), 32, dtype, 4, ("const", 1), ("uniform",), "sum", seed=5)
    dt = harness.make_device_tables(cfg)
    for t in range(cfg.T):
        want = W.full_table_storage(cfg, t, int(dt.rows[t]))
        got = dt.tables[t].cpu()
        got = got.view(torch.int16).numpy().view(np.uint16) if dtype != "f32" else got.numpy()
        want = want.view(np.uint16) if dtype != "f32" else want
        assert np.array_equal(got, want)


# --------------------------------------------------------------------------------------------------
# plan (a1 + a2): bit-exact
# --------------------------------------------------------------------------------------------------
def _plan_parity(lengths: np.ndarray, T: int, B: int, K: int, max_indices=None):
    N = int(lengths.astype(np.int64).sum())
    plan = binding.Plan([10] * T, 16, binding.DPI_F32, B, N if max_indices is None else max_indices)
    plan.set_quantum(K)
    dev = torch.from_numpy(np.ascontiguousarray(lengths, dtype=np.int32)).cuda()
    for _ in range(2):  # the second build reuses the look-back status words (epoch tagging)
        plan.build(dev)
        off, seg, S, n, seg_off = plan.export(with_seg_off=True)
        o_off, o_seg, o_S, o_seg_off = oracle.plan(lengths, K, with_seg_off=True)
        assert n == N and S == o_S
        assert np.array_equal(off, o_off)
        assert np.array_equal(seg, o_seg)
        assert np.array_equal(seg_off, o_seg_off)
        assert plan.stats() == oracle.plan_stats(lengths)      # a1's min / max bag length
        assert plan.status() == 0                              # nothing overflowed
    plan.destroy()


@pytest.mark.parametrize("K", [1, 3, 32, 64, 1000])
def test_plan_small_ragged(K):
    rng = np.random.default_rng(K)
    for T, B in [(1, 1), (3, 7), (4, 128), (5, 1000), (7, 2049 // 7 + 1)]:
        ln = rng.integers(0, 9, size=T * B).astype(np.int32)
        _plan_parity(ln, T, B, K)


@pytest.mark.parametrize("name", ["c1", "c2", "c3", "c4", "c5"])
@pytest.mark.parametrize("K", [32, 48])
def test_plan_full_size_configs(name, K):
    cfg = W.CONFIGS[name]
    ln = W.make_lengths(cfg, cfg.seed)
    _plan_parity(ln, cfg.T, cfg.B, K)


def test_plan_degenerate_cases():
    _plan_parity(np.zeros(5000, np.int32), 5, 1000, 32)               # all empty
    _plan_parity(np.array([100000], np.int32), 1, 1, 32)              # one long bag spans many quanta
    ln = np.zeros(4099, np.int32); ln[0] = 7; ln[-1] = 900; ln[2048] = 33
    _plan_parity(ln, 1, 4099, 16)                                     # tile boundaries, ragged tail
    _plan_parity(np.full(2048 * 3, 1, np.int32), 3, 2048, 32)         # exact multiple of the scan tile
    _plan_parity(np.full(10, 64, np.int32), 2, 5, 7)                  # K does not divide anything


def test_plan_many_tiles_lookback_window():
    """More than 32 tiles behind: the look-back window has to slide."""
    rng = np.random.default_rng(3)
    B, T = 40000, 5  # 200000 bags = 98 tiles
    ln = rng.integers(0, 5, size=B * T).astype(np.int32)
    _plan_parity(ln, T, B, 32)


def test_plan_overflow_is_reported_not_out_of_bounds():
    ln = np.full(100, 10, np.int32)
    plan = binding.Plan([10], 16, binding.DPI_F32, 100, 500)  # capacity 500 < N = 1000
    plan.build(torch.from_numpy(ln).cuda())
    with pytest.raises(binding.DpiError) as e:
        plan.export()
    assert e.value.status == 1 and "max_indices" in e.value.detail
    # ... and without exporting anything: the sticky device counter (dpi_plan_status) counts overflowed builds once
    plan.build(torch.from_numpy(ln).cuda())
    assert plan.status() == 2
    assert plan.status() == 0
    # N = max_indices + 1: the segment buffer (sized for max_indices + G) still has room, the plan is marked S = 0 all the same
    one_over = np.full(100, 5, np.int32)
    one_over[17] = 6
    plan.build(torch.from_numpy(one_over).cuda())
    _, _, meta_ptr = plan.device_views()
    meta = torch.zeros(12, dtype=torch.int32, device="cuda")
    binding.copy_device_words(meta, meta_ptr, 12)
    meta = meta.cpu().numpy()
    assert meta[0] == 0 and meta[1] == 501 and meta[3] == 1      # S, N, overflow flag
    assert plan.status() == 1
    ok = np.full(100, 5, np.int32)
    plan.build(torch.from_numpy(ok).cuda())
    assert plan.status() == 0 and plan.export()[3] == 500
    plan.destroy()


# --------------------------------------------------------------------------------------------------
# lookup (a3)
# --------------------------------------------------------------------------------------------------
def _run_gpu(cfg, dt, batch, pooling, K=0, opts=None, via_explicit_offsets=False, input_first=False):
    db = harness.upload_batch(batch)
    # no bag-length hint by default: these tests are about the balanced-segment kernel on every bag shape; the short-bag
    # variant has its own tests (mode 6 / DPI_OPT_MAX_BAG_HINT) further down
    plan = harness.make_plan(cfg, dt.rows, max(batch.N, 1), bag_hint=bool((opts or {}).get("bag_hint", False)))
    broken_promise = bool((opts or {}).get("broken_promise", False))   # the bag-length hint is violated on purpose
    opts = {k: v for k, v in (opts or {}).items() if k not in ("bag_hint", "broken_promise")}
    if K:
        plan.set_quantum(K)
    for k, v in (opts or {}).items():
        plan.set_option(k, v)
    plan.build(db.lengths)
    if broken_promise:
        with pytest.raises(binding.DpiError):
            plan.check_indices(db.indices)
    else:
        assert plan.check_indices(db.indices) == 0
    out = harness.new_output(cfg, fill_nan=True)
    off_dev = None
    if via_explicit_offsets:
        off_dev = torch.from_numpy(host_offsets(batch.lengths)).cuda()
    if input_first:
        plan.lookup_input_first(dt.ptrs, db.indices, out, pooling=pooling, offsets_dev=off_dev)
    else:
        plan.lookup(dt.ptrs, db.indices, out, pooling=pooling, offsets_dev=off_dev)
    torch.cuda.synchronize()
    res = harness.out_to_f64(out)
    plan.destroy()
    return res


def _full_parity(cfg, K=0, opts=None, batch_seed=None, pooling=None, input_first=False):
    rows = cfg.table_rows()
    host_tables = [W.full_table_storage(cfg, t, int(rows[t])) for t in range(cfg.T)]
    dt = harness.tables_from_host(cfg, host_tables)
    batch = W.make_batch(cfg, rows, batch_seed)
    pooling = cfg.pooling_modes() if pooling is None else pooling
    got = _run_gpu(cfg, dt, batch, pooling, K, opts, input_first=input_first)
    ref = oracle_reference(host_tables, cfg.dtype, cfg.B, batch.lengths, batch.indices, pooling)
    return assert_outputs_match(got, ref, batch.lengths, cfg.T, cfg.D, cfg.dtype, cfg.out)


def test_c1_exact_config():
    _full_parity(W.C1)


@pytest.mark.parametrize("dtype,D,out", [("f32", 4, None), ("f32", 16, None), ("f32", 24, None), ("f32", 64, None),
                                         ("f32", 128, None),
                                         ("f16", 8, None), ("f16", 32, None), ("f16", 72, None), ("f16", 256, None),
                                         ("f16", 8, "f32"), ("f16", 64, "f32"),
                                         ("bf16", 8, None), ("bf16", 64, None), ("bf16", 128, None), ("bf16", 256, None),
                                         ("bf16", 8, "f32"), ("bf16", 24, "f32"), ("bf16", 64, "f32"), ("bf16", 256, "f32")])
@pytest.mark.parametrize("lengths", [("const", 1), ("uniform", 1, 4), ("poisson", 20.0, 100, 0.05)])
def test_shapes_dtypes_and_length_mixes(dtype, D, out, lengths):
    """Several tiles, a ragged tail, every lanes-per-row instantiation (incl. non-power-of-two row sizes),
    mixed sum/mean pooling, empty bags, both output types of the 16-bit tables."""
    cfg = W.Config("s", 5, (1000, 17, 4000, 1, 250), D, dtype, 333, lengths, ("zipf", 1.05), "half", seed=11,
                   out_dtype=out)
    _full_parity(cfg)


@pytest.mark.parametrize("unroll", [2, 4, 8, 16])
@pytest.mark.parametrize("mode", [0, 1, 2, 3])
def test_every_kernel_variant_gives_the_same_answer(unroll, mode):
    cfg = W.Config("v", 6, (500, 30, 2000, 7, 100, 1000), 64, "f32", 257, ("uniform", 0, 70), ("uniform",), "half", 3)
    _full_parity(cfg, K=32, opts={binding.OPT_UNROLL: unroll, binding.OPT_MODE: mode})
    cfg16 = cfg.scaled(dtype="bf16", D=32, lengths=("uniform", 0, 5))
    _full_parity(cfg16, K=16, opts={binding.OPT_UNROLL: unroll, binding.OPT_MODE: mode, binding.OPT_BLOCK_THREADS: 128})


@pytest.mark.parametrize("K", [1, 5, 32, 200, 100000])
def test_any_quantum_gives_the_same_answer(K):
    cfg = W.Config("k", 3, (100, 1000, 10), 32, "f16", 500, ("poisson", 6.0, 40, 0.2), ("zipf", 1.2), "mean", 4)
    _full_parity(cfg, K=K)


@pytest.mark.parametrize("dtype,D,out", [("f32", 16, None), ("f32", 24, None), ("f16", 32, None), ("bf16", 64, "f32"),
                                         ("bf16", 8, None)])
@pytest.mark.parametrize("lengths", [("const", 1), ("uniform", 0, 5), ("poisson", 20.0, 100, 0.05)])
def test_input_first_ablation_kernel_matches_the_oracle(dtype, D, out, lengths):
    """The strawman mapping of PAPER.md:172-176 (one thread per sample) computes the same block."""
    cfg = W.Config("if", 5, (1000, 17, 4000, 1, 250), D, dtype, 333, lengths, ("zipf", 1.05), "half", seed=12,
                   out_dtype=out)
    _full_parity(cfg, input_first=True)


def test_input_first_c2_full_size_equals_output_first_bit_for_bit():
    """One-hot (the paper's case): both mappings are pure row copies, so the blocks are identical."""
    cfg = W.C2
    dt = harness.make_device_tables(cfg)
    batch = W.make_batch(cfg, dt.rows)
    a = _run_gpu(cfg, dt, batch, cfg.pooling_modes())
    b = _run_gpu(cfg, dt, batch, cfg.pooling_modes(), input_first=True)
    assert np.array_equal(a, b)


def test_degenerate_inputs():
    # all bags empty -> zero matrix, N = 0
    cfg = W.Config("e", 3, (5, 5, 5), 16, "f32", 64, ("const", 0), ("uniform",), "mean", 0)
    _full_parity(cfg)
    # single sample, single table, one long bag (spans many quanta)
    cfg = W.Config("l", 1, (1000,), 64, "f32", 1, ("const", 5000), ("uniform",), "mean", 0)
    _full_parity(cfg, K=32)
    # B = 1, many tables
    cfg = W.Config("b1", 100, ("loguniform", 10, 1000), 16, "bf16", 1, ("uniform", 0, 3), ("uniform",), "half", 2)
    _full_parity(cfg)
    # one-row tables: every index is 0
    cfg = W.Config("r1", 4, (1, 1, 1, 1), 32, "f32", 77, ("uniform", 0, 9), ("uniform",), "sum", 2)
    _full_parity(cfg)


def test_first_and_last_bag_empty_and_explicit_offsets():
    cfg = W.Config("x", 2, (50, 60), 16, "f32", 40, ("uniform", 1, 4), ("uniform",), "sum", 9)
    rows = cfg.table_rows()
    host_tables = [W.full_table_storage(cfg, t, int(rows[t])) for t in range(cfg.T)]
    dt = harness.tables_from_host(cfg, host_tables)
    batch = W.make_batch(cfg, rows)
    ln = batch.lengths.copy()
    off = host_offsets(ln)
    keep = np.ones(batch.N, bool)
    keep[off[0]:off[1]] = False
    keep[off[-2]:off[-1]] = False
    ln[0] = 0
    ln[-1] = 0
    b2 = W.Batch(ln, batch.indices[keep])
    pooling = np.array([1, 0], np.uint8)
    got = _run_gpu(cfg, dt, b2, pooling, via_explicit_offsets=True)
    ref = oracle_reference(host_tables, cfg.dtype, cfg.B, b2.lengths, b2.indices, pooling)
    assert_outputs_match(got, ref, b2.lengths, cfg.T, cfg.D, cfg.dtype)


def test_onehot_is_alg1_bit_exact_with_index_encoding_tables():
    """Alg. 1: every output element decodes to its own (t, IDs[b,t], c)."""
    T, B, D = 7, 1000, 16
    rows = [7, 300, 1, 4095, 64, 4096, 33]
    tables = [(t * 65536 + np.arange(rows[t])[:, None] * 16 + np.arange(D)[None, :]).astype(np.float32)
              for t in range(T)]
    cfg = W.Config("enc", T, tuple(rows), D, "f32", B, ("const", 1), ("uniform",), "sum", 1)
    dt = harness.tables_from_host(cfg, tables)
    batch = W.make_batch(cfg, np.asarray(rows, np.int64))
    got = _run_gpu(cfg, dt, batch, np.zeros(T, np.uint8)).astype(np.int64).reshape(B, T, D)
    ids = batch.indices.reshape(B, T)
    assert np.array_equal(got >> 16, np.broadcast_to(np.arange(T)[None, :, None], (B, T, D)))
    assert np.array_equal((got >> 4) & 0xFFF, np.broadcast_to(ids[:, :, None], (B, T, D)))
    assert np.array_equal(got & 0xF, np.broadcast_to(np.arange(D)[None, None, :], (B, T, D)))
    want = oracle.alg1_onehot(tables, oracle.F32, ids)
    assert np.array_equal(got.reshape(B, T * D).astype(np.float64), want)


@pytest.mark.parametrize("dtype", ["f16", "bf16"])
def test_16bit_exactly_representable_values_are_bit_exact(dtype):
    rng = np.random.default_rng(10)
    T, B, D = 3, 300, 32
    rows = [12, 100, 5]
    ks = [rng.integers(-3, 4, size=(rows[t], D)) for t in range(T)]
    host_tables = [W.to_storage((k / 1024.0).astype(np.float32), dtype) for k in ks]
    cfg = W.Config("x16", T, tuple(rows), D, dtype, B, ("uniform", 0, 64), ("uniform",), "sum", 6)
    dt = harness.tables_from_host(cfg, host_tables)
    batch = W.make_batch(cfg, np.asarray(rows, np.int64))
    got = _run_gpu(cfg, dt, batch, np.zeros(T, np.uint8))
    ref = oracle_reference(host_tables, dtype, B, batch.lengths, batch.indices, np.zeros(T, np.uint8))
    assert np.array_equal(got, ref)


def test_check_indices_counts_out_of_range():
    cfg = W.Config("oob", 2, (10, 20), 16, "f32", 8, ("const", 2), ("uniform",), "sum", 0)
    batch = W.make_batch(cfg)
    idx = batch.indices.copy()
    idx[0] = 10      # table 0 has rows 0..9
    idx[3] = -1
    idx[5] = 19      # fine for table 0? entry 5 belongs to bag 2 = (b=1,t=0) -> 19 >= 10 is bad
    db = harness.upload_batch(W.Batch(batch.lengths, idx))
    plan = harness.make_plan(cfg, cfg.table_rows(), batch.N)
    plan.build(db.lengths)
    assert plan.check_indices(db.indices) == 3
    plan.destroy()


def test_forward_host_equals_device_path():
    cfg = W.Config("h", 4, (100, 2000, 50, 7), 32, "bf16", 513, ("uniform", 0, 6), ("zipf", 1.1), "half", 8)
    rows = cfg.table_rows()
    host_tables = [W.full_table_storage(cfg, t, int(rows[t])) for t in range(cfg.T)]
    dt = harness.tables_from_host(cfg, host_tables)
    batch = W.make_batch(cfg, rows)
    pooling = cfg.pooling_modes()
    dev = _run_gpu(cfg, dt, batch, pooling)
    plan = harness.make_plan(cfg, rows, harness.max_indices_bound(cfg))
    ln = torch.from_numpy(batch.lengths).pin_memory()
    idx = torch.from_numpy(batch.indices).pin_memory()
    out = torch.empty((cfg.B, cfg.T * cfg.D), dtype=torch.bfloat16).pin_memory()
    plan.forward_host(dt.ptrs, ln, idx, out, pooling=pooling)
    assert np.array_equal(out.double().numpy(), dev)
    ref = oracle_reference(host_tables, cfg.dtype, cfg.B, batch.lengths, batch.indices, pooling)
    assert_outputs_match(out.double().numpy(), ref, batch.lengths, cfg.T, cfg.D, cfg.dtype, cfg.out)   # and against the oracle
    # the pipelined variant (chunks of whole samples over three streams) gives the same block, ragged last chunk included
    for chunks in (2, 3, 7, 64):
        plan.set_option(binding.OPT_HOST_CHUNKS, chunks)
        out.fill_(float("nan"))
        plan.forward_host(dt.ptrs, ln, idx, out, pooling=pooling)
        assert np.array_equal(out.double().numpy(), dev), f"{chunks} chunks"
    # output path: staged block + D2H copy (1) and the lookup storing straight into the pinned host block (2, and what
    # auto picked above) give the same bytes, pipelined or not
    for direct in (1, 2):
        plan.set_option(binding.OPT_HOST_DIRECT_OUT, direct)
        for chunks in (1, 5):
            plan.set_option(binding.OPT_HOST_CHUNKS, chunks)
            out.fill_(float("nan"))
            plan.forward_host(dt.ptrs, ln, idx, out, pooling=pooling)
            assert np.array_equal(out.double().numpy(), dev), f"direct_out={direct}, {chunks} chunks"
    pageable = torch.empty((cfg.B, cfg.T * cfg.D), dtype=torch.bfloat16)
    with pytest.raises(binding.DpiError):   # "require direct" on memory the device cannot store into
        plan.forward_host(dt.ptrs, ln, idx, pageable, pooling=pooling)
    plan.set_option(binding.OPT_HOST_DIRECT_OUT, 0)
    plan.set_option(binding.OPT_HOST_CHUNKS, 0)
    # pageable host memory works as well
    out2 = torch.empty((cfg.B, cfg.T * cfg.D), dtype=torch.bfloat16)
    plan.forward_host(dt.ptrs, torch.from_numpy(batch.lengths), torch.from_numpy(batch.indices), out2, pooling=pooling)
    assert np.array_equal(out2.double().numpy(), dev)
    with pytest.raises(binding.DpiError):  # lengths that do not add up to n_indices are caught before any copy
        plan.forward_host(dt.ptrs, ln, idx[:-1].clone().pin_memory(), out, pooling=pooling)
    plan.destroy()


def test_c4_with_bf16_output_meets_the_derived_bound():
    """Same workload as c4 but the output block in bf16 (the table dtype): held to 2^-8 relative (R6)."""
    _sampled_full_size(W.C4.scaled(out_dtype=None, B=1024), 256)


def test_out_dtype_validation():
    plan = binding.Plan([10], 16, binding.DPI_F16, 4, 10)
    plan.set_out_dtype(binding.DPI_F32)
    plan.set_out_dtype(binding.DPI_F16)
    with pytest.raises(binding.DpiError) as e:
        plan.set_out_dtype(binding.DPI_BF16)
    assert e.value.status == 2
    plan.destroy()


# --------------------------------------------------------------------------------------------------
# BASELINE.json configs at full size, in the launch configuration bench.py times (library defaults)
# --------------------------------------------------------------------------------------------------
def _sampled_full_size(cfg, n_samples, rotate=1):
    dt = harness.make_device_tables(cfg)
    rng = np.random.default_rng(123)
    worst = 0.0
    for r in range(rotate):
        batch = W.make_batch(cfg, dt.rows, cfg.seed + r)
        pooling = cfg.pooling_modes()
        got = _run_gpu(cfg, dt, batch, pooling)
        # properties that hold at any size: written everywhere, empty bags are +0.0
        L = batch.lengths.reshape(cfg.B, cfg.T)
        g3 = got.reshape(cfg.B, cfg.T, cfg.D)
        assert not np.isnan(got).any()
        assert not g3[L == 0].any()
        samples = np.sort(rng.choice(cfg.B, size=min(n_samples, cfg.B), replace=False))
        samples[0] = 0
        samples[-1] = cfg.B - 1  # both ends of the batch (first and last warp-task)
        sub = W.compact_subproblem(cfg, batch, samples)
        ref = oracle.lookup(sub.tables, W.DTYPE_CODE[cfg.dtype], len(samples), sub.indices,
                            host_offsets(sub.lengths), pooling)
        worst = max(worst, assert_outputs_match(got[samples], ref, sub.lengths, cfg.T, cfg.D, cfg.dtype, cfg.out))
    del dt
    torch.cuda.empty_cache()
    return worst


def test_c2_full_size_every_sample():
    _sampled_full_size(W.C2, W.C2.B, rotate=2)


def test_c3_full_size_every_sample():
    _sampled_full_size(W.C3, W.C3.B)


def test_c4_full_size_sampled():
    _sampled_full_size(W.C4, 512)


def test_c5_full_size_sampled():
    free, _ = torch.cuda.mem_get_info()
    if free < 90e9:
        pytest.fail(f"config 5 needs ~82 GB of tables; only {free / 1e9:.0f} GB free on this device")
    _sampled_full_size(W.C5, 4096)


def _via_forward(cfg, dt, batch, pooling):
    """dpi_forward (what bench.py times for `value`): planner + lookup, or one fused launch, library defaults."""
    db = harness.upload_batch(batch)
    plan = harness.make_plan(cfg, dt.rows, max(batch.N, 1))
    out = harness.new_output(cfg, fill_nan=True)
    plan.forward(db.lengths, dt.ptrs, db.indices, out, pooling=pooling)
    torch.cuda.synchronize()
    res = harness.out_to_f64(out)
    plan.destroy()
    return res


def _via_forward_host(cfg, dt, batch, pooling, direct_out):
    """dpi_forward_host (the call behind bench.py's `e2e`): pinned host buffers, library-default chunking (c5: 8 sample chunks
    on three streams, first chunk a quarter of the rest), NaN-filled host block. direct_out: 0 = auto (the lookup stores
    straight into the pinned block over PCIe), 1 = staged block + D2H copy."""
    plan = harness.make_plan(cfg, dt.rows, max(batch.N, 1))
    plan.set_option(binding.OPT_HOST_DIRECT_OUT, direct_out)
    ln = torch.from_numpy(np.ascontiguousarray(batch.lengths)).pin_memory()
    idx = torch.from_numpy(np.ascontiguousarray(batch.indices)).pin_memory()
    out = torch.full((cfg.B, cfg.T * cfg.D), float("nan"), dtype=harness.TORCH_DTYPE[cfg.out]).pin_memory()
    plan.forward_host(dt.ptrs, ln, idx, out, pooling=pooling)
    res = out.to(torch.float64).numpy()
    plan.destroy()
    return res


def _every_sample_full_size(cfg, samples_per_pass):
    """Every output element of one full-size batch against the oracle, through every entry point bench.py times: dpi_plan_build +
    dpi_lookup, dpi_forward (`value`), dpi_forward_host with the library defaults and with the staged output (`e2e`). The tables do
    not fit on the host (c5) or are slow to mirror (c4), so the oracle works through the batch in passes of `samples_per_pass`
    samples, each on tables compacted to the rows that pass references (values recomputed from the counter-based generator,
    never read back from the device); each pass's reference is compared with all four blocks."""
    dt = harness.make_device_tables(cfg)
    batch = W.make_batch(cfg, dt.rows, cfg.seed)
    pooling = cfg.pooling_modes()
    gots = {"plan_build + lookup": _run_gpu(cfg, dt, batch, pooling),
            "forward": _via_forward(cfg, dt, batch, pooling),
            "forward_host (auto)": _via_forward_host(cfg, dt, batch, pooling, 0),
            "forward_host (staged out)": _via_forward_host(cfg, dt, batch, pooling, 1)}
    worst = 0.0
    for lo in range(0, cfg.B, samples_per_pass):
        samples = np.arange(lo, min(cfg.B, lo + samples_per_pass))
        sub = W.compact_subproblem(cfg, batch, samples)
        ref = oracle.lookup(sub.tables, W.DTYPE_CODE[cfg.dtype], len(samples), sub.indices, host_offsets(sub.lengths), pooling)
        for name, got in gots.items():
            try:
                worst = max(worst, assert_outputs_match(got[samples], ref, sub.lengths, cfg.T, cfg.D, cfg.dtype, cfg.out))
            except AssertionError as e:
                raise AssertionError(f"{name}, samples {lo}..{samples[-1]}: {e}") from e
    del dt
    torch.cuda.empty_cache()
    return worst


def test_c4_full_size_every_sample():
    _every_sample_full_size(W.C4, 1024)


def test_c5_full_size_every_sample():
    free, _ = torch.cuda.mem_get_info()
    if free < 90e9:
        pytest.fail(f"config 5 needs ~82 GB of tables; only {free / 1e9:.0f} GB free on this device")
    _every_sample_full_size(W.C5, 8192)


# --------------------------------------------------------------------------------------------------
# dpi_lookup_onehot: Algorithm 1 itself, no built plan
# --------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("dtype,D", [("f32", 4), ("f32", 16), ("f32", 24), ("f32", 64), ("f32", 128), ("f16", 8), ("f16", 32),
                                     ("bf16", 40), ("bf16", 64), ("bf16", 256)])
@pytest.mark.parametrize("B,T", [(1, 1), (5, 3), (333, 26), (2049, 7)])
def test_lookup_onehot_is_alg1_bit_exact(dtype, D, B, T):
    rows = tuple(int(r) for r in (np.arange(T) * 37 % 211 + 1))
    cfg = W.Config("oh", T, rows, D, dtype, B, ("const", 1), ("uniform",), "sum", 3)
    host_tables = [W.full_table_storage(cfg, t, rows[t]) for t in range(T)]
    dt = harness.tables_from_host(cfg, host_tables)
    batch = W.make_batch(cfg, np.asarray(rows, np.int64))
    ids = batch.indices.reshape(B, T)
    plan = harness.make_plan(cfg, dt.rows, batch.N)          # never built: Alg. 1 needs no plan
    out = harness.new_output(cfg, fill_nan=True)
    plan.lookup_onehot(dt.ptrs, torch.from_numpy(batch.indices).cuda(), out)
    torch.cuda.synchronize()
    want = oracle.alg1_onehot(host_tables, W.DTYPE_CODE[dtype], ids)
    assert np.array_equal(harness.out_to_f64(out), want)
    plan.destroy()


def test_lookup_onehot_c2_full_size_int64_ids_and_equals_the_planned_path():
    cfg = W.C2
    dt = harness.make_device_tables(cfg)
    batch = W.make_batch(cfg, dt.rows)
    host_tables = [W.full_table_storage(cfg, t, int(dt.rows[t])) for t in range(cfg.T)]
    want = oracle.alg1_onehot(host_tables, oracle.F32, batch.indices.reshape(cfg.B, cfg.T))
    planned = _run_gpu(cfg, dt, batch, cfg.pooling_modes())
    assert np.array_equal(planned, want)
    plan = harness.make_plan(cfg, dt.rows, batch.N)
    out = harness.new_output(cfg, fill_nan=True)
    plan.lookup_onehot(dt.ptrs, torch.from_numpy(batch.indices).cuda(), out)
    torch.cuda.synchronize()
    assert np.array_equal(harness.out_to_f64(out), want)
    plan.set_layout(binding.BAGS_SAMPLE_MAJOR, binding.IDX_I64)
    out.fill_(float("nan"))
    plan.lookup_onehot(dt.ptrs, torch.from_numpy(batch.indices.astype(np.int64)).cuda(), out)
    torch.cuda.synchronize()
    assert np.array_equal(harness.out_to_f64(out), want)
    plan.destroy()


def test_lookup_onehot_rejects_what_it_does_not_cover():
    cfg = W.Config("ohv", 2, (10, 10), 16, "bf16", 4, ("const", 1), ("uniform",), "sum", 3)
    dt = harness.make_device_tables(cfg)
    ids = torch.zeros(8, dtype=torch.int32, device="cuda")
    out = harness.new_output(cfg)
    plan = harness.make_plan(cfg, dt.rows, 8)
    plan.set_out_dtype(W.DTYPE_CODE["f32"])
    with pytest.raises(binding.DpiError) as e:
        plan.lookup_onehot(dt.ptrs, ids, out)
    assert e.value.status == 2
    plan.set_out_dtype(W.DTYPE_CODE["bf16"])
    plan.set_layout(binding.BAGS_TABLE_MAJOR, binding.IDX_I32)
    with pytest.raises(binding.DpiError):
        plan.lookup_onehot(dt.ptrs, ids, out)
    plan.set_layout(binding.BAGS_SAMPLE_MAJOR, binding.IDX_I32)
    with pytest.raises(binding.DpiError):
        plan.lookup_onehot(dt.ptrs, None, out)
    plan.lookup_onehot(dt.ptrs, ids, out)
    torch.cuda.synchronize()
    plan.destroy()


# --------------------------------------------------------------------------------------------------
# maximum sizes of the boundary (include/dpi.h): T = DPI_MAX_TABLES, table_rows = 2^31 - 1, 512-byte rows
# --------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("lengths", [("const", 1), ("uniform", 0, 3)])
def test_max_table_count_2048(lengths):
    """DPI_MAX_TABLES tables: the per-table pointer block in shared memory (16 KB), the 2048-bit pooling mask passed by
    value, the table id stepping across bags; B = 3 keeps the oracle quick. Mixed sum / mean pooling."""
    T = 2048
    rows = tuple(int(r) for r in (np.arange(T) * 7 % 13 + 1))
    cfg = W.Config("t2048", T, rows, 16, "f32", 3, lengths, ("uniform",), "half", seed=21)
    _full_parity(cfg)
    _full_parity(cfg.scaled(dtype="bf16", D=8, out_dtype="f32"), K=64)
    if lengths[0] == "const":       # Alg. 1 plan-free kernel at the same table count
        host_tables = [W.full_table_storage(cfg, t, rows[t]) for t in range(T)]
        dt = harness.tables_from_host(cfg, host_tables)
        batch = W.make_batch(cfg, np.asarray(rows, np.int64))
        plan = harness.make_plan(cfg, dt.rows, batch.N)
        out = harness.new_output(cfg, fill_nan=True)
        plan.lookup_onehot(dt.ptrs, torch.from_numpy(batch.indices).cuda(), out)
        torch.cuda.synchronize()
        assert np.array_equal(harness.out_to_f64(out), oracle.alg1_onehot(host_tables, oracle.F32, batch.indices.reshape(3, T)))
        plan.destroy()


def test_one_table_more_than_the_limit_is_refused():
    with pytest.raises(binding.DpiError) as e:
        binding.Plan([5] * 2049, np.full(2049, 16, np.int32), 0, 2, 10)
    assert e.value.status == 2


def test_max_table_height_row_ids_up_to_2_pow_31_minus_2():
    """One table of 2^31 - 1 rows x 16 B (34 GB): row ids need all 31 bits and byte offsets 35 bits. Only the referenced
    rows are given values on the device; the oracle sees the same rows compacted (ids remapped), so nothing it reads
    comes from the CUDA path. A second, small table checks the column block order next to it."""
    n_big = 2 ** 31 - 1
    free, _ = torch.cuda.mem_get_info()
    if free < 40 * 2 ** 30:
        pytest.skip("needs 40 GB of free device memory")
    D, B, T = 4, 64, 2
    big = torch.empty((n_big, D), dtype=torch.float32, device="cuda")      # uninitialised except the referenced rows
    small32 = W.dense_values_f32(3, 1, (10, D), 0.05)
    small = torch.from_numpy(small32).cuda()
    h = W.hash_u64(W.stream_key(8, W.STREAM_DENSE, 0), np.arange(3 * B, dtype=np.uint64))
    ids_big = (h % np.uint64(n_big)).astype(np.int64)
    ids_big[:6] = [0, 1, n_big - 1, n_big - 2, 2 ** 30, 2 ** 31 - 4097]     # the corners
    uniq, inv = np.unique(ids_big, return_inverse=True)
    vals32 = W.dense_values_f32(3, 2, (uniq.shape[0], D), 0.05)
    big[torch.from_numpy(uniq).cuda()] = torch.from_numpy(vals32).cuda()
    lengths = np.tile(np.array([3, 2], np.int32), B)                      # bag (b, big) has 3 entries, (b, small) 2
    ids_small = (W.hash_u64(W.stream_key(8, W.STREAM_DENSE, 1), np.arange(2 * B, dtype=np.uint64)) % np.uint64(10)).astype(np.int64)
    gpu_idx = np.empty(5 * B, np.int32)
    ora_idx = np.empty(5 * B, np.int32)
    for b in range(B):
        gpu_idx[5 * b: 5 * b + 3] = ids_big[3 * b: 3 * b + 3]
        ora_idx[5 * b: 5 * b + 3] = inv[3 * b: 3 * b + 3]
        gpu_idx[5 * b + 3: 5 * b + 5] = ora_idx[5 * b + 3: 5 * b + 5] = ids_small[2 * b: 2 * b + 2]
    ptrs = torch.tensor([big.data_ptr(), small.data_ptr()], dtype=torch.int64, device="cuda")
    pooling = np.array([1, 0], np.uint8)
    plan = binding.Plan([n_big, 10], np.array([D, D], np.int32), 0, B, 5 * B)
    plan.build(torch.from_numpy(lengths).cuda())
    idx_dev = torch.from_numpy(gpu_idx).cuda()
    assert plan.check_indices(idx_dev) == 0
    out = torch.full((B, T * D), float("nan"), device="cuda")
    plan.lookup(ptrs, idx_dev, out, pooling=pooling)
    torch.cuda.synchronize()
    ref = oracle_reference([vals32, small32], "f32", B, lengths, ora_idx, pooling)
    assert_outputs_match(harness.out_to_f64(out), ref, lengths, T, D, "f32")
    plan.destroy()
    del big


def test_widest_rows_512_bytes_full_warp_per_row():
    cfg = W.Config("w512", 3, (300, 5, 2000), 128, "f32", 515, ("poisson", 9.0, 60, 0.1), ("zipf", 1.05), "half", seed=5)
    _full_parity(cfg)
    _full_parity(cfg.scaled(dtype="f16", D=256, out_dtype="f32"))


# --------------------------------------------------------------------------------------------------
# DPI_OPT_MODE = 6: the short-bag variant (one lane group per bag straight from the plan's offsets, lookup_direct.cu)
# --------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("dtype,D,out", [("f32", 4, None), ("f32", 16, None), ("f32", 24, None), ("f32", 64, None), ("f32", 128, None),
                                         ("f16", 8, None), ("f16", 32, None), ("f16", 72, "f32"), ("bf16", 64, "f32"),
                                         ("bf16", 256, None)])
@pytest.mark.parametrize("lengths", [("const", 1), ("uniform", 0, 3), ("uniform", 1, 4), ("poisson", 20.0, 100, 0.05),
                                     ("const", 0)])
def test_direct_short_bag_variant_matches_the_oracle(dtype, D, out, lengths):
    """Same contract as the default kernel (tolerances of tests/parity.py, bit-exact for bags of length <= 1, +0.0 for empty
    bags), several tiles and a ragged tail; the Poisson(20) case checks that long bags are still correct here."""
    cfg = W.Config("d", 5, (1000, 17, 4000, 1, 250), D, dtype, 333, lengths, ("zipf", 1.05), "half", seed=12, out_dtype=out)
    _full_parity(cfg, opts={binding.OPT_MODE: 6})


def test_direct_short_bag_variant_full_size_c3_c2_c1_and_degenerate_shapes():
    _full_parity(W.C3, opts={binding.OPT_MODE: 6})
    _full_parity(W.C2, opts={binding.OPT_MODE: 6})
    _full_parity(W.C1, opts={binding.OPT_MODE: 6})
    _full_parity(W.Config("dl", 2, (1000, 50), 64, "f32", 3, ("const", 5000), ("uniform",), "mean", 0), opts={binding.OPT_MODE: 6})
    _full_parity(W.Config("d1", 100, ("loguniform", 10, 1000), 16, "bf16", 1, ("uniform", 0, 3), ("uniform",), "half", 2),
                 opts={binding.OPT_MODE: 6})
    T = 2048
    rows = tuple(int(r) for r in (np.arange(T) * 7 % 13 + 1))
    _full_parity(W.Config("dt", T, rows, 16, "f32", 3, ("uniform", 0, 3), ("uniform",), "half", seed=21), opts={binding.OPT_MODE: 6})


def test_bag_length_hint_selects_the_short_bag_variant_and_a_broken_promise_is_still_correct():
    """DPI_OPT_MAX_BAG_HINT is a promise about bag lengths; it only selects the kernel. c3 with its true bound (3), a config
    whose bags are far longer than the promised 2 (correct, just not load-balanced), and a hint above 8 (planned kernel)."""
    _full_parity(W.C3, opts={"bag_hint": True})
    cfg = W.Config("hp", 3, (100, 1000, 10), 32, "f16", 500, ("poisson", 6.0, 40, 0.2), ("zipf", 1.2), "mean", 4)
    _full_parity(cfg, opts={binding.OPT_MAX_BAG_HINT: 2, "broken_promise": True})
    _full_parity(cfg, opts={binding.OPT_MAX_BAG_HINT: 40})
    with pytest.raises(binding.DpiError):
        binding.Plan([5], 16, 0, 4, 10).set_option(binding.OPT_MAX_BAG_HINT, -1)
    # the promise is checkable off the hot path, like the index range
    rows = cfg.table_rows()
    batch = W.make_batch(cfg, rows)
    db = harness.upload_batch(batch)
    plan = harness.make_plan(cfg, rows, max(batch.N, 1), bag_hint=False)
    plan.build(db.lengths)
    longest = int(batch.lengths.max())
    plan.set_option(binding.OPT_MAX_BAG_HINT, longest)
    assert plan.check_indices(db.indices) == 0
    plan.set_option(binding.OPT_MAX_BAG_HINT, longest - 1)
    with pytest.raises(binding.DpiError) as e:
        plan.check_indices(db.indices)
    assert e.value.status == 1 and "DPI_OPT_MAX_BAG_HINT" in e.value.detail
    plan.destroy()


# --------------------------------------------------------------------------------------------------
# 256-bit row vectors (DPI_OPT_VEC_BYTES): every Wide<Traits> instantiation against the oracle
# --------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("dtype,D,out", [("f32", 8, None), ("f32", 16, None), ("f32", 24, None), ("f32", 64, None), ("f32", 128, None),
                                         ("f16", 16, None), ("f16", 48, None), ("f16", 64, "f32"), ("f16", 256, None),
                                         ("bf16", 16, "f32"), ("bf16", 64, None), ("bf16", 64, "f32"), ("bf16", 256, "f32")])
@pytest.mark.parametrize("lengths", [("const", 1), ("uniform", 0, 5), ("poisson", 20.0, 100, 0.05)])
@pytest.mark.parametrize("unroll", [0, 2, 8])
def test_256bit_row_vectors_match_the_oracle(dtype, D, out, lengths, unroll):
    """Rows of 32 ... 512 B (1 ... 16 lanes per row, incl. the non-power-of-two 96-byte row), all three task shapes and the
    device-picked short-bag body, table-dtype and fp32 output, one / two / four 256-bit loads per batch and lane."""
    cfg = W.Config("w", 5, (1000, 17, 4000, 1, 250), D, dtype, 333, lengths, ("zipf", 1.05), "half", seed=12, out_dtype=out)
    _full_parity(cfg, opts={binding.OPT_VEC_BYTES: 32, binding.OPT_UNROLL: unroll})


def test_256bit_row_vectors_modes_c5_shape_and_fallbacks():
    cfg = W.Config("w5", 8, (5000,) * 8, 64, "f32", 300, ("uniform", 1, 64), ("uniform",), "sum", seed=2)
    for mode in (0, 1, 2, 3):   # auto rule: fp32 rows of 256 B take the 256-bit kernel without being asked
        _full_parity(cfg, opts={binding.OPT_MODE: mode})
    _full_parity(cfg, opts={binding.OPT_VEC_BYTES: 16})
    _full_parity(cfg, K=7, opts={binding.OPT_VEC_BYTES: 32, binding.OPT_UNROLL: 16, binding.OPT_BLOCK_THREADS: 128})
    # rows that are not a multiple of 32 B cannot take 256-bit vectors; asking for them is refused, auto stays at 128 bit
    plan = binding.Plan([10, 10], np.asarray([12, 12], np.int32), 0, 4, 8)
    with pytest.raises(binding.DpiError) as e:
        plan.set_option(binding.OPT_VEC_BYTES, 32)
    assert e.value.status == 2
    plan.destroy()
    # an output block that is only 16-byte aligned silently runs the 128-bit kernel (same results)
    rows = cfg.table_rows()
    host_tables = [W.full_table_storage(cfg, t, int(rows[t])) for t in range(cfg.T)]
    dt = harness.tables_from_host(cfg, host_tables)
    batch = W.make_batch(cfg, rows, None)
    db = harness.upload_batch(batch)
    plan = harness.make_plan(cfg, rows, batch.N)
    plan.build(db.lengths)
    flat = torch.full((cfg.B * cfg.T * cfg.D + 4,), float("nan"), dtype=torch.float32, device="cuda")
    out = flat[4:].view(cfg.B, cfg.T * cfg.D)          # 16 bytes past a 512-byte aligned allocation
    assert out.data_ptr() % 32 == 16
    plan.lookup(dt.ptrs, db.indices, out, pooling=cfg.pooling_modes())
    torch.cuda.synchronize()
    ref = oracle_reference(host_tables, cfg.dtype, cfg.B, batch.lengths, batch.indices, cfg.pooling_modes())
    assert_outputs_match(harness.out_to_f64(out), ref, batch.lengths, cfg.T, cfg.D, cfg.dtype, cfg.out)
    plan.destroy()
