"""GPU parity tests (`-m gpu`) of the launch modes bench.py times and of the one-call path:

* dpi_forward (a1 + a2 + a3 in one call; ONE fused launch on small / short-bag batches) against the oracle: plan bit-exact,
  outputs within the north_star tolerances (tests/parity.py);
* plan + lookup and dpi_forward under CUDA-graph replay with programmatic dependent launch on and off, rotating batches,
  every step writing its own NaN-filled block (the planner's self-resetting ticket / epoch state is what replay stresses);
* the device picking the a3 variant from a1's max_len (no DPI_OPT_MAX_BAG_HINT);
* the north-star spelling dpi_plan and dpi_plan_device_views put to use; two plans driven from two host threads.
"""
import threading

import numpy as np
import pytest
import torch

import oracle
from paper_2606_21101_b200 import binding, harness, nongemm, workloads as W
from tests.parity import assert_outputs_match, host_offsets, oracle_reference

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module", autouse=True)
def _lib():
    from paper_2606_21101_b200 import build
    build.build()
    binding.load_library()
    harness.require_cuda()


def _tables(cfg):
    rows = cfg.table_rows()
    host_tables = [W.full_table_storage(cfg, t, int(rows[t])) for t in range(cfg.T)]
    return rows, host_tables, harness.tables_from_host(cfg, host_tables)


def _check_plan(plan, lengths):
    K = plan.info()["K"]
    off, seg, S, N, seg_off = plan.export(with_seg_off=True)
    o_off, o_seg, o_S, o_seg_off = oracle.plan(lengths, K, with_seg_off=True)
    assert N == int(lengths.astype(np.int64).sum()) and S == o_S
    assert np.array_equal(off, o_off) and np.array_equal(seg, o_seg) and np.array_equal(seg_off, o_seg_off)
    assert plan.stats() == oracle.plan_stats(lengths)


def _forward_parity(cfg, fused=0, K=0, idx64=False, batch_seed=None, max_indices=None, twice=True):
    """dpi_forward on one batch: output block vs oracle, plan left behind vs oracle (bit-exact)."""
    rows, host_tables, dt = _tables(cfg)
    batch = W.make_batch(cfg, rows, batch_seed)
    pooling = cfg.pooling_modes()
    plan = harness.make_plan(cfg, rows, max(batch.N, 1) if max_indices is None else max_indices, bag_hint=False)
    plan.set_option(binding.OPT_FUSED, fused)
    if K:
        plan.set_quantum(K)
    if idx64:
        plan.set_layout(binding.BAGS_SAMPLE_MAJOR, binding.IDX_I64)
    db = harness.upload_batch(batch)
    idx_dev = torch.from_numpy(np.ascontiguousarray(batch.indices.astype(np.int64) if idx64 else batch.indices)).cuda() \
        if batch.N else db.indices.to(torch.int64 if idx64 else torch.int32)
    ref = oracle_reference(host_tables, cfg.dtype, cfg.B, batch.lengths, batch.indices, pooling)
    worst = 0.0
    for _ in range(2 if twice else 1):   # the second call reuses the look-back records (epoch tagging)
        out = harness.new_output(cfg, fill_nan=True)
        before = binding.launch_count()
        plan.forward(db.lengths, dt.ptrs, idx_dev, out, pooling=pooling)
        launches = binding.launch_count() - before
        torch.cuda.synchronize()
        worst = max(worst, assert_outputs_match(harness.out_to_f64(out), ref, batch.lengths, cfg.T, cfg.D, cfg.dtype, cfg.out))
        _check_plan(plan, batch.lengths)
        assert plan.status() == 0
    # the plan dpi_forward leaves behind drives a later dpi_lookup on the same batch (both a3 kernels)
    for mode in (0, 3):
        plan.set_option(binding.OPT_MODE, mode)
        out = harness.new_output(cfg, fill_nan=True)
        plan.lookup(dt.ptrs, idx_dev, out, pooling=pooling)
        torch.cuda.synchronize()
        assert_outputs_match(harness.out_to_f64(out), ref, batch.lengths, cfg.T, cfg.D, cfg.dtype, cfg.out)
    plan.destroy()
    return launches, worst


# --------------------------------------------------------------------------------------------------
# dpi_forward: the fused single launch
# --------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("name", ["c1", "c2", "c3"])
def test_forward_fused_is_one_launch_and_matches_the_oracle_full_size(name):
    launches, _ = _forward_parity(W.CONFIGS[name])          # auto rule: small, short bags -> fused
    assert launches == 1
    launches, _ = _forward_parity(W.CONFIGS[name], fused=2)  # forced off: planner + lookup
    assert launches == 2


@pytest.mark.parametrize("dtype,D,out", [("f32", 4, None), ("f32", 16, None), ("f32", 24, None), ("f32", 64, None), ("f32", 128, None),
                                         ("f16", 8, None), ("f16", 32, None), ("f16", 72, "f32"), ("f16", 256, None),
                                         ("bf16", 8, "f32"), ("bf16", 64, "f32"), ("bf16", 64, None), ("bf16", 256, None)])
@pytest.mark.parametrize("lengths", [("const", 1), ("uniform", 0, 3), ("uniform", 1, 4), ("poisson", 20.0, 100, 0.05), ("const", 0),
                                     ("uniform", 0, 40)])
def test_forward_fused_shapes_dtypes_and_length_mixes(dtype, D, out, lengths):
    """Every lanes-per-row instantiation, both output types, several 512-bag tiles and a ragged tail, mixed sum / mean,
    empty bags; Poisson(20) and U{0..40} bags run the warp-per-bag tile path (fused forced on: their capacity says long)."""
    cfg = W.Config("ff", 5, (1000, 17, 4000, 1, 250), D, dtype, 333, lengths, ("zipf", 1.05), "half", seed=13, out_dtype=out)
    launches, _ = _forward_parity(cfg, fused=1)
    assert launches == 1


@pytest.mark.parametrize("B,T", [(1, 1), (1, 100), (3, 2048), (127, 4), (129, 4), (1000, 5), (4099, 3), (20000, 7)])
@pytest.mark.parametrize("K", [0, 1, 7, 1000])
def test_forward_fused_chunking_and_any_quantum(B, T, K):
    """Chunk / tile boundaries: fewer bags than one lane-group round, exactly one tile, one more than a tile, several chunks
    of several tiles (140 000 bags); T up to DPI_MAX_TABLES; the plan for any quantum."""
    rows = tuple(int(r) for r in (np.arange(T) * 7 % 13 + 1))
    cfg = W.Config("fc", T, rows, 16, "f32", B, ("uniform", 0, 5), ("uniform",), "half", seed=B + T)
    launches, _ = _forward_parity(cfg, fused=1, K=K, twice=False)
    assert launches == 1


def test_forward_fused_degenerate_and_long_bags():
    _forward_parity(W.Config("e", 3, (5, 5, 5), 16, "f32", 64, ("const", 0), ("uniform",), "mean", 0), fused=1)
    # one bag far longer than a tile's staging buffer, spanning many quanta: indices come straight from global memory
    _forward_parity(W.Config("l", 1, (1000,), 64, "f32", 1, ("const", 20000), ("uniform",), "mean", 0), fused=1, K=32)
    _forward_parity(W.Config("l2", 2, (1000, 50), 64, "bf16", 3, ("const", 5000), ("uniform",), "half", 0), fused=1)
    # bags of 17 entries in a tile of 512: 8704 entries > the staging buffer, lane-group path would not apply (17 > 16)
    _forward_parity(W.Config("l3", 4, (100, 200, 300, 50), 32, "f16", 300, ("const", 17), ("uniform",), "half", 0), fused=1)
    # bags of exactly 16: lane-group path with four rounds of four entries, staging buffer overflow (8192 entries)
    _forward_parity(W.Config("l4", 4, (100, 200, 300, 50), 32, "f16", 300, ("const", 16), ("uniform",), "half", 0), fused=1)
    _forward_parity(W.Config("r1", 4, (1, 1, 1, 1), 32, "f32", 77, ("uniform", 0, 9), ("uniform",), "sum", 2), fused=1)


def test_forward_fused_int64_ids():
    cfg = W.Config("i64", 5, (1000, 17, 4000, 1, 250), 32, "f16", 700, ("uniform", 0, 4), ("zipf", 1.05), "half", seed=14)
    launches, _ = _forward_parity(cfg, fused=1, idx64=True)
    assert launches == 1


def test_forward_falls_back_to_two_launches_for_long_bag_capacities_and_variants():
    cfg = W.Config("fb", 5, (1000, 17, 4000, 1, 250), 64, "bf16", 333, ("poisson", 20.0, 100, 0.05), ("zipf", 1.05), "half",
                   seed=15, out_dtype="f32")
    launches, _ = _forward_parity(cfg)                       # auto: capacity ~19 entries per bag -> plan + balanced lookup
    assert launches == 2
    launches, _ = _forward_parity(W.C1, max_indices=9 * W.C1.G)   # capacity 9 per bag: not "short on average"
    assert launches == 2


def test_forward_honours_a_one_id_per_bag_promise_below_4e5_bags():
    """DPI_OPT_MAX_BAG_HINT = 1 on a small batch: dpi_forward takes planner + the short-bag launch (measured faster there,
    profiles/r02_forward_crossover.md), two launches, same block; without the promise the same call is one launch."""
    cfg = W.C2.scaled(name="c2-small", B=256)
    rows, host_tables, dt = _tables(cfg)
    batch = W.make_batch(cfg, rows, None)
    db = harness.upload_batch(batch)
    ref = oracle_reference(host_tables, cfg.dtype, cfg.B, batch.lengths, batch.indices, cfg.pooling_modes())
    for hint, want in ((True, 2), (False, 1)):
        plan = harness.make_plan(cfg, rows, batch.N, bag_hint=hint)
        out = harness.new_output(cfg, fill_nan=True)
        before = binding.launch_count()
        plan.forward(db.lengths, dt.ptrs, db.indices, out, pooling=cfg.pooling_modes())
        assert binding.launch_count() - before == want
        torch.cuda.synchronize()
        assert_outputs_match(harness.out_to_f64(out), ref, batch.lengths, cfg.T, cfg.D, cfg.dtype, cfg.out)
        _check_plan(plan, batch.lengths)
        plan.destroy()


def test_forward_overflow_is_counted():
    cfg = W.C1
    rows, host_tables, dt = _tables(cfg)
    batch = W.make_batch(cfg, rows)
    db = harness.upload_batch(batch)
    plan = harness.make_plan(cfg, rows, batch.N - 1, bag_hint=False)     # one entry short
    out = harness.new_output(cfg, fill_nan=True)
    plan.forward(db.lengths, dt.ptrs, db.indices, out, pooling=cfg.pooling_modes())
    assert plan.status() == 1 and plan.status() == 0
    with pytest.raises(binding.DpiError):
        plan.export()
    # The plan it left behind carries S = 0 (N = max_indices + 1 still fits the segment buffer: the case ADVICE r2 found), so
    # no later lookup on it reads or writes anything: balanced segments, the device-picked and the host-picked short-bag body
    for mode, hint in ((0, 0), (3, 0), (6, 0), (0, 4)):
        plan.set_option(binding.OPT_MODE, mode)
        plan.set_option(binding.OPT_MAX_BAG_HINT, hint)
        out2 = harness.new_output(cfg, fill_nan=True)
        plan.lookup(dt.ptrs, db.indices, out2, pooling=cfg.pooling_modes())
        torch.cuda.synchronize()
        assert bool(torch.isnan(out2).all()), (mode, hint)
    # ... and the two-launch dpi_forward (planner + lookup) leaves the block untouched as a whole
    plan.set_option(binding.OPT_MODE, 0)
    plan.set_option(binding.OPT_MAX_BAG_HINT, 0)
    plan.set_option(binding.OPT_FUSED, 2)
    out3 = harness.new_output(cfg, fill_nan=True)
    plan.forward(db.lengths, dt.ptrs, db.indices, out3, pooling=cfg.pooling_modes())
    torch.cuda.synchronize()
    assert bool(torch.isnan(out3).all()) and plan.status() == 1
    plan.destroy()


# --------------------------------------------------------------------------------------------------
# CUDA-graph replay, PDL on / off, rotating batches: the mode bench.py times for c1-c3
# --------------------------------------------------------------------------------------------------
def _graph_replay(cfg, call, pdl, steps=16, R=8, opts=None):
    rows, host_tables, dt = _tables(cfg)
    pooling = cfg.pooling_modes()
    batches = [W.make_batch(cfg, rows, cfg.seed + r) for r in range(R)]
    dbs = [harness.upload_batch(b) for b in batches]
    refs = [oracle_reference(host_tables, cfg.dtype, cfg.B, b.lengths, b.indices, pooling) for b in batches]
    plan = harness.make_plan(cfg, rows, harness.max_indices_bound(cfg), bag_hint=False)
    plan.set_option(binding.OPT_PDL, pdl)
    for k, v in (opts or {}).items():
        plan.set_option(k, v)
    outs = [harness.new_output(cfg, fill_nan=True) for _ in range(steps)]
    stream = torch.cuda.Stream()

    def step(i, s):
        b = dbs[i % R]
        if call == "forward":
            plan.forward(b.lengths, dt.ptrs, b.indices, outs[i], pooling=pooling, stream=s)
        else:
            plan.build(b.lengths, s)
            plan.lookup(dt.ptrs, b.indices, outs[i], pooling=pooling, stream=s)

    with torch.cuda.stream(stream):
        for i in range(2):
            step(i, stream)           # warm-up outside the capture (lazy module loading)
    torch.cuda.synchronize()
    graph = torch.cuda.CUDAGraph()
    with torch.cuda.graph(graph, stream=stream):
        for i in range(steps):
            step(i, torch.cuda.current_stream())
    for replay in range(2):
        for o in outs:
            o.fill_(float("nan"))
        torch.cuda.synchronize()
        graph.replay()
        torch.cuda.synchronize()
        for i in range(steps):
            b = batches[i % R]
            assert_outputs_match(harness.out_to_f64(outs[i]), refs[i % R], b.lengths, cfg.T, cfg.D, cfg.dtype, cfg.out)
        _check_plan(plan, batches[(steps - 1) % R].lengths)   # the plan of the last step, bit-exact
        assert plan.status() == 0
    plan.destroy()


@pytest.mark.parametrize("pdl", [1, 0])
@pytest.mark.parametrize("name", ["c1", "c3"])
@pytest.mark.parametrize("variant", ["device-picked", "balanced", "short-bag launch", "fused"])
def test_graph_replay_of_rotating_batches_matches_the_oracle(name, variant, pdl):
    cfg = W.CONFIGS[name]
    if variant == "fused":
        _graph_replay(cfg, "forward", pdl)
    else:
        opts = {"device-picked": {}, "balanced": {binding.OPT_MODE: 3}, "short-bag launch": {binding.OPT_MODE: 6}}[variant]
        _graph_replay(cfg, "plan+lookup", pdl, opts=opts)


def test_graph_replay_long_bags_balanced_kernel():
    cfg = W.Config("gl", 6, (500, 30, 2000, 7, 100, 1000), 64, "f32", 700, ("uniform", 0, 70), ("uniform",), "half", 3)
    _graph_replay(cfg, "plan+lookup", 1, steps=16, R=4)
    _graph_replay(cfg, "forward", 1, steps=16, R=4)


# --------------------------------------------------------------------------------------------------
# the device picks the a3 variant from a1's max_len
# --------------------------------------------------------------------------------------------------
def test_the_device_picks_the_variant_without_any_hint():
    """Same plan object, batches whose longest bag changes from call to call: 3 (short-bag body), 40 (balanced segments),
    1 (one-hot), 0 (all empty). No DPI_OPT_MAX_BAG_HINT anywhere."""
    base = W.Config("dp", 5, (1000, 17, 4000, 1, 250), 32, "f16", 600, ("uniform", 0, 3), ("zipf", 1.05), "half", seed=16)
    rows, host_tables, dt = _tables(base)
    plan = harness.make_plan(base, rows, base.G * 40, bag_hint=False)
    assert plan.get_option(binding.OPT_MAX_BAG_HINT) == 0
    for lengths in [("uniform", 0, 3), ("uniform", 0, 40), ("const", 1), ("const", 0), ("uniform", 1, 8), ("uniform", 1, 9)]:
        cfg = base.scaled(lengths=lengths)
        batch = W.make_batch(cfg, rows)
        db = harness.upload_batch(batch)
        pooling = cfg.pooling_modes()
        plan.build(db.lengths)
        out = harness.new_output(cfg, fill_nan=True)
        plan.lookup(dt.ptrs, db.indices, out, pooling=pooling)
        torch.cuda.synchronize()
        ref = oracle_reference(host_tables, cfg.dtype, cfg.B, batch.lengths, batch.indices, pooling)
        assert_outputs_match(harness.out_to_f64(out), ref, batch.lengths, cfg.T, cfg.D, cfg.dtype, cfg.out)
        assert plan.stats() == oracle.plan_stats(batch.lengths)
    plan.destroy()


# --------------------------------------------------------------------------------------------------
# dpi_plan (north-star spelling) and dpi_plan_device_views
# --------------------------------------------------------------------------------------------------
def test_dpi_plan_north_star_spelling_and_device_views_feed_the_lr_operator():
    """dpi_plan(table_rows, dims, lengths, B) builds in one call; the borrowed views are the plan: offsets feed the first-order
    (LR) operator of NEXT-4 directly, the interleaved segment records and meta equal the oracle's plan."""
    cfg = W.Config("ns", 4, (100, 2000, 50, 7), 16, "f32", 300, ("uniform", 0, 5), ("zipf", 1.1), "sum", 18)
    rows, host_tables, dt = _tables(cfg)
    batch = W.make_batch(cfg, rows)
    db = harness.upload_batch(batch)
    plan = binding.dpi_plan(rows, cfg.D, W.DTYPE_CODE[cfg.dtype], db.lengths, cfg.B, batch.N)
    K = plan.info()["K"]
    o_off, o_seg, o_S, o_seg_off = oracle.plan(batch.lengths, K, with_seg_off=True)
    off_p, seg_p, meta_p = plan.device_views()
    torch.cuda.synchronize()

    def view(ptr, n):
        t = torch.empty(n, dtype=torch.int32, device="cuda")
        binding.copy_device_words(t, ptr, n)
        return t.cpu().numpy()

    meta = view(meta_p, 8)
    lo, hi = oracle.plan_stats(batch.lengths)
    assert meta.tolist() == [o_S, batch.N, int(np.maximum(batch.lengths, 1).sum()), 0, K, cfg.G, lo, hi]
    assert np.array_equal(view(off_p, cfg.G + 1), o_off)
    seg = view(seg_p, 2 * (o_S + 1)).reshape(-1, 2)
    assert np.array_equal(seg[:, 0], o_seg) and np.array_equal(seg[:, 1], o_seg_off)
    # north-star spelling of the lookup on that plan
    out = harness.new_output(cfg, fill_nan=True)
    binding.dpi_lookup(dt.ptrs, db.indices, None, plan, cfg.pooling_modes(), out)
    torch.cuda.synchronize()
    ref = oracle_reference(host_tables, cfg.dtype, cfg.B, batch.lengths, batch.indices, cfg.pooling_modes())
    assert_outputs_match(harness.out_to_f64(out), ref, batch.lengths, cfg.T, cfg.D, cfg.dtype, cfg.out)
    # the offsets view as the CSR offsets of dpi_lr_first_order (small-integer weights: exact)
    w_host = [(np.arange(int(r)) % 7 - 3).astype(np.float32) for r in rows]
    w_dev = [torch.from_numpy(w).cuda() for w in w_host]
    w_ptrs = torch.tensor([w.data_ptr() for w in w_dev], dtype=torch.int64, device="cuda")
    y = torch.full((cfg.B,), float("nan"), device="cuda")
    nongemm.lr_first_order(w_ptrs, db.indices, off_p, cfg.B, cfg.T, 2.0, y)
    torch.cuda.synchronize()
    want = oracle.lr_first_order([w.astype(np.float64) for w in w_host], cfg.B, batch.indices, o_off, bias=2.0)
    assert np.array_equal(y.double().cpu().numpy(), want)
    plan.destroy()


# --------------------------------------------------------------------------------------------------
# distinct plans are independent: two host threads, two streams, two different instantiations
# --------------------------------------------------------------------------------------------------
def test_two_plans_on_two_host_threads_and_streams():
    cfgs = [W.Config("ta", 6, (500, 30, 2000, 7, 100, 1000), 64, "f32", 300, ("uniform", 0, 30), ("uniform",), "half", 3),
            W.Config("tb", 2048, tuple(int(r) for r in (np.arange(2048) * 7 % 13 + 1)), 8, "bf16", 4, ("uniform", 0, 3), ("uniform",),
                     "half", seed=21, out_dtype="f32")]   # the second one needs > 48 KB of shared memory in the general kernel
    prepared = []
    for cfg in cfgs:
        rows, host_tables, dt = _tables(cfg)
        batch = W.make_batch(cfg, rows)
        prepared.append((cfg, rows, dt, batch, harness.upload_batch(batch),
                         oracle_reference(host_tables, cfg.dtype, cfg.B, batch.lengths, batch.indices, cfg.pooling_modes())))
    errors = []

    def worker(i):
        try:
            torch.cuda.set_device(0)
            cfg, rows, dt, batch, db, ref = prepared[i]
            stream = torch.cuda.Stream()
            for rep in range(20):
                plan = harness.make_plan(cfg, rows, max(batch.N, 1), bag_hint=False)    # create inside the thread: per-plan state only
                out = harness.new_output(cfg, fill_nan=True)
                with torch.cuda.stream(stream):
                    if rep % 2:
                        plan.forward(db.lengths, dt.ptrs, db.indices, out, pooling=cfg.pooling_modes(), stream=stream)
                    else:
                        plan.build(db.lengths, stream)
                        plan.lookup_ex(dt.ptrs, db.indices, out, pooling=cfg.pooling_modes(), flags=binding.LOOKUP_FORCE_GENERAL,
                                       stream=stream)
                stream.synchronize()
                assert_outputs_match(harness.out_to_f64(out), ref, batch.lengths, cfg.T, cfg.D, cfg.dtype, cfg.out)
                plan.destroy()
        except BaseException as e:  # noqa: BLE001 -- reported by the main thread
            errors.append((i, repr(e)))

    threads = [threading.Thread(target=worker, args=(i,)) for i in range(2)]
    for t in threads:
        t.start()
    for t in threads:
        t.join()
    assert not errors, errors


def test_set_quantum_invalidates_the_built_plan():
    cfg = W.C1
    rows, host_tables, dt = _tables(cfg)
    batch = W.make_batch(cfg, rows)
    db = harness.upload_batch(batch)
    plan = harness.make_plan(cfg, rows, batch.N, bag_hint=False)
    plan.build(db.lengths)
    plan.set_quantum(1)          # re-allocates the segment buffer: what was built is gone
    out = harness.new_output(cfg)
    with pytest.raises(binding.DpiError) as e:
        plan.lookup(dt.ptrs, db.indices, out, pooling=cfg.pooling_modes())
    assert e.value.status == 1 and "built" in e.value.detail
    plan.build(db.lengths)
    plan.lookup(dt.ptrs, db.indices, out, pooling=cfg.pooling_modes())
    torch.cuda.synchronize()
    _check_plan(plan, batch.lengths)
    plan.destroy()
