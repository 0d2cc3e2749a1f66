"""GPU parity for SURVEY.md 8(f) NEXT-4 (include/dpi_nongemm.h) against oracle/nongemm_oracle.c, element by element, through
the C ABI. Tolerances, u = 2^-24 the fp32 unit roundoff, A_c = sum_t |x_tc|:
  FM   v:  |err| <= 2 (T + 2) u A_c^2                       (T-term sums s and q, one fma, one halving)
       y:  |err| <= sum_c tol_v[c] + 8 u sum_c |v_c|        (tree sum over the D columns)
       bit-exact when every intermediate is an integer below 2^24
  cross:   |err| <= 2 u (|x0 (u + b)| + |xl|) + eps_out |ref|
  bias_act identity / relu: |err| <= 2 u |u + b| + eps_out |ref|;  sigmoid: 2^-21 + eps_out |ref|
  eps_out = 0 (fp32 out), 2^-11 (fp16), 2^-8 (bf16): one round-to-nearest-even cast at the store; fp16 adds the absolute
  floor 2^-25 (half the spacing of its subnormals: results below 2^-14 are not relatively accurate)."""
import numpy as np
import pytest
import torch

import oracle
from paper_2606_21101_b200 import binding, harness, nongemm
from paper_2606_21101_b200 import workloads as W

pytestmark = pytest.mark.gpu

U32 = 2.0 ** -24
EPS_OUT = {"f32": 0.0, "f16": 2.0 ** -11, "bf16": 2.0 ** -8}
FLOOR_OUT = {"f32": 1e-30, "f16": 2.0 ** -25, "bf16": 1e-30}
TORCH = {"f32": torch.float32, "f16": torch.float16, "bf16": torch.bfloat16}


def to_device(x32: np.ndarray, dtype: str):
    """float32 values -> (device tensor of `dtype`, float64 array of exactly the values the device holds)."""
    st = W.to_storage(x32, dtype)
    exact = W.storage_to_f64(st, dtype)
    if dtype == "bf16":
        t = torch.from_numpy(st.view(np.int16).copy()).cuda().view(torch.bfloat16)
    else:
        t = torch.from_numpy(st.copy()).cuda()
    return t, exact


def f64(t: torch.Tensor) -> np.ndarray:
    return t.detach().to("cpu").to(torch.float64).numpy()


# ---------------------------------------------------------------------------------------------------------------
# FM second-order term
# ---------------------------------------------------------------------------------------------------------------
def run_fm(x32, dtype, T, D, pad=0, want_y=True, want_v=True):
    B = x32.shape[0]
    if pad:
        wide = np.full((B, T * D + pad), 7.0, dtype=np.float32)   # the padding columns must not be read into the result
        wide[:, : T * D] = x32
        x32 = wide
    xd, exact = to_device(x32, dtype)
    y = torch.full((B,), float("nan"), device="cuda") if want_y else None
    v = torch.full((B, D), float("nan"), device="cuda") if want_v else None
    nongemm.fm_interaction(xd, W.DTYPE_CODE[dtype], B, T, D, y=y, v=v, x_ld=x32.shape[1] if pad else 0)
    torch.cuda.synchronize()
    ref_y, ref_v = oracle.fm_pairwise(exact, T, D)
    A2 = np.abs(exact[:, : T * D]).reshape(B, T, D).sum(axis=1) ** 2
    tol_v = 2 * (T + 2) * U32 * A2
    if want_v:
        got_v = f64(v)
        assert not np.isnan(got_v).any()
        assert (np.abs(got_v - ref_v) <= tol_v).all(), f"v: max err {np.abs(got_v - ref_v).max():.3e}"
    if want_y:
        got_y = f64(y)
        tol_y = tol_v.sum(axis=1) + 8 * U32 * np.abs(ref_v).sum(axis=1)
        assert not np.isnan(got_y).any()
        assert (np.abs(got_y - ref_y) <= tol_y).all(), f"y: max err {np.abs(got_y - ref_y).max():.3e}"
    return (f64(y) if want_y else None), (f64(v) if want_v else None), ref_y, ref_v


@pytest.mark.parametrize("dtype,D", [("f32", 4), ("f32", 16), ("f32", 24), ("f32", 64), ("f32", 128), ("f16", 8),
                                     ("f16", 32), ("f16", 40), ("bf16", 64), ("bf16", 256)])
@pytest.mark.parametrize("B,T", [(1, 1), (3, 2), (203, 26), (1037, 39), (77, 100)])
def test_fm_shapes_dtypes(dtype, D, B, T):
    x = W.dense_values_f32(11, T * 1000 + D, (B, T * D), 0.25)
    run_fm(x, dtype, T, D)


@pytest.mark.parametrize("dtype", ["f32", "f16", "bf16"])
def test_fm_row_pitch_and_single_outputs(dtype):
    T, D, B = 7, 16, 130
    x = W.dense_values_f32(12, 0, (B, T * D), 0.25)
    y0, v0, _, _ = run_fm(x, dtype, T, D)
    y1, _, _, _ = run_fm(x, dtype, T, D, pad=8, want_v=False)
    _, v2, _, _ = run_fm(x, dtype, T, D, pad=24, want_y=False)
    assert np.array_equal(y0, y1) and np.array_equal(v0, v2)      # same arithmetic, whatever the pitch / outputs


@pytest.mark.parametrize("dtype", ["f32", "f16", "bf16"])
def test_fm_small_integers_are_bit_exact(dtype):
    T, D, B = 26, 16, 300
    h = W.hash_u64(W.stream_key(5, W.STREAM_DENSE, 3), np.arange(B * T * D, dtype=np.uint64))
    x = ((h % np.uint64(17)).astype(np.float32) - 8.0).reshape(B, T * D)     # integers in [-8, 8]
    y, v, ref_y, ref_v = run_fm(x, dtype, T, D)
    assert np.array_equal(v, ref_v) and np.array_equal(y, ref_y)


def test_fm_degenerate_cases():
    T, D = 5, 16
    z = torch.zeros((4, T * D), device="cuda")
    y = torch.full((4,), float("nan"), device="cuda")
    nongemm.fm_interaction(z, 0, 4, T, D, y=y)
    nongemm.fm_interaction(z, 0, 0, T, D, y=y)          # B = 0: no launch, no error
    torch.cuda.synchronize()
    assert (y == 0).all()
    one = torch.ones((2, 1 * D), device="cuda")          # a single field has no pairs
    y1 = torch.full((2,), float("nan"), device="cuda")
    nongemm.fm_interaction(one, 0, 2, 1, D, y=y1)
    torch.cuda.synchronize()
    assert (y1 == 0).all()


def test_fm_on_the_lookup_output_of_c2_full_size():
    """The chain the paper describes (embedding block -> explicit interaction): plan + lookup on BASELINE.json
    configs[1], FM on the block the lookup wrote. c2 is one-hot fp32, so the lookup output is bit-identical to the
    oracle's block (Alg. 1) and the oracle FM can run on the ORACLE's block, not on anything the GPU produced."""
    cfg = W.C2
    dt = harness.make_device_tables(cfg)
    batch = W.make_batch(cfg, dt.rows)
    db = harness.upload_batch(batch)
    plan = harness.make_plan(cfg, dt.rows, batch.N)
    plan.build(db.lengths)
    out = harness.new_output(cfg, fill_nan=True)
    plan.lookup(dt.ptrs, db.indices, out, pooling=cfg.pooling_modes())
    y = torch.full((cfg.B,), float("nan"), device="cuda")
    nongemm.fm_interaction(out, 0, cfg.B, cfg.T, cfg.D, y=y)
    torch.cuda.synchronize()
    host_tables = [W.full_table_storage(cfg, t, int(dt.rows[t])) for t in range(cfg.T)]
    block = oracle.alg1_onehot(host_tables, 0, batch.indices.reshape(cfg.B, cfg.T))
    assert np.array_equal(harness.out_to_f64(out), block)
    ref_y, ref_v = oracle.fm_pairwise(block, cfg.T, cfg.D)
    A2 = np.abs(block).reshape(cfg.B, cfg.T, cfg.D).sum(axis=1) ** 2
    tol = (2 * (cfg.T + 2) * U32 * A2).sum(axis=1) + 8 * U32 * np.abs(ref_v).sum(axis=1)
    assert (np.abs(f64(y) - ref_y) <= tol).all()
    plan.destroy()


@pytest.mark.parametrize("dtype,B,T,D", [("f16", 16384, 22, 32), ("f32", 65536, 8, 64), ("f32", 8192, 100, 64)])
def test_fm_full_size_block_shapes(dtype, B, T, D):
    """X_embed blocks with the shapes of c3, c5 and c4 (fp32 output): every sample against the oracle."""
    x = W.dense_values_f32(13, T, (B, T * D), 0.25)
    run_fm(x, dtype, T, D, want_v=False)


# ---------------------------------------------------------------------------------------------------------------
# element-wise operators
# ---------------------------------------------------------------------------------------------------------------
def run_cross(dtype, B, F, with_bias=True, seed=21, in_place=None):
    x0, e0 = to_device(W.dense_values_f32(seed, 1, (B, F), 0.5), dtype)
    xl, el = to_device(W.dense_values_f32(seed, 2, (B, F), 0.5), dtype)
    u, eu = to_device(W.dense_values_f32(seed, 3, (B, F), 2.0), dtype)
    bias32 = W.dense_values_f32(seed, 4, (F,), 1.0) if with_bias else None
    bias = torch.from_numpy(bias32).cuda() if with_bias else None
    out = {None: torch.full((B, F), float("nan"), dtype=TORCH[dtype], device="cuda"), "xl": xl, "u": u}[in_place]
    nongemm.cross_combine(x0, xl, u, bias, out, W.DTYPE_CODE[dtype], B, F)
    torch.cuda.synchronize()
    ref = oracle.cross_combine(e0, el, eu, None if bias32 is None else bias32.astype(np.float64))
    b64 = 0.0 if bias32 is None else bias32.astype(np.float64)[None, :]
    tol = 2 * U32 * (np.abs(e0 * (eu + b64)) + np.abs(el)) + EPS_OUT[dtype] * np.abs(ref) + FLOOR_OUT[dtype]
    got = f64(out)
    assert not np.isnan(got).any()
    assert (np.abs(got - ref) <= tol).all(), f"max err {np.abs(got - ref).max():.3e}"
    return got


@pytest.mark.parametrize("dtype", ["f32", "f16", "bf16"])
@pytest.mark.parametrize("B,F", [(1, 8), (5, 416), (203, 704), (1037, 24), (64, 8200), (3000, 512)])
def test_cross_combine_shapes(dtype, B, F):
    run_cross(dtype, B, F)
    run_cross(dtype, B, F, with_bias=False)


@pytest.mark.parametrize("dtype", ["f32", "bf16"])
def test_cross_combine_in_place_equals_out_of_place(dtype):
    a = run_cross(dtype, 333, 416)
    assert np.array_equal(a, run_cross(dtype, 333, 416, in_place="xl"))
    assert np.array_equal(a, run_cross(dtype, 333, 416, in_place="u"))


@pytest.mark.parametrize("dtype", ["f32", "f16", "bf16"])
def test_cross_combine_small_integers_are_bit_exact(dtype):
    B, F = 129, 416
    h = W.hash_u64(W.stream_key(6, W.STREAM_DENSE, 9), np.arange(4 * B * F, dtype=np.uint64)).reshape(4, B, F)
    ints = [(h[i] % np.uint64(m)).astype(np.float32) - float(m // 2) for i, m in enumerate((9, 17, 9))]   # |x0|<=4, |xl|<=8, |u|<=4
    bias32 = ((h[3][0] % np.uint64(9)).astype(np.float32) - 4.0)                                            # |b|<=4
    (x0, e0), (xl, el), (u, eu) = (to_device(a, dtype) for a in ints)
    out = torch.empty((B, F), dtype=TORCH[dtype], device="cuda")
    nongemm.cross_combine(x0, xl, u, torch.from_numpy(bias32).cuda(), out, W.DTYPE_CODE[dtype], B, F)
    torch.cuda.synchronize()
    ref = oracle.cross_combine(e0, el, eu, bias32.astype(np.float64))      # |ref| <= 4*8 + 8 = 40: exact in bf16 too
    assert np.array_equal(f64(out), ref)


@pytest.mark.parametrize("dtype", ["f32", "f16", "bf16"])
@pytest.mark.parametrize("act", [nongemm.ACT_IDENTITY, nongemm.ACT_RELU, nongemm.ACT_SIGMOID])
@pytest.mark.parametrize("B,F", [(1, 8), (203, 400), (1037, 1024), (31, 8200)])
def test_bias_act_shapes(dtype, act, B, F):
    u, eu = to_device(W.dense_values_f32(31, 1, (B, F), 4.0), dtype)
    bias32 = W.dense_values_f32(31, 2, (F,), 1.0)
    out = torch.full((B, F), float("nan"), dtype=TORCH[dtype], device="cuda")
    nongemm.bias_act(u, torch.from_numpy(bias32).cuda(), out, W.DTYPE_CODE[dtype], B, F, act)
    torch.cuda.synchronize()
    ref = oracle.bias_act(eu, bias32.astype(np.float64), act)
    s = np.abs(eu + bias32.astype(np.float64)[None, :])
    tol = (2.0 ** -21 if act == nongemm.ACT_SIGMOID else 2 * U32 * s) + EPS_OUT[dtype] * np.abs(ref) + FLOOR_OUT[dtype]
    got = f64(out)
    assert not np.isnan(got).any()
    assert (np.abs(got - ref) <= tol).all(), f"max err {np.abs(got - ref).max():.3e}"


def test_bias_act_exact_cases_and_in_place():
    B, F = 77, 416
    u32 = W.dense_values_f32(32, 1, (B, F), 3.0)
    u = torch.from_numpy(u32).cuda()
    out = torch.empty_like(u)
    nongemm.bias_act(u, None, out, 0, B, F, nongemm.ACT_IDENTITY)
    assert torch.equal(out, u)                                           # identity without bias: a copy
    nongemm.bias_act(u, None, out, 0, B, F, nongemm.ACT_RELU)
    ref = oracle.bias_act(u32.astype(np.float64), None, oracle.ACT_RELU)
    assert np.array_equal(f64(out), ref)                                 # relu without bias: exact
    nongemm.bias_act(u, None, u, 0, B, F, nongemm.ACT_RELU)              # in place
    torch.cuda.synchronize()
    assert torch.equal(out, u)


# ---------------------------------------------------------------------------------------------------------------
# Algorithm 2
# ---------------------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("ne,ni", [(0, 0), (0, 3), (1, 1), (2, 5), (5, 2), (4, 4), (7, 6)])
def test_bfs_schedule_equals_the_oracle_queue(ne, ni):
    assert nongemm.bfs_schedule(ne, ni) == oracle.bfs_queue(ne, ni)


@pytest.mark.parametrize("n_streams", [1, 2])
@pytest.mark.parametrize("ne,ni", [(1, 3), (3, 1), (2, 2), (0, 2), (3, 0)])
def test_launcher_runs_algorithm_2_and_joins(n_streams, ne, ni):
    """Explicit module: ne chained in-place relu/bias steps on buffer E; implicit module: ni chained steps on buffer I.
    The launch order seen by the callbacks must be the oracle's queue; each module's operators must land on one
    stream of its own (two streams) or on the caller's stream (one stream); after the join the caller's stream sees
    both results, equal to running the chains one after the other."""
    B, F = 257, 416
    e32, i32 = W.dense_values_f32(41, 1, (B, F), 1.0), W.dense_values_f32(41, 2, (B, F), 1.0)
    bias32 = W.dense_values_f32(41, 3, (F,), 0.25)
    bias = torch.from_numpy(bias32).cuda()
    main = torch.cuda.Stream()
    order, streams = [], {0: set(), 1: set()}
    with torch.cuda.stream(main):
        E, I = torch.from_numpy(e32).cuda(), torch.from_numpy(i32).cuda()

        def op(module, k, buf):
            def launch(s):
                order.append((module, k))
                streams[module].add(s)
                nongemm.bias_act(buf, bias, buf, 0, B, F, nongemm.ACT_IDENTITY, stream=s)
            return launch

        main.synchronize()      # the H2D copies above ran on `main`; the module streams fork from it anyway
        L = nongemm.Launcher()
        L.run([op(0, k, E) for k in range(ne)], [op(1, k, I) for k in range(ni)], n_streams=n_streams, stream=main)
        got_e, got_i = E.clone(), I.clone()      # enqueued on `main`: ordered after the join
    main.synchronize()
    assert order == oracle.bfs_queue(ne, ni)
    if n_streams == 2:
        assert all(len(streams[m]) <= 1 for m in (0, 1))
        if ne and ni:
            assert streams[0] != streams[1] and main.cuda_stream not in (streams[0] | streams[1])
    else:
        assert (streams[0] | streams[1]) <= {main.cuda_stream}
    ref_e, ref_i = e32.astype(np.float64), i32.astype(np.float64)
    for _ in range(ne):
        ref_e = oracle.bias_act(ref_e, bias32.astype(np.float64), oracle.ACT_IDENTITY).astype(np.float32).astype(np.float64)
    for _ in range(ni):
        ref_i = oracle.bias_act(ref_i, bias32.astype(np.float64), oracle.ACT_IDENTITY).astype(np.float32).astype(np.float64)
    assert np.array_equal(f64(got_e), ref_e) and np.array_equal(f64(got_i), ref_i)   # one fp32 add per step: exact match
    L.destroy()


def test_launcher_is_graph_capturable():
    B, F = 128, 64
    a = torch.zeros((B, F), device="cuda")
    b = torch.zeros((B, F), device="cuda")
    one = torch.ones((F,), device="cuda")
    L = nongemm.Launcher()
    mk = lambda buf: (lambda s: nongemm.bias_act(buf, one, buf, 0, B, F, nongemm.ACT_IDENTITY, stream=s))
    g = torch.cuda.CUDAGraph()
    side = torch.cuda.Stream()
    with torch.cuda.stream(side):
        with torch.cuda.graph(g, stream=side):
            L.run([mk(a)], [mk(b), mk(b), mk(b)], n_streams=2, stream=side)
    torch.cuda.synchronize()
    for _ in range(5):
        g.replay()
    torch.cuda.synchronize()
    assert (a == 5).all() and (b == 15).all()
    L.destroy()


# ---------------------------------------------------------------------------------------------------------------
# DeepFM first-order (logistic regression) term
# ---------------------------------------------------------------------------------------------------------------
def _lr_problem(T, B, lengths, seed=17):
    rows = tuple(int(r) for r in (np.arange(T) * 131 % 997 + 1))
    cfg = W.Config("lr", T, rows, 4, "f32", B, lengths, ("zipf", 1.05), "sum", seed)
    batch = W.make_batch(cfg, np.asarray(rows, np.int64))
    w32 = [W.dense_values_f32(seed, 100 + t, (rows[t],), 0.5) for t in range(T)]
    w_dev = [torch.from_numpy(w).cuda() for w in w32]
    ptrs = torch.tensor([w.data_ptr() for w in w_dev], dtype=torch.int64, device="cuda")
    return batch, w32, w_dev, ptrs


@pytest.mark.parametrize("T,B", [(1, 1), (3, 5), (26, 1037), (39, 333), (100, 77)])
@pytest.mark.parametrize("lengths", [("const", 1), ("uniform", 0, 4), ("poisson", 20.0, 100, 0.05)])
def test_lr_first_order_matches_the_oracle(T, B, lengths):
    batch, w32, w_dev, ptrs = _lr_problem(T, B, lengths)
    off = np.concatenate(([0], np.cumsum(batch.lengths.astype(np.int64)))).astype(np.int32)
    idx_dev = torch.from_numpy(batch.indices if batch.N else np.zeros(1, np.int32)).cuda()
    off_dev = torch.from_numpy(off).cuda()
    y = torch.full((B,), float("nan"), device="cuda")
    nongemm.lr_first_order(ptrs, idx_dev, off_dev, B, T, 0.25, y)
    torch.cuda.synchronize()
    w64 = [w.astype(np.float64) for w in w32]
    ref = oracle.lr_first_order(w64, B, batch.indices, off, bias=0.25)
    # fp32 sum of n terms in tree / lane order: |err| <= (n + 2) u sum|w| (+ the bias add)
    n = batch.lengths.reshape(B, T).sum(axis=1)
    absum = oracle.lr_first_order([np.abs(w) for w in w64], B, batch.indices, off, bias=0.25)
    tol = (n + 2) * U32 * absum + 1e-30
    got = f64(y)
    assert not np.isnan(got).any()
    assert (np.abs(got - ref) <= tol).all(), f"max err {np.abs(got - ref).max():.3e}"
    if lengths[0] == "const":       # one-hot: the same numbers without offsets
        y1 = torch.full((B,), float("nan"), device="cuda")
        nongemm.lr_first_order(ptrs, idx_dev, None, B, T, 0.25, y1)
        torch.cuda.synchronize()
        assert torch.equal(y, y1)


def test_lr_integer_weights_are_exact_and_accumulate_adds_onto_fm():
    T, B, D = 26, 300, 16
    batch, _, _, _ = _lr_problem(T, B, ("uniform", 0, 3))
    rows = [int(r) for r in (np.arange(T) * 131 % 997 + 1)]
    wi = [((np.arange(rows[t]) * 7 + t) % 41 - 20).astype(np.float32) for t in range(T)]
    w_dev = [torch.from_numpy(w).cuda() for w in wi]
    ptrs = torch.tensor([w.data_ptr() for w in w_dev], dtype=torch.int64, device="cuda")
    off = np.concatenate(([0], np.cumsum(batch.lengths.astype(np.int64)))).astype(np.int32)
    idx_dev, off_dev = torch.from_numpy(batch.indices).cuda(), torch.from_numpy(off).cuda()
    y = torch.full((B,), float("nan"), device="cuda")
    nongemm.lr_first_order(ptrs, idx_dev, off_dev, B, T, -3.0, y)
    torch.cuda.synchronize()
    ref = oracle.lr_first_order([w.astype(np.float64) for w in wi], B, batch.indices, off, bias=-3.0)
    assert np.array_equal(f64(y), ref)                                   # small integers: every partial sum is exact
    # DeepFM explicit module = FM + LR: FM writes y, LR accumulates onto it (integers again, so the sum is exact)
    h = W.hash_u64(W.stream_key(5, W.STREAM_DENSE, 3), np.arange(B * T * D, dtype=np.uint64))
    x = ((h % np.uint64(9)).astype(np.float32) - 4.0).reshape(B, T * D)
    xd = torch.from_numpy(x).cuda()
    nongemm.fm_interaction(xd, 0, B, T, D, y=y)
    nongemm.lr_first_order(ptrs, idx_dev, off_dev, B, T, -3.0, y, accumulate=True)
    torch.cuda.synchronize()
    fm_ref, _ = oracle.fm_pairwise(x.astype(np.float64), T, D)
    assert np.array_equal(f64(y), fm_ref + ref)


def test_lr_all_empty_and_validation():
    T, B = 4, 9
    w_dev = [torch.ones(3, device="cuda") for _ in range(T)]
    ptrs = torch.tensor([w.data_ptr() for w in w_dev], dtype=torch.int64, device="cuda")
    off = torch.zeros(B * T + 1, dtype=torch.int32, device="cuda")
    idx = torch.zeros(1, dtype=torch.int32, device="cuda")
    y = torch.full((B,), float("nan"), device="cuda")
    nongemm.lr_first_order(ptrs, idx, off, B, T, 1.5, y)
    torch.cuda.synchronize()
    assert (y == 1.5).all()
    from paper_2606_21101_b200 import binding
    with pytest.raises(binding.DpiError):
        nongemm.lr_first_order(None, idx, off, B, T, 0.0, y)
    with pytest.raises(binding.DpiError):
        nongemm.lr_first_order(ptrs, idx, off, B, 0, 0.0, y)


# ---------------------------------------------------------------------------------------------------------------
# dpi_forward_fm: the lookup and its first non-GEMM consumer as one operator
# ---------------------------------------------------------------------------------------------------------------
def _lookup_tol(ref, lengths, T, D, dtype):
    """Per-element tolerance of the pooled block (tests/parity.py) as an array [B, T*D]."""
    L = np.repeat(np.maximum(lengths.reshape(-1, T), 1), D, axis=1).astype(np.float64)
    if dtype == "f32":
        return 1e-5 * L
    return np.maximum(2e-3 * np.abs(ref), 1e-6 * L)


def _forward_fm_case(cfg, batch_seed=None, fused=0, expect_launches=None):
    from tests.parity import assert_outputs_match, oracle_reference
    rows = cfg.table_rows()
    host_tables = [W.full_table_storage(cfg, t, int(rows[t])) for t in range(cfg.T)]
    dt = harness.tables_from_host(cfg, host_tables)
    batch = W.make_batch(cfg, rows, batch_seed)
    db = harness.upload_batch(batch)
    pooling = cfg.pooling_modes()
    plan = harness.make_plan(cfg, rows, max(batch.N, 1))
    plan.set_option(binding.OPT_FUSED, fused)
    B, T, D = cfg.B, cfg.T, cfg.D
    out = harness.new_output(cfg, fill_nan=True)
    y = torch.full((B,), float("nan"), device="cuda")
    v = torch.full((B, D), float("nan"), device="cuda")
    before = binding.launch_count()
    nongemm.forward_fm(plan, db.lengths, dt.ptrs, db.indices, out, y=y, v=v, pooling=pooling)
    launches = binding.launch_count() - before
    torch.cuda.synchronize()
    if expect_launches is not None:
        assert launches == expect_launches
    # the block and the plan are exactly what dpi_forward leaves behind
    ref = oracle_reference(host_tables, cfg.dtype, B, batch.lengths, batch.indices, pooling)
    assert_outputs_match(harness.out_to_f64(out), ref, batch.lengths, T, D, cfg.dtype, cfg.out)
    off, seg, S, N = plan.export()
    o_off, o_seg, o_S = oracle.plan(batch.lengths, plan.info()["K"])
    assert N == batch.N and S == o_S and np.array_equal(off, o_off) and np.array_equal(seg, o_seg)
    # FM by its definition on the ORACLE's block; tolerance = the FM operator's own bound + the pooled block's tolerance
    # carried through v_c = sum_{t<u} x_t x_u:  |dv_c| <= A_c E_c + E_c^2,  A_c = sum_t |x_tc|,  E_c = sum_t tol_tc
    ref_y, ref_v = oracle.fm_pairwise(ref, T, D)
    A = np.abs(ref).reshape(B, T, D).sum(axis=1)
    E = _lookup_tol(ref, batch.lengths, T, D, cfg.dtype).reshape(B, T, D).sum(axis=1)
    tol_v = 2 * (T + 2) * U32 * (A + E) ** 2 + A * E + E * E
    got_v, got_y = f64(v), f64(y)
    assert not np.isnan(got_v).any() and not np.isnan(got_y).any()
    assert (np.abs(got_v - ref_v) <= tol_v).all(), f"v: max err {np.abs(got_v - ref_v).max():.3e}"
    tol_y = tol_v.sum(axis=1) + 8 * U32 * np.abs(ref_v).sum(axis=1)
    assert (np.abs(got_y - ref_y) <= tol_y).all(), f"y: max err {np.abs(got_y - ref_y).max():.3e}"
    # and y / v are bit-identical to dpi_fm_interaction applied to the block this very call wrote (the same per-sample code
    # runs in the epilogue and in fm_kernel; the block itself may differ from plan + lookup in summation order only)
    y2 = torch.full((B,), float("nan"), device="cuda")
    v2 = torch.full((B, D), float("nan"), device="cuda")
    nongemm.fm_interaction(out, W.DTYPE_CODE[cfg.out], B, T, D, y=y2, v=v2)
    torch.cuda.synchronize()
    assert torch.equal(y, y2) and torch.equal(v, v2)
    plan.destroy()
    return launches


@pytest.mark.parametrize("name", ["c1", "c2", "c3"])
def test_forward_fm_is_one_launch_on_the_small_configs_full_size(name):
    assert _forward_fm_case(W.CONFIGS[name], expect_launches=1) == 1


@pytest.mark.parametrize("dtype,D,lengths,pool", [("f32", 16, ("uniform", 0, 4), "half"), ("f16", 32, ("uniform", 1, 3), "mean"),
                                                   ("bf16", 64, ("const", 1), "sum"), ("f32", 64, ("poisson", 20.0, 100, 0.05), "half"),
                                                   ("f16", 8, ("uniform", 0, 40), "sum")])
@pytest.mark.parametrize("B,T", [(1, 1), (37, 3), (300, 22), (2049, 7), (129, 100)])
def test_forward_fm_shapes_whole_sample_chunks_and_long_bags(dtype, D, lengths, pool, B, T):
    """T that does not divide the natural chunk size (chunks are rounded up to whole samples), one sample, more tables than
    lane groups, bags long enough for the warp-per-bag chunk path; fused forced on so every shape takes the single launch."""
    cfg = W.Config("ffm", T, tuple(int(7 + 13 * t) for t in range(T)), D, dtype, B, lengths, ("zipf", 1.1), pool, seed=5)
    assert _forward_fm_case(cfg, fused=1, expect_launches=1) == 1


def test_forward_fm_falls_back_to_the_chain_and_validates():
    # fp32 output of bf16 tables and batches beyond the fused rule: planner + lookup + FM kernel, same results
    cfg = W.Config("ffm2", 5, (100, 20, 7, 300, 50), 32, "bf16", 200, ("uniform", 0, 5), ("uniform",), "half", seed=3, out_dtype="f32")
    assert _forward_fm_case(cfg, expect_launches=None) >= 2
    cfg = W.Config("ffm3", 4, (100, 20, 7, 300), 16, "f32", 64, ("poisson", 20.0, 100, 0.0), ("uniform",), "sum", seed=3)
    assert _forward_fm_case(cfg, fused=2, expect_launches=3) == 3
    plan = binding.Plan([10, 10], np.asarray([16, 8], np.int32), 0, 4, 8)     # mixed dims: no FM
    z = torch.zeros(64, device="cuda")
    with pytest.raises(binding.DpiError) as e:
        nongemm.forward_fm(plan, z.view(torch.int32), z, z.view(torch.int32), z, y=z)
    assert e.value.status == 2
    plan.destroy()
