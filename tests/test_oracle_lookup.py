"""Pins for oracle.lookup / oracle.alg1_onehot (CPU only).

Each test checks the oracle against something that is NOT the oracle: the paper's Alg. 1 identity, a
hand-worked fixture, closed forms, the one-hot-matrix product view, a library routine
(torch-CPU embedding_bag), or structural invariants (PAPER.md:83 independence, sample permutation).
"""
import numpy as np
import pytest
import torch

import oracle
from paper_2606_21101_b200 import workloads as W
from tests.golden.load_golden import fig5_tables, load


def _offsets(lengths):
    return np.concatenate(([0], np.cumsum(np.asarray(lengths, dtype=np.int64)))).astype(np.int32)


def _rand_problem(rng, T, B, D, rows, max_len, p_empty=0.2):
    tables = [rng.uniform(-0.05, 0.05, size=(rows[t], D)).astype(np.float32) for t in range(T)]
    lengths = rng.integers(0, max_len + 1, size=B * T)
    lengths[rng.random(B * T) < p_empty] = 0
    idx = np.concatenate([rng.integers(0, rows[g % T], size=lengths[g]) for g in range(B * T)] + [np.zeros(0, int)])
    return tables, lengths.astype(np.int32), idx.astype(np.int32)


# --------------------------------------------------------------------------------------------------
# hand-worked fixture (PAPER.md:133 shape, Alg. 1)
# --------------------------------------------------------------------------------------------------
def test_golden_fig5_onehot():
    g = load("fig5_shape_example.txt")
    ids = np.array(g["onehot.ids"], dtype=np.int32)
    want = np.array(g["onehot.out"], dtype=np.float64)
    got = oracle.alg1_onehot(fig5_tables(), oracle.F32, ids)
    assert np.array_equal(got, want)
    # the pooled entry point with every bag of length 1 is the same thing
    got2 = oracle.lookup(fig5_tables(), oracle.F32, 2, ids.reshape(-1), np.arange(9, dtype=np.int32),
                         np.zeros(4, np.uint8))
    assert np.array_equal(got2, want)


def test_golden_fig5_multihot_sum_and_mixed():
    g = load("fig5_shape_example.txt")
    lengths = np.array(g["multihot.lengths"], dtype=np.int32).reshape(-1)
    indices = np.array(sum(g["multihot.indices"], []), dtype=np.int32)
    off = _offsets(lengths)
    got = oracle.lookup(fig5_tables(), oracle.F32, 2, indices, off, np.zeros(4, np.uint8))
    assert np.array_equal(got, np.array(g["multihot.sum"]))
    pooling = np.array(g["multihot.pooling"], dtype=np.uint8).reshape(-1)
    got = oracle.lookup(fig5_tables(), oracle.F32, 2, indices, off, pooling)
    np.testing.assert_allclose(got, np.array(g["multihot.mixed"]), rtol=1e-15, atol=0)


# --------------------------------------------------------------------------------------------------
# Alg. 1: gather identity + column-block order
# --------------------------------------------------------------------------------------------------
def test_alg1_is_row_gather_and_blocks_in_table_order():
    """Index-encoding tables: E_t[r][c] = t*2^16 + r*2^4 + c (exact in fp32). Every output element must
    decode to its own (t, IDs[b,t], c) -- catches transposed layouts, wrong table, wrong column."""
    rng = np.random.default_rng(1)
    T, B, D = 5, 37, 16
    rows = [7, 300, 1, 4095, 64]
    tables = [(t * 65536 + np.arange(rows[t])[:, None] * 16 + np.arange(D)[None, :]).astype(np.float32)
              for t in range(T)]
    ids = np.stack([rng.integers(0, rows[t], size=B) for t in range(T)], axis=1).astype(np.int32)
    out = oracle.alg1_onehot(tables, oracle.F32, ids)
    assert out.shape == (B, T * D)
    code = out.astype(np.int64).reshape(B, T, D)
    assert np.array_equal(code >> 16, np.broadcast_to(np.arange(T)[None, :, None], (B, T, D)))
    assert np.array_equal((code >> 4) & 0xFFF, np.broadcast_to(ids[:, :, None], (B, T, D)))
    assert np.array_equal(code & 0xF, np.broadcast_to(np.arange(D)[None, None, :], (B, T, D)))
    # the pooled entry point agrees bit for bit when every bag has length 1 (sum and mean)
    for pool in (0, 1):
        out2 = oracle.lookup(tables, oracle.F32, B, ids.reshape(-1), np.arange(B * T + 1, dtype=np.int32),
                             np.full(T, pool, np.uint8))
        assert np.array_equal(out2, out)


def test_length_one_equals_library_gather():
    """results indistinguishable from PyTorch -> one-hot == torch index_select + cat."""
    rng = np.random.default_rng(2)
    T, B, D = 6, 50, 8
    rows = [10, 1000, 3, 77, 500, 2]
    tables = [rng.standard_normal((rows[t], D)).astype(np.float32) for t in range(T)]
    ids = np.stack([rng.integers(0, rows[t], size=B) for t in range(T)], axis=1).astype(np.int32)
    want = torch.cat([torch.from_numpy(tables[t]).index_select(0, torch.from_numpy(ids[:, t].astype(np.int64)))
                      for t in range(T)], dim=1).double().numpy()
    got = oracle.alg1_onehot(tables, oracle.F32, ids)
    assert np.array_equal(got, want)


# --------------------------------------------------------------------------------------------------
# closed forms
# --------------------------------------------------------------------------------------------------
def test_constant_tables_sum_is_len_times_kappa_and_mean_is_kappa():
    rng = np.random.default_rng(3)
    T, B, D = 4, 33, 4
    rows = [5, 9, 2, 100]
    kappa = [0.5, -0.25, 2.0, 0.125]
    tables = [np.full((rows[t], D), kappa[t], dtype=np.float32) for t in range(T)]
    _, lengths, idx = _rand_problem(rng, T, B, D, rows, 9)
    off = _offsets(lengths)
    s = oracle.lookup(tables, oracle.F32, B, idx, off, np.zeros(T, np.uint8)).reshape(B, T, D)
    m = oracle.lookup(tables, oracle.F32, B, idx, off, np.ones(T, np.uint8)).reshape(B, T, D)
    L = lengths.reshape(B, T)
    for t in range(T):
        assert np.array_equal(s[:, t, :], np.broadcast_to((L[:, t] * kappa[t])[:, None], (B, D)))
        want_m = np.where(L[:, t] > 0, kappa[t], 0.0)
        assert np.array_equal(m[:, t, :], np.broadcast_to(want_m[:, None], (B, D)))


def test_row_id_tables_sum_of_indices():
    """E_t[r][c] = r + c*2^-3: out = sum(indices) + L*c/8 exactly -- catches dropped/duplicated entries and
    off-by-one bag boundaries (neighbouring bags have different index sums)."""
    rng = np.random.default_rng(4)
    T, B, D = 3, 64, 4
    rows = [1000, 17, 300]
    tables = [(np.arange(rows[t])[:, None] + np.arange(D)[None, :] / 8.0).astype(np.float32) for t in range(T)]
    _, lengths, idx = _rand_problem(rng, T, B, D, rows, 12)
    off = _offsets(lengths)
    got = oracle.lookup(tables, oracle.F32, B, idx, off, np.zeros(T, np.uint8)).reshape(B * T, D)
    for g in range(B * T):
        seg = idx[off[g]:off[g + 1]].astype(np.int64)
        want = seg.sum() + len(seg) * np.arange(D) / 8.0
        assert np.array_equal(got[g], want), g


def test_mean_is_sum_over_len_and_empty_is_positive_zero():
    rng = np.random.default_rng(5)
    T, B, D = 5, 40, 8
    rows = [11, 13, 17, 19, 23]
    tables, lengths, idx = _rand_problem(rng, T, B, D, rows, 7, p_empty=0.3)
    lengths[0] = 0
    lengths[-1] = 0  # first and last bag empty: boundaries of offsets
    idx = np.concatenate([rng.integers(0, rows[g % T], size=lengths[g]) for g in range(B * T)]).astype(np.int32)
    off = _offsets(lengths)
    s = oracle.lookup(tables, oracle.F32, B, idx, off, np.zeros(T, np.uint8)).reshape(B * T, D)
    m = oracle.lookup(tables, oracle.F32, B, idx, off, np.ones(T, np.uint8)).reshape(B * T, D)
    for g in range(B * T):
        if lengths[g] == 0:
            for arr in (s, m):
                assert np.all(arr[g] == 0.0) and not np.any(np.signbit(arr[g]))
        else:
            assert np.array_equal(m[g], s[g] / float(lengths[g]))


def test_all_empty_batch_is_zero_matrix():
    T, B, D = 3, 5, 4
    tables = [np.ones((4, D), np.float32) for _ in range(T)]
    off = np.zeros(B * T + 1, np.int32)
    for pool in (0, 1):
        out = oracle.lookup(tables, oracle.F32, B, np.zeros(0, np.int32), off, np.full(T, pool, np.uint8))
        assert out.shape == (B, T * D) and not out.any() and not np.signbit(out).any()


# --------------------------------------------------------------------------------------------------
# independent formulations
# --------------------------------------------------------------------------------------------------
def test_one_hot_matrix_product_formulation():
    """fields are "encoded with one-hot encoding" and then represented as IDs; a pooled lookup
    is the multi-hot count matrix times the table: out_t = M_t @ E_t (numpy matmul in float64)."""
    rng = np.random.default_rng(6)
    T, B, D = 4, 20, 6
    rows = [9, 30, 4, 15]
    tables, lengths, idx = _rand_problem(rng, T, B, D, rows, 6)
    off = _offsets(lengths)
    got = oracle.lookup(tables, oracle.F32, B, idx, off, np.zeros(T, np.uint8))
    for t in range(T):
        M = np.zeros((B, rows[t]))
        for b in range(B):
            g = b * T + t
            for j in range(off[g], off[g + 1]):
                M[b, idx[j]] += 1.0
        want = M @ tables[t].astype(np.float64)
        np.testing.assert_allclose(got[:, t * D:(t + 1) * D], want, rtol=0, atol=1e-15)


@pytest.mark.parametrize("mode", ["sum", "mean"])
def test_torch_embedding_bag_library_cross_check(mode):
    rng = np.random.default_rng(7)
    T, B, D = 5, 64, 16
    rows = [100, 7, 1000, 33, 2]
    tables, lengths, idx = _rand_problem(rng, T, B, D, rows, 10)
    off = _offsets(lengths)
    got = oracle.lookup(tables, oracle.F32, B, idx, off, np.full(T, 0 if mode == "sum" else 1, np.uint8))
    L = lengths.reshape(B, T)
    for t in range(T):
        bag_idx = np.concatenate([idx[off[b * T + t]:off[b * T + t + 1]] for b in range(B)] + [np.zeros(0, np.int32)])
        bag_off = np.concatenate(([0], np.cumsum(L[:, t])))
        want = torch.nn.functional.embedding_bag(
            torch.from_numpy(bag_idx.astype(np.int64)), torch.from_numpy(tables[t]).double(),
            torch.from_numpy(bag_off.astype(np.int64)), mode=mode, include_last_offset=True).numpy()
        np.testing.assert_allclose(got[:, t * D:(t + 1) * D], want, rtol=1e-14, atol=1e-16)


def test_fused_equals_hstack_of_single_table_lookups():
    """lookups across fields are independent and never share a table."""
    rng = np.random.default_rng(8)
    T, B, D = 6, 31, 8
    rows = [5, 50, 500, 2, 20, 200]
    tables, lengths, idx = _rand_problem(rng, T, B, D, rows, 5)
    off = _offsets(lengths)
    pooling = np.array([0, 1, 0, 1, 1, 0], np.uint8)
    fused = oracle.lookup(tables, oracle.F32, B, idx, off, pooling)
    L = lengths.reshape(B, T)
    for t in range(T):
        one_idx = np.concatenate([idx[off[b * T + t]:off[b * T + t + 1]] for b in range(B)] + [np.zeros(0, np.int32)])
        single = oracle.lookup([tables[t]], oracle.F32, B, one_idx, _offsets(L[:, t]), pooling[t:t + 1])
        assert np.array_equal(fused[:, t * D:(t + 1) * D], single)


def test_sample_permutation_permutes_rows():
    rng = np.random.default_rng(9)
    T, B, D = 3, 25, 4
    rows = [40, 8, 300]
    tables, lengths, idx = _rand_problem(rng, T, B, D, rows, 6)
    off = _offsets(lengths)
    base = oracle.lookup(tables, oracle.F32, B, idx, off, np.array([0, 1, 0], np.uint8))
    perm = rng.permutation(B)
    L2 = lengths.reshape(B, T)[perm].reshape(-1)
    idx2 = np.concatenate([idx[off[b * T + t]:off[b * T + t + 1]] for b in perm for t in range(T)])
    out2 = oracle.lookup(tables, oracle.F32, B, idx2.astype(np.int32), _offsets(L2), np.array([0, 1, 0], np.uint8))
    assert np.array_equal(out2, base[perm])


def test_duplicates_count_with_multiplicity():
    tables = [np.array([[1.0, 2.0], [10.0, 20.0]], np.float32)]
    out = oracle.lookup(tables, oracle.F32, 1, np.array([1, 1, 1, 0], np.int32), np.array([0, 4], np.int32),
                        np.zeros(1, np.uint8))
    assert np.array_equal(out, [[31.0, 62.0]])


# --------------------------------------------------------------------------------------------------
# 16-bit storage
# --------------------------------------------------------------------------------------------------
def test_f16_decoder_exhaustive_against_numpy():
    bits = np.arange(65536, dtype=np.uint16)
    want = bits.view(np.float16).astype(np.float64)
    for b in range(0, 65536, 1):
        w = want[b]
        got = oracle.decode_f16(b)
        if np.isnan(w):
            assert np.isnan(got)
        else:
            assert got == w and np.signbit(got) == np.signbit(w), b


def test_bf16_decoder_exhaustive_against_torch():
    bits = torch.arange(65536, dtype=torch.int32).to(torch.uint16)
    want = bits.view(torch.bfloat16).double().numpy()
    for b in range(65536):
        got = oracle.decode_bf16(b)
        if np.isnan(want[b]):
            assert np.isnan(got)
        else:
            assert got == want[b], b


@pytest.mark.parametrize("dtype", ["f16", "bf16"])
def test_16bit_tables_exactly_representable_values_are_bit_exact(dtype):
    """Values k*2^-10 with |k| <= 3 are exact in fp16 and bf16; sums of <= 64 of them are exact integers/1024
    so the float64 oracle must equal the integer computation exactly."""
    rng = np.random.default_rng(10)
    T, B, D = 3, 40, 8
    rows = [12, 100, 5]
    ks = [rng.integers(-3, 4, size=(rows[t], D)) for t in range(T)]
    tables = [W.to_storage((k / 1024.0).astype(np.float32), dtype) for k in ks]
    lengths = rng.integers(0, 65, size=B * T).astype(np.int32)
    idx = np.concatenate([rng.integers(0, rows[g % T], size=lengths[g]) for g in range(B * T)]).astype(np.int32)
    off = _offsets(lengths)
    got = oracle.lookup(tables, W.DTYPE_CODE[dtype], B, idx, off, np.zeros(T, np.uint8)).reshape(B * T, D)
    for g in range(B * T):
        want = ks[g % T][idx[off[g]:off[g + 1]]].sum(axis=0) / 1024.0
        assert np.array_equal(got[g], want)


def test_16bit_storage_roundtrip_of_workload_values():
    """The oracle reads what the generator stored: decode(to_storage(x)) equals the library conversion."""
    x = W.table_values_f32(0, 3, 32, np.arange(50))
    h = W.to_storage(x, "f16")
    b = W.to_storage(x, "bf16")
    assert np.array_equal(h.astype(np.float64), torch.from_numpy(x).half().double().numpy())
    assert np.array_equal(W.storage_to_f64(b, "bf16"), torch.from_numpy(x).bfloat16().double().numpy())
    tabs = [b]
    out = oracle.lookup(tabs, oracle.BF16, 1, np.array([7], np.int32), np.array([0, 1], np.int32), np.zeros(1, np.uint8))
    assert np.array_equal(out[0], torch.from_numpy(x[7]).bfloat16().double().numpy())


# --------------------------------------------------------------------------------------------------
# error behaviour
# --------------------------------------------------------------------------------------------------
def test_out_of_range_index_is_rejected():
    tables = [np.zeros((4, 2), np.float32)]
    for bad in (-1, 4):
        with pytest.raises(oracle.OracleError):
            oracle.lookup(tables, oracle.F32, 1, np.array([bad], np.int32), np.array([0, 1], np.int32),
                          np.zeros(1, np.uint8))


# --------------------------------------------------------------------------------------------------
# the all-cores timing leg (bench.py cpu_baseline): same bags, same per-bag order, samples split over threads
# --------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("dtype", ["f32", "f16", "bf16"])
def test_lookup_par_is_bit_identical_to_the_single_thread_oracle(dtype):
    rng = np.random.default_rng(21)
    T, B, D = 7, 257, 24
    rows = [100, 7, 1000, 33, 2, 500, 64]
    tables32, lengths, idx = _rand_problem(rng, T, B, D, rows, 12)
    tables = [W.to_storage(t, dtype) for t in tables32]
    off = _offsets(lengths)
    pooling = (np.arange(T) % 2).astype(np.uint8)
    one = oracle.lookup(tables, W.DTYPE_CODE[dtype], B, idx, off, pooling)
    par, team = oracle.lookup_par(tables, W.DTYPE_CODE[dtype], B, idx, off, pooling)
    assert team >= 1
    assert np.array_equal(one.view(np.uint64), par.view(np.uint64))   # bit for bit, signed zeros included


def test_lookup_par_golden_fig5_and_error_status():
    g = load("fig5_shape_example.txt")
    lengths = np.array(g["multihot.lengths"], dtype=np.int32).reshape(-1)
    idx = np.array(sum(g["multihot.indices"], []), dtype=np.int32)
    pooling = np.array(g["multihot.pooling"][0], dtype=np.uint8)
    got, _ = oracle.lookup_par(fig5_tables(), oracle.F32, 2, idx, _offsets(lengths), pooling)
    np.testing.assert_allclose(got, np.array(g["multihot.mixed"]), rtol=1e-15)
    bad = idx.copy()
    bad[3] = 3   # tables have rows 0..2
    with pytest.raises(oracle.OracleError):
        oracle.lookup_par(fig5_tables(), oracle.F32, 2, bad, _offsets(lengths), pooling)
