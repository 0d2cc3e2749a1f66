"""Pins for oracle.lookup_general -- the interface variants of SURVEY.md §8(f) NEXT-2 (CPU only).

The paper only hints at these ("marking offset information" PAPER.md:168; 64-bit ids from the framework
PAPER.md:336), so each pin is something other than the oracle: the torch-CPU embedding_bag library routine with
per_sample_weights in float64, closed forms for exactly representable weights, index-encoding tables that decode
every output element to its own (table, row, column) under mixed dims, PAPER.md:83 independence (hstack of
single-table calls), and a tiny pure-Python brute force that walks the table-major bag grid.
"""
import numpy as np
import pytest
import torch

import oracle


def _offsets(lengths):
    return np.concatenate(([0], np.cumsum(np.asarray(lengths, dtype=np.int64))))


def _problem(rng, T, B, dims, rows, max_len, order=oracle.SAMPLE_MAJOR, p_empty=0.2):
    """Random bags in the requested bag order; returns tables, lengths[G], indices[N] (int64), table_of_bag[G]."""
    tables = [rng.uniform(-0.05, 0.05, size=(rows[t], dims[t])).astype(np.float32) for t in range(T)]
    G = B * T
    tab = (np.arange(G) % T) if order == oracle.SAMPLE_MAJOR else (np.arange(G) // B)
    lengths = rng.integers(0, max_len + 1, size=G)
    lengths[rng.random(G) < p_empty] = 0
    idx = np.concatenate([rng.integers(0, rows[tab[g]], size=lengths[g]) for g in range(G)] + [np.zeros(0, int)])
    return tables, lengths.astype(np.int64), idx.astype(np.int64), tab


def test_reduces_to_the_pinned_lookup_when_nothing_is_generalised():
    rng = np.random.default_rng(0)
    T, B, D = 5, 40, 8
    tables, ln, idx, _ = _problem(rng, T, B, [D] * T, [50, 3, 700, 11, 1], 6)
    pooling = np.array([0, 1, 0, 1, 1], np.uint8)
    want = oracle.lookup(tables, oracle.F32, B, idx.astype(np.int32), _offsets(ln).astype(np.int32), pooling)
    got = oracle.lookup_general(tables, oracle.F32, B, idx, _offsets(ln), pooling)
    assert np.array_equal(got, want)


def test_mixed_dims_index_encoding_tables_decode_to_their_own_slot():
    """E_t[r][c] = t*2^16 + r*2^5 + c (exact in fp32), one-hot bags: every output element must decode to
    (t, ids[b,t], c) at column col[t] + c -- catches a wrong column prefix, a wrong per-table width or row stride."""
    rng = np.random.default_rng(1)
    dims = [4, 16, 8, 32, 4, 12]
    T, B = len(dims), 17
    rows = [9, 100, 3, 64, 1, 30]
    tables = [(t * 65536 + np.arange(rows[t])[:, None] * 32 + np.arange(dims[t])[None, :]).astype(np.float32)
              for t in range(T)]
    ids = np.stack([rng.integers(0, rows[t], size=B) for t in range(T)], axis=1)  # [B, T]
    got = oracle.lookup_general(tables, oracle.F32, B, ids.reshape(-1), np.arange(B * T + 1), np.zeros(T, np.uint8))
    assert got.shape == (B, sum(dims))
    col = np.concatenate(([0], np.cumsum(dims)))
    for t in range(T):
        blk = got[:, col[t]:col[t + 1]].astype(np.int64)
        assert np.array_equal(blk >> 16, np.full_like(blk, t))
        assert np.array_equal((blk >> 5) & 0x7FF, np.repeat(ids[:, t:t + 1], dims[t], axis=1))
        assert np.array_equal(blk & 31, np.tile(np.arange(dims[t]), (B, 1)))


@pytest.mark.parametrize("order", [oracle.SAMPLE_MAJOR, oracle.TABLE_MAJOR])
def test_mixed_dims_equal_hstack_of_single_table_calls(order):
    """fields are independent, so the fused block is the hstack of per-table blocks. A single
    table has only one bag order, so this also pins table-major against sample-major."""
    rng = np.random.default_rng(2)
    dims = [8, 4, 24, 16]
    T, B = 4, 29
    rows = [20, 500, 7, 90]
    tables, ln, idx, tab = _problem(rng, T, B, dims, rows, 5, order)
    off = _offsets(ln)
    pooling = np.array([0, 1, 1, 0], np.uint8)
    got = oracle.lookup_general(tables, oracle.F32, B, idx, off, pooling, bag_order=order)
    col = np.concatenate(([0], np.cumsum(dims)))
    for t in range(T):
        bags = np.nonzero(tab == t)[0]  # in sample order for both layouts
        sub_idx = np.concatenate([idx[off[g]:off[g + 1]] for g in bags] + [np.zeros(0, np.int64)])
        sub = oracle.lookup([tables[t]], oracle.F32, B, sub_idx.astype(np.int32), _offsets(ln[bags]).astype(np.int32),
                            pooling[t:t + 1])
        assert np.array_equal(got[:, col[t]:col[t + 1]], sub)


def test_table_major_brute_force_on_a_tiny_grid():
    """Pure-Python walk of the [T, B] bag grid: bag (b,t) is g = t*B + b."""
    rng = np.random.default_rng(3)
    dims, rows = [4, 8, 4], [5, 3, 9]
    T, B = 3, 4
    tables, ln, idx, _ = _problem(rng, T, B, dims, rows, 3, oracle.TABLE_MAJOR, p_empty=0.25)
    off = _offsets(ln)
    pooling = np.array([0, 1, 0], np.uint8)
    want = np.zeros((B, sum(dims)))
    col = 0
    for t in range(T):
        for b in range(B):
            g = t * B + b
            rws = [tables[t][idx[j]].astype(np.float64) for j in range(off[g], off[g + 1])]
            if rws:
                v = np.sum(rws, axis=0)
                want[b, col:col + dims[t]] = v / len(rws) if pooling[t] else v
        col += dims[t]
    got = oracle.lookup_general(tables, oracle.F32, B, idx, off, pooling, bag_order=oracle.TABLE_MAJOR)
    np.testing.assert_allclose(got, want, rtol=1e-15, atol=0)


def test_table_major_is_the_bag_grid_transpose_of_sample_major():
    rng = np.random.default_rng(4)
    dims, rows = [8, 8, 16, 4, 4], [30, 2, 11, 400, 77]
    T, B = 5, 23
    tables, ln, idx, _ = _problem(rng, T, B, dims, rows, 4)
    off = _offsets(ln)
    pooling = np.array([0, 0, 1, 1, 0], np.uint8)
    want = oracle.lookup_general(tables, oracle.F32, B, idx, off, pooling)
    perm = np.arange(B * T).reshape(B, T).T.reshape(-1)  # table-major position -> sample-major bag id
    idx_tm = np.concatenate([idx[off[g]:off[g + 1]] for g in perm] + [np.zeros(0, np.int64)])
    got = oracle.lookup_general(tables, oracle.F32, B, idx_tm, _offsets(ln[perm]), pooling, bag_order=oracle.TABLE_MAJOR)
    assert np.array_equal(got, want)


def test_weights_torch_embedding_bag_library_cross_check():
    rng = np.random.default_rng(5)
    dims, rows = [16, 8, 4], [100, 7, 1000]
    T, B = 3, 50
    tables, ln, idx, _ = _problem(rng, T, B, dims, rows, 9)
    off = _offsets(ln)
    w = rng.uniform(-2, 2, size=idx.shape[0]).astype(np.float32)
    got = oracle.lookup_general(tables, oracle.F32, B, idx, off, np.zeros(T, np.uint8), weights=w)
    col = np.concatenate(([0], np.cumsum(dims)))
    for t in range(T):
        bags = np.arange(B) * T + t
        sel = np.concatenate([np.arange(off[g], off[g + 1]) for g in bags] + [np.zeros(0, np.int64)]).astype(np.int64)
        want = torch.nn.functional.embedding_bag(
            torch.from_numpy(idx[sel]), torch.from_numpy(tables[t]).double(), torch.from_numpy(_offsets(ln[bags])),
            mode="sum", include_last_offset=True, per_sample_weights=torch.from_numpy(w[sel]).double()).numpy()
        np.testing.assert_allclose(got[:, col[t]:col[t + 1]], want, rtol=1e-13, atol=1e-16)


def test_weights_closed_forms():
    """Unit weights change nothing; a power-of-two weight scales exactly; a zero weight drops the entry; and the
    result is linear in the weights (exactly, for weights and values that are small dyadic rationals)."""
    rng = np.random.default_rng(6)
    dims, rows = [8, 4], [40, 9]
    T, B = 2, 30
    tables = [(rng.integers(-8, 9, size=(rows[t], dims[t])) / 64.0).astype(np.float32) for t in range(T)]
    _, ln, idx, _ = _problem(rng, T, B, dims, rows, 6)
    off = _offsets(ln)
    pool = np.zeros(T, np.uint8)
    base = oracle.lookup_general(tables, oracle.F32, B, idx, off, pool)
    n = idx.shape[0]
    assert np.array_equal(oracle.lookup_general(tables, oracle.F32, B, idx, off, pool, weights=np.ones(n, np.float32)), base)
    assert np.array_equal(oracle.lookup_general(tables, oracle.F32, B, idx, off, pool, weights=np.full(n, 0.25, np.float32)),
                          0.25 * base)
    # zero weight == entry removed
    keep = rng.random(n) < 0.6
    w = keep.astype(np.float32)
    kept_len = np.array([keep[off[g]:off[g + 1]].sum() for g in range(B * T)])
    dropped = oracle.lookup_general(tables, oracle.F32, B, idx[keep], _offsets(kept_len), pool)
    assert np.array_equal(oracle.lookup_general(tables, oracle.F32, B, idx, off, pool, weights=w), dropped)
    # linearity
    w1 = (rng.integers(-4, 5, size=n) / 4.0).astype(np.float32)
    w2 = (rng.integers(-4, 5, size=n) / 4.0).astype(np.float32)
    a = oracle.lookup_general(tables, oracle.F32, B, idx, off, pool, weights=w1)
    b = oracle.lookup_general(tables, oracle.F32, B, idx, off, pool, weights=w2)
    ab = oracle.lookup_general(tables, oracle.F32, B, idx, off, pool, weights=w1 + w2)
    assert np.array_equal(ab, a + b)


def test_weights_with_mean_pooling_and_bad_arguments_are_rejected():
    tables = [np.zeros((3, 4), np.float32)]
    with pytest.raises(oracle.OracleError):
        oracle.lookup_general(tables, oracle.F32, 1, np.zeros(1, np.int64), np.array([0, 1]), np.ones(1, np.uint8),
                              weights=np.ones(1, np.float32))
    with pytest.raises(oracle.OracleError):  # index beyond the table, only representable in 64 bits
        oracle.lookup_general(tables, oracle.F32, 1, np.array([1 << 33]), np.array([0, 1]), np.zeros(1, np.uint8))
    with pytest.raises(oracle.OracleError):
        oracle.lookup_general(tables, oracle.F32, 1, np.zeros(1, np.int64), np.array([0, 1]), np.zeros(1, np.uint8),
                              bag_order=2)


@pytest.mark.parametrize("dtype", ["f16", "bf16"])
def test_16bit_mixed_dims_weighted_exactly_representable(dtype):
    """Values k/64, weights in {0.5, 1, 2}: every product and sum is exact in any of the formats involved."""
    from paper_2606_21101_b200 import workloads as W
    rng = np.random.default_rng(7)
    dims, rows = [8, 16], [12, 5]
    T, B = 2, 11
    vals = [(rng.integers(-3, 4, size=(rows[t], dims[t])) / 64.0).astype(np.float32) for t in range(T)]
    tables = [W.to_storage(v, dtype) for v in vals]
    _, ln, idx, _ = _problem(rng, T, B, dims, rows, 5)
    off = _offsets(ln)
    w = rng.choice(np.array([0.5, 1.0, 2.0], np.float32), size=idx.shape[0])
    got = oracle.lookup_general(tables, W.DTYPE_CODE[dtype], B, idx, off, np.zeros(T, np.uint8), weights=w)
    want = oracle.lookup_general(vals, oracle.F32, B, idx, off, np.zeros(T, np.uint8), weights=w)
    assert np.array_equal(got, want)
