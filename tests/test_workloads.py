"""The seeded input recipe: determinism, ranges and the shapes BASELINE.json names."""
import math

import numpy as np
import pytest

from paper_2606_21101_b200 import workloads as W


def test_hash_is_splitmix_stream_and_deterministic():
    key = W.stream_key(0, W.STREAM_VAL, 3)
    a = W.hash_u64(key, np.arange(5))
    b = W.hash_u64(key, np.arange(5))
    assert np.array_equal(a, b) and len(set(a.tolist())) == 5
    # scalar python re-computation of one element
    z = (key + 3 * W.GAMMA) & ((1 << 64) - 1)
    assert int(a[3]) == W._fmix64_int(z)
    assert W.stream_key(0, W.STREAM_VAL, 3) != W.stream_key(0, W.STREAM_VAL, 4) != W.stream_key(1, W.STREAM_VAL, 3)


def test_bf16_rne_matches_torch():
    import torch
    rng = np.random.default_rng(0)
    x = np.concatenate([rng.uniform(-0.05, 0.05, 100000).astype(np.float32),
                        np.array([0.0, 1.0, 1.00390625, 1.01171875, -1.00390625, 3.0e-39], np.float32)])
    got = W.f32_to_bf16_bits(x)
    want = torch.from_numpy(x).bfloat16().view(torch.int16).numpy().view(np.uint16)
    assert np.array_equal(got, want)
    assert np.array_equal(W.bf16_bits_to_f32(got), torch.from_numpy(x).bfloat16().float().numpy())


def test_table_values_range_and_row_recompute():
    v = W.table_values_f32(0, 2, 64, np.arange(2000))
    assert v.dtype == np.float32 and v.min() >= -0.05 and v.max() < 0.05
    assert abs(float(v.mean())) < 5e-4 and abs(float(v.std()) - 0.1 / math.sqrt(12)) < 5e-4
    some = np.array([1999, 0, 77])
    assert np.array_equal(W.table_values_f32(0, 2, 64, some), v[some])
    assert not np.array_equal(W.table_values_f32(0, 3, 64, some), v[some])


@pytest.mark.parametrize("cfg", [W.C1, W.C2, W.C3, W.C4, W.C5], ids=lambda c: c.name)
def test_table_rows_match_baseline_shapes(cfg):
    rows = cfg.table_rows()
    assert rows.shape == (cfg.T,) and rows.dtype == np.int64
    if isinstance(cfg.rows[0], str):
        assert rows.min() >= cfg.rows[1] and rows.max() <= cfg.rows[2]
        assert np.array_equal(rows, cfg.table_rows())
    else:
        assert rows.tolist() == list(cfg.rows)
    assert cfg.row_bytes % 16 == 0


def test_c1_batch():
    b = W.make_batch(W.C1)
    assert b.lengths.shape == (512,) and b.lengths.min() >= 1 and b.lengths.max() <= 4
    assert b.N == b.lengths.sum()
    rows = W.C1.table_rows()
    t = np.repeat(np.arange(512) % 4, b.lengths)
    assert np.all(b.indices >= 0) and np.all(b.indices < rows[t])
    b2 = W.make_batch(W.C1)
    assert np.array_equal(b.indices, b2.indices)
    b3 = W.make_batch(W.C1, batch_seed=1)
    assert not np.array_equal(b.lengths, b3.lengths)


def test_c2_onehot_zipf_is_skewed_and_scattered():
    cfg = W.C2
    rows = cfg.table_rows()
    b = W.make_batch(cfg, rows)
    assert b.N == cfg.G and np.all(b.lengths == 1)
    ids = b.indices.reshape(cfg.B, cfg.T)
    assert np.all(ids >= 0) and np.all(ids < rows[None, :])
    t = int(np.argmax(rows))
    col = ids[:, t]
    top = np.bincount(col).max() / cfg.B
    assert top > 0.03  # rank-1 mass of Zipf(1.05) over ~1e6 rows is ~7 %
    hot_row = int(np.bincount(col).argmax())
    assert hot_row == 0  # rank 1 maps to row (0 * a) mod n = 0; rank 2 is scattered far from it
    second = int(np.argsort(np.bincount(col))[-2])
    assert second > rows[t] // 2


def test_c4_lengths_poisson_with_empties():
    ln = W.make_lengths(W.C4, 0)
    assert ln.shape == (W.C4.G,) and ln.max() <= 100 and ln.min() == 0
    assert abs((ln == 0).mean() - 0.05) < 0.003
    assert abs(ln[ln > 0].mean() - 20.0) < 0.1


def test_c5_shape_and_bytes():
    cfg = W.C5
    ln = W.make_lengths(cfg, 0)
    assert ln.min() == 1 and ln.max() == 64 and abs(ln.mean() - 32.5) < 0.1
    rows = cfg.table_rows()
    assert rows.sum() * cfg.row_bytes == 81_920_000_000
    by = W.algorithmic_bytes(cfg, cfg.G, int(ln.sum()))
    assert abs(by["lookup"] / 4.5666e9 - 1) < 0.01  # 4 566.6 MB


def test_zipf_bijection_is_a_permutation():
    for n in (10, 97, 1000, 4096):
        a = W._coprime_multiplier(n)
        assert math.gcd(a, n) == 1 and a >= 0.618 * n
        assert len(set(((np.arange(n) * a) % n).tolist())) == n


def test_compact_subproblem_matches_full_tables():
    cfg = W.C1
    rows = cfg.table_rows()
    batch = W.make_batch(cfg, rows)
    full = [W.full_table_storage(cfg, t, int(rows[t])) for t in range(cfg.T)]
    samples = np.array([5, 0, 127, 64])
    sub = W.compact_subproblem(cfg, batch, samples)
    starts = np.concatenate(([0], np.cumsum(batch.lengths)))
    pos = 0
    for i, b in enumerate(samples):
        for t in range(cfg.T):
            g = b * cfg.T + t
            L = batch.lengths[g]
            assert sub.lengths[i * cfg.T + t] == L
            orig = batch.indices[starts[g]:starts[g] + L]
            got_rows = sub.tables[t][sub.indices[pos:pos + L]]
            assert np.array_equal(got_rows, full[t][orig])
            pos += L
    assert pos == sub.indices.shape[0]


def test_to_table_major_is_the_bag_grid_transpose():
    rng = np.random.default_rng(0)
    T, B = 3, 5
    ln = rng.integers(0, 4, size=B * T).astype(np.int32)
    idx = np.arange(int(ln.sum()), dtype=np.int32) + 100
    w = W.make_weights(1, idx.shape[0])
    assert w.dtype == np.float32 and (w >= 0).all() and (w < 2).all()
    ln_tm, idx_tm, w_tm = W.to_table_major(T, B, ln, idx, w)
    starts = np.concatenate(([0], np.cumsum(ln)))
    pos = 0
    for t in range(T):
        for b in range(B):
            g = b * T + t
            assert ln_tm[t * B + b] == ln[g]
            seg = slice(starts[g], starts[g + 1])
            assert np.array_equal(idx_tm[pos:pos + ln[g]], idx[seg]) and np.array_equal(w_tm[pos:pos + ln[g]], w[seg])
            pos += ln[g]
