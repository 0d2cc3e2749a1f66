"""Pins for oracle.plan (CPU only): hand-worked fixture, numpy cumsum, closed form for equal lengths,
cover / monotone / bounded-cost invariants and an O(G*S) brute force written straight from the definition
in DESIGN.md §3."""
import numpy as np
import pytest

import oracle
from tests.golden.load_golden import load


def brute_plan(lengths, K):
    """Definition, slowest possible: seg_bag[s] = min(G, min{g in [0,G] : C[g] >= s*K}) by linear search."""
    G = len(lengths)
    C = [0]
    for L in lengths:
        C.append(C[-1] + max(int(L), 1))
    S = -(-C[G] // K)
    seg = []
    for s in range(S + 1):
        cand = [g for g in range(G + 1) if C[g] >= s * K]
        seg.append(min(G, min(cand)) if cand else G)
    return seg, S


def test_golden_fig5_plan():
    g = load("fig5_shape_example.txt")
    lengths = np.array(g["multihot.lengths"], dtype=np.int32).reshape(-1)
    K = int(g["plan.K"][0][0])
    off, seg, S, seg_off = oracle.plan(lengths, K, with_seg_off=True)
    assert off.tolist() == [int(x) for x in g["plan.offsets"][0]]
    assert S == int(g["plan.S"][0][0])
    assert seg.tolist() == [int(x) for x in g["plan.seg_bag"][0]]
    assert seg_off.tolist() == [int(x) for x in g["plan.seg_off"][0]]


@pytest.mark.parametrize("seed", range(6))
@pytest.mark.parametrize("K", [1, 2, 3, 7, 32, 1000])
def test_plan_matches_brute_force_and_cumsum(seed, K):
    rng = np.random.default_rng(seed)
    G = int(rng.integers(1, 60))
    lengths = rng.integers(0, 9, size=G).astype(np.int32)
    if seed % 3 == 0:
        lengths[rng.random(G) < 0.5] = 0
    off, seg, S = oracle.plan(lengths, K)
    assert off[0] == 0 and np.array_equal(np.diff(off), lengths) and off[-1] == lengths.sum()
    assert np.array_equal(off[1:], np.cumsum(lengths))
    bseg, bS = brute_plan(lengths.tolist(), K)
    assert S == bS and seg.tolist() == bseg
    seg_off = oracle.plan(lengths, K, with_seg_off=True)[3]
    assert seg_off.tolist() == [int(np.sum(lengths[:g])) for g in bseg]  # entries before the task's first bag


@pytest.mark.parametrize("ell", [1, 2, 3, 5, 64])
@pytest.mark.parametrize("K", [1, 4, 32, 33])
def test_equal_lengths_closed_form(ell, K):
    """len == ell >= 1 for every bag: C[g] = g*ell, so seg_bag[s] = min(G, ceil(s*K/ell)), S = ceil(G*ell/K)."""
    G = 1000
    off, seg, S = oracle.plan(np.full(G, ell, np.int32), K)
    assert S == -(-G * ell // K)
    want = [min(G, -(-s * K // ell)) for s in range(S + 1)]
    assert seg.tolist() == want
    assert np.array_equal(off, np.arange(G + 1) * ell)


def test_all_empty_bags():
    G, K = 1000, 32
    off, seg, S = oracle.plan(np.zeros(G, np.int32), K)
    assert not off.any()
    assert S == -(-G // K)
    assert seg.tolist() == [min(G, s * K) for s in range(S + 1)]


@pytest.mark.parametrize("K", [1, 8, 32, 100])
def test_invariants_on_ctr_shaped_lengths(K):
    rng = np.random.default_rng(11)
    G = 20000
    lengths = np.minimum(rng.poisson(20, size=G), 100).astype(np.int32)
    lengths[rng.random(G) < 0.05] = 0
    off, seg, S = oracle.plan(lengths, K)
    cost = np.maximum(lengths, 1).astype(np.int64)
    C = np.concatenate(([0], np.cumsum(cost)))
    assert seg[0] == 0 and seg[S] == G and len(seg) == S + 1
    assert np.all(np.diff(seg) >= 0)  # monotone -> every bag lies in exactly one [seg[s], seg[s+1])
    seg_cost = C[seg[1:]] - C[seg[:-1]]
    assert seg_cost.sum() == C[G]
    assert np.all(seg_cost < K + cost.max())  # bounded: a segment overshoots its quantum by < one bag
    # lower-bound property, both sides
    s_arr = np.arange(S + 1) * K
    assert np.all((C[seg] >= s_arr) | (seg == G))
    inner = seg > 0
    assert np.all(C[seg[inner] - 1] < s_arr[inner])


def test_single_long_bag_spans_several_quanta():
    off, seg, S = oracle.plan(np.array([100], np.int32), 32)
    assert S == 4 and seg.tolist() == [0, 1, 1, 1, 1] and off.tolist() == [0, 100]


def test_zero_bags():
    off, seg, S = oracle.plan(np.zeros(0, np.int32), 32)
    assert off.tolist() == [0] and S == 0 and seg.tolist() == [0]


def test_rejects_negative_length_and_overflow():
    with pytest.raises(oracle.OracleError):
        oracle.plan(np.array([1, -1], np.int32), 4)
    with pytest.raises(oracle.OracleError):
        oracle.plan(np.full(3, 2 ** 30, np.int32), 2 ** 20)


# --------------------------------------------------------------------------------------------------
# a1's min / max bag length (SURVEY.md 8(a) a1 "uniform-length flag"): DESIGN.md §3
# --------------------------------------------------------------------------------------------------
def test_golden_fig5_plan_stats():
    g = load("fig5_shape_example.txt")
    lengths = np.array(g["multihot.lengths"], dtype=np.int32).reshape(-1)
    assert oracle.plan_stats(lengths) == (int(g["plan.min_len"][0][0]), int(g["plan.max_len"][0][0]))
    onehot = np.ones(np.array(g["onehot.ids"]).size, dtype=np.int32)   # Alg. 1: one id per (sample, field)
    assert oracle.plan_stats(onehot) == (int(g["onehot.min_len"][0][0]), int(g["onehot.max_len"][0][0]))


@pytest.mark.parametrize("ell", [0, 1, 7, 2 ** 31 - 1])
def test_plan_stats_constant_lengths(ell):
    assert oracle.plan_stats(np.full(1000, ell, np.int32)) == (ell, ell)


def test_plan_stats_closed_forms_and_invariants():
    # arithmetic progression a, a+1, ..., a+n-1 in any order: min = a, max = a+n-1
    rng = np.random.default_rng(5)
    for a, n in [(0, 1), (3, 10), (1, 4096), (100, 2049)]:
        ln = (a + rng.permutation(n)).astype(np.int32)
        assert oracle.plan_stats(ln) == (a, a + n - 1)
    # the extreme sits first / last / alone
    assert oracle.plan_stats(np.array([9, 1, 1, 1], np.int32)) == (1, 9)
    assert oracle.plan_stats(np.array([1, 1, 1, 0], np.int32)) == (0, 1)
    assert oracle.plan_stats(np.array([5], np.int32)) == (5, 5)
    assert oracle.plan_stats(np.zeros(0, np.int32)) == (0, 0)
    # brute force through a sort; invariants min <= N/G <= max; invariance under permutation; concatenation rule
    for seed in range(5):
        r = np.random.default_rng(seed)
        ln = r.integers(0, 50, size=int(r.integers(1, 300))).astype(np.int32)
        lo, hi = oracle.plan_stats(ln)
        srt = sorted(ln.tolist())
        assert (lo, hi) == (srt[0], srt[-1])
        assert lo * len(ln) <= int(ln.sum()) <= hi * len(ln)
        assert oracle.plan_stats(r.permutation(ln)) == (lo, hi)
        other = r.integers(0, 80, size=17).astype(np.int32)
        lo2, hi2 = oracle.plan_stats(other)
        assert oracle.plan_stats(np.concatenate([ln, other])) == (min(lo, lo2), max(hi, hi2))
    with pytest.raises(oracle.OracleError):
        oracle.plan_stats(np.array([1, -2], np.int32))


def test_plan_stats_on_the_five_configs():
    """The recipes fix the extremes: c2 is one-hot (uniform flag), c1 U{1..4}, c3 U{1..3}, c5 U{1..64} hit both ends at
    these batch sizes; c4 = Poisson(20) capped at 100 with 5 % empty bags -> min 0."""
    from paper_2606_21101_b200 import workloads as W
    assert oracle.plan_stats(W.make_lengths(W.C2, 0)) == (1, 1)
    assert oracle.plan_stats(W.make_lengths(W.C1, 0)) == (1, 4)
    assert oracle.plan_stats(W.make_lengths(W.C3, 0)) == (1, 3)
    assert oracle.plan_stats(W.make_lengths(W.C5, 0)) == (1, 64)
    lo, hi = oracle.plan_stats(W.make_lengths(W.C4, 0))
    assert lo == 0 and 30 <= hi <= 100


# --------------------------------------------------------------------------------------------------
# the plan with 64-bit offsets: same definition, N may pass 2^31
# --------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("seed", range(4))
@pytest.mark.parametrize("K", [1, 3, 32, 1000])
def test_plan64_equals_the_32_bit_plan_and_brute_force_where_both_exist(seed, K):
    rng = np.random.default_rng(100 + seed)
    lengths = rng.integers(0, 9, size=int(rng.integers(1, 80))).astype(np.int32)
    off, seg, S, seg_off = oracle.plan(lengths, K, with_seg_off=True)
    off64, seg64, S64, seg_off64 = oracle.plan64(lengths, K)
    assert off64.dtype == np.int64 and seg_off64.dtype == np.int64
    assert S64 == S and np.array_equal(off64, off) and np.array_equal(seg64, seg) and np.array_equal(seg_off64, seg_off)
    bseg, bS = brute_plan(lengths.tolist(), K)
    assert S64 == bS and seg64.tolist() == bseg


def test_plan64_golden_fig5():
    g = load("fig5_shape_example.txt")
    lengths = np.array(g["multihot.lengths"], dtype=np.int32).reshape(-1)
    off, seg, S, seg_off = oracle.plan64(lengths, int(g["plan.K"][0][0]))
    assert off.tolist() == [int(x) for x in g["plan.offsets"][0]] and S == int(g["plan.S"][0][0])
    assert seg.tolist() == [int(x) for x in g["plan.seg_bag"][0]]
    assert seg_off.tolist() == [int(x) for x in g["plan.seg_off"][0]]


@pytest.mark.parametrize("ell,G,K", [(2 ** 30, 3, 2 ** 20), (2 ** 31 - 1, 5, 2 ** 31 - 1), (3 * 2 ** 20, 1024, 12345),
                                     (2 ** 29, 9, 2 ** 33)])
def test_plan64_equal_lengths_closed_form_beyond_2_pow_31(ell, G, K):
    """len == ell for every bag: offsets[g] = g*ell, C[g] = g*ell, S = ceil(G*ell/K), seg_bag[s] = min(G, ceil(s*K/ell)),
    seg_off[s] = seg_bag[s]*ell -- with N = G*ell >= 2^31, where the 32-bit plan refuses."""
    lengths = np.full(G, ell, np.int32)
    assert G * ell >= 2 ** 31
    with pytest.raises(oracle.OracleError):
        oracle.plan(lengths, min(K, 2 ** 31 - 1))
    off, seg, S, seg_off = oracle.plan64(lengths, K)
    assert S == -(-G * ell // K)
    assert off.tolist() == [g * ell for g in range(G + 1)]
    want = [min(G, -(-s * K // ell)) for s in range(S + 1)]
    assert seg.tolist() == want and seg_off.tolist() == [w * ell for w in want]


def test_plan64_mixed_lengths_past_2_pow_31_invariants():
    rng = np.random.default_rng(9)
    G, K = 4000, 2 ** 16
    lengths = rng.integers(0, 2 ** 21, size=G).astype(np.int32)
    lengths[rng.random(G) < 0.1] = 0
    off, seg, S, seg_off = oracle.plan64(lengths, K)
    assert int(off[-1]) == int(lengths.astype(np.int64).sum()) >= 2 ** 31
    assert np.array_equal(np.diff(off), lengths)
    C = np.concatenate(([0], np.cumsum(np.maximum(lengths, 1).astype(np.int64))))
    assert S == -(-int(C[G]) // K) and seg[0] == 0 and seg[S] == G and np.all(np.diff(seg) >= 0)
    s_arr = np.arange(S + 1, dtype=np.int64) * K
    assert np.all((C[seg] >= s_arr) | (seg == G))
    inner = seg > 0
    assert np.all(C[seg[inner] - 1] < s_arr[inner])
    assert np.array_equal(seg_off, off[seg])
