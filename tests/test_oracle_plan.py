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
