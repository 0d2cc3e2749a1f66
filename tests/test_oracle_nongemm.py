"""Pins for oracle/nongemm_oracle.c: every check is against something other
than the oracle's own formula -- hand-worked fixtures, closed forms, exact integer / rational arithmetic, library
routines, invariants.  CPU only."""
from fractions import Fraction
from itertools import combinations

import numpy as np
import pytest

import oracle
from tests.golden.load_golden import load

GOLD = load("nongemm_examples.txt")


# ---------------------------------------------------------------------------------------------------------------
# FM second-order term
# ---------------------------------------------------------------------------------------------------------------
def test_fm_hand_worked_fixture():
    x = np.array(GOLD["fm.x"])
    y, v = oracle.fm_pairwise(x, 3, 2)
    assert np.array_equal(v, np.array(GOLD["fm.v"]))
    assert np.array_equal(y, np.array(GOLD["fm.y"][0]))


def test_fm_two_fields_is_a_dot_product():
    rng = np.random.default_rng(0)
    x = rng.standard_normal((7, 2 * 12))
    y, v = oracle.fm_pairwise(x, 2, 12)
    for b in range(7):
        assert y[b] == pytest.approx(np.dot(x[b, :12], x[b, 12:]), rel=1e-14, abs=1e-14)
    assert np.allclose(v, x[:, :12] * x[:, 12:], rtol=1e-15, atol=0)


@pytest.mark.parametrize("T,D", [(1, 4), (2, 4), (5, 3), (26, 16), (39, 8)])
def test_fm_closed_forms(T, D):
    ones = np.ones((3, T * D))
    y, v = oracle.fm_pairwise(ones, T, D)
    assert np.array_equal(y, np.full(3, T * (T - 1) // 2 * D))          # C(T,2) pairs, D ones each
    assert np.array_equal(v, np.full((3, D), T * (T - 1) // 2))
    # field t = a_t * e (same direction, integer magnitudes): y = D * sum_{t<u} a_t a_u
    a = np.arange(1, T + 1)
    x = np.repeat(a, D)[None, :].astype(np.float64)
    y, _ = oracle.fm_pairwise(x, T, D)
    assert y[0] == D * sum(int(p) * int(q) for p, q in combinations(a, 2))


def test_fm_orthogonal_fields_give_zero_and_single_field_gives_zero():
    D = 6
    x = np.zeros((1, 6 * D))
    for t in range(6):
        x[0, t * D + t] = t + 1.5       # field t is a multiple of the unit vector e_t
    y, v = oracle.fm_pairwise(x, 6, D)
    assert y[0] == 0.0 and not v.any()
    y, _ = oracle.fm_pairwise(np.arange(8.0)[None, :], 1, 8)
    assert y[0] == 0.0


def test_fm_square_of_sum_identity_in_exact_integer_arithmetic():
    """0.5 * ((sum_t x_t)^2 - sum_t x_t^2), the rearrangement named by the paper's operators ("element-wise square and
    reduce-sum"), evaluated in Python integers: must equal the pairwise definition exactly."""
    rng = np.random.default_rng(1)
    T, D, B = 9, 5, 4
    xi = rng.integers(-50, 51, size=(B, T, D))
    y, v = oracle.fm_pairwise(xi.reshape(B, T * D).astype(np.float64), T, D)
    for b in range(B):
        tot = 0
        for c in range(D):
            col = [int(z) for z in xi[b, :, c]]
            twice = sum(col) ** 2 - sum(z * z for z in col)
            assert twice % 2 == 0 and v[b, c] == twice // 2
            tot += twice // 2
        assert y[b] == tot


def test_fm_field_permutation_invariance_homogeneity_and_row_pitch():
    rng = np.random.default_rng(2)
    T, D, B = 7, 4, 5
    x = rng.integers(-8, 9, size=(B, T, D)).astype(np.float64)      # integers: every product and sum is exact
    y, v = oracle.fm_pairwise(x.reshape(B, -1), T, D)
    perm = rng.permutation(T)
    y2, v2 = oracle.fm_pairwise(x[:, perm, :].reshape(B, -1), T, D)
    assert np.array_equal(y, y2) and np.array_equal(v, v2)
    y3, _ = oracle.fm_pairwise(4.0 * x.reshape(B, -1), T, D)           # degree-2 homogeneous; 4 and 16 are powers of two
    assert np.array_equal(y3, 16.0 * y)
    wide = np.full((B, T * D + 3), 1e30)                                # columns past T*D are not part of the block
    wide[:, : T * D] = x.reshape(B, -1)
    y4, _ = oracle.fm_pairwise(wide, T, D)
    assert np.array_equal(y4, y)


# ---------------------------------------------------------------------------------------------------------------
# DCNv2 cross combine
# ---------------------------------------------------------------------------------------------------------------
def test_cross_hand_worked_fixture():
    out = oracle.cross_combine(GOLD["cross.x0"], GOLD["cross.xl"], GOLD["cross.u"], GOLD["cross.bias"][0])
    assert np.array_equal(out, np.array(GOLD["cross.out"]))


def test_cross_special_cases():
    rng = np.random.default_rng(3)
    x0, xl, u = (rng.integers(-9, 10, size=(4, 6)).astype(np.float64) for _ in range(3))
    b = rng.integers(-3, 4, size=6).astype(np.float64)
    z = np.zeros_like(x0)
    assert np.array_equal(oracle.cross_combine(x0, xl, z, None), xl)                 # W = 0, b = 0: identity layer
    assert np.array_equal(oracle.cross_combine(z, xl, u, b), xl)                     # x0 = 0
    assert np.array_equal(oracle.cross_combine(x0, z, np.ones_like(u), None), x0)    # u = 1, xl = 0
    assert np.array_equal(oracle.cross_combine(x0, xl, -b[None, :].repeat(4, 0), b), xl)   # u = -bias
    # bias is per FEATURE (column), not per row: a one-hot bias touches exactly one column
    e = np.zeros(6); e[2] = 1.0
    d = oracle.cross_combine(x0, xl, u, e) - oracle.cross_combine(x0, xl, u, None)
    assert np.array_equal(d[:, 2], x0[:, 2]) and not np.delete(d, 2, axis=1).any()


def test_cross_scalar_recurrence_in_exact_rationals():
    """F = 1: x_{l+1} = x0 (w x_l + b) + x_l (DCNv2 with a 1x1 weight), three layers, against Fractions."""
    x0, w, b = Fraction(3, 4), Fraction(-5, 8), Fraction(1, 2)
    xl_f, xl = x0, np.array([[float(x0)]])
    for _ in range(3):
        u = np.array([[float(w)]]) * xl                       # the GEMM part (1x1), exact in binary
        xl = oracle.cross_combine(np.array([[float(x0)]]), xl, u, np.array([float(b)]))
        xl_f = x0 * (w * xl_f + b) + xl_f
        assert Fraction(float(xl[0, 0])) == xl_f                # dyadic rationals: float64 holds them exactly


# ---------------------------------------------------------------------------------------------------------------
# bias + activation
# ---------------------------------------------------------------------------------------------------------------
def test_bias_act_hand_worked_fixture():
    u, b = GOLD["act.u"], GOLD["act.bias"][0]
    assert np.array_equal(oracle.bias_act(u, b, oracle.ACT_IDENTITY), np.array(GOLD["act.identity"]))
    assert np.array_equal(oracle.bias_act(u, b, oracle.ACT_RELU), np.array(GOLD["act.relu"]))
    s = oracle.bias_act(u, b, oracle.ACT_SIGMOID)
    assert s[0, 1] == 0.5 and s[0, 2] == 0.5


def test_relu_properties():
    rng = np.random.default_rng(4)
    u = rng.standard_normal((5, 9))
    r = oracle.bias_act(u, None, oracle.ACT_RELU)
    assert np.array_equal(r, (u + np.abs(u)) / 2)                                   # relu(v) = (v + |v|) / 2
    assert np.array_equal(oracle.bias_act(r, None, oracle.ACT_RELU), r)             # idempotent
    assert (r >= 0).all() and np.array_equal(r[u > 0], u[u > 0])
    assert np.array_equal(oracle.bias_act(u, None, oracle.ACT_RELU) - oracle.bias_act(-u, None, oracle.ACT_RELU), u)


def test_sigmoid_against_library_and_symmetry():
    from scipy.special import expit
    rng = np.random.default_rng(5)
    u = rng.standard_normal((6, 7)) * 4
    b = rng.standard_normal(7)
    s = oracle.bias_act(u, b, oracle.ACT_SIGMOID)
    assert np.allclose(s, expit(u + b[None, :]), rtol=1e-14, atol=1e-16)
    s_neg = oracle.bias_act(-u, -b, oracle.ACT_SIGMOID)
    assert np.allclose(s + s_neg, 1.0, rtol=0, atol=1e-15)
    assert oracle.bias_act(np.zeros((1, 1)), None, oracle.ACT_SIGMOID)[0, 0] == 0.5


# ---------------------------------------------------------------------------------------------------------------
# DeepFM first-order (logistic regression) term
# ---------------------------------------------------------------------------------------------------------------
LR_W = [np.array([1.0, 2, 3]), np.array([10.0, 20]), np.array([100.0, 200, 300, 400])]


def test_lr_hand_worked_fixture():
    ln = np.array(GOLD["lr.lengths"]).reshape(-1).astype(np.int64)
    idx = np.concatenate([np.array(r) for r in GOLD["lr.indices"]]).astype(np.int32)
    off = np.concatenate(([0], np.cumsum(ln))).astype(np.int32)
    assert np.array_equal(oracle.lr_first_order(LR_W, 2, idx, off, bias=0.5), np.array(GOLD["lr.y"][0]))
    ids = np.array(GOLD["lr.onehot_ids"]).reshape(-1).astype(np.int32)
    assert np.array_equal(oracle.lr_first_order(LR_W, 2, ids, None, bias=0.5), np.array(GOLD["lr.onehot_y"][0]))


def test_lr_closed_forms_and_library_routines():
    rng = np.random.default_rng(7)
    T, B = 6, 40
    rows = [5, 1, 300, 17, 64, 9]
    ln = rng.integers(0, 5, size=B * T)
    off = np.concatenate(([0], np.cumsum(ln))).astype(np.int32)
    idx = np.concatenate([rng.integers(0, rows[g % T], size=ln[g]) for g in range(B * T)]).astype(np.int32)
    # constant weights kappa_t = 2^t: y = bias + sum_t 2^t * len(b, t), exactly
    w = [np.full(rows[t], 2.0 ** t) for t in range(T)]
    y = oracle.lr_first_order(w, B, idx, off, bias=-3.0)
    assert np.array_equal(y, -3.0 + (ln.reshape(B, T) * 2.0 ** np.arange(T)).sum(axis=1))
    # integer weights: numpy take + add.reduceat-free brute force in Python ints
    wi = [rng.integers(-50, 51, size=rows[t]).astype(np.float64) for t in range(T)]
    y = oracle.lr_first_order(wi, B, idx, off)
    for b in range(B):
        tot = 0
        for t in range(T):
            g = b * T + t
            tot += int(sum(int(wi[t][r]) for r in idx[off[g]:off[g + 1]]))
        assert y[b] == tot
    # one-hot: numpy take per table, summed over tables
    ids = np.stack([rng.integers(0, rows[t], size=B) for t in range(T)], axis=1).astype(np.int32)
    y1 = oracle.lr_first_order(wi, B, ids.reshape(-1), None, bias=1.0)
    assert np.array_equal(y1, 1.0 + sum(np.take(wi[t], ids[:, t]) for t in range(T)))
    # the same thing through the separately pinned pooled lookup: width-1 tables, sum pooling, then a row sum
    ref = oracle.lookup([w_.astype(np.float32).reshape(-1, 1) for w_ in wi], oracle.F32, B, idx, off, np.zeros(T, np.uint8))
    assert np.array_equal(y, ref.sum(axis=1))


def test_bad_arguments_are_rejected():
    with pytest.raises(oracle.OracleError):
        oracle.bias_act(np.zeros((1, 1)), None, 7)
    with pytest.raises(ValueError):
        oracle.cross_combine(np.zeros((2, 3)), np.zeros((2, 3)), np.zeros((2, 4)))
    with pytest.raises(oracle.OracleError):
        oracle.fm_pairwise(np.zeros((2, 5)), 2, 3)      # row shorter than T*D


# ---------------------------------------------------------------------------------------------------------------
# Algorithm 2
# ---------------------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("key", ["bfs.2_4", "bfs.3_3", "bfs.3_1", "bfs.0_2"])
def test_bfs_queue_hand_expansions(key):
    ne, ni = (int(z) for z in key.split(".")[1].split("_"))
    flat = [int(z) for z in GOLD[key][0]]
    want = list(zip(flat[0::2], flat[1::2]))
    assert oracle.bfs_queue(ne, ni) == want


@pytest.mark.parametrize("ne", range(0, 7))
@pytest.mark.parametrize("ni", range(0, 7))
def test_bfs_queue_invariants(ne, ni):
    q = oracle.bfs_queue(ne, ni)
    assert sorted(q) == [(0, i) for i in range(ne)] + [(1, i) for i in range(ni)]          # every op exactly once
    for m in (0, 1):
        assert [i for mm, i in q if mm == m] == list(range(ne if m == 0 else ni))          # per-module order kept
    if q:
        first = 1 if ni > ne else 0                # "The module that has more operators launches first"
        assert q[0][0] == first
    k = min(ne, ni)
    head = q[: 2 * k]
    assert all(head[i][0] != head[i + 1][0] for i in range(len(head) - 1))                 # alternating pattern
    assert all(mm == (1 if ni > ne else 0) for mm, _ in q[2 * k:])                          # tail = the longer module
