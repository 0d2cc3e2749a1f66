"""Shared helpers of the GPU parity tests: the comparison rule of BASELINE.json's north_star and a driver
that runs the CUDA path through the C ABI (binding) and the oracle on the same seeded inputs."""
from __future__ import annotations

import numpy as np

import oracle
from paper_2606_21101_b200 import workloads as W


def host_offsets(lengths: np.ndarray) -> np.ndarray:
    """Layout helper for handing bags to the oracle (numpy cumsum; the oracle's own plan is checked elsewhere)."""
    return np.concatenate(([0], np.cumsum(np.asarray(lengths, dtype=np.int64)))).astype(np.int32)


def assert_outputs_match(gpu_f64: np.ndarray, ref: np.ndarray, lengths: np.ndarray, T: int, D: int, dtype: str,
                         out_dtype: str = None):
    """north_star: fp32 tables max|err| <= 1e-5 * bag length; fp16/bf16 tables <= 2e-3 relative (fp32
    accumulate), with the absolute floor 1e-6*L for cancellation. Against the UNROUNDED
    float64 reference. Bit-exact when L <= 1; an empty bag is exactly +0.0.
    Only a bf16 OUTPUT cannot meet 2e-3: one correct RNE to 8 significand bits already costs up to
    2^-8 = 3.906e-3 relative, so that variant is held to 2^-8*|ref| + 1e-6*L (reading R6)."""
    out_dtype = out_dtype or dtype
    B = ref.shape[0]
    g = gpu_f64.reshape(B * T, D)
    r = ref.reshape(B * T, D)
    L = np.asarray(lengths, dtype=np.int64).reshape(B * T)
    assert not np.isnan(g).any(), "an output element was never written (NaN sentinel survived)"
    err = np.abs(g - r)
    Lm = np.maximum(L, 1).astype(np.float64)[:, None]
    if dtype == "f32":
        tol = 1e-5 * Lm * np.ones_like(r)
    elif out_dtype == "bf16":
        tol = 2.0 ** -8 * np.abs(r) + 1e-6 * Lm
    else:
        tol = np.maximum(2e-3 * np.abs(r), 1e-6 * Lm)
    bad = err > tol
    assert not bad.any(), (f"{int(bad.sum())} elements out of tolerance; worst err {err.max():.3e} at bag "
                           f"{int(np.argmax(err.max(axis=1)))} (L={int(L[np.argmax(err.max(axis=1))])})")
    short = L <= 1
    if dtype == "f32":
        assert np.array_equal(g[short], r[short]), "bags of length <= 1 must be bit-exact (Alg. 1 is a copy)"
    else:
        # the reference is unrounded float64 of 16-bit values: a single row is exactly representable
        assert np.array_equal(g[short], r[short]), "bags of length <= 1 must be bit-exact"
    empty = L == 0
    assert not g[empty].any() and not np.signbit(g[empty]).any(), "empty bag must be +0.0"
    return float(err.max()) if err.size else 0.0


def oracle_reference(host_tables, dtype: str, B: int, lengths: np.ndarray, indices: np.ndarray, pooling: np.ndarray):
    return oracle.lookup(host_tables, W.DTYPE_CODE[dtype], B, indices, host_offsets(lengths), pooling)


def assert_outputs_match_general(gpu_f64: np.ndarray, ref: np.ndarray, L_bt: np.ndarray, dims, dtype: str,
                                 out_dtype: str = None, weighted: bool = False):
    """The same rule as assert_outputs_match for the interface variants: per-table dims (table t at columns
    [col[t], col[t]+dims[t])), L_bt[b, t] = length of bag (b, t). With per-entry weights a single row is no longer a
    copy: w*x is rounded once to fp32, so bags of length 1 are compared with the fp32 rounding of the reference
    (fp32 output only); |w| <= 2 keeps the stated absolute bounds valid."""
    out_dtype = out_dtype or dtype
    dims = np.asarray(dims, dtype=np.int64)
    B, T = L_bt.shape
    assert gpu_f64.shape == ref.shape == (B, int(dims.sum()))
    assert not np.isnan(gpu_f64).any(), "an output element was never written (NaN sentinel survived)"
    L = np.repeat(np.asarray(L_bt, dtype=np.int64), dims, axis=1)  # [B, sum dims]
    Lm = np.maximum(L, 1).astype(np.float64)
    err = np.abs(gpu_f64 - ref)
    if dtype == "f32":
        tol = 1e-5 * Lm
    elif out_dtype == "bf16":
        tol = 2.0 ** -8 * np.abs(ref) + 1e-6 * Lm
    else:
        tol = np.maximum(2e-3 * np.abs(ref), 1e-6 * Lm)
    bad = err > tol
    assert not bad.any(), f"{int(bad.sum())} elements out of tolerance; worst err {err.max():.3e}"
    short = L <= 1
    if not weighted:
        assert np.array_equal(gpu_f64[short], ref[short]), "bags of length <= 1 must be bit-exact"
    elif out_dtype == "f32":
        assert np.array_equal(gpu_f64[short], ref[short].astype(np.float32).astype(np.float64)), \
            "a weighted single row must be the fp32 rounding of w*x"
    empty = L == 0
    assert not gpu_f64[empty].any() and not np.signbit(gpu_f64[empty]).any(), "empty bag must be +0.0"
    return float(err.max()) if err.size else 0.0
