"""ctypes loader for the plain-C CPU oracle (``dpi_oracle.c``).

TEST INFRASTRUCTURE ONLY. May be imported by ``tests/``, ``__graft_entry__.smoke()`` and ``bench.py``'s
``cpu_baseline`` / ``--impl reference`` legs; never by ``paper_2606_21101_b200``. It imports nothing from
the CUDA path. Argument marshalling only: every number comes out of ``dpi_oracle.c``.
"""
from __future__ import annotations

import ctypes
import os
import subprocess
import threading
from typing import Sequence

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "dpi_oracle.c")
_SRC_NONGEMM = os.path.join(_HERE, "nongemm_oracle.c")
_LIB = os.path.join(_HERE, "liboracle.so")
_lock = threading.Lock()
_lib = None

F32, F16, BF16 = 0, 1, 2
SUM, MEAN = 0, 1
_STATUS = {0: "ok", 1: "bad argument", 2: "index out of range", 3: "offset overflow (N >= 2^31)",
           4: "seg_bag capacity too small"}


class OracleError(RuntimeError):
    pass


def build(force: bool = False) -> str:
    """Compile dpi_oracle.c -> liboracle.so with gcc (-O2, no fast-math, no FMA contraction)."""
    with _lock:
        newest = max(os.path.getmtime(_SRC), os.path.getmtime(_SRC_NONGEMM))
        if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < newest:
            tmp = _LIB + f".tmp{os.getpid()}"
            # -fopenmp only serves oracle_lookup_par (the all-cores timing leg); every other function is a plain loop
            subprocess.check_call(["gcc", "-O2", "-std=c11", "-ffp-contract=off", "-fopenmp", "-fPIC", "-shared",
                                   "-Wall", "-Wextra", "-o", tmp, _SRC, _SRC_NONGEMM, "-lm"])
            os.replace(tmp, _LIB)
    return _LIB


def _load():
    global _lib
    if _lib is None:
        lib = ctypes.CDLL(build())
        vp, i32, i64 = ctypes.c_void_p, ctypes.c_int32, ctypes.c_int64
        lib.oracle_alg1_onehot.argtypes = [i32, i32, i32, ctypes.c_int, vp, vp, vp, vp]
        lib.oracle_alg1_onehot.restype = ctypes.c_int
        lib.oracle_lookup.argtypes = [i32, i32, i32, ctypes.c_int, vp, vp, vp, vp, vp, vp]
        lib.oracle_lookup.restype = ctypes.c_int
        lib.oracle_lookup_general.argtypes = [i32, i32, vp, ctypes.c_int, vp, vp, vp, vp, vp, vp, ctypes.c_int, vp]
        lib.oracle_lookup_general.restype = ctypes.c_int
        lib.oracle_plan.argtypes = [vp, i64, i32, vp, vp, vp, i64, vp]
        lib.oracle_plan.restype = ctypes.c_int
        lib.oracle_lookup_par.argtypes = [i32, i32, i32, ctypes.c_int, vp, vp, vp, vp, vp, vp, vp]
        lib.oracle_lookup_par.restype = ctypes.c_int
        lib.oracle_plan_stats.argtypes = [vp, i64, vp, vp]
        lib.oracle_plan_stats.restype = ctypes.c_int
        lib.oracle_plan64.argtypes = [vp, i64, i64, vp, vp, vp, i64, vp]
        lib.oracle_plan64.restype = ctypes.c_int
        lib.oracle_decode_f16.argtypes = [ctypes.c_uint16]
        lib.oracle_decode_f16.restype = ctypes.c_double
        lib.oracle_decode_bf16.argtypes = [ctypes.c_uint16]
        lib.oracle_decode_bf16.restype = ctypes.c_double
        lib.oracle_fm_pairwise.argtypes = [i32, i32, i32, vp, i64, vp, vp]
        lib.oracle_fm_pairwise.restype = ctypes.c_int
        lib.oracle_cross_combine.argtypes = [i32, i32, vp, vp, vp, vp, vp]
        lib.oracle_cross_combine.restype = ctypes.c_int
        lib.oracle_bias_act.argtypes = [i32, i32, vp, vp, ctypes.c_int, vp]
        lib.oracle_bias_act.restype = ctypes.c_int
        lib.oracle_lr_first_order.argtypes = [i32, i32, vp, vp, vp, vp, ctypes.c_double, vp]
        lib.oracle_lr_first_order.restype = ctypes.c_int
        lib.oracle_bfs_queue.argtypes = [i32, i32, vp, vp]
        lib.oracle_bfs_queue.restype = ctypes.c_int
        _lib = lib
    return _lib


def _check(rc: int):
    if rc != 0:
        raise OracleError(_STATUS.get(rc, f"status {rc}"))


_STORAGE = {F32: np.float32, F16: np.float16, BF16: np.uint16}


def _table_ptrs(tables: Sequence[np.ndarray], dtype: int, D):
    """D: the common embedding dim, or a per-table sequence of dims."""
    keep = []
    dims = [int(D)] * len(tables) if np.isscalar(D) else [int(d) for d in D]
    for t, D in zip(tables, dims):
        a = np.ascontiguousarray(t)
        if dtype == F16 and a.dtype == np.uint16:
            pass  # raw binary16 bits are accepted as well
        elif a.dtype != _STORAGE[dtype]:
            raise TypeError(f"table dtype {a.dtype} does not match oracle dtype code {dtype}")
        if a.ndim != 2 or a.shape[1] != D:
            raise ValueError("table must be [rows, D]")
        keep.append(a)
    arr = (ctypes.c_void_p * len(keep))(*[a.ctypes.data for a in keep])
    rows = np.asarray([a.shape[0] for a in keep], dtype=np.int64)
    return arr, rows, keep


def alg1_onehot(tables: Sequence[np.ndarray], dtype: int, ids: np.ndarray) -> np.ndarray:
    """Algorithm 1. ids int32[b, k] -> float64[b, k*d]."""
    ids = np.ascontiguousarray(ids, dtype=np.int32)
    b, k = ids.shape
    d = int(np.asarray(tables[0]).shape[1])
    ptrs, rows, keep = _table_ptrs(tables, dtype, d)
    out = np.empty((b, k * d), dtype=np.float64)
    _check(_load().oracle_alg1_onehot(b, k, d, dtype, ctypes.cast(ptrs, ctypes.c_void_p), rows.ctypes.data,
                                      ids.ctypes.data, out.ctypes.data))
    del keep
    return out


def _out_block(out, B: int, width: int) -> np.ndarray:
    """The caller's float64 [B, width] block (timing loops reuse one), or a fresh one."""
    if out is None:
        return np.empty((B, width), dtype=np.float64)
    if out.dtype != np.float64 or out.shape != (B, width) or not out.flags.c_contiguous:
        raise ValueError("out must be a C-contiguous float64 [B, T*D] array")
    return out


def lookup(tables: Sequence[np.ndarray], dtype: int, B: int, indices: np.ndarray, offsets: np.ndarray,
           pooling: np.ndarray, out: np.ndarray = None) -> np.ndarray:
    """Pooled multi-hot lookup. Returns the unrounded float64 reference [B, T*D] (written into `out` when
    given)."""
    T = len(tables)
    D = int(np.asarray(tables[0]).shape[1])
    indices = np.ascontiguousarray(indices, dtype=np.int32)
    offsets = np.ascontiguousarray(offsets, dtype=np.int32)
    pooling = np.ascontiguousarray(pooling, dtype=np.uint8)
    if offsets.shape[0] != B * T + 1 or pooling.shape[0] != T:
        raise ValueError("offsets must be [B*T+1], pooling [T]")
    if int(offsets[-1]) > indices.shape[0]:
        raise ValueError("offsets[-1] exceeds len(indices)")
    ptrs, rows, keep = _table_ptrs(tables, dtype, D)
    ref = _out_block(out, B, T * D)
    _check(_load().oracle_lookup(T, B, D, dtype, ctypes.cast(ptrs, ctypes.c_void_p), rows.ctypes.data,
                                 indices.ctypes.data, offsets.ctypes.data, pooling.ctypes.data,
                                 ref.ctypes.data))
    del keep
    return ref


def lookup_par(tables: Sequence[np.ndarray], dtype: int, B: int, indices: np.ndarray, offsets: np.ndarray,
               pooling: np.ndarray, out: np.ndarray = None):
    """oracle_lookup on all host cores (OpenMP over samples; bit-identical block). Returns (ref float64[B, T*D],
    threads used). bench.py's cpu_baseline timing leg; the tests pin it to lookup()."""
    T = len(tables)
    D = int(np.asarray(tables[0]).shape[1])
    indices = np.ascontiguousarray(indices, dtype=np.int32)
    offsets = np.ascontiguousarray(offsets, dtype=np.int32)
    pooling = np.ascontiguousarray(pooling, dtype=np.uint8)
    if offsets.shape[0] != B * T + 1 or pooling.shape[0] != T:
        raise ValueError("offsets must be [B*T+1], pooling [T]")
    if int(offsets[-1]) > indices.shape[0]:
        raise ValueError("offsets[-1] exceeds len(indices)")
    ptrs, rows, keep = _table_ptrs(tables, dtype, D)
    ref = _out_block(out, B, T * D)
    team = ctypes.c_int32(0)
    _check(_load().oracle_lookup_par(T, B, D, dtype, ctypes.cast(ptrs, ctypes.c_void_p), rows.ctypes.data,
                                     indices.ctypes.data, offsets.ctypes.data, pooling.ctypes.data,
                                     ref.ctypes.data, ctypes.byref(team)))
    del keep
    return ref, int(team.value)


SAMPLE_MAJOR, TABLE_MAJOR = 0, 1


def lookup_general(tables: Sequence[np.ndarray], dtype: int, B: int, indices: np.ndarray, offsets: np.ndarray,
                   pooling: np.ndarray, weights: np.ndarray = None, bag_order: int = SAMPLE_MAJOR) -> np.ndarray:
    """Interface variants (mixed per-table dims, int64 indices/offsets, per-entry fp32 weights, table-major bags).
    Returns the unrounded float64 reference [B, sum(dims)]."""
    T = len(tables)
    dims = np.asarray([np.asarray(t).shape[1] for t in tables], dtype=np.int32)
    indices = np.ascontiguousarray(indices, dtype=np.int64)
    offsets = np.ascontiguousarray(offsets, dtype=np.int64)
    pooling = np.ascontiguousarray(pooling, dtype=np.uint8)
    if offsets.shape[0] != B * T + 1 or pooling.shape[0] != T:
        raise ValueError("offsets must be [B*T+1], pooling [T]")
    if int(offsets[-1]) > indices.shape[0]:
        raise ValueError("offsets[-1] exceeds len(indices)")
    w = None
    if weights is not None:
        w = np.ascontiguousarray(weights, dtype=np.float32)
        if w.shape[0] != indices.shape[0]:
            raise ValueError("weights must have one entry per index")
    ptrs, rows, keep = _table_ptrs(tables, dtype, dims)
    ref = np.empty((B, int(dims.sum())), dtype=np.float64)
    _check(_load().oracle_lookup_general(T, B, dims.ctypes.data, dtype, ctypes.cast(ptrs, ctypes.c_void_p),
                                         rows.ctypes.data, indices.ctypes.data, offsets.ctypes.data,
                                         None if w is None else w.ctypes.data, pooling.ctypes.data, int(bag_order),
                                         ref.ctypes.data))
    del keep
    return ref


def plan(lengths: np.ndarray, K: int, with_seg_off: bool = False):
    """Workload plan. Returns (offsets int32[G+1], seg_bag int32[S+1], S) and, with
    with_seg_off=True, seg_off int32[S+1] as a fourth element."""
    lengths = np.ascontiguousarray(lengths, dtype=np.int32)
    G = lengths.shape[0]
    cap = (int(lengths.astype(np.int64).sum()) + G) // max(K, 1) + 3  # upper bound on S+1 (C[G] <= N + G)
    offsets = np.empty(G + 1, dtype=np.int32)
    seg_bag = np.empty(cap, dtype=np.int32)
    seg_off = np.empty(cap, dtype=np.int32)
    S = ctypes.c_int32(0)
    _check(_load().oracle_plan(lengths.ctypes.data, G, K, offsets.ctypes.data, seg_bag.ctypes.data,
                               seg_off.ctypes.data, cap, ctypes.byref(S)))
    res = (offsets, seg_bag[: S.value + 1].copy(), int(S.value))
    return res + (seg_off[: S.value + 1].copy(),) if with_seg_off else res


def plan_stats(lengths: np.ndarray):
    """(min_len, max_len) of the bag-length sequence (both 0 for G == 0)."""
    lengths = np.ascontiguousarray(lengths, dtype=np.int32)
    lo, hi = ctypes.c_int32(0), ctypes.c_int32(0)
    _check(_load().oracle_plan_stats(lengths.ctypes.data, lengths.shape[0], ctypes.byref(lo), ctypes.byref(hi)))
    return int(lo.value), int(hi.value)


def plan64(lengths: np.ndarray, K: int):
    """The plan with 64-bit offsets (N may be >= 2^31). Returns (offsets int64[G+1], seg_bag int32[S+1], S,
    seg_off int64[S+1])."""
    lengths = np.ascontiguousarray(lengths, dtype=np.int32)
    G = lengths.shape[0]
    cap = (int(lengths.astype(np.int64).sum()) + G) // max(int(K), 1) + 3
    offsets = np.empty(G + 1, dtype=np.int64)
    seg_bag = np.empty(cap, dtype=np.int32)
    seg_off = np.empty(cap, dtype=np.int64)
    S = ctypes.c_int64(0)
    _check(_load().oracle_plan64(lengths.ctypes.data, G, int(K), offsets.ctypes.data, seg_bag.ctypes.data,
                                 seg_off.ctypes.data, cap, ctypes.byref(S)))
    return offsets, seg_bag[: S.value + 1].copy(), int(S.value), seg_off[: S.value + 1].copy()


def decode_f16(bits: int) -> float:
    return float(_load().oracle_decode_f16(int(bits)))


def decode_bf16(bits: int) -> float:
    return float(_load().oracle_decode_bf16(int(bits)))


# ---- non-GEMM consumers of X_embed and Algorithm 2 (nongemm_oracle.c) -----------------------
ACT_IDENTITY, ACT_RELU, ACT_SIGMOID = 0, 1, 2
MODULE_EXPLICIT, MODULE_IMPLICIT = 0, 1


def _f64_2d(a) -> np.ndarray:
    a = np.ascontiguousarray(a, dtype=np.float64)
    if a.ndim != 2:
        raise ValueError("expected a [B, F] matrix")
    return a


def fm_pairwise(x: np.ndarray, T: int, D: int):
    """FM second-order term by its definition (DESIGN.md 11.4 N1). x float64[B, >= T*D] ->
    (y float64[B], v float64[B, D]) with v[b,c] = sum_{t<u} x[b,t,c] x[b,u,c] and y = v.sum(1)."""
    x = _f64_2d(x)
    B, ld = x.shape
    y = np.empty(B, dtype=np.float64)
    v = np.empty((B, D), dtype=np.float64)
    _check(_load().oracle_fm_pairwise(B, T, D, x.ctypes.data, ld, y.ctypes.data, v.ctypes.data))
    return y, v


def cross_combine(x0, xl, u, bias=None) -> np.ndarray:
    """DCNv2 cross layer, non-GEMM part (DESIGN.md 11.4 N2): x0 * (u + bias) + xl, float64[B, F]."""
    x0, xl, u = _f64_2d(x0), _f64_2d(xl), _f64_2d(u)
    if not (x0.shape == xl.shape == u.shape):
        raise ValueError("shape mismatch")
    B, F = x0.shape
    bias = None if bias is None else np.ascontiguousarray(bias, dtype=np.float64)
    if bias is not None and bias.shape != (F,):
        raise ValueError("bias must be [F]")
    out = np.empty((B, F), dtype=np.float64)
    _check(_load().oracle_cross_combine(B, F, x0.ctypes.data, xl.ctypes.data, u.ctypes.data,
                                        None if bias is None else bias.ctypes.data, out.ctypes.data))
    return out


def bias_act(u, bias=None, act: int = ACT_RELU) -> np.ndarray:
    """MLP layer, non-GEMM part (DESIGN.md 11.4 N3): act(u + bias), float64[B, F]."""
    u = _f64_2d(u)
    B, F = u.shape
    bias = None if bias is None else np.ascontiguousarray(bias, dtype=np.float64)
    if bias is not None and bias.shape != (F,):
        raise ValueError("bias must be [F]")
    out = np.empty((B, F), dtype=np.float64)
    _check(_load().oracle_bias_act(B, F, u.ctypes.data, None if bias is None else bias.ctypes.data, int(act),
                                   out.ctypes.data))
    return out


def lr_first_order(weights: Sequence[np.ndarray], B: int, indices: np.ndarray, offsets=None, bias: float = 0.0) -> np.ndarray:
    """DeepFM first-order (logistic-regression) term (DESIGN.md 11.4 N7): weights[t] is float64[rows_t]; sample-major CSR
    bags as in lookup(); offsets=None means one-hot. Returns float64[B]."""
    keep = [np.ascontiguousarray(w, dtype=np.float64).reshape(-1) for w in weights]
    T = len(keep)
    ptrs = (ctypes.c_void_p * T)(*[a.ctypes.data for a in keep])
    rows = np.asarray([a.shape[0] for a in keep], dtype=np.int64)
    indices = np.ascontiguousarray(indices, dtype=np.int32)
    off = None if offsets is None else np.ascontiguousarray(offsets, dtype=np.int32)
    y = np.empty(B, dtype=np.float64)
    _check(_load().oracle_lr_first_order(B, T, ctypes.cast(ptrs, ctypes.c_void_p), rows.ctypes.data, indices.ctypes.data,
                                         None if off is None else off.ctypes.data, float(bias), y.ctypes.data))
    del keep
    return y


def bfs_queue(n_explicit: int, n_implicit: int):
    """Algorithm 2: launch queue as a list of (module, op index), module 0 = explicit,
    1 = implicit."""
    n = int(n_explicit) + int(n_implicit)
    qm = np.empty(max(n, 1), dtype=np.int32)
    qo = np.empty(max(n, 1), dtype=np.int32)
    _check(_load().oracle_bfs_queue(int(n_explicit), int(n_implicit), qm.ctypes.data, qo.ctypes.data))
    return [(int(qm[i]), int(qo[i])) for i in range(n)]
