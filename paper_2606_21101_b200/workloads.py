"""Seeded synthetic CTR-shaped inputs for the fused multi-table embedding lookup.

This module serves BOTH the CPU oracle's tests and the CUDA path's tests/bench. It holds none of the
method's arithmetic (no offsets, no plan, no pooling): it only draws table heights, bag lengths, indices
and table values. numpy only; imports neither ``oracle`` nor the CUDA binding.

The paper measures on Criteo (39 fields) / Avazu (24 fields) through FuxiCTR models (PAPER.md:261-265,
§V-A); neither dataset is available, so the five configs of BASELINE.json are synthetic stand-ins that
take the *shapes* of those workloads (tens of fields, per-field cardinality spread over orders of
magnitude PAPER.md:137, D in {16,32,64}, batch 128..65536 PAPER.md:366-376, skewed ID popularity).
No dataset record appears anywhere.

Recipe (also stated in DESIGN.md §5)
------------------------------------
Counter-based generator: ``h(key, i) = fmix64(key + i*GAMMA)`` (SplitMix64 finaliser over a Weyl
sequence); ``key(seed, stream, sub) = fmix64(fmix64(seed + GAMMA*(stream+1)) ^ (sub*SUBMUL))``.
``U(h) = (h >> 11) * 2**-53`` in float64.

* table heights  : given list, or log-uniform ``floor(exp(ln lo + U*(ln hi - ln lo)))`` per table.
* bag lengths    : constant; uniform a..b ``a + floor(U*(b-a+1))``; Poisson(mean) by inverse CDF capped,
                   then set to 0 where ``U_EMPTY < p_empty``. Bag order is sample-major, g = b*T + t
                   (Alg. 1 line 7 ``IDs[row*k + table_id]``).
* indices        : per flat entry e (bag-contiguous), sub-stream = table id. uniform ``floor(U*rows_t)``;
                   bounded Zipf(alpha) on ranks 1..rows_t by inverse CDF (float64 cumulative table +
                   searchsorted), rank->row through the affine bijection ``row = (rank*a_t) mod rows_t``
                   with ``a_t`` the smallest integer >= 0.618*rows_t coprime to rows_t (hot rows scattered).
* table values   : ``v(t,r,c) = ((h(key(seed,VAL,t), r*D+c) >> 40) * 2**-24 - 0.5) * 0.1`` evaluated in
                   float32 -> uniform in [-0.05, 0.05), then RNE-cast to the table dtype. Any row can be
                   recomputed on the host, which is what lets tests check an 82 GB device table without a
                   host mirror. ``csrc/synth_fill.cu`` implements the same generator on the device.
"""
from __future__ import annotations

import math
from dataclasses import dataclass, field, replace
from typing import List, Optional, Sequence, Tuple, Union

import numpy as np

GAMMA = 0x9E3779B97F4A7C15
SUBMUL = 0xD1B54A32D192ED03
_M64 = (1 << 64) - 1

STREAM_ROWS, STREAM_LEN, STREAM_EMPTY, STREAM_IDX, STREAM_VAL, STREAM_WGT = 1, 2, 3, 4, 5, 6

DTYPES = ("f32", "f16", "bf16")
DTYPE_BYTES = {"f32": 4, "f16": 2, "bf16": 2}
DTYPE_CODE = {"f32": 0, "f16": 1, "bf16": 2}  # == dpi_dtype_t in include/dpi.h
POOL_SUM, POOL_MEAN = 0, 1


# ----------------------------------------------------------------------------------------------------
# counter-based generator
# ----------------------------------------------------------------------------------------------------
def _fmix64_int(z: int) -> int:
    z &= _M64
    z = ((z ^ (z >> 30)) * 0xBF58476D1CE4E5B9) & _M64
    z = ((z ^ (z >> 27)) * 0x94D049BB133111EB) & _M64
    return z ^ (z >> 31)


def stream_key(seed: int, stream: int, sub: int = 0) -> int:
    """64-bit key of one random stream (python ints; passed verbatim to the device fill kernel)."""
    k = _fmix64_int((seed + GAMMA * (stream + 1)) & _M64)
    return _fmix64_int(k ^ ((sub * SUBMUL) & _M64))


def hash_u64(key: Union[int, np.ndarray], i: np.ndarray) -> np.ndarray:
    """h(key, i) for an array of counters (uint64 wrap-around arithmetic)."""
    with np.errstate(over="ignore"):
        z = np.asarray(i, dtype=np.uint64) * np.uint64(GAMMA)
        z = z + (np.asarray(key, dtype=np.uint64) if isinstance(key, np.ndarray) else np.uint64(key))
        z = (z ^ (z >> np.uint64(30))) * np.uint64(0xBF58476D1CE4E5B9)
        z = (z ^ (z >> np.uint64(27))) * np.uint64(0x94D049BB133111EB)
        z = z ^ (z >> np.uint64(31))
    return z


def unit_f64(h: np.ndarray) -> np.ndarray:
    """U in [0,1) with 53 random bits."""
    return (h >> np.uint64(11)).astype(np.float64) * (2.0 ** -53)


# ----------------------------------------------------------------------------------------------------
# 16-bit storage formats (inputs only; the oracle has its own decoders)
# ----------------------------------------------------------------------------------------------------
def f32_to_bf16_bits(x: np.ndarray) -> np.ndarray:
    """Round-to-nearest-even float32 -> bfloat16 bit pattern (uint16). Inputs are finite."""
    u = np.ascontiguousarray(x, dtype=np.float32).view(np.uint32)
    rounded = u + (np.uint32(0x7FFF) + ((u >> np.uint32(16)) & np.uint32(1)))
    return (rounded >> np.uint32(16)).astype(np.uint16)


def bf16_bits_to_f32(b: np.ndarray) -> np.ndarray:
    return (np.ascontiguousarray(b, dtype=np.uint16).astype(np.uint32) << np.uint32(16)).view(np.float32)


def to_storage(x32: np.ndarray, dtype: str) -> np.ndarray:
    """float32 values -> storage array (float32 / float16 / uint16 holding bf16 bits)."""
    if dtype == "f32":
        return np.ascontiguousarray(x32, dtype=np.float32)
    if dtype == "f16":
        return np.ascontiguousarray(x32, dtype=np.float32).astype(np.float16)
    if dtype == "bf16":
        return f32_to_bf16_bits(x32)
    raise ValueError(dtype)


def storage_to_f64(a: np.ndarray, dtype: str) -> np.ndarray:
    """storage array -> float64 (exact)."""
    if dtype == "bf16":
        return bf16_bits_to_f32(a).astype(np.float64)
    return np.asarray(a).astype(np.float64)


def storage_numpy_dtype(dtype: str):
    return {"f32": np.float32, "f16": np.float16, "bf16": np.uint16}[dtype]


# ----------------------------------------------------------------------------------------------------
# configs
# ----------------------------------------------------------------------------------------------------
@dataclass(frozen=True)
class Config:
    """One synthetic workload shape. ``rows`` is a list of table heights or ("loguniform", lo, hi)."""
    name: str
    T: int
    rows: Union[Tuple[int, ...], Tuple[str, float, float]]
    D: int
    dtype: str
    B: int
    lengths: Tuple  # ("const", L) | ("uniform", a, b) | ("poisson", mean, cap, p_empty)
    index_dist: Tuple  # ("uniform",) | ("zipf", alpha)
    pooling: str  # "sum" | "mean" | "half"  (half: t < T//2 sum, else mean -- DESIGN.md reading R11)
    seed: int = 0
    out_dtype: Optional[str] = None  # None = table dtype; "f32" = fp32 output block from 16-bit tables

    @property
    def out(self) -> str:
        return self.out_dtype or self.dtype

    @property
    def out_row_bytes(self) -> int:
        return self.D * DTYPE_BYTES[self.out]

    @property
    def G(self) -> int:
        return self.B * self.T

    @property
    def row_bytes(self) -> int:
        return self.D * DTYPE_BYTES[self.dtype]

    def pooling_modes(self) -> np.ndarray:
        if self.pooling == "sum":
            return np.zeros(self.T, dtype=np.uint8)
        if self.pooling == "mean":
            return np.ones(self.T, dtype=np.uint8)
        if self.pooling == "half":
            p = np.zeros(self.T, dtype=np.uint8)
            p[self.T // 2:] = POOL_MEAN
            return p
        raise ValueError(self.pooling)

    def table_rows(self) -> np.ndarray:
        """int64[T] table heights (seeded draw for log-uniform specs)."""
        if isinstance(self.rows[0], str):
            kind, lo, hi = self.rows
            assert kind == "loguniform"
            u = unit_f64(hash_u64(stream_key(self.seed, STREAM_ROWS), np.arange(self.T)))
            r = np.floor(np.exp(math.log(lo) + u * (math.log(hi) - math.log(lo)))).astype(np.int64)
            return np.clip(r, int(lo), int(hi))
        r = np.asarray(self.rows, dtype=np.int64)
        assert r.shape == (self.T,)
        return r

    def scaled(self, **kw) -> "Config":
        return replace(self, **kw)


# BASELINE.json configs[0..4]
C1 = Config("c1", 4, (1000, 500, 2000, 100), 16, "f32", 128, ("uniform", 1, 4), ("uniform",), "sum", 0)
C2 = Config("c2", 26, ("loguniform", 10, 1e6), 16, "f32", 4096, ("const", 1), ("zipf", 1.05), "sum", 0)
C3 = Config("c3", 22, ("loguniform", 100, 5e6), 32, "f16", 16384, ("uniform", 1, 3), ("zipf", 1.2), "mean", 0)
# c4: BASELINE.json names no output type; fp32 output keeps the stated 2e-3 relative tolerance reachable
# (a correctly rounded bf16 output alone carries up to 2^-8 = 3.9e-3; reading R6).
C4 = Config("c4", 100, ("loguniform", 1e5, 5e6), 64, "bf16", 8192, ("poisson", 20.0, 100, 0.05),
            ("zipf", 1.05), "half", 0, out_dtype="f32")
C5 = Config("c5", 8, (40_000_000,) * 8, 64, "f32", 65536, ("uniform", 1, 64), ("uniform",), "sum", 0)
CONFIGS = {c.name: c for c in (C1, C2, C3, C4, C5)}


# ----------------------------------------------------------------------------------------------------
# bag lengths and indices
# ----------------------------------------------------------------------------------------------------
def _poisson_cdf(mean: float, cap: int) -> np.ndarray:
    p = math.exp(-mean)
    cdf = np.empty(cap + 1, dtype=np.float64)
    acc = 0.0
    for k in range(cap + 1):
        acc += p
        cdf[k] = acc
        p = p * mean / (k + 1)
    return cdf


def make_lengths(cfg: Config, batch_seed: int, bag_base: int = 0) -> np.ndarray:
    """int32[G] bag lengths, sample-major (g = b*T + t). ``bag_base`` offsets the bag counter: the lengths of
    bags [bag_base, bag_base + G) of a larger (global) batch of the same seed -- used to draw one rank's
    shard of a batch-sharded global batch without drawing the rest (bag_base must be a multiple of T)."""
    G = cfg.G
    assert bag_base % cfg.T == 0
    g = np.arange(bag_base, bag_base + G, dtype=np.uint64)
    kind = cfg.lengths[0]
    if kind == "const":
        return np.full(G, int(cfg.lengths[1]), dtype=np.int32)
    u = unit_f64(hash_u64(stream_key(batch_seed, STREAM_LEN), g))
    if kind == "uniform":
        a, b = int(cfg.lengths[1]), int(cfg.lengths[2])
        return (a + np.floor(u * (b - a + 1))).astype(np.int32).clip(a, b)
    if kind == "poisson":
        mean, cap, p_empty = float(cfg.lengths[1]), int(cfg.lengths[2]), float(cfg.lengths[3])
        cdf = _poisson_cdf(mean, cap)
        ln = np.minimum(np.searchsorted(cdf, u, side="right"), cap).astype(np.int32)
        ue = unit_f64(hash_u64(stream_key(batch_seed, STREAM_EMPTY), g))
        ln[ue < p_empty] = 0
        return ln
    raise ValueError(kind)


def _coprime_multiplier(n: int) -> int:
    a = max(1, int(math.ceil(0.618 * n)))
    while math.gcd(a, n) != 1:
        a += 1
    return a


class _ZipfTable:
    """Inverse-CDF sampler of the bounded Zipf(alpha) law on ranks 1..n (float64 cumulative table)."""

    def __init__(self, n: int, alpha: float):
        self.n = n
        w = np.arange(1, n + 1, dtype=np.float64) ** (-alpha)
        self.cdf = np.cumsum(w)
        self.a = _coprime_multiplier(n)

    def rows(self, u: np.ndarray) -> np.ndarray:
        rank0 = np.searchsorted(self.cdf, u * self.cdf[-1], side="right")
        rank0 = np.minimum(rank0, self.n - 1).astype(np.int64)
        return (rank0 * self.a) % self.n


def make_indices(cfg: Config, rows: np.ndarray, lengths: np.ndarray, batch_seed: int,
                 entry_base: int = 0) -> np.ndarray:
    """int32[N] per-table local row ids, bag-contiguous in sample-major bag order. ``entry_base`` offsets the
    per-entry counter (the flat position of this shard's first entry inside the global batch)."""
    T = cfg.T
    lengths = np.asarray(lengths, dtype=np.int64)
    N = int(lengths.sum())
    if N == 0:
        return np.zeros(0, dtype=np.int32)
    table_of_entry = (np.repeat(np.arange(cfg.G, dtype=np.int64), lengths) % T).astype(np.int32)
    keys = np.array([stream_key(batch_seed, STREAM_IDX, t) for t in range(T)], dtype=np.uint64)
    u = unit_f64(hash_u64(keys[table_of_entry], np.arange(entry_base, entry_base + N, dtype=np.uint64)))
    out = np.empty(N, dtype=np.int32)
    if cfg.index_dist[0] == "uniform":
        r = rows[table_of_entry].astype(np.float64)
        out[:] = np.minimum(np.floor(u * r), r - 1).astype(np.int32)
        return out
    if cfg.index_dist[0] == "zipf":
        alpha = float(cfg.index_dist[1])
        order = np.argsort(table_of_entry, kind="stable")
        counts = np.bincount(table_of_entry, minlength=T)
        pos = 0
        for t in range(T):
            sel = order[pos:pos + counts[t]]
            pos += counts[t]
            if sel.size:
                out[sel] = _ZipfTable(int(rows[t]), alpha).rows(u[sel]).astype(np.int32)
        return out
    raise ValueError(cfg.index_dist)


@dataclass
class Batch:
    """One batch of sparse inputs (host arrays)."""
    lengths: np.ndarray  # int32[G]
    indices: np.ndarray  # int32[N]

    @property
    def N(self) -> int:
        return int(self.indices.shape[0])


def make_batch(cfg: Config, rows: Optional[np.ndarray] = None, batch_seed: Optional[int] = None) -> Batch:
    rows = cfg.table_rows() if rows is None else rows
    bs = cfg.seed if batch_seed is None else batch_seed
    ln = make_lengths(cfg, bs)
    return Batch(ln, make_indices(cfg, rows, ln, bs))


# ----------------------------------------------------------------------------------------------------
# table values
# ----------------------------------------------------------------------------------------------------
def value_key(cfg_seed: int, t: int) -> int:
    return stream_key(cfg_seed, STREAM_VAL, t)


def table_values_f32(seed: int, t: int, D: int, row_ids: np.ndarray) -> np.ndarray:
    """float32[len(row_ids), D] values of the requested rows of table t (before the storage cast)."""
    row_ids = np.asarray(row_ids, dtype=np.uint64)
    ctr = row_ids[:, None] * np.uint64(D) + np.arange(D, dtype=np.uint64)[None, :]
    h = hash_u64(value_key(seed, t), ctr)
    x = (h >> np.uint64(40)).astype(np.float32) * np.float32(2.0 ** -24)
    return (x - np.float32(0.5)) * np.float32(0.1)


def table_rows_storage(cfg: Config, t: int, row_ids: np.ndarray) -> np.ndarray:
    """Requested rows of table t in storage format."""
    return to_storage(table_values_f32(cfg.seed, t, cfg.D, row_ids), cfg.dtype)


def full_table_storage(cfg: Config, t: int, n_rows: int, chunk: int = 1 << 18) -> np.ndarray:
    """Whole table t on the host (small tables only)."""
    out = np.empty((n_rows, cfg.D), dtype=storage_numpy_dtype(cfg.dtype))
    for lo in range(0, n_rows, chunk):
        hi = min(n_rows, lo + chunk)
        out[lo:hi] = table_rows_storage(cfg, t, np.arange(lo, hi))
    return out


STREAM_DENSE = 97  # dense activations for the NEXT-4 operators (X_embed-shaped blocks, GEMM outputs, biases)


def dense_values_f32(seed: int, sub: int, shape, scale: float = 0.25) -> np.ndarray:
    """float32 array of `shape`, uniform in [-scale, scale): element i (row-major) comes from counter i of stream
    (seed, STREAM_DENSE, sub). Stand-in for pooled embedding blocks / layer activations."""
    n = int(np.prod(shape))
    h = hash_u64(stream_key(seed, STREAM_DENSE, sub), np.arange(n, dtype=np.uint64))
    x = (h >> np.uint64(40)).astype(np.float32) * np.float32(2.0 ** -24)
    return ((x - np.float32(0.5)) * np.float32(2.0 * scale)).reshape(shape)


# ----------------------------------------------------------------------------------------------------
# sub-problems for sampled parity at full size
# ----------------------------------------------------------------------------------------------------
@dataclass
class CompactProblem:
    """A lookup problem restricted to some samples, with tables compacted to the rows it references.

    ``tables[t]`` holds only the referenced rows of table t (storage format) and ``indices`` are remapped
    into those compact tables, so a host oracle can evaluate outputs of a workload whose real tables do
    not fit on the host. Pure data movement: no pooling, no offsets.
    """
    cfg: Config
    sample_ids: np.ndarray  # int64[B'] rows of the full batch
    lengths: np.ndarray  # int32[B'*T]
    indices: np.ndarray  # int32[N'] remapped
    tables: List[np.ndarray]
    table_rows: np.ndarray  # int64[T] compact heights (>=1)


def compact_subproblem(cfg: Config, batch: Batch, sample_ids: Sequence[int]) -> CompactProblem:
    T = cfg.T
    sample_ids = np.asarray(sample_ids, dtype=np.int64)
    ln_full = batch.lengths.astype(np.int64)
    starts = np.concatenate(([0], np.cumsum(ln_full)))  # entry position of each bag (layout only)
    bag_ids = (sample_ids[:, None] * T + np.arange(T)[None, :]).reshape(-1)
    ln = ln_full[bag_ids]
    n = int(ln.sum())
    # flat entry positions of the selected bags, in order
    rep_start = np.repeat(starts[bag_ids], ln)
    within = np.arange(n) - np.repeat(np.cumsum(ln) - ln, ln)
    idx = batch.indices[rep_start + within].astype(np.int64)
    tab = np.repeat(np.arange(bag_ids.size) % T, ln)
    new_idx = np.empty(n, dtype=np.int32)
    tables, heights = [], []
    for t in range(T):
        sel = np.nonzero(tab == t)[0]
        uniq, inv = np.unique(idx[sel], return_inverse=True)
        if uniq.size == 0:
            uniq = np.zeros(1, dtype=np.int64)
        else:
            new_idx[sel] = inv.astype(np.int32)
        tables.append(table_rows_storage(cfg, t, uniq))
        heights.append(uniq.size)
    return CompactProblem(cfg, sample_ids, ln.astype(np.int32), new_idx, tables,
                          np.asarray(heights, dtype=np.int64))


# ----------------------------------------------------------------------------------------------------
# interface variants: data movement and draws only
# ----------------------------------------------------------------------------------------------------
def make_weights(batch_seed: int, n: int, lo: float = 0.0, hi: float = 2.0) -> np.ndarray:
    """float32[n] per-entry weights, uniform in [lo, hi) (one per flat index entry, sample-major entry order)."""
    u = unit_f64(hash_u64(stream_key(batch_seed, STREAM_WGT), np.arange(n, dtype=np.uint64)))
    return (lo + u * (hi - lo)).astype(np.float32)


def to_table_major(T: int, B: int, lengths: np.ndarray, *per_entry: np.ndarray):
    """Re-order a sample-major batch (bag g = b*T + t) into table-major order (bag g' = t*B + b): returns the
    permuted lengths and every per-entry array (indices, weights, ...) with its bags moved along. Pure permutation."""
    lengths = np.asarray(lengths, dtype=np.int64)
    perm = np.arange(B * T).reshape(B, T).T.reshape(-1)  # table-major position -> sample-major bag id
    starts = np.concatenate(([0], np.cumsum(lengths)))[:-1]
    ln_tm = lengths[perm]
    n = int(lengths.sum())
    src = np.repeat(starts[perm], ln_tm) + (np.arange(n) - np.repeat(np.cumsum(ln_tm) - ln_tm, ln_tm))
    return (ln_tm.astype(np.int32),) + tuple(np.ascontiguousarray(np.asarray(a)[src]) for a in per_entry)


def mixed_dim_tables(seed: int, dims: Sequence[int], rows: Sequence[int], dtype: str) -> List[np.ndarray]:
    """Host tables of different widths with the seeded value recipe (storage format), small tables only."""
    return [to_storage(table_values_f32(seed, t, int(dims[t]), np.arange(int(rows[t]))), dtype) for t in range(len(dims))]


def algorithmic_bytes(cfg: Config, G: int, N: int, S: int = 0) -> dict:
    """Bytes the path must move: per gathered row rowB+4, per bag 4 (offset) + D*elt (output)
    for the lookup; planner 4 read + 4 written per bag + 4 per segment."""
    lookup = N * (cfg.row_bytes + 4) + G * (4 + cfg.out_row_bytes)
    plan = G * 8 + 4 * (S + 1)
    return {"lookup": lookup, "plan": plan, "total": lookup + plan}
