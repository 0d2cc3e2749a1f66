"""Thin ctypes binding over ``libdpi.so`` (include/dpi.h). Argument marshalling only: every step of the
path runs in the CUDA library. PyTorch appears here only as the owner of device memory and streams.

There is no CPU fallback: if the library is missing, import-time use raises ``DpiLibraryMissing``; if no
CUDA device is present the library itself returns ``DPI_ERR_CUDA``.
"""
from __future__ import annotations

import ctypes
import os
from typing import Optional, Sequence

import numpy as np

from . import build as _build

DPI_OK = 0
STATUS_NAMES = {0: "DPI_OK", 1: "DPI_ERR_INVALID_ARG", 2: "DPI_ERR_UNSUPPORTED", 3: "DPI_ERR_ALLOC",
                4: "DPI_ERR_CUDA", 5: "DPI_ERR_INDEX_RANGE"}
DPI_F32, DPI_F16, DPI_BF16 = 0, 1, 2
DPI_POOL_SUM, DPI_POOL_MEAN = 0, 1
OPT_UNROLL, OPT_BLOCK_THREADS, OPT_BLOCKS_PER_SM, OPT_MODE, OPT_ROW_L1_NO_ALLOC, OPT_PDL, OPT_HOST_CHUNKS, OPT_HOST_DIRECT_OUT, OPT_MAX_BAG_HINT, OPT_FUSED, OPT_FUSED_MAX_BAGS, OPT_VEC_BYTES = range(12)
BAGS_SAMPLE_MAJOR, BAGS_TABLE_MAJOR = 0, 1
IDX_I32, IDX_I64 = 0, 1
OFF_I32, OFF_I64 = 0, 1
LOOKUP_FORCE_GENERAL = 1

# every symbol include/dpi.h declares (tests check the .so exports each one)
EXPORTS = ["dpi_plan_create", "dpi_plan_set_out_dtype", "dpi_plan_set_layout", "dpi_plan_set_columns", "dpi_plan_out_width", "dpi_lookup_ex",
           "dpi_plan_set_quantum", "dpi_plan_set_option", "dpi_plan_get_option",
           "dpi_plan_build", "dpi_plan", "dpi_plan_device_views", "dpi_plan_info", "dpi_plan_export", "dpi_plan_stats",
           "dpi_lookup", "dpi_forward", "dpi_plan_status", "dpi_lookup_onehot", "dpi_lookup_input_first", "dpi_forward_host", "dpi_check_indices", "dpi_plan_destroy", "dpi_launch_count",
           "dpi_version", "dpi_status_string", "dpi_last_error", "dpi_peer_alloc", "dpi_peer_open", "dpi_peer_close", "dpi_peer_free",
           "dpi_plan_set_offset_type", "dpi_plan_export64", "dpi_forward_noalloc"]


class LookupArgs(ctypes.Structure):
    """dpi_lookup_args_t of include/dpi.h."""
    _fields_ = [("struct_size", ctypes.c_uint32), ("flags", ctypes.c_uint32), ("table_ptrs_dev", ctypes.c_void_p),
                ("indices_dev", ctypes.c_void_p), ("offsets_dev", ctypes.c_void_p), ("weights_dev", ctypes.c_void_p),
                ("pooling", ctypes.c_void_p), ("out_dev", ctypes.c_void_p), ("out_ld", ctypes.c_int64),
                ("out_peers_dev", ctypes.c_void_p), ("n_peers", ctypes.c_int32), ("rows_per_peer", ctypes.c_int32)]


class DpiLibraryMissing(RuntimeError):
    pass


class DpiError(RuntimeError):
    def __init__(self, status: int, detail: str):
        super().__init__(f"{STATUS_NAMES.get(status, status)}: {detail}")
        self.status = status
        self.detail = detail


_lib = None


def load_library(path: Optional[str] = None) -> ctypes.CDLL:
    """dlopen libdpi.so (built in-tree by ``python -m paper_2606_21101_b200.build``)."""
    global _lib
    if _lib is not None and path is None:
        return _lib
    path = path or _build.lib_path("libdpi.so")
    if not os.path.exists(path):
        raise DpiLibraryMissing(f"{path} not found: run `python -m paper_2606_21101_b200.build` "
                                "(the CUDA library is the only implementation; there is no fallback)")
    lib = ctypes.CDLL(path)
    vp, i32, i64, st = ctypes.c_void_p, ctypes.c_int32, ctypes.c_int64, ctypes.c_int
    sig = {
        "dpi_plan_create": (st, [i32, vp, vp, ctypes.c_int, i32, i64, vp]),
        "dpi_plan_set_out_dtype": (st, [vp, ctypes.c_int]),
        "dpi_plan_set_layout": (st, [vp, ctypes.c_int, ctypes.c_int]),
        "dpi_plan_out_width": (st, [vp, vp]),
        "dpi_plan_set_columns": (st, [vp, vp]),
        "dpi_lookup_ex": (st, [vp, vp, vp]),
        "dpi_plan_set_quantum": (st, [vp, i32]),
        "dpi_plan_set_option": (st, [vp, ctypes.c_int, i32]),
        "dpi_plan_get_option": (st, [vp, ctypes.c_int, vp]),
        "dpi_plan_build": (st, [vp, vp, vp]),
        "dpi_plan": (st, [vp, i32, vp, ctypes.c_int, vp, i32, i64, vp, vp]),
        "dpi_plan_device_views": (st, [vp, vp, vp, vp]),
        "dpi_plan_info": (st, [vp, vp, vp, vp, vp, vp, vp, vp]),
        "dpi_plan_export": (st, [vp, vp, vp, vp, i64, vp, vp, vp]),
        "dpi_plan_stats": (st, [vp, vp, vp, vp]),
        "dpi_plan_set_offset_type": (st, [vp, ctypes.c_int, i64]),
        "dpi_plan_export64": (st, [vp, vp, vp, vp, i64, vp, vp, vp]),
        "dpi_lookup": (st, [vp, vp, vp, vp, vp, vp, vp]),
        "dpi_lookup_input_first": (st, [vp, vp, vp, vp, vp, vp, vp]),
        "dpi_forward": (st, [vp, vp, vp, vp, vp, vp, vp]),
        "dpi_plan_status": (st, [vp, vp, vp]),
        "dpi_forward_noalloc": (st, [i32, i32, ctypes.c_int, i32, vp, vp, vp, vp, vp, vp]),
        "dpi_lookup_onehot": (st, [vp, vp, vp, vp, vp]),
        "dpi_forward_host": (st, [vp, vp, vp, vp, i64, vp, vp, vp]),
        "dpi_check_indices": (st, [vp, vp, vp, vp]),
        "dpi_plan_destroy": (st, [vp]),
        "dpi_peer_alloc": (st, [i64, vp, vp]),
        "dpi_peer_open": (st, [vp, vp]),
        "dpi_peer_close": (st, [vp]),
        "dpi_peer_free": (st, [vp]),
        "dpi_launch_count": (i64, []),
        "dpi_version": (i32, []),
        "dpi_status_string": (ctypes.c_char_p, [ctypes.c_int]),
        "dpi_last_error": (ctypes.c_char_p, []),
    }
    for name, (res, args) in sig.items():
        fn = getattr(lib, name)
        fn.restype = res
        fn.argtypes = args
    _lib = lib
    return lib


def _check(status: int):
    if status != DPI_OK:
        raise DpiError(status, load_library().dpi_last_error().decode(errors="replace"))


def _ptr(x) -> int:
    """Device/host address of a torch tensor, numpy array, int or None."""
    if x is None:
        return 0
    if isinstance(x, int):
        return x
    if isinstance(x, np.ndarray):
        return x.ctypes.data
    return x.data_ptr()  # torch.Tensor


def _stream_handle(stream) -> int:
    if stream is None:
        import torch
        return torch.cuda.current_stream().cuda_stream
    if isinstance(stream, int):
        return stream
    return stream.cuda_stream


PEER_HANDLE_BYTES = 64


def peer_alloc(nbytes: int):
    """dpi_peer_alloc: (device pointer, 64-byte IPC handle) of a dedicated allocation on the current device."""
    ptr = ctypes.c_void_p()
    handle = (ctypes.c_uint8 * PEER_HANDLE_BYTES)()
    _check(load_library().dpi_peer_alloc(int(nbytes), ctypes.byref(ptr), handle))
    return int(ptr.value), bytes(handle)


def peer_open(handle: bytes) -> int:
    """dpi_peer_open: map another process's dpi_peer_alloc block; returns the device pointer in this process."""
    ptr = ctypes.c_void_p()
    buf = (ctypes.c_uint8 * PEER_HANDLE_BYTES).from_buffer_copy(handle)
    _check(load_library().dpi_peer_open(buf, ctypes.byref(ptr)))
    return int(ptr.value)


def peer_close(ptr: int):
    _check(load_library().dpi_peer_close(ctypes.c_void_p(ptr)))


def peer_free(ptr: int):
    _check(load_library().dpi_peer_free(ctypes.c_void_p(ptr)))


NOALLOC_MAX_BAGS = 524288


def forward_noalloc(T: int, D: int, dtype: int, B: int, lengths_dev, table_ptrs_dev, indices_dev, out_dev, pooling=None, stream=None):
    """dpi_forward_noalloc: the one-launch forward path on the library's built-in scratch array -- no plan object and no
    device allocation, for callers that cannot call cudaMalloc (include/dpi.h). At most NOALLOC_MAX_BAGS bags; calls that
    may overlap on one GPU race on the shared array."""
    pool = None if pooling is None else np.ascontiguousarray(pooling, dtype=np.uint8)
    _check(load_library().dpi_forward_noalloc(int(T), int(D), int(dtype), int(B), _ptr(lengths_dev), _ptr(table_ptrs_dev),
                                              _ptr(indices_dev), _ptr(pool), _ptr(out_dev), _stream_handle(stream)))


def launch_count() -> int:
    return int(load_library().dpi_launch_count())


def version() -> int:
    return int(load_library().dpi_version())


class Plan:
    """Owner of a ``dpi_plan_t*``. Method names mirror the C entry points."""

    def __init__(self, table_rows: Sequence[int], dims, dtype: int, B: int, max_indices: int):
        lib = load_library()
        self._lib = lib
        rows = np.ascontiguousarray(table_rows, dtype=np.int64)
        T = rows.shape[0]
        dims = np.ascontiguousarray(np.broadcast_to(np.asarray(dims, dtype=np.int32), (T,)))
        handle = ctypes.c_void_p()
        _check(lib.dpi_plan_create(T, rows.ctypes.data, dims.ctypes.data, int(dtype), int(B), int(max_indices),
                                   ctypes.byref(handle)))
        self._h = handle
        self.T, self.B, self.D, self.dtype = T, int(B), int(dims.max()), int(dtype)
        self.dims = dims.copy()
        self.out_width = int(dims.sum())
        self.out_dtype = int(dtype)
        self.G = self.T * self.B
        self.max_indices = int(max_indices)

    @classmethod
    def _adopt(cls, handle, rows, dims, dtype, B, max_indices) -> "Plan":
        """Wrap a handle the library already created (dpi_plan)."""
        self = cls.__new__(cls)
        self._lib = load_library()
        self._h = handle
        self.T, self.B, self.D, self.dtype = int(rows.shape[0]), int(B), int(dims.max()), int(dtype)
        self.dims = dims.copy()
        self.out_width = int(dims.sum())
        self.out_dtype = int(dtype)
        self.G = self.T * self.B
        self.max_indices = int(max_indices)
        return self

    # -- lifetime --------------------------------------------------------------------------------------
    def destroy(self):
        if getattr(self, "_h", None):
            self._lib.dpi_plan_destroy(self._h)
            self._h = None

    def __del__(self):
        try:
            self.destroy()
        except Exception:
            pass

    # -- dpi_plan_set_out_dtype ------------------------------------------------------------------------------
    def set_out_dtype(self, out_dtype: int):
        _check(self._lib.dpi_plan_set_out_dtype(self._h, int(out_dtype)))
        self.out_dtype = int(out_dtype)

    # -- dpi_plan_set_layout / dpi_plan_out_width -----------------------------------------------------------
    def set_layout(self, bag_order: int = BAGS_SAMPLE_MAJOR, index_type: int = IDX_I32):
        _check(self._lib.dpi_plan_set_layout(self._h, int(bag_order), int(index_type)))

    def set_columns(self, columns=None):
        cols = None if columns is None else np.ascontiguousarray(columns, dtype=np.int64)
        _check(self._lib.dpi_plan_set_columns(self._h, _ptr(cols)))
        self.out_width = self.plan_out_width()

    def plan_out_width(self) -> int:
        w = ctypes.c_int64()
        _check(self._lib.dpi_plan_out_width(self._h, ctypes.byref(w)))
        return int(w.value)

    # -- dpi_plan_set_quantum / options ---------------------------------------------------------------------
    def set_quantum(self, K: int):
        _check(self._lib.dpi_plan_set_quantum(self._h, int(K)))

    def set_option(self, opt: int, value: int):
        _check(self._lib.dpi_plan_set_option(self._h, int(opt), int(value)))

    def get_option(self, opt: int) -> int:
        v = ctypes.c_int32()
        _check(self._lib.dpi_plan_get_option(self._h, int(opt), ctypes.byref(v)))
        return v.value

    def info(self) -> dict:
        T, B, D, dt, K = (ctypes.c_int32() for _ in range(5))
        G, cap = ctypes.c_int64(), ctypes.c_int64()
        _check(self._lib.dpi_plan_info(self._h, ctypes.byref(T), ctypes.byref(B), ctypes.byref(D), ctypes.byref(dt),
                                       ctypes.byref(G), ctypes.byref(K), ctypes.byref(cap)))
        return {"T": T.value, "B": B.value, "D": D.value, "dtype": dt.value, "G": G.value, "K": K.value,
                "seg_capacity": cap.value}

    # -- dpi_plan_build -------------------------------------------------------------------------------------
    def build(self, lengths_dev, stream=None):
        _check(self._lib.dpi_plan_build(self._h, _ptr(lengths_dev), _stream_handle(stream)))

    # -- dpi_plan_device_views ------------------------------------------------------------------------------
    def device_views(self):
        o, s, m = ctypes.c_void_p(), ctypes.c_void_p(), ctypes.c_void_p()
        _check(self._lib.dpi_plan_device_views(self._h, ctypes.byref(o), ctypes.byref(s), ctypes.byref(m)))
        return o.value, s.value, m.value

    # -- dpi_plan_export ------------------------------------------------------------------------------------
    def export(self, stream=None, with_seg_off: bool = False):
        """Returns (offsets int32[G+1], seg_bag int32[S+1], S, N) as host numpy arrays (synchronises);
        with_seg_off=True appends seg_off int32[S+1]."""
        cap = self.info()["seg_capacity"]
        offsets = np.empty(self.G + 1, dtype=np.int32)
        seg = np.empty(cap, dtype=np.int32)
        seg_off = np.empty(cap, dtype=np.int32)
        S, N = ctypes.c_int32(), ctypes.c_int64()
        _check(self._lib.dpi_plan_export(self._h, offsets.ctypes.data, seg.ctypes.data, seg_off.ctypes.data, cap,
                                         ctypes.byref(S), ctypes.byref(N), _stream_handle(stream)))
        res = (offsets, seg[: S.value + 1].copy(), int(S.value), int(N.value))
        return res + (seg_off[: S.value + 1].copy(),) if with_seg_off else res

    # -- dpi_plan_set_offset_type / dpi_plan_export64 (NEXT-2: 64-bit offsets) ------------------------------
    def set_offset_type(self, offset_type: int, max_indices: int = 0):
        _check(self._lib.dpi_plan_set_offset_type(self._h, int(offset_type), int(max_indices)))

    def export64(self, stream=None):
        """Plan with 64-bit offsets -> (offsets int64[G+1], seg_bag int32[S+1], S, N, seg_off int64[S+1]) (synchronises)."""
        cap = self.info()["seg_capacity"]
        offsets = np.empty(self.G + 1, dtype=np.int64)
        seg = np.empty(cap, dtype=np.int32)
        seg_off = np.empty(cap, dtype=np.int64)
        S, N = ctypes.c_int64(), ctypes.c_int64()
        _check(self._lib.dpi_plan_export64(self._h, offsets.ctypes.data, seg.ctypes.data, seg_off.ctypes.data, cap,
                                           ctypes.byref(S), ctypes.byref(N), _stream_handle(stream)))
        return offsets, seg[: S.value + 1].copy(), int(S.value), int(N.value), seg_off[: S.value + 1].copy()

    # -- dpi_plan_stats -------------------------------------------------------------------------------------
    def stats(self, stream=None):
        """(min_len, max_len) of the last built batch (synchronises)."""
        lo, hi = ctypes.c_int32(), ctypes.c_int32()
        _check(self._lib.dpi_plan_stats(self._h, ctypes.byref(lo), ctypes.byref(hi), _stream_handle(stream)))
        return int(lo.value), int(hi.value)

    # -- dpi_lookup -----------------------------------------------------------------------------------------
    def lookup(self, table_ptrs_dev, indices_dev, out_dev, pooling=None, offsets_dev=None, stream=None):
        pool = None if pooling is None else np.ascontiguousarray(pooling, dtype=np.uint8)
        _check(self._lib.dpi_lookup(_ptr(table_ptrs_dev), _ptr(indices_dev), _ptr(offsets_dev), self._h,
                                    _ptr(pool), _ptr(out_dev), _stream_handle(stream)))

    # -- dpi_forward (a1 + a2 + a3 in one call; one fused launch on small / short-bag batches) ------------------
    def forward(self, lengths_dev, table_ptrs_dev, indices_dev, out_dev, pooling=None, stream=None):
        pool = None if pooling is None else np.ascontiguousarray(pooling, dtype=np.uint8)
        _check(self._lib.dpi_forward(self._h, _ptr(lengths_dev), _ptr(table_ptrs_dev), _ptr(indices_dev), _ptr(pool),
                                     _ptr(out_dev), _stream_handle(stream)))

    # -- dpi_plan_status ------------------------------------------------------------------------------------
    def status(self, stream=None) -> int:
        """Number of builds since the last call that overflowed the plan's capacity (synchronises; clears the count)."""
        n = ctypes.c_int32(0)
        st = self._lib.dpi_plan_status(self._h, ctypes.byref(n), _stream_handle(stream))
        if st not in (DPI_OK, 1):
            _check(st)
        return int(n.value)

    # -- dpi_lookup_ex ----------------------------------------------------------------------------------------
    def lookup_ex(self, table_ptrs_dev, indices_dev, out_dev, pooling=None, offsets_dev=None, weights_dev=None,
                  out_ld: int = 0, flags: int = 0, out_peers_dev=None, n_peers: int = 0, rows_per_peer: int = 0, stream=None):
        pool = None if pooling is None else np.ascontiguousarray(pooling, dtype=np.uint8)
        a = LookupArgs(ctypes.sizeof(LookupArgs), int(flags), _ptr(table_ptrs_dev), _ptr(indices_dev), _ptr(offsets_dev),
                       _ptr(weights_dev), _ptr(pool), _ptr(out_dev), int(out_ld), _ptr(out_peers_dev), int(n_peers),
                       int(rows_per_peer))
        _check(self._lib.dpi_lookup_ex(ctypes.byref(a), self._h, _stream_handle(stream)))

    # -- dpi_lookup_input_first (ablation) ---------------------------------------------------
    def lookup_input_first(self, table_ptrs_dev, indices_dev, out_dev, pooling=None, offsets_dev=None, stream=None):
        pool = None if pooling is None else np.ascontiguousarray(pooling, dtype=np.uint8)
        _check(self._lib.dpi_lookup_input_first(_ptr(table_ptrs_dev), _ptr(indices_dev), _ptr(offsets_dev), self._h,
                                                _ptr(pool), _ptr(out_dev), _stream_handle(stream)))

    # -- dpi_lookup_onehot (Algorithm 1, no built plan needed) ------------------------------------------------
    def lookup_onehot(self, table_ptrs_dev, ids_dev, out_dev, stream=None):
        _check(self._lib.dpi_lookup_onehot(_ptr(table_ptrs_dev), _ptr(ids_dev), self._h, _ptr(out_dev),
                                           _stream_handle(stream)))

    # -- dpi_forward_host -----------------------------------------------------------------------------------
    def forward_host(self, table_ptrs_dev, lengths_host, indices_host, out_host, pooling=None, stream=None):
        pool = None if pooling is None else np.ascontiguousarray(pooling, dtype=np.uint8)
        n = int(indices_host.numel() if hasattr(indices_host, "numel") else indices_host.shape[0])
        _check(self._lib.dpi_forward_host(self._h, _ptr(table_ptrs_dev), _ptr(lengths_host), _ptr(indices_host), n,
                                          _ptr(pool), _ptr(out_host), _stream_handle(stream)))

    # -- dpi_check_indices ----------------------------------------------------------------------------------
    def check_indices(self, indices_dev, stream=None) -> int:
        n_bad = ctypes.c_int64()
        st = self._lib.dpi_check_indices(self._h, _ptr(indices_dev), ctypes.byref(n_bad), _stream_handle(stream))
        if st not in (DPI_OK, 5):
            _check(st)
        return int(n_bad.value)


def dpi_plan(table_rows, dims, dtype: int, lengths_dev, B: int, max_indices: int, stream=None) -> Plan:
    """north_star spelling, the C entry point `dpi_plan` (create + build in one call)."""
    lib = load_library()
    rows = np.ascontiguousarray(table_rows, dtype=np.int64)
    T = rows.shape[0]
    dims_a = np.ascontiguousarray(np.broadcast_to(np.asarray(dims, dtype=np.int32), (T,)))
    handle = ctypes.c_void_p()
    _check(lib.dpi_plan(rows.ctypes.data, T, dims_a.ctypes.data, int(dtype), _ptr(lengths_dev), int(B), int(max_indices),
                        _stream_handle(stream), ctypes.byref(handle)))
    return Plan._adopt(handle, rows, dims_a, dtype, B, max_indices)


def dpi_lookup(table_ptrs_dev, indices_dev, offsets_dev, plan: Plan, pooling, out_dev, stream=None):
    plan.lookup(table_ptrs_dev, indices_dev, out_dev, pooling=pooling, offsets_dev=offsets_dev, stream=stream)


# ----------------------------------------------------------------------------------------------------
# bench/test helper library (synthetic table fill on the device) -- not part of the method
# ----------------------------------------------------------------------------------------------------
_synth = None


def _synth_lib():
    global _synth
    if _synth is None:
        path = _build.lib_path("libdpi_synth.so")
        if not os.path.exists(path):
            raise DpiLibraryMissing(f"{path} not found: run `python -m paper_2606_21101_b200.build`")
        _synth = ctypes.CDLL(path)
        _synth.dpi_synth_fill_table.restype = ctypes.c_int
        _synth.dpi_synth_fill_table.argtypes = [ctypes.c_void_p, ctypes.c_uint64, ctypes.c_int, ctypes.c_uint64,
                                                ctypes.c_void_p]
        _synth.dpi_synth_row_read_probe.restype = ctypes.c_int
        _synth.dpi_synth_row_read_probe.argtypes = [ctypes.c_void_p, ctypes.c_uint64, ctypes.c_uint32, ctypes.c_uint64,
                                                    ctypes.c_uint64, ctypes.c_int, ctypes.c_int, ctypes.c_int,
                                                    ctypes.c_void_p, ctypes.c_void_p]
        _synth.dpi_synth_copy_words.restype = ctypes.c_int
        _synth.dpi_synth_copy_words.argtypes = [ctypes.c_void_p, ctypes.c_void_p, ctypes.c_uint64]
    return _synth


def copy_device_words(dst_dev, src_ptr: int, n_words: int):
    """Test helper: device-to-device copy of n_words 32-bit words from a raw device address (e.g. a borrowed pointer of
    dpi_plan_device_views) into a tensor; synchronous."""
    rc = _synth_lib().dpi_synth_copy_words(_ptr(dst_dev), int(src_ptr), int(n_words))
    if rc != 0:
        raise RuntimeError(f"dpi_synth_copy_words failed with cudaError {rc}")


def synth_row_read_probe(base_dev, span_rows: int, row_bytes: int, n_rows: int, key: int, random: bool, unroll: int,
                         ctas_per_sm: int, sink_dev, stream=None):
    """Bench context only: read n_rows whole rows at hashed (or consecutive) positions of a span_rows-row buffer."""
    rc = _synth_lib().dpi_synth_row_read_probe(_ptr(base_dev), int(span_rows), int(row_bytes), int(n_rows), int(key),
                                               int(bool(random)), int(unroll), int(ctas_per_sm), _ptr(sink_dev),
                                               _stream_handle(stream))
    if rc != 0:
        raise RuntimeError(f"dpi_synth_row_read_probe failed with cudaError {rc}")


def synth_fill_table(dst_dev, n_elems: int, dtype: int, key: int, stream=None):
    _synth = _synth_lib()
    rc = _synth.dpi_synth_fill_table(_ptr(dst_dev), int(n_elems), int(dtype), int(key), _stream_handle(stream))
    if rc != 0:
        raise RuntimeError(f"dpi_synth_fill_table failed with cudaError {rc}")
