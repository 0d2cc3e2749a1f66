"""ctypes binding of include/dpi_nongemm.h: the fused non-GEMM consumers of X_embed
 and the breadth-first two-stream launcher (Algorithm 2).

Argument marshalling only; same names as the C entry points; every number is produced by the CUDA kernels in
``csrc/nongemm_kernels.cu``. There is no CPU fallback (``bfs_schedule`` is host logic in the C library itself)."""
from __future__ import annotations

import ctypes
from typing import Callable, List, Optional, Sequence, Tuple

import numpy as np

from . import binding
from .binding import _check, _ptr, _stream_handle

EXPORTS = ["dpi_forward_fm", "dpi_fm_interaction", "dpi_lr_first_order", "dpi_cross_combine", "dpi_bias_act", "dpi_bfs_schedule", "dpi_launcher_create",
           "dpi_launcher_destroy", "dpi_launcher_run"]

ACT_IDENTITY, ACT_RELU, ACT_SIGMOID = 0, 1, 2
MODULE_EXPLICIT, MODULE_IMPLICIT = 0, 1

OP_FN = ctypes.CFUNCTYPE(None, ctypes.c_void_p, ctypes.c_void_p)  # dpi_op_fn(user, stream)


class Op(ctypes.Structure):
    """dpi_op_t"""
    _fields_ = [("launch", OP_FN), ("user", ctypes.c_void_p)]


_ready = False


def _lib() -> ctypes.CDLL:
    global _ready
    lib = binding.load_library()
    if not _ready:
        vp, i32, i64, st = ctypes.c_void_p, ctypes.c_int32, ctypes.c_int64, ctypes.c_int
        sig = {
            "dpi_fm_interaction": (st, [vp, ctypes.c_int, i32, i32, i32, i64, vp, vp, vp]),
            "dpi_forward_fm": (st, [vp, vp, vp, vp, vp, vp, vp, vp, vp]),
            "dpi_cross_combine": (st, [vp, vp, vp, vp, vp, ctypes.c_int, i32, i32, vp]),
            "dpi_lr_first_order": (st, [vp, vp, vp, i32, i32, ctypes.c_float, vp, i32, vp]),
            "dpi_bias_act": (st, [vp, vp, vp, ctypes.c_int, i32, i32, ctypes.c_int, vp]),
            "dpi_bfs_schedule": (st, [i32, i32, vp, vp]),
            "dpi_launcher_create": (st, [vp]),
            "dpi_launcher_destroy": (st, [vp]),
            "dpi_launcher_run": (st, [vp, vp, i32, vp, i32, i32, vp]),
        }
        for name, (res, args) in sig.items():
            fn = getattr(lib, name)
            fn.restype = res
            fn.argtypes = args
        _ready = True
    return lib


def fm_interaction(x, dtype: int, B: int, T: int, D: int, y=None, v=None, x_ld: int = 0, stream=None) -> None:
    """dpi_fm_interaction: x [B, x_ld] device tensor of `dtype`; y fp32[B] and / or v fp32[B, D] device tensors."""
    _check(_lib().dpi_fm_interaction(_ptr(x), int(dtype), int(B), int(T), int(D), int(x_ld), _ptr(y), _ptr(v),
                                     _stream_handle(stream)))


def forward_fm(plan, lengths_dev, table_ptrs_dev, indices_dev, out_dev, y=None, v=None, pooling=None, stream=None) -> None:
    """dpi_forward_fm: dpi_forward (plan + fused lookup into out_dev) plus the FM second-order term y fp32[B] / v fp32[B, D] of
    every sample -- one launch on small / short-bag batches. `plan` is a binding.Plan."""
    import numpy as np
    pool = None if pooling is None else np.ascontiguousarray(pooling, dtype=np.uint8)
    _check(_lib().dpi_forward_fm(plan._h, _ptr(lengths_dev), _ptr(table_ptrs_dev), _ptr(indices_dev), _ptr(pool), _ptr(out_dev),
                                 _ptr(y), _ptr(v), _stream_handle(stream)))


def lr_first_order(w_ptrs, indices, offsets, B: int, T: int, bias: float, y, accumulate: bool = False, stream=None) -> None:
    """dpi_lr_first_order: y[b] (+)= bias + sum of the scalar weights of sample b's entries. w_ptrs: device int64[T] of
    pointers to fp32 weight vectors; indices int32 (CSR, sample-major); offsets int32[B*T+1] or None (one-hot)."""
    _check(_lib().dpi_lr_first_order(_ptr(w_ptrs), _ptr(indices), _ptr(offsets), int(B), int(T), float(bias), _ptr(y),
                                     int(bool(accumulate)), _stream_handle(stream)))


def cross_combine(x0, xl, u, bias, out, dtype: int, B: int, F: int, stream=None) -> None:
    """dpi_cross_combine: out = x0 * (u + bias) + xl over [B, F] device tensors of `dtype`; bias fp32[F] or None."""
    _check(_lib().dpi_cross_combine(_ptr(x0), _ptr(xl), _ptr(u), _ptr(bias), _ptr(out), int(dtype), int(B), int(F),
                                    _stream_handle(stream)))


def bias_act(u, bias, out, dtype: int, B: int, F: int, act: int = ACT_RELU, stream=None) -> None:
    """dpi_bias_act: out = act(u + bias) over [B, F] device tensors of `dtype`; bias fp32[F] or None."""
    _check(_lib().dpi_bias_act(_ptr(u), _ptr(bias), _ptr(out), int(dtype), int(B), int(F), int(act),
                               _stream_handle(stream)))


def bfs_schedule(n_explicit: int, n_implicit: int) -> List[Tuple[int, int]]:
    """dpi_bfs_schedule: Algorithm 2's launch queue as [(module, op index)], module 0 = explicit, 1 = implicit."""
    n = max(int(n_explicit), 0) + max(int(n_implicit), 0)
    qm = np.empty(max(n, 1), dtype=np.int32)
    qo = np.empty(max(n, 1), dtype=np.int32)
    _check(_lib().dpi_bfs_schedule(int(n_explicit), int(n_implicit), qm.ctypes.data, qo.ctypes.data))
    return [(int(qm[i]), int(qo[i])) for i in range(n)]


class Launcher:
    """Owner of a ``dpi_launcher_t*`` (two non-blocking module streams + fork/join events)."""

    def __init__(self):
        self._h = ctypes.c_void_p()
        _check(_lib().dpi_launcher_create(ctypes.byref(self._h)))

    def run(self, explicit_ops: Sequence[Callable[[int], None]], implicit_ops: Sequence[Callable[[int], None]],
            n_streams: int = 2, stream=None) -> None:
        """dpi_launcher_run. Each op is a Python callable taking the raw cudaStream_t handle (an int) and enqueuing
        its work there; it is wrapped into a dpi_op_t whose `launch` calls it."""
        keep = []

        def wrap(fn):
            def tramp(_user, s):
                fn(int(s) if s else 0)
            cb = OP_FN(tramp)
            keep.append(cb)
            return cb

        def pack(ops):
            arr = (Op * max(len(ops), 1))()
            for i, fn in enumerate(ops):
                arr[i].launch = wrap(fn)
                arr[i].user = None
            return arr

        e_arr, i_arr = pack(explicit_ops), pack(implicit_ops)
        _check(_lib().dpi_launcher_run(self._h, ctypes.cast(e_arr, ctypes.c_void_p), len(explicit_ops),
                                       ctypes.cast(i_arr, ctypes.c_void_p), len(implicit_ops), int(n_streams),
                                       _stream_handle(stream)))
        del keep

    def destroy(self) -> None:
        if self._h:
            _check(_lib().dpi_launcher_destroy(self._h))
            self._h = ctypes.c_void_p()

    def __del__(self):
        try:
            self.destroy()
        except Exception:
            pass
