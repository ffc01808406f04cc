"""Thin ctypes binding of libqcf.so (include/qcf.h): argument marshalling only.

Every step of the path runs in the library's CUDA kernels; torch is used by callers for device memory and streams.
Names mirror the C ABI.  There is no CPU fallback: a missing library or device raises.
"""
from __future__ import annotations

import ctypes as C
import os
from typing import List, Optional, Sequence

import numpy as np

_PKG_DIR = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_PKG_DIR, "libqcf.so")

QCF_OK, QCF_ERR_INVALID_ARG, QCF_ERR_UNSUPPORTED, QCF_ERR_WORKSPACE, QCF_ERR_CUDA = range(5)
_STATUS = {0: "QCF_OK", 1: "QCF_ERR_INVALID_ARG", 2: "QCF_ERR_UNSUPPORTED", 3: "QCF_ERR_WORKSPACE", 4: "QCF_ERR_CUDA"}

# every symbol include/qcf.h declares (tests/test_abi.py checks the header against this list and the .so)
EXPORTS = (
    "qcf_create", "qcf_destroy", "qcf_last_error", "qcf_version", "qcf_batch_create", "qcf_batch_destroy",
    "qcf_batch_get_info", "qcf_n_select", "qcf_rope_reposition", "qcf_score", "qcf_select_topk", "qcf_recompute_attn",
    "qcf_full_prefill_attn", "qcf_layer_step", "qcf_layer_step_host", "qcf_set_profiling", "qcf_get_stage_ms",
)


class QcfError(RuntimeError):
    def __init__(self, status: int, message: str):
        super().__init__("%s: %s" % (_STATUS.get(status, status), message))
        self.status = status


class qcf_layout(C.Structure):
    _fields_ = [("n_q_heads", C.c_int32), ("n_kv_heads", C.c_int32), ("head_dim", C.c_int32),
                ("rope_theta", C.c_float), ("softmax_scale", C.c_float)]


class qcf_request(C.Structure):
    _fields_ = [("n_chunks", C.c_int32), ("n_query", C.c_int32),
                ("chunk_len", C.POINTER(C.c_int32)), ("chunk_row", C.POINTER(C.c_int64))]


class qcf_batch_info(C.Structure):
    _fields_ = [("batch", C.c_int32), ("t_stride", C.c_int32), ("n_stride", C.c_int32), ("q_stride", C.c_int32),
                ("total_ctx", C.c_int64)]


class qcf_layer_args(C.Structure):
    _fields_ = [("k_pool", C.c_void_p), ("v_pool", C.c_void_p), ("k_fused", C.c_void_p), ("v_fused", C.c_void_p),
                ("q_probe", C.c_void_p), ("scores", C.c_void_p), ("sel", C.c_void_p), ("n_sel", C.c_void_p),
                ("q_new", C.c_void_p), ("k_new", C.c_void_p), ("v_new", C.c_void_p), ("out", C.c_void_p),
                ("lse", C.c_void_p), ("ratio", C.c_double), ("rows_by_position", C.c_int32),
                ("is_critical_layer", C.c_int32), ("accumulate", C.c_int32), ("select_now", C.c_int32)]


_lib = None


def load_library(build_if_missing: bool = True) -> C.CDLL:
    """dlopen libqcf.so (building it in-tree first if it is absent and nvcc is available)."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(LIB_PATH):
        if not build_if_missing:
            raise FileNotFoundError(LIB_PATH)
        from . import build as _build
        _build.build()
    lib = C.CDLL(LIB_PATH)
    vp, i32, i64, f64 = C.c_void_p, C.c_int32, C.c_int64, C.c_double
    sigs = {
        "qcf_create": (i32, [C.POINTER(vp), C.POINTER(qcf_layout), i32, i32, i32]),
        "qcf_destroy": (None, [vp]),
        "qcf_last_error": (C.c_char_p, [vp]),
        "qcf_version": (C.c_char_p, []),
        "qcf_batch_create": (i32, [vp, C.POINTER(qcf_request), i32, C.POINTER(vp)]),
        "qcf_batch_destroy": (None, [vp]),
        "qcf_batch_get_info": (i32, [vp, C.POINTER(qcf_batch_info)]),
        "qcf_n_select": (i32, [i32, f64]),
        "qcf_rope_reposition": (i32, [vp, vp, vp, vp, vp, vp, vp]),
        "qcf_score": (i32, [vp, vp, vp, vp, vp, i32, vp]),
        "qcf_select_topk": (i32, [vp, vp, vp, f64, vp, vp, vp]),
        "qcf_recompute_attn": (i32, [vp, vp, vp, vp, vp, vp, vp, i32, vp, vp, vp, vp, vp]),
        "qcf_full_prefill_attn": (i32, [vp, vp, vp, vp, vp, vp, vp, vp]),
        "qcf_layer_step": (i32, [vp, vp, C.POINTER(qcf_layer_args), vp]),
        "qcf_layer_step_host": (i32, [vp, vp, C.POINTER(qcf_layer_args), i64, vp]),
        "qcf_set_profiling": (i32, [vp, i32]),
        "qcf_get_stage_ms": (i32, [vp, C.POINTER(C.c_float)]),
    }
    for name, (res, args) in sigs.items():
        fn = getattr(lib, name)
        fn.restype, fn.argtypes = res, args
    _lib = lib
    return lib


def _ptr(x) -> Optional[int]:
    """Device/host address of a torch tensor, numpy array, int or None."""
    if x is None:
        return None
    if isinstance(x, int):
        return x
    if isinstance(x, np.ndarray):
        return x.ctypes.data
    return x.data_ptr()          # torch.Tensor


def _stream(stream) -> Optional[int]:
    if stream is None:
        import torch
        return torch.cuda.current_stream().cuda_stream
    if isinstance(stream, int):
        return stream
    return stream.cuda_stream


def qcf_n_select(n_ctx: int, ratio: float) -> int:
    return int(load_library().qcf_n_select(n_ctx, ratio))


class Batch:
    """qcf_batch: device-resident description of a batch of requests (chunk lengths + PIC pool rows)."""

    def __init__(self, ctx: "Context", chunk_lens: Sequence[Sequence[int]], chunk_rows: Sequence[Sequence[int]],
                 n_query: Sequence[int]):
        self.ctx = ctx
        n = len(chunk_lens)
        reqs = (qcf_request * max(n, 1))()
        self._keep = []
        for b in range(n):
            cl = np.ascontiguousarray(chunk_lens[b], dtype=np.int32)
            cr = np.ascontiguousarray(chunk_rows[b], dtype=np.int64)
            assert cl.shape == cr.shape
            self._keep += [cl, cr]
            reqs[b].n_chunks = len(cl)
            reqs[b].n_query = int(n_query[b])
            reqs[b].chunk_len = cl.ctypes.data_as(C.POINTER(C.c_int32))
            reqs[b].chunk_row = cr.ctypes.data_as(C.POINTER(C.c_int64))
        h = C.c_void_p()
        ctx._check(ctx.lib.qcf_batch_create(ctx.handle, reqs, n, C.byref(h)))
        self.handle = h
        info = qcf_batch_info()
        ctx.lib.qcf_batch_get_info(self.handle, C.byref(info))
        self.batch, self.t_stride, self.n_stride, self.q_stride = info.batch, info.t_stride, info.n_stride, info.q_stride
        self.total_ctx = info.total_ctx
        self.n_ctx = [int(np.sum(c)) for c in chunk_lens]
        self.n_query = [int(q) for q in n_query]

    def close(self):
        if self.handle:
            self.ctx.lib.qcf_batch_destroy(self.handle)
            self.handle = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass


class Context:
    """qcf_ctx for one head layout on the current CUDA device."""

    def __init__(self, n_q_heads: int, n_kv_heads: int, head_dim: int, rope_theta: float, max_batch: int,
                 max_ctx: int, max_query: int, softmax_scale: float = 0.0):
        self.lib = load_library()
        self.layout = qcf_layout(n_q_heads, n_kv_heads, head_dim, rope_theta, softmax_scale)
        h = C.c_void_p()
        st = self.lib.qcf_create(C.byref(h), C.byref(self.layout), max_batch, max_ctx, max_query)
        if st != QCF_OK:
            raise QcfError(st, self.lib.qcf_last_error(None).decode())
        self.handle = h

    def _check(self, st: int):
        if st != QCF_OK:
            raise QcfError(st, self.lib.qcf_last_error(self.handle).decode())

    def close(self):
        if getattr(self, "handle", None):
            self.lib.qcf_destroy(self.handle)
            self.handle = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def batch(self, chunk_lens, chunk_rows, n_query) -> Batch:
        return Batch(self, chunk_lens, chunk_rows, n_query)

    # ---- stage entry points (names and argument order of include/qcf.h)
    def qcf_rope_reposition(self, b: Batch, k_pool, v_pool, k_fused, v_fused, stream=None):
        self._check(self.lib.qcf_rope_reposition(self.handle, b.handle, _ptr(k_pool), _ptr(v_pool), _ptr(k_fused),
                                                 _ptr(v_fused), _stream(stream)))

    def qcf_score(self, b: Batch, q_probe, k_fused, scores, accumulate: bool = False, stream=None):
        self._check(self.lib.qcf_score(self.handle, b.handle, _ptr(q_probe), _ptr(k_fused), _ptr(scores),
                                       int(bool(accumulate)), _stream(stream)))

    def qcf_select_topk(self, b: Batch, scores, ratio: float, sel, n_sel, stream=None):
        self._check(self.lib.qcf_select_topk(self.handle, b.handle, _ptr(scores), float(ratio), _ptr(sel), _ptr(n_sel),
                                             _stream(stream)))

    def qcf_recompute_attn(self, b: Batch, sel, n_sel, q_new, k_new, v_new, rows_by_position: bool, k_fused, v_fused,
                           out, lse=None, stream=None):
        self._check(self.lib.qcf_recompute_attn(self.handle, b.handle, _ptr(sel), _ptr(n_sel), _ptr(q_new), _ptr(k_new),
                                                _ptr(v_new), int(bool(rows_by_position)), _ptr(k_fused), _ptr(v_fused),
                                                _ptr(out), _ptr(lse), _stream(stream)))

    def qcf_full_prefill_attn(self, b: Batch, q, k, v, out, lse=None, stream=None):
        self._check(self.lib.qcf_full_prefill_attn(self.handle, b.handle, _ptr(q), _ptr(k), _ptr(v), _ptr(out), _ptr(lse),
                                                   _stream(stream)))

    @staticmethod
    def layer_args(*, k_pool, v_pool, k_fused, v_fused, q_probe, scores, sel, n_sel, q_new, k_new, v_new, out,
                   lse=None, ratio: float = 0.0, rows_by_position: bool = True, is_critical_layer: bool = True,
                   accumulate: bool = False, select_now: bool = True) -> qcf_layer_args:
        return qcf_layer_args(_ptr(k_pool), _ptr(v_pool), _ptr(k_fused), _ptr(v_fused), _ptr(q_probe), _ptr(scores),
                              _ptr(sel), _ptr(n_sel), _ptr(q_new), _ptr(k_new), _ptr(v_new), _ptr(out), _ptr(lse),
                              float(ratio), int(bool(rows_by_position)), int(bool(is_critical_layer)),
                              int(bool(accumulate)), int(bool(select_now)))

    def qcf_layer_step(self, b: Batch, args: qcf_layer_args, stream=None):
        self._check(self.lib.qcf_layer_step(self.handle, b.handle, C.byref(args), _stream(stream)))

    def qcf_layer_step_host(self, b: Batch, args: qcf_layer_args, pool_rows: int, stream=None):
        self._check(self.lib.qcf_layer_step_host(self.handle, b.handle, C.byref(args), int(pool_rows), _stream(stream)))

    def qcf_set_profiling(self, enable: bool):
        self._check(self.lib.qcf_set_profiling(self.handle, int(bool(enable))))

    def qcf_get_stage_ms(self) -> List[float]:
        ms = (C.c_float * 5)()
        self._check(self.lib.qcf_get_stage_ms(self.handle, ms))
        return [float(x) for x in ms]
