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
    "qcf_full_prefill_attn", "qcf_layer_step", "qcf_layer_step_host", "qcf_set_profiling", "qcf_get_stage_ms", "qcf_set_head_shards", "qcf_debug_set",
    "qcf_anchor_rank", "qcf_anchor_gather", "qcf_linear", "qcf_stack_create", "qcf_stack_destroy", "qcf_stack_prefill", "qcf_stack_layer", "qcf_stack_fuse", "qcf_stack_first_token",
    "qcf_decode_attn", "qcf_decode_attn_static", "qcf_stack_decode", "qcf_score_exchange_bytes", "qcf_set_score_exchange",
)

QCF_EPI_STORE, QCF_EPI_ADD_RESIDUAL, QCF_EPI_SWIGLU = 0, 1, 2
QCF_ANCHOR_SINK, QCF_ANCHOR_KNORM = 0, 1
QCF_DEBUG_PDL, QCF_DEBUG_ATTN_CLUSTER, QCF_DEBUG_GEMM_MT = 0, 1, 2


class QcfError(RuntimeError):
    def __init__(self, status: int, message: str):
        super().__init__("%s: %s" % (_STATUS.get(status, status), message))
        self.status = status


class qcf_layout(C.Structure):
    _fields_ = [("n_q_heads", C.c_int32), ("n_kv_heads", C.c_int32), ("head_dim", C.c_int32),
                ("rope_theta", C.c_float), ("softmax_scale", C.c_float)]


class qcf_request(C.Structure):
    _fields_ = [("n_chunks", C.c_int32), ("n_query", C.c_int32),
                ("chunk_len", C.POINTER(C.c_int32)), ("chunk_row", C.POINTER(C.c_int64)),
                ("chunk_pos", C.POINTER(C.c_int32))]


class qcf_batch_info(C.Structure):
    _fields_ = [("batch", C.c_int32), ("t_stride", C.c_int32), ("n_stride", C.c_int32), ("q_stride", C.c_int32),
                ("total_ctx", C.c_int64), ("pool_rows_touched", C.c_int64)]


class qcf_layer_args(C.Structure):
    _fields_ = [("k_pool", C.c_void_p), ("v_pool", C.c_void_p), ("k_fused", C.c_void_p), ("v_fused", C.c_void_p),
                ("q_probe", C.c_void_p), ("scores", C.c_void_p), ("sel", C.c_void_p), ("n_sel", C.c_void_p),
                ("q_new", C.c_void_p), ("k_new", C.c_void_p), ("v_new", C.c_void_p), ("out", C.c_void_p),
                ("lse", C.c_void_p), ("ratio", C.c_double), ("rows_by_position", C.c_int32),
                ("is_critical_layer", C.c_int32), ("accumulate", C.c_int32), ("select_now", C.c_int32)]


class qcf_stack_dims(C.Structure):
    _fields_ = [("n_layers", C.c_int32), ("hidden", C.c_int32), ("ffn", C.c_int32), ("vocab", C.c_int32),
                ("rms_eps", C.c_float)]


class qcf_layer_weights(C.Structure):
    _fields_ = [(n, C.c_void_p) for n in ("w_qkv", "w_o", "w_gate_up", "w_down", "g_attn", "g_ffn", "g_q", "g_k")]


class qcf_fuse_args(C.Structure):
    _fields_ = [
        ("k_pic", C.POINTER(C.c_void_p)), ("v_pic", C.POINTER(C.c_void_p)), ("pool_rows", C.c_int64),
        ("k_anchor", C.POINTER(C.c_void_p)), ("v_anchor", C.POINTER(C.c_void_p)), ("anchor_rows", C.c_int64),
        ("crit_layers", C.POINTER(C.c_int32)), ("n_crit", C.c_int32), ("ratio", C.c_double), ("tokens", C.c_void_p),
        ("k_fused", C.POINTER(C.c_void_p)), ("v_fused", C.POINTER(C.c_void_p)), ("scores", C.c_void_p),
        ("sel", C.c_void_p), ("n_sel", C.c_void_p), ("hidden_out", C.c_void_p), ("overlap", C.c_int32), ("stages", C.c_int32), ("load_gbps", C.c_double),
    ]


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
        "qcf_set_head_shards": (i32, [vp, i32]),
        "qcf_debug_set": (i32, [vp, i32, i32]),
        "qcf_score_exchange_bytes": (i64, [i32, i64]),
        "qcf_set_score_exchange": (i32, [vp, i32, i32, C.POINTER(vp), i64]),
        "qcf_get_stage_ms": (i32, [vp, C.POINTER(C.c_float)]),
        "qcf_anchor_rank": (i32, [vp, vp, vp, i32, f64, vp, i32, i32, vp, vp, vp]),
        "qcf_anchor_gather": (i32, [vp, vp, vp, vp, vp, vp, vp, vp, vp]),
        "qcf_linear": (i32, [vp, vp, vp, vp, vp, i32, i32, i32, i32, vp]),
        "qcf_stack_create": (i32, [vp, C.POINTER(qcf_stack_dims), C.POINTER(qcf_layer_weights), vp, i32, i32, i64,
                                   C.POINTER(vp)]),
        "qcf_stack_destroy": (None, [vp]),
        "qcf_stack_prefill": (i32, [vp, vp, vp, C.POINTER(vp), C.POINTER(vp), vp, vp]),
        "qcf_stack_layer": (i32, [vp, i32, vp, vp, vp, i32, i32, vp, vp, vp, vp, vp]),
        "qcf_stack_fuse": (i32, [vp, vp, vp, C.POINTER(qcf_fuse_args), vp]),
        "qcf_stack_first_token": (i32, [vp, vp, i32, vp, vp, vp, vp, vp]),
        "qcf_decode_attn": (i32, [vp, vp, vp, vp, i32, vp, vp, vp]),
        "qcf_decode_attn_static": (i32, [C.POINTER(qcf_layout), vp, vp, vp, i32, vp, vp, vp]),
        "qcf_stack_decode": (i32, [vp, vp, i32, i32, C.POINTER(vp), C.POINTER(vp), vp, vp, vp, vp, vp]),
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


def qcf_score_exchange_bytes(n_shards: int, slot_elems: int) -> int:
    return int(load_library().qcf_score_exchange_bytes(int(n_shards), int(slot_elems)))


def qcf_decode_attn_static(n_q_heads: int, n_kv_heads: int, head_dim: int, q, k_cache, v_cache, n_keys: int, out, lse=None,
                           softmax_scale: float = 0.0, stream=None) -> None:
    """qcf_decode_attn without a Context: for callers that must not allocate device memory (the kernel's workspace is a
    fixed array inside libqcf.so; limits and sharing rules in include/qcf.h).  Marshals the arguments, nothing else."""
    lib = load_library()
    lay = qcf_layout(int(n_q_heads), int(n_kv_heads), int(head_dim), 0.0, float(softmax_scale))
    st = lib.qcf_decode_attn_static(C.byref(lay), _ptr(q), _ptr(k_cache), _ptr(v_cache), int(n_keys), _ptr(out), _ptr(lse),
                                    _stream(stream))
    if st != QCF_OK:
        raise QcfError(st, (lib.qcf_last_error(None) or b"").decode())


def qcf_n_select(n_ctx: int, ratio: float) -> int:
    return int(load_library().qcf_n_select(n_ctx, ratio))


class Batch:
    """qcf_batch: device-resident description of a batch of requests (chunk lengths + PIC pool rows)."""

    def __init__(self, ctx: "Context", chunk_lens: Sequence[Sequence[int]], chunk_rows: Sequence[Sequence[int]],
                 n_query: Sequence[int], chunk_pos: Optional[Sequence[Sequence[int]]] = None):
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
            if chunk_pos is not None:              # anchor stitch (Eq. 15-16): rotate by the chunk's ORIGINAL offset
                cp = np.ascontiguousarray(chunk_pos[b], dtype=np.int32)
                assert cp.shape == cl.shape
                self._keep.append(cp)
                reqs[b].chunk_pos = cp.ctypes.data_as(C.POINTER(C.c_int32))
        h = C.c_void_p()
        ctx._check(ctx.lib.qcf_batch_create(ctx.handle, reqs, n, C.byref(h)))
        self.handle = h
        info = qcf_batch_info()
        ctx.lib.qcf_batch_get_info(self.handle, C.byref(info))
        self.batch, self.t_stride, self.n_stride, self.q_stride = info.batch, info.t_stride, info.n_stride, info.q_stride
        self.total_ctx = info.total_ctx
        self.pool_rows_touched = info.pool_rows_touched
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

    def batch(self, chunk_lens, chunk_rows, n_query, chunk_pos=None) -> Batch:
        return Batch(self, chunk_lens, chunk_rows, n_query, chunk_pos)

    def qcf_anchor_rank(self, chunks: Batch, k_pool, rule: int, r_a: float, scores, anchor_idx, n_anchor,
                        accumulate: bool = False, select_now: bool = True, stream=None):
        self._check(self.lib.qcf_anchor_rank(self.handle, chunks.handle, _ptr(k_pool), int(rule), float(r_a), _ptr(scores),
                                             int(bool(accumulate)), int(bool(select_now)), _ptr(anchor_idx), _ptr(n_anchor),
                                             _stream(stream)))

    def qcf_anchor_gather(self, chunks: Batch, k_pool, v_pool, anchor_idx, n_anchor, k_anchor, v_anchor, stream=None):
        self._check(self.lib.qcf_anchor_gather(self.handle, chunks.handle, _ptr(k_pool), _ptr(v_pool), _ptr(anchor_idx),
                                               _ptr(n_anchor), _ptr(k_anchor), _ptr(v_anchor), _stream(stream)))

    def qcf_linear(self, a, w, residual, c, M: int, N: int, K: int, epilogue: int = QCF_EPI_STORE, stream=None):
        self._check(self.lib.qcf_linear(self.handle, _ptr(a), _ptr(w), _ptr(residual), _ptr(c), M, N, K, epilogue,
                                        _stream(stream)))

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

    def qcf_set_head_shards(self, n_shards: int):
        self._check(self.lib.qcf_set_head_shards(self.handle, int(n_shards)))

    def qcf_decode_attn(self, q, k_cache, v_cache, n_keys: int, out, lse=None, stream=None):
        self._check(self.lib.qcf_decode_attn(self.handle, _ptr(q), _ptr(k_cache), _ptr(v_cache), int(n_keys), _ptr(out),
                                             _ptr(lse), _stream(stream)))

    def qcf_debug_set(self, knob: int, value: int):
        self._check(self.lib.qcf_debug_set(self.handle, int(knob), int(value)))

    def qcf_set_score_exchange(self, rank: int, n_shards: int, peer_bufs, slot_elems: int):
        """peer_bufs: sequence of n_shards device pointers / tensors (rank p's exchange buffer mapped into this process);
        None turns the exchange off."""
        if peer_bufs is None:
            self._check(self.lib.qcf_set_score_exchange(self.handle, 0, 1, None, 0))
            return
        self._exch_keep = list(peer_bufs)
        self._check(self.lib.qcf_set_score_exchange(self.handle, int(rank), int(n_shards), _ptr_array(self._exch_keep),
                                                    int(slot_elems)))

    def qcf_set_profiling(self, enable: bool):
        self._check(self.lib.qcf_set_profiling(self.handle, int(bool(enable))))

    def qcf_get_stage_ms(self) -> List[float]:
        ms = (C.c_float * 5)()
        self._check(self.lib.qcf_get_stage_ms(self.handle, ms))
        return [float(x) for x in ms]


def _ptr_array(ptrs):
    arr = (C.c_void_p * len(ptrs))()
    for i, p in enumerate(ptrs):
        arr[i] = _ptr(p)
    return arr


class Stack:
    """qcf_stack (config 3).  `layers`: list of dicts of device tensors keyed by the field names of qcf_layer_weights;
    the tensors are kept alive by this object."""

    def __init__(self, ctx: Context, n_layers: int, hidden: int, ffn: int, vocab: int, rms_eps: float, layers, embed,
                 max_rows: int, max_pos: int, max_pool_rows: int = 0):
        self.ctx, self.lib, self.handle = ctx, ctx.lib, None
        self._keep = (layers, embed)
        self.n_layers, self.hidden, self.ffn = n_layers, hidden, ffn
        dims = qcf_stack_dims(n_layers, hidden, ffn, vocab, rms_eps)
        lw = (qcf_layer_weights * n_layers)()
        for i, d in enumerate(layers):
            for name, _ in qcf_layer_weights._fields_:
                setattr(lw[i], name, _ptr(d[name]))
        h = C.c_void_p()
        ctx._check(self.lib.qcf_stack_create(ctx.handle, C.byref(dims), lw, _ptr(embed), max_rows, max_pos,
                                             max_pool_rows, C.byref(h)))
        self.handle = h

    def close(self):
        if self.handle:
            self.lib.qcf_stack_destroy(self.handle)
            self.handle = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def qcf_stack_prefill(self, b: Batch, tokens, k_cache, v_cache, hidden_out=None, stream=None):
        self.ctx._check(self.lib.qcf_stack_prefill(self.handle, b.handle, _ptr(tokens), _ptr_array(k_cache),
                                                   _ptr_array(v_cache), _ptr(hidden_out), _stream(stream)))

    def qcf_stack_layer(self, layer: int, b: Batch, sel, n_sel, n_rows: int, x, k_fused, v_fused, query_pos0: int = -1,
                        q_tap=None, stream=None):
        self.ctx._check(self.lib.qcf_stack_layer(self.handle, layer, b.handle, _ptr(sel), _ptr(n_sel), n_rows,
                                                 query_pos0, _ptr(x), _ptr(k_fused), _ptr(v_fused), _ptr(q_tap),
                                                 _stream(stream)))

    def qcf_stack_first_token(self, hidden, row: int, g_final, w_lm, logits, token, stream=None):
        self.ctx._check(self.lib.qcf_stack_first_token(self.handle, _ptr(hidden), int(row), _ptr(g_final), _ptr(w_lm),
                                                       _ptr(logits), _ptr(token), _stream(stream)))

    def qcf_stack_decode(self, token_in, pos0: int, n_new: int, k_cache, v_cache, g_final, w_lm, logits, tokens_out,
                         stream=None):
        self.ctx._check(self.lib.qcf_stack_decode(self.handle, _ptr(token_in), int(pos0), int(n_new), _ptr_array(k_cache),
                                                  _ptr_array(v_cache), _ptr(g_final), _ptr(w_lm), _ptr(logits),
                                                  _ptr(tokens_out), _stream(stream)))

    def qcf_stack_fuse(self, main: Batch, probe: Batch, *, k_pic, v_pic, pool_rows: int, k_anchor, v_anchor,
                       anchor_rows: int, crit_layers, ratio: float, tokens, k_fused, v_fused, scores, sel, n_sel,
                       hidden_out=None, overlap: bool = True, stages: int = 0, load_gbps: float = 0.0, stream=None):
        crit = (C.c_int32 * len(crit_layers))(*[int(c) for c in crit_layers])
        keep = [_ptr_array(x) for x in (k_pic, v_pic, k_anchor, v_anchor, k_fused, v_fused)]
        a = qcf_fuse_args(keep[0], keep[1], pool_rows, keep[2], keep[3], anchor_rows, crit, len(crit_layers), ratio,
                          _ptr(tokens), keep[4], keep[5], _ptr(scores), _ptr(sel), _ptr(n_sel), _ptr(hidden_out),
                          1 if overlap else 0, int(stages), float(load_gbps))
        self.ctx._check(self.lib.qcf_stack_fuse(self.handle, main.handle, probe.handle, C.byref(a), _stream(stream)))
