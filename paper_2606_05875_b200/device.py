"""Device-side plumbing shared by tests/, bench.py and __graft_entry__.smoke(): puts a seeded `inputs.Workload` into
device (or pinned host) buffers laid out as include/qcf.h expects and owns the output buffers.

Torch is used for memory and streams only; all arithmetic happens inside libqcf.so.
"""
from __future__ import annotations

from typing import Dict, List

import numpy as np
import torch

from . import binding
from .inputs import Workload


def _bits_to_tensor(bits: np.ndarray, device, pin: bool = False) -> torch.Tensor:
    """uint16 bf16 bit patterns -> torch.bfloat16 tensor (same bits)."""
    t = torch.from_numpy(np.ascontiguousarray(bits).view(np.int16)).view(torch.bfloat16)
    if device == "cpu":
        return t.pin_memory() if pin else t
    return t.to(device)


class DeviceWorkload:
    """One batch of requests resident on `device` ("cuda:0", or "cpu" for pinned-host buffers of the e2e leg)."""

    def __init__(self, wl: Workload, ctx: binding.Context, device="cuda:0", pin: bool = False):
        cfg = wl.cfg
        self.wl, self.ctx, self.cfg, self.device = wl, ctx, cfg, device
        hq, hkv, d = cfg.n_q_heads, cfg.n_kv_heads, cfg.head_dim
        # PIC pool: chunks back to back; chunk_row = first pool row of each chunk
        lens = [k.shape[0] for k in wl.pool_k]
        starts = np.concatenate([[0], np.cumsum(lens)]).astype(np.int64)
        self.pool_rows = int(starts[-1])
        cat = lambda xs: np.concatenate(xs, axis=0) if xs else np.zeros((0, hkv, d), np.uint16)
        self.k_pool = _bits_to_tensor(cat(wl.pool_k), device, pin)
        self.v_pool = _bits_to_tensor(cat(wl.pool_v), device, pin)
        chunk_lens = [r.chunk_len for r in wl.requests]
        chunk_rows = [starts[np.asarray(r.chunk_ids, dtype=np.int64)] if len(r.chunk_ids) else np.zeros(0, np.int64)
                      for r in wl.requests]
        n_query = [r.n_query for r in wl.requests]
        self.batch = ctx.batch(chunk_lens, chunk_rows, n_query)
        B, T, Nn, Q = self.batch.batch, self.batch.t_stride, self.batch.n_stride, self.batch.q_stride
        self.B, self.T, self.Nn, self.Q = B, T, Nn, Q

        def padded(rows_list: List[np.ndarray], stride: int, heads: int) -> torch.Tensor:
            buf = np.zeros((B, stride, heads, d), dtype=np.uint16)
            for b, x in enumerate(rows_list):
                buf[b, : x.shape[0]] = x
            return _bits_to_tensor(buf, device, pin)

        self.q_probe = padded([r.q_probe for r in wl.requests], Q, hq)
        self.q_new = padded([r.q_new for r in wl.requests], T, hq)
        self.k_new = padded([r.k_new for r in wl.requests], T, hkv)
        self.v_new = padded([r.v_new for r in wl.requests], T, hkv)

        def empty(shape, dtype):
            t = torch.zeros(shape, dtype=dtype, device=device)
            return t.pin_memory() if (device == "cpu" and pin) else t

        self.k_fused = empty((B, T, hkv, d), torch.bfloat16)
        self.v_fused = empty((B, T, hkv, d), torch.bfloat16)
        self.scores = empty((B, max(Nn, 1)), torch.float32)
        self.sel = empty((B, max(Nn, 1)), torch.int32)
        self.n_sel = empty((B,), torch.int32)
        self.out = empty((B, T, hq, d), torch.bfloat16)
        self.lse = empty((B, T, hq), torch.float32)

    def layer_args(self, ratio=None, **kw) -> binding.qcf_layer_args:
        return self.ctx.layer_args(
            k_pool=self.k_pool, v_pool=self.v_pool, k_fused=self.k_fused, v_fused=self.v_fused, q_probe=self.q_probe,
            scores=self.scores, sel=self.sel, n_sel=self.n_sel, q_new=self.q_new, k_new=self.k_new, v_new=self.v_new,
            out=self.out, lse=kw.pop("lse", None), ratio=self.cfg.ratio if ratio is None else ratio, **kw)

    def algorithmic_work(self, ratio=None) -> Dict[str, float]:
        """Per-launch algorithmic bytes / flops of each stage."""
        cfg = self.cfg
        ratio = cfg.ratio if ratio is None else ratio
        hq, hkv, d = cfg.n_q_heads, cfg.n_kv_heads, cfg.head_dim
        row = hkv * d * 2
        tot_n = sum(self.batch.n_ctx)
        pairs = 0
        n_rows = 0
        for n, lq in zip(self.batch.n_ctx, self.batch.n_query):
            k = binding.qcf_n_select(n, ratio)
            # expected causal extent of k uniformly spread positions + exact extent of the query rows
            pairs += k * (n + 1) / 2.0 + sum(n + i + 1 for i in range(lq))
            n_rows += k + lq
        return {
            "a1_bytes": 4.0 * row * tot_n,
            "a2_flops": sum(2.0 * lq * hq * n * d for n, lq in zip(self.batch.n_ctx, self.batch.n_query)),
            "a2_bytes": float(row // 2 * tot_n),
            "a2_exps": float(sum(lq * hq * n for n, lq in zip(self.batch.n_ctx, self.batch.n_query))),
            "a4_bytes": 4.0 * row * n_rows,
            # a5: the fused K and V of every request once + the Q rows read and the O rows written
            "a5_bytes": float(sum(2 * row * (n + lq) for n, lq in zip(self.batch.n_ctx, self.batch.n_query))
                              + 2 * n_rows * hq * d * 2),
            "a5_flops_expected": 4.0 * d * hq * pairs,
            "n_rows": n_rows,
        }


def attn_flops(cfg, n_ctx: int, positions: np.ndarray) -> float:
    """Exact a5 flops of one request: 4 d Hq sum_r (p_r + 1)."""
    return 4.0 * cfg.head_dim * cfg.n_q_heads * float(np.sum(positions.astype(np.int64) + 1))
