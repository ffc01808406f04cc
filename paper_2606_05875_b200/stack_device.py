"""Device-side plumbing of BASELINE config 3 for bench.py (and the full-size GPU tests): random-init weights drawn on the
device, Phase-I artifacts (per-chunk PIC caches, compact anchor pools) built with the library's own prefill and parked
in pinned host memory, and the buffers qcf_stack_fuse / qcf_stack_prefill write.

Torch is used for memory, random initialisation and streams only; every step of the path runs inside libqcf.so.
"""
from __future__ import annotations

from typing import Dict, List

import numpy as np
import torch

from . import binding
from .inputs import StackWorkload


def device_weights(sp, seed: int, device) -> tuple:
    """Random-init bf16 weights in the layout of qcf_layer_weights (N(0, 0.02^2); gains 1 + 0.1 N(0,1); embeddings
    N(0,1)).  13.9 GB at config 3, drawn on the device (there are no checkpoints in this container)."""
    g = torch.Generator(device=device)
    g.manual_seed(seed)
    hq, hkv, d, hid, ffn = sp.n_q_heads, sp.n_kv_heads, sp.head_dim, sp.hidden, sp.ffn

    def w(rows, cols):
        return (torch.randn((rows, cols), generator=g, device=device, dtype=torch.float32) * 0.02).to(torch.bfloat16)

    def gain(n):
        return (1.0 + 0.1 * torch.randn((n,), generator=g, device=device, dtype=torch.float32)).to(torch.bfloat16)

    layers = []
    for _ in range(sp.n_layers):
        layers.append({"w_qkv": w((hq + 2 * hkv) * d, hid), "w_o": w(hid, hq * d), "w_gate_up": w(2 * ffn, hid),
                       "w_down": w(hid, ffn), "g_attn": gain(hid), "g_ffn": gain(hid), "g_q": gain(d), "g_k": gain(d)})
    embed = torch.randn((sp.vocab, hid), generator=g, device=device, dtype=torch.float32).to(torch.bfloat16)
    return layers, embed


class StackRun:
    """One config-3 request resident on `device`: stack handle, batches, Phase-I artifacts, output buffers."""

    def __init__(self, wl: StackWorkload, ctx: binding.Context, layers, embed, device="cuda:0"):
        sp = wl.spec
        self.wl, self.sp, self.ctx, self.device = wl, sp, ctx, device
        n, lq, L = sp.n_ctx, sp.n_query, sp.n_layers
        hkv, d = sp.n_kv_heads, sp.head_dim
        self.t = n + lq
        self.stack = binding.Stack(ctx, L, sp.hidden, sp.ffn, sp.vocab, sp.rms_eps, layers, embed, self.t, self.t,
                                   max_pool_rows=n)
        lens = [sp.chunk_len] * sp.n_chunks
        off = [i * sp.chunk_len for i in range(sp.n_chunks)]
        self.main = ctx.batch([lens], [off], [lq])
        self.probe = ctx.batch([np.diff(wl.anchor_ptr)], [wl.anchor_ptr[:-1]], [lq], chunk_pos=[off])
        self.full = self.main                      # dense prefill of the whole prompt uses the same geometry
        self.tokens = torch.from_numpy(np.concatenate(wl.chunk_tokens + [wl.query_tokens]).astype(np.int32)).to(device)
        self.k_sel = binding.qcf_n_select(n, sp.ratio)
        self.n_rows = self.k_sel + lq
        self.anchor_rows = int(wl.anchor_ptr[-1])
        kv = lambda rows: torch.zeros((rows, hkv, d), dtype=torch.bfloat16, device=device)
        self.k_fused = [kv(self.t) for _ in range(L)]
        self.v_fused = [kv(self.t) for _ in range(L)]
        self.scores = torch.zeros(n, dtype=torch.float32, device=device)
        self.sel = torch.zeros(n, dtype=torch.int32, device=device)
        self.n_sel = torch.zeros(1, dtype=torch.int32, device=device)
        self.hidden = torch.zeros((self.n_rows, sp.hidden), dtype=torch.bfloat16, device=device)
        self.k_pic: List[torch.Tensor] = []
        self.v_pic: List[torch.Tensor] = []
        self.k_anchor: List[torch.Tensor] = []
        self.v_anchor: List[torch.Tensor] = []

    def build_phase1(self, pinned: bool = True):
        """Eq. 3 with the library's prefill, chunk by chunk at chunk-local positions; pools go to pinned host memory
        (the paper's KV store is off-device) or stay on the device (pinned=False)."""
        sp, dev = self.sp, self.device
        L, hkv, d = sp.n_layers, sp.n_kv_heads, sp.head_dim
        pool_k = [torch.zeros((sp.n_ctx, hkv, d), dtype=torch.bfloat16, device=dev) for _ in range(L)]
        pool_v = [torch.zeros_like(p) for p in pool_k]
        cb = self.ctx.batch([[sp.chunk_len]], [[0]], [0])
        for i in range(sp.n_chunks):
            r0, r1 = i * sp.chunk_len, (i + 1) * sp.chunk_len
            self.stack.qcf_stack_prefill(cb, self.tokens[r0:r1], [p[r0:r1] for p in pool_k], [p[r0:r1] for p in pool_v])
        torch.cuda.synchronize()
        a_rows = np.concatenate([i * sp.chunk_len + self.wl.anchor_idx[self.wl.anchor_ptr[i]: self.wl.anchor_ptr[i + 1]]
                                 for i in range(sp.n_chunks)]).astype(np.int64)
        a_rows = torch.from_numpy(a_rows).to(dev)
        park = (lambda t: t.cpu().pin_memory()) if pinned else (lambda t: t)
        for l in range(L):
            self.k_anchor.append(park(pool_k[l][a_rows].contiguous()))
            self.v_anchor.append(park(pool_v[l][a_rows].contiguous()))
            self.k_pic.append(park(pool_k[l]))
            self.v_pic.append(park(pool_v[l]))
        torch.cuda.synchronize()

    def use_selector(self, kind: str):
        """Which view stage 1 sees (include/qcf.h, qcf_stack_fuse): 'qcfuse' = per-chunk anchors + the critical layers
        (the default, set by build_phase1), 'fullview' = every token of every chunk as an anchor + every layer
        (ProphetKV-style, Eq. 9-11), 'final' = no anchors, last layer only.  Call after build_phase1."""
        sp, ctx = self.sp, self.ctx
        lens = [sp.chunk_len] * sp.n_chunks
        off = [i * sp.chunk_len for i in range(sp.n_chunks)]
        if not hasattr(self, "_qcfuse_view"):
            self._qcfuse_view = (self.probe, self.k_anchor, self.v_anchor, self.anchor_rows, tuple(sp.crit_layers))
        if kind == "qcfuse":
            self.probe, self.k_anchor, self.v_anchor, self.anchor_rows, self.crit = self._qcfuse_view
        elif kind == "fullview":
            self.probe = ctx.batch([lens], [off], [sp.n_query], chunk_pos=[off])
            self.k_anchor, self.v_anchor, self.anchor_rows = self.k_pic, self.v_pic, sp.n_ctx
            self.crit = tuple(range(sp.n_layers))
        elif kind == "final":
            self.probe = ctx.batch([[0] * sp.n_chunks], [[0] * sp.n_chunks], [sp.n_query], chunk_pos=[off])
            self.k_anchor, self.v_anchor, self.anchor_rows = self.k_pic, self.v_pic, 0
            self.crit = (sp.n_layers - 1,)
        else:
            raise ValueError(kind)

    def fuse(self, overlap: bool = True, stream=None, stages: int = 0, load_gbps: float = 0.0):
        sp = self.sp
        self.stack.qcf_stack_fuse(self.main, self.probe, k_pic=self.k_pic, v_pic=self.v_pic, pool_rows=sp.n_ctx,
                                  k_anchor=self.k_anchor, v_anchor=self.v_anchor, anchor_rows=self.anchor_rows,
                                  crit_layers=getattr(self, "crit", sp.crit_layers), ratio=sp.ratio, tokens=self.tokens, k_fused=self.k_fused,
                                  v_fused=self.v_fused, scores=self.scores, sel=self.sel, n_sel=self.n_sel,
                                  hidden_out=self.hidden, overlap=overlap, stages=stages, load_gbps=load_gbps, stream=stream)

    def full_prefill(self, k_cache, v_cache, hidden_out=None, stream=None):
        self.stack.qcf_stack_prefill(self.full, self.tokens, k_cache, v_cache, hidden_out, stream)

    def flops(self) -> Dict[str, float]:
        """Algorithmic flops: GEMMs 2 M (params per layer) per layer, attention 4 d Hq pairs."""
        sp = self.sp
        hq, hkv, d, hid, ffn = sp.n_q_heads, sp.n_kv_heads, sp.head_dim, sp.hidden, sp.ffn
        per_row = 2.0 * (hid * (hq + 2 * hkv) * d + hq * d * hid + 3 * hid * ffn)
        n, lq, L = sp.n_ctx, sp.n_query, sp.n_layers
        sel = self.sel[: self.k_sel].cpu().numpy().astype(np.int64)
        pos = np.concatenate([sel, np.arange(n, n + lq)])
        attn_sel = 4.0 * d * hq * float(np.sum(pos + 1))
        attn_full = 4.0 * d * hq * float(np.sum(np.arange(n + lq) + 1))
        l_probe = max(sp.crit_layers) + 1
        attn_probe = 4.0 * d * hq * float(np.sum(self.anchor_rows + np.arange(lq) + 1))
        score = 2.0 * lq * hq * n * d * len(sp.crit_layers)
        return {"gemm_fuse": per_row * (self.n_rows * L + lq * l_probe), "attn_fuse": attn_sel * L + attn_probe * l_probe + score,
                "gemm_full": per_row * (n + lq) * L, "attn_full": attn_full * L}
