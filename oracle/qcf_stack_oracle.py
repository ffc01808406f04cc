"""fp64 CPU oracle for BASELINE config 3: the QCFuse two-stage pipeline on a Qwen3-shaped decoder stack.

TEST INFRASTRUCTURE — NOT A PRODUCT PATH.  Only `tests/`, `__graft_entry__.smoke()` and `bench.py`'s
`cpu_baseline` / `--impl reference` legs may import this module.  It shares no code with the CUDA path
(`paper_2606_05875_b200/`) and imports nothing from it; it builds on `oracle/qcf_oracle.py` (same rules).

What is computed (citations are /root/reference/PAPER.md lines + equation):

  full_prefill     Eq. 2  KV^Full(X) = LLM(X): every row through every layer
  build_pic        Eq. 3  per-chunk offline caches at chunk-local positions
  probe_stage      Eq. 15-20, Fig. 9 stage 1: forward U over the stitched
                   anchor cache up to the deepest critical layer, tap Q_U^l(C_A) at l in L*, score the original
                   context positions against the stitched PIC keys of those layers, top-k -> P
  fuse_stage       Eq. 6-7, Fig. 9 stage 2: per layer, rows R = P u U only:
                   projections, refreshed K/V scattered into the fused cache, causal attention over it, MLP
  decode_step /    generation over KV^Fuse ("the fused KV cache and the user query states are handed to
  greedy_decode    decoding"; TTFT ends at the first token, decoding continues from it): one new token at
                   position p attends over cache rows 0..p of every layer and appends its own K/V at row p

The decoder layer is the "Qwen3-8B-shaped" block BASELINE.json names (the paper fixes nothing about it;
DESIGN.md readings (l), (q)): pre-norm residual block, RMSNorm (eps 1e-6), GQA attention with per-head RMSNorm on
q and k ("QK-norm") before RoPE, no biases, SwiGLU MLP:

      h = RMSNorm(x; g_attn);  q, k, v = h W_q^T, h W_k^T, h W_v^T
      q = RoPE(RMSNorm_head(q; g_q), pos);  k = RoPE(RMSNorm_head(k; g_k), pos)
      cache[pos] = bf16(k), bf16(v)                       (the KV cache is a bf16 object, reading (t))
      a = CausalGQA(q, cache);  x = x + a W_o^T
      h = RMSNorm(x; g_ffn);    x = x + (silu(h W_g^T) * (h W_u^T)) W_d^T

All arithmetic is numpy float64; only K/V written to a cache are rounded (to bf16).  Attention always reads the
cache (rounded values), in every path, so that "fused with rho = 1" and "full prefill" are the same function.

Pins (tests/test_stack_oracle_pins.py, `-m "not gpu"`): each dense op against torch CPU fp64 library routines
(F.rms_norm, F.linear, F.silu, F.scaled_dot_product_attention); W_o = W_d = 0 leaves x unchanged; W_g = 0 kills the
MLP; causality (perturbing a later token leaves earlier rows unchanged); prefill at positions shifted by D gives the
same hidden states and K caches equal to Pi(D) of the unshifted ones (ties the stack's RoPE to Eq. 4);
single-chunk prompt fused == full prefill at every layer for any P; rho = 1 multi-chunk == full prefill;
rho = 0 == the probe path with every token an anchor (two independent code paths);
decode_step on the caches of a T-token full prefill == the last row of a (T+1)-token full prefill (hidden state and the
appended K/V), its attention == torch fp64 SDPA of one query row over the cache; greedy_decode == re-running the full
prefill on the growing sequence and taking the argmax each time (brute force).
Parity unpinned: selection QUALITY versus the paper's Recall@10 % / F1 (needs datasets and trained weights).
"""
from __future__ import annotations

from dataclasses import dataclass, field
from typing import Dict, List, Optional, Sequence, Tuple

import numpy as np

from . import qcf_oracle as O


@dataclass
class StackConfig:
    n_layers: int
    hidden: int
    ffn: int
    n_q_heads: int
    n_kv_heads: int
    head_dim: int
    rope_theta: float
    rms_eps: float = 1e-6


@dataclass
class LayerWeights:
    """float64 arrays, nn.Linear layout [out, in]."""
    wq: np.ndarray        # [Hq*d, hidden]
    wk: np.ndarray        # [Hkv*d, hidden]
    wv: np.ndarray        # [Hkv*d, hidden]
    wo: np.ndarray        # [hidden, Hq*d]
    wg: np.ndarray        # [ffn, hidden]
    wu: np.ndarray        # [ffn, hidden]
    wd: np.ndarray        # [hidden, ffn]
    g_attn: np.ndarray    # [hidden]
    g_ffn: np.ndarray     # [hidden]
    g_q: np.ndarray       # [d]
    g_k: np.ndarray       # [d]


# --------------------------------------------------------------------------- dense ops


def rms_norm(x: np.ndarray, g: np.ndarray, eps: float) -> np.ndarray:
    """y = x / sqrt(mean(x^2) + eps) * g along the last axis."""
    ms = np.mean(np.square(x), axis=-1, keepdims=True)
    return x / np.sqrt(ms + np.float64(eps)) * g


def linear(x: np.ndarray, w: np.ndarray) -> np.ndarray:
    """y = x W^T (W in [out, in] layout, no bias)."""
    return x @ w.T


def silu(x: np.ndarray) -> np.ndarray:
    return x / (1.0 + np.exp(-x))


def layer_qkv(x: np.ndarray, pos: np.ndarray, w: LayerWeights, cfg: StackConfig):
    """Projections of rows x[n, hidden] sitting at request positions pos[n].
    Returns q [n, Hq, d] (unrounded), k, v [n, Hkv, d] rounded to bf16 (they are cache entries)."""
    n = x.shape[0]
    hq, hkv, d = cfg.n_q_heads, cfg.n_kv_heads, cfg.head_dim
    h = rms_norm(x, w.g_attn, cfg.rms_eps)
    q = linear(h, w.wq).reshape(n, hq, d)
    k = linear(h, w.wk).reshape(n, hkv, d)
    v = linear(h, w.wv).reshape(n, hkv, d)
    q = O.rope(rms_norm(q, w.g_q, cfg.rms_eps), pos, cfg.rope_theta)
    k = O.rope(rms_norm(k, w.g_k, cfg.rms_eps), pos, cfg.rope_theta)
    return q, O.bf16_round(k), O.bf16_round(v)


def layer_finish(x: np.ndarray, attn: np.ndarray, w: LayerWeights, cfg: StackConfig) -> np.ndarray:
    """Output projection + residual, then the SwiGLU MLP + residual."""
    n = x.shape[0]
    x = x + linear(attn.reshape(n, cfg.n_q_heads * cfg.head_dim), w.wo)
    h = rms_norm(x, w.g_ffn, cfg.rms_eps)
    return x + linear(silu(linear(h, w.wg)) * linear(h, w.wu), w.wd)


# --------------------------------------------------------------------------- Eq. 2 / Eq. 3


def full_prefill(x0: np.ndarray, layers: Sequence[LayerWeights], cfg: StackConfig, pos0: int = 0,
                 return_hidden: bool = False):
    """Eq. 2: all T rows x0[T, hidden] (embeddings) at positions pos0..pos0+T-1 through every
    layer with dense causal attention.  Returns (x_L, K[l], V[l]) with K/V [T, Hkv, d] bf16-rounded caches, and the
    list of layer inputs x_l if return_hidden."""
    t = x0.shape[0]
    pos = np.arange(pos0, pos0 + t)
    x, ks, vs, hid = np.asarray(x0, dtype=np.float64), [], [], []
    for w in layers:
        hid.append(x)
        q, k, v = layer_qkv(x, pos, w, cfg)
        a = O.recompute_attn(q, np.arange(t), k, v)          # row i sees cache rows j <= i
        x = layer_finish(x, a, w, cfg)
        ks.append(k)
        vs.append(v)
    return (x, ks, vs, hid) if return_hidden else (x, ks, vs)


def build_pic(chunk_x0: Sequence[np.ndarray], layers: Sequence[LayerWeights], cfg: StackConfig):
    """Eq. 3: KV_i^PIC = LLM(c_i), each chunk alone at chunk-local positions 0..|c_i|-1.
    Returns k_pic[l][i], v_pic[l][i]."""
    n_l = len(layers)
    k_pic: List[List[np.ndarray]] = [[] for _ in range(n_l)]
    v_pic: List[List[np.ndarray]] = [[] for _ in range(n_l)]
    for x0 in chunk_x0:
        _, ks, vs = full_prefill(x0, layers, cfg, 0)
        for l in range(n_l):
            k_pic[l].append(ks[l])
            v_pic[l].append(vs[l])
    return k_pic, v_pic


# --------------------------------------------------------------------------- stage 1: selective token localization


def probe_stage(xq0: np.ndarray, k_pic, v_pic, anchor_idx: np.ndarray, anchor_ptr: np.ndarray,
                layers: Sequence[LayerWeights], cfg: StackConfig, crit_layers: Sequence[int], ratio: float,
                return_hidden: bool = False) -> dict:
    """Fig. 9 stage 1 = Eq. 15-17 + Eq. 18/20 + Eq. 11.

    The user query U (embeddings xq0[Lq, hidden], positions N..N+Lq-1) runs through layers
    0..max(L*) with the stitched ANCHOR cache KV^A(C_A) (Eq. 16) as its prefix: every anchor keeps its original request
    position, all of them precede the query, so every query row sees every anchor plus the query rows up to itself.
    At l in L* the post-RoPE query states are tapped as Q_U^l(C_A) (Eq. 17) and scored against the stitched PIC keys of
    the ORIGINAL context positions of that layer (Eq. 18); the sum over L* (Eq. 20) feeds TopK (Eq. 11).
    crit_layers are 0-based layer indices.
    """
    lq = xq0.shape[0]
    n = int(sum(k.shape[0] for k in k_pic[0]))
    pos_u = np.arange(n, n + lq)
    x = np.asarray(xq0, dtype=np.float64)
    scores = np.zeros(n, dtype=np.float64)
    taps: Dict[int, np.ndarray] = {}
    hid = []
    for l in range(max(crit_layers) + 1):
        hid.append(x)
        w = layers[l]
        k_a, v_a, _pos_a = O.anchor_stitch(k_pic[l], v_pic[l], anchor_idx, anchor_ptr, cfg.rope_theta)
        q, k_u, v_u = layer_qkv(x, pos_u, w, cfg)
        n_a = k_a.shape[0]
        # compact cache [anchors ; query rows]: query row i sees compact rows j <= n_a + i
        a = O.recompute_attn(q, n_a + np.arange(lq), np.concatenate([k_a, k_u], 0), np.concatenate([v_a, v_u], 0))
        if l in crit_layers:
            taps[l] = q
            k_ctx, _ = O.reposition(k_pic[l], v_pic[l], cfg.rope_theta)
            scores += O.score(q, k_ctx)
        x = layer_finish(x, a, w, cfg)
    sel = O.select_topk(scores, O.n_select(n, ratio))
    out = {"scores": scores, "sel": sel, "q_probe": taps}
    if return_hidden:
        out["hidden"] = hid
    return out


# --------------------------------------------------------------------------- stage 2: pipeline cache fusion


def fuse_layer(x_rows: np.ndarray, rows: np.ndarray, n_sel: int, k_ctx: np.ndarray, v_ctx: np.ndarray,
               w: LayerWeights, cfg: StackConfig) -> dict:
    """One layer of Fig. 9 stage 2 for the rows R = P u U (rows[:n_sel] = P ascending, then the query positions).
    k_ctx / v_ctx [N, Hkv, d] are the stitched PIC entries of this layer (Eq. 4).  Refreshed K/V replace the PIC
    entries at P, the query's own K/V are appended (Eq. 7); every row attends causally over the fused cache
    (reading (k): all refreshed K/V depend only on the layer input, so scatter first, then attend)."""
    n = k_ctx.shape[0]
    q, k_new, v_new = layer_qkv(x_rows, rows, w, cfg)
    t = n + (len(rows) - n_sel)
    k_pos = np.zeros((t,) + k_new.shape[1:])
    v_pos = np.zeros((t,) + v_new.shape[1:])
    k_pos[rows], v_pos[rows] = k_new, v_new                   # fresh rows indexed by request position
    k_f, v_f = O.fuse(k_ctx, v_ctx, rows[:n_sel], k_pos, v_pos)
    a = O.recompute_attn(q, rows, k_f, v_f)
    return {"x": layer_finish(x_rows, a, w, cfg), "q": q, "k_new": k_new, "v_new": v_new, "attn": a,
            "k_fused": k_f, "v_fused": v_f}


def fuse_stage(x_rows0: np.ndarray, sel: np.ndarray, n_ctx: int, k_pic, v_pic, layers: Sequence[LayerWeights],
               cfg: StackConfig, return_hidden: bool = False):
    """Fig. 9 stage 2: x_rows0 = embeddings of rows R = P u U (layer-1 input, reading (l)); each
    layer starts from the loaded PIC entries (Eq. 4) and recomputes only R.  Returns the final hidden states of R."""
    sel = np.asarray(sel, dtype=np.int64)
    lq = x_rows0.shape[0] - len(sel)
    rows = np.concatenate([sel, np.arange(n_ctx, n_ctx + lq)])
    x, hid = np.asarray(x_rows0, dtype=np.float64), []
    for l, w in enumerate(layers):
        hid.append(x)
        k_ctx, v_ctx = O.reposition(k_pic[l], v_pic[l], cfg.rope_theta)
        x = fuse_layer(x, rows, len(sel), k_ctx, v_ctx, w, cfg)["x"]
    return (x, hid) if return_hidden else x


# --------------------------------------------------------------------------- first token (end of TTFT)


def first_token(x_last: np.ndarray, g_final: np.ndarray, w_lm: np.ndarray, eps: float):
    """The first generated token (TTFT) from the final hidden state of the last query row:
    logits = RMSNorm(x_last; g_final) W_lm^T, token = argmax (ties to the lower id).  Returns (token, logits)."""
    logits = linear(rms_norm(np.asarray(x_last, dtype=np.float64), g_final, eps), w_lm)
    return int(np.argmax(logits)), logits


# --------------------------------------------------------------------------- decoding over KV^Fuse


def decode_step(x_tok: np.ndarray, pos: int, k_cache: Sequence[np.ndarray], v_cache: Sequence[np.ndarray],
                layers: Sequence[LayerWeights], cfg: StackConfig):
    """One generated token through the stack: x_tok[hidden] is its embedding, `pos` its request
    position (= number of rows already in every layer's cache: N + Lq + tokens generated so far).  Per layer: project the
    single row at position pos, APPEND its bf16 K/V as cache row pos, attend causally over rows 0..pos of that layer's
    cache (KV^Fuse followed by earlier generated tokens), finish the block.  k_cache[l] / v_cache[l] are [pos, Hkv, d];
    returns (x_out[hidden], k_cache', v_cache') with caches of pos + 1 rows (new lists; inputs are not modified)."""
    x = np.asarray(x_tok, dtype=np.float64)[None, :]
    p = np.array([pos])
    k_out, v_out = [], []
    for l, w in enumerate(layers):
        assert k_cache[l].shape[0] == pos and v_cache[l].shape[0] == pos
        q, k_new, v_new = layer_qkv(x, p, w, cfg)
        k_l = np.concatenate([k_cache[l], k_new], 0)
        v_l = np.concatenate([v_cache[l], v_new], 0)
        a = O.recompute_attn(q, p, k_l, v_l)                  # the row at position pos sees cache rows j <= pos
        x = layer_finish(x, a, w, cfg)
        k_out.append(k_l)
        v_out.append(v_l)
    return x[0], k_out, v_out


def greedy_decode(first_tok: int, n_new: int, embed: np.ndarray, k_cache: Sequence[np.ndarray],
                  v_cache: Sequence[np.ndarray], layers: Sequence[LayerWeights], cfg: StackConfig, g_final: np.ndarray,
                  w_lm: np.ndarray):
    """Greedy generation after TTFT: `first_tok` is the token first_token() produced from the last query row; each step
    embeds the previous token, runs decode_step at the next position and takes argmax(RMSNorm(x) W_lm^T) (ties to the lower
    id).  Returns (tokens[n_new] generated AFTER first_tok, logits[n_new][vocab], k_cache, v_cache)."""
    toks, logs = [], []
    tok = int(first_tok)
    pos = k_cache[0].shape[0]
    for _ in range(n_new):
        x, k_cache, v_cache = decode_step(embed[tok], pos, k_cache, v_cache, layers, cfg)
        tok, lg = first_token(x, g_final, w_lm, cfg.rms_eps)
        toks.append(tok)
        logs.append(lg)
        pos += 1
    return np.asarray(toks, dtype=np.int64), np.asarray(logs), k_cache, v_cache
