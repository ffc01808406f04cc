"""Seeded synthetic workloads for the QCFuse layer step.

This module only *synthesises inputs*: bf16 bit patterns for per-chunk PIC caches, probe
queries and fresh Q/K/V rows, chunk tables, anchor lists.  It holds none of the method's
arithmetic (no re-positioning, scoring, top-k or attention) and is imported by tests and
bench.py only — neither `oracle/` nor the CUDA binding imports it.

The positional encoding applied here (`_encode_positions`) is the *offline model's* RoPE that
a PIC cache carries when it arrives ("key cache is encoded at chunk-local
positions starting from zero"); it is written as a complex multiplication, independently of
both the oracle's and the kernel's rotation code.

They stand in for the paper's workloads (Qwen3-8B-class GQA layers, 512/1024-token chunks,
rho in 0.1..0.5): the datasets and weights are not in the container.
"""
from __future__ import annotations

from dataclasses import dataclass, field, replace
from typing import Dict, List, Optional, Tuple

import numpy as np

# --------------------------------------------------------------------------- bf16 bit helpers


def f32_to_bf16_bits(x: np.ndarray) -> np.ndarray:
    """float32 -> bf16 bit pattern (uint16), round-to-nearest-even."""
    x = np.ascontiguousarray(x, dtype=np.float32)
    u = x.view(np.uint32)
    lsb = (u >> np.uint32(16)) & np.uint32(1)
    r = u + np.uint32(0x7FFF) + lsb
    return (r >> np.uint32(16)).astype(np.uint16)


def bf16_bits_to_f32(b: np.ndarray) -> np.ndarray:
    b = np.ascontiguousarray(b, dtype=np.uint16)
    return (b.astype(np.uint32) << np.uint32(16)).view(np.float32)


def bf16_bits_to_f64(b: np.ndarray) -> np.ndarray:
    return bf16_bits_to_f32(b).astype(np.float64)


# --------------------------------------------------------------------------- configs


@dataclass(frozen=True)
class LayerConfig:
    """One BASELINE.json config of the single-layer step."""

    name: str
    seed: int
    batch: int
    n_chunks: int          # m, per request
    chunk_len: int         # tokens per chunk
    n_query: int           # Lq
    n_q_heads: int         # Hq
    n_kv_heads: int        # Hkv
    head_dim: int          # d
    rope_theta: float
    ratio: float           # rho
    pool_chunks: int = 0   # >0: chunks are drawn from a shared pool of this many caches (config 4)
    heavy_frac: float = 0.0    # fraction of tokens whose keys are scaled (config 5)
    heavy_scale: float = 1.0
    ragged: bool = False       # chunk lengths vary (edge-case configs used by tests)

    @property
    def n_ctx(self) -> int:
        return self.n_chunks * self.chunk_len


CONFIGS: Dict[str, LayerConfig] = {
    # BASELINE.json configs[0]
    "c1": LayerConfig("c1", 1001, 1, 2, 64, 16, 4, 2, 64, 1e6, 0.3),
    # configs[1] — the bench workload
    "c2": LayerConfig("c2", 1002, 1, 10, 512, 64, 32, 8, 128, 1e6, 0.3),
    # configs[3] — batched serving, ratio swept by the caller
    "c4": LayerConfig("c4", 1004, 16, 8, 1024, 128, 32, 8, 128, 1e6, 0.3, pool_chunks=256),
    # configs[4] — long context, heavy hitters
    "c5": LayerConfig("c5", 1005, 1, 32, 1024, 128, 64, 8, 128, 1e6, 0.15,
                      heavy_frac=0.05, heavy_scale=4.0),
    # reduced shapes for fast parity runs (several tiles + ragged tails)
    "t_ragged": LayerConfig("t_ragged", 2001, 1, 5, 0, 19, 8, 2, 128, 1e6, 0.3, ragged=True),
    "t_ragged64": LayerConfig("t_ragged64", 2002, 1, 3, 0, 7, 4, 2, 64, 1e4, 0.37, ragged=True),
    "t_batch": LayerConfig("t_batch", 2003, 3, 4, 96, 24, 8, 2, 128, 1e6, 0.3, pool_chunks=9),
    "t_g8": LayerConfig("t_g8", 2004, 1, 4, 160, 40, 16, 2, 128, 1e6, 0.15,
                        heavy_frac=0.05, heavy_scale=4.0),
    "t_mid": LayerConfig("t_mid", 2005, 1, 4, 256, 32, 32, 8, 128, 1e6, 0.3),
}

_RAGGED_LENS = {
    "t_ragged": [131, 64, 1, 257, 77],
    "t_ragged64": [33, 5, 90],
}


@dataclass
class Request:
    """One RAG request C=[c_1..c_m] + U: per-chunk PIC caches and fresh rows."""

    chunk_ids: List[int]                 # index into Workload.pool_k / pool_v
    chunk_len: np.ndarray                # int32 [m]
    n_ctx: int                           # N
    n_query: int                         # Lq
    q_probe: np.ndarray                  # uint16 [Lq, Hq, d]  bf16 bits, positions N..N+Lq-1
    q_new: np.ndarray                    # uint16 [N+Lq, Hq, d]  rows indexed by request position
    k_new: np.ndarray                    # uint16 [N+Lq, Hkv, d]
    v_new: np.ndarray                    # uint16 [N+Lq, Hkv, d]
    anchor_idx: np.ndarray               # int32, chunk-local anchor positions, CSR values
    anchor_ptr: np.ndarray               # int32 [m+1]


@dataclass
class Workload:
    cfg: LayerConfig
    pool_k: List[np.ndarray] = field(default_factory=list)   # each uint16 [len, Hkv, d]
    pool_v: List[np.ndarray] = field(default_factory=list)
    requests: List[Request] = field(default_factory=list)


def shard_heads(wl: Workload, rank: int, world: int) -> Workload:
    """The slice of `wl` a rank of a KV-head-sharded step holds: kv-heads
    [rank*Hkv/world, (rank+1)*Hkv/world) of every cache and the q heads that read them.  Slicing only."""
    cfg = wl.cfg
    if cfg.n_kv_heads % world:
        raise ValueError("Hkv = %d is not divisible by %d shards" % (cfg.n_kv_heads, world))
    per = cfg.n_kv_heads // world
    g = cfg.n_q_heads // cfg.n_kv_heads
    kv = slice(rank * per, (rank + 1) * per)
    qh = slice(rank * per * g, (rank + 1) * per * g)
    cut = lambda x, sl: np.ascontiguousarray(x[:, sl])
    out = Workload(replace(cfg, n_q_heads=per * g, n_kv_heads=per))
    out.pool_k = [cut(k, kv) for k in wl.pool_k]
    out.pool_v = [cut(v, kv) for v in wl.pool_v]
    for r in wl.requests:
        out.requests.append(Request(r.chunk_ids, r.chunk_len, r.n_ctx, r.n_query, cut(r.q_probe, qh), cut(r.q_new, qh),
                                    cut(r.k_new, kv), cut(r.v_new, kv), r.anchor_idx, r.anchor_ptr))
    return out


# --------------------------------------------------------------------------- synthesis


def _encode_positions(x: np.ndarray, pos: np.ndarray, theta: float) -> np.ndarray:
    """Offline-model RoPE on raw rows x[T, H, d] at integer positions pos[T] (fp64, complex form).

    Pair (j, j+d/2) is read as the complex number x_j + i*x_{j+d/2} and multiplied by
    exp(i * pos * theta^(-2j/d)) — the half-split ("rotate_half") convention, reading (a).
    """
    t, h, d = x.shape
    half = d // 2
    inv_freq = np.float64(theta) ** (-2.0 * np.arange(half, dtype=np.float64) / d)
    ang = pos.astype(np.float64)[:, None] * inv_freq[None, :]            # [T, half]
    z = x[..., :half].astype(np.float64) + 1j * x[..., half:].astype(np.float64)
    z = z * np.exp(1j * ang)[:, None, :]
    out = np.empty((t, h, d), dtype=np.float32)
    out[..., :half] = z.real
    out[..., half:] = z.imag
    return out


def _normal_bf16(rng: np.random.Generator, shape) -> np.ndarray:
    return rng.standard_normal(shape, dtype=np.float32)


def _anchors_for_chunk(rng: np.random.Generator, length: int, r_a: float) -> np.ndarray:
    """DESIGN.md reading (o): first 4 positions (sink-style) + seeded random others, ascending."""
    n_a = int(np.ceil(r_a * length))
    n_a = min(max(n_a, 0), length)
    head = np.arange(min(4, n_a), dtype=np.int64)
    rest_pool = np.arange(len(head), length, dtype=np.int64)
    rest = rng.choice(rest_pool, size=n_a - len(head), replace=False) if n_a > len(head) else \
        np.empty(0, dtype=np.int64)
    return np.sort(np.concatenate([head, rest])).astype(np.int32)


def make_workload(name: str, *, ratio: Optional[float] = None, batch: Optional[int] = None,
                  r_a: float = 0.1) -> Workload:
    """Build the seeded workload of config `name` (see CONFIGS)."""
    cfg = CONFIGS[name]
    if ratio is not None or batch is not None:
        cfg = LayerConfig(**{**cfg.__dict__,
                             "ratio": cfg.ratio if ratio is None else ratio,
                             "batch": cfg.batch if batch is None else batch})
    ss = np.random.SeedSequence(cfg.seed)
    (s_kraw, s_vpic, s_qp, s_qn, s_kn, s_vn, s_heavy, s_draw, s_anchor) = ss.spawn(9)
    rng_k, rng_v = np.random.default_rng(s_kraw), np.random.default_rng(s_vpic)
    rng_qp, rng_qn = np.random.default_rng(s_qp), np.random.default_rng(s_qn)
    rng_kn, rng_vn = np.random.default_rng(s_kn), np.random.default_rng(s_vn)
    rng_heavy, rng_draw = np.random.default_rng(s_heavy), np.random.default_rng(s_draw)
    rng_anchor = np.random.default_rng(s_anchor)

    hq, hkv, d, theta = cfg.n_q_heads, cfg.n_kv_heads, cfg.head_dim, cfg.rope_theta
    wl = Workload(cfg)

    # ---- chunk pool: PIC caches at chunk-local positions 0..len-1
    if cfg.ragged:
        lens = list(_RAGGED_LENS[cfg.name])
        n_pool = len(lens)
    else:
        n_pool = cfg.pool_chunks if cfg.pool_chunks > 0 else cfg.n_chunks * cfg.batch
        lens = [cfg.chunk_len] * n_pool
    heavy_masks = []
    for ln in lens:
        k_raw = _normal_bf16(rng_k, (ln, hkv, d))
        heavy = rng_heavy.random(ln) < cfg.heavy_frac if cfg.heavy_frac > 0 else np.zeros(ln, bool)
        if cfg.heavy_frac > 0:
            k_raw[heavy] *= np.float32(cfg.heavy_scale)
        heavy_masks.append(heavy)
        k_pic = _encode_positions(k_raw, np.arange(ln), theta)
        wl.pool_k.append(f32_to_bf16_bits(k_pic))
        wl.pool_v.append(f32_to_bf16_bits(_normal_bf16(rng_v, (ln, hkv, d))))

    # ---- requests
    for b in range(cfg.batch):
        if cfg.ragged:
            ids = list(range(n_pool))
        elif cfg.pool_chunks > 0:
            # without replacement inside a request, independently across requests (reading (u))
            ids = [int(i) for i in rng_draw.choice(n_pool, size=cfg.n_chunks, replace=False)]
        else:
            ids = list(range(b * cfg.n_chunks, (b + 1) * cfg.n_chunks))
        clen = np.array([lens[i] for i in ids], dtype=np.int32)
        n_ctx = int(clen.sum())
        lq = cfg.n_query
        pos_all = np.arange(n_ctx + lq)
        q_probe = _encode_positions(_normal_bf16(rng_qp, (lq, hq, d)), pos_all[n_ctx:], theta)
        q_new = _encode_positions(_normal_bf16(rng_qn, (n_ctx + lq, hq, d)), pos_all, theta)
        k_new_raw = _normal_bf16(rng_kn, (n_ctx + lq, hkv, d))
        if cfg.heavy_frac > 0:   # the fresh keys of heavy tokens are heavy too
            hv = np.concatenate([heavy_masks[i] for i in ids] + [np.zeros(lq, bool)])
            k_new_raw[hv] *= np.float32(cfg.heavy_scale)
        k_new = _encode_positions(k_new_raw, pos_all, theta)
        v_new = _normal_bf16(rng_vn, (n_ctx + lq, hkv, d))
        a_list = [_anchors_for_chunk(rng_anchor, int(ln), r_a) for ln in clen]
        a_ptr = np.zeros(len(ids) + 1, dtype=np.int32)
        a_ptr[1:] = np.cumsum([len(a) for a in a_list])
        wl.requests.append(Request(
            chunk_ids=ids, chunk_len=clen, n_ctx=n_ctx, n_query=lq,
            q_probe=f32_to_bf16_bits(q_probe), q_new=f32_to_bf16_bits(q_new),
            k_new=f32_to_bf16_bits(k_new), v_new=f32_to_bf16_bits(v_new),
            anchor_idx=np.concatenate(a_list).astype(np.int32) if a_list else np.empty(0, np.int32),
            anchor_ptr=a_ptr))
    return wl


# --------------------------------------------------------------------------- config 3: full-stack workload


@dataclass(frozen=True)
class StackSpec:
    """BASELINE.json configs[2] ("c3") and its reduced test shapes: a Qwen3-shaped decoder stack with random-init
    weights plus one multi-chunk request.  No arithmetic of the method lives here: only seeded tensors."""

    name: str
    seed: int
    n_layers: int
    hidden: int
    ffn: int
    vocab: int
    n_q_heads: int
    n_kv_heads: int
    head_dim: int
    rope_theta: float
    n_chunks: int
    chunk_len: int
    n_query: int
    ratio: float
    crit_layers: Tuple[int, ...]      # 0-based layer indices of L* (reading (p): the three middle layers)
    r_a: float = 0.1                  # anchor retained ratio
    rms_eps: float = 1e-6

    @property
    def n_ctx(self) -> int:
        return self.n_chunks * self.chunk_len


STACKS: Dict[str, StackSpec] = {
    # configs[2]: 36 layers, hidden 4096, FFN 12288, GQA 32/8, d 128; 20 x 512 context + 64-token query; L* = {17,18,19} (1-based)
    "c3": StackSpec("c3", 1003, 36, 4096, 12288, 32768, 32, 8, 128, 1e6, 20, 512, 64, 0.3, (16, 17, 18)),
    # free-running parity stack: 4 layers, hidden 512, FFN 1536, 8/2 heads, d 64, 4 x 128 tokens
    "s_small": StackSpec("s_small", 3001, 4, 512, 1536, 1024, 8, 2, 64, 1e6, 4, 128, 16, 0.3, (1, 2)),
    # d = 128 variant with ragged GEMM tails (hidden 384 = 1.5 K-blocks of 256, n_R not a multiple of 128)
    "s_d128": StackSpec("s_d128", 3002, 3, 384, 1152, 512, 8, 2, 128, 1e6, 3, 160, 24, 0.35, (0, 2)),
    # one c3-shaped layer slice for teacher-forced full-width checks: real widths, 2 layers, short context
    "s_wide": StackSpec("s_wide", 3003, 2, 4096, 12288, 2048, 32, 8, 128, 1e6, 3, 256, 32, 0.3, (0, 1)),
}

_W_NAMES = ("wq", "wk", "wv", "wo", "wg", "wu", "wd")


@dataclass
class StackWorkload:
    spec: StackSpec
    embed: np.ndarray                            # uint16 [vocab, hidden]  bf16 bits, N(0, 1)
    layers: List[Dict[str, np.ndarray]]          # per layer: wq.. wd uint16 [out, in] (N(0, 0.02^2)); g_* uint16 gains
    chunk_tokens: List[np.ndarray]               # int32 [chunk_len] each
    query_tokens: np.ndarray                     # int32 [Lq]
    anchor_idx: np.ndarray                       # int32 CSR values (chunk-local anchor positions, ascending)
    anchor_ptr: np.ndarray                       # int32 [m+1]


def make_stack_workload(name: str, *, ratio: Optional[float] = None, with_weights: bool = True,
                        n_layers: Optional[int] = None) -> StackWorkload:
    """Seeded stack + request.  Weights ~ N(0, 0.02^2), embeddings ~ N(0, 1), norm gains 1 + 0.1 N(0, 1) (so that a
    dropped gain is visible to the parity tests), all rounded to bf16 (both the oracle and the library read these
    bit patterns); token ids uniform over the synthetic vocabulary; anchors as in make_workload (reading (o))."""
    sp = STACKS[name]
    if ratio is not None:
        sp = StackSpec(**{**sp.__dict__, "ratio": ratio})
    if n_layers is not None:          # the first n_layers layers of the same seeded stack (full-size single-layer tests)
        sp = StackSpec(**{**sp.__dict__, "n_layers": n_layers,
                          "crit_layers": tuple(c for c in sp.crit_layers if c < n_layers) or (0,)})
    ss = np.random.SeedSequence(sp.seed)
    s_emb, s_w, s_tok, s_anchor = ss.spawn(4)
    rng_e, rng_w = np.random.default_rng(s_emb), np.random.default_rng(s_w)
    rng_t, rng_a = np.random.default_rng(s_tok), np.random.default_rng(s_anchor)
    hq, hkv, d, hid, ffn = sp.n_q_heads, sp.n_kv_heads, sp.head_dim, sp.hidden, sp.ffn
    shapes = {"wq": (hq * d, hid), "wk": (hkv * d, hid), "wv": (hkv * d, hid), "wo": (hid, hq * d),
              "wg": (ffn, hid), "wu": (ffn, hid), "wd": (hid, ffn)}
    # with_weights=False: tokens and anchors only (c3's 13.9 GB of weights are drawn on the device by the bench)
    embed = f32_to_bf16_bits(rng_e.standard_normal((sp.vocab, hid), dtype=np.float32)) if with_weights else None
    layers = []
    for _ in range(sp.n_layers if with_weights else 0):
        lw = {n: f32_to_bf16_bits(rng_w.standard_normal(shapes[n], dtype=np.float32) * np.float32(0.02))
              for n in _W_NAMES}
        for n, sz in (("g_attn", hid), ("g_ffn", hid), ("g_q", d), ("g_k", d)):
            lw[n] = f32_to_bf16_bits(np.float32(1.0) + np.float32(0.1) * rng_w.standard_normal(sz, dtype=np.float32))
        layers.append(lw)
    chunk_tokens = [rng_t.integers(0, sp.vocab, size=sp.chunk_len, dtype=np.int32) for _ in range(sp.n_chunks)]
    query_tokens = rng_t.integers(0, sp.vocab, size=sp.n_query, dtype=np.int32)
    a_list = [_anchors_for_chunk(rng_a, sp.chunk_len, sp.r_a) for _ in range(sp.n_chunks)]
    a_ptr = np.zeros(sp.n_chunks + 1, dtype=np.int32)
    a_ptr[1:] = np.cumsum([len(a) for a in a_list])
    return StackWorkload(sp, embed, layers, chunk_tokens, query_tokens,
                         np.concatenate(a_list).astype(np.int32), a_ptr)
