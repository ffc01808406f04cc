"""fp64 CPU oracle for the QCFuse per-layer selective-recompute step.

TEST INFRASTRUCTURE — NOT A PRODUCT PATH.  Only `tests/`, `__graft_entry__.smoke()` and
`bench.py`'s `cpu_baseline` / `--impl reference` legs may import this module.  It shares no
code with the CUDA path (`paper_2606_05875_b200/`) and imports nothing from it.

Every function restates, step by step and in the paper's order and notation, what
/root/reference/PAPER.md defines (citations are PAPER.md line numbers + equation).  All
arithmetic is numpy float64; `numpy.matmul` / `numpy.exp` / `numpy.argsort` serve as library
steps.  No blocking, fusion or re-ordering beyond what the definitions state.  Where the paper
is silent the reading is the one listed in DESIGN.md ("Readings", letters (a)..(v)).

Pins (tests/test_oracle_pins.py, `-m "not gpu"`): closed-form RoPE composition, complex-number
restatement, relative-position invariance, softmax sums, torch fp64 SDPA for rho=1 / rho=0 /
single-chunk cases, brute-force top-k, hand-computed fixtures under tests/golden/, anchor counts and
brute-force Sink / Knorm rankings (Eq. 14).
Parity unpinned: none of the functions below; *selection quality versus the paper's
Recall@10% / F1 claims* is unpinned (needs the datasets and trained weights).

Conventions: tensors are float64 numpy arrays; caches are token-major [T, Hkv, d]; queries
[T, Hq, d]; q-head h reads kv-head g = h // (Hq // Hkv).
"""
from __future__ import annotations

from typing import List, Sequence, Tuple

import numpy as np

# --------------------------------------------------------------------------- bf16 rounding


def bf16_round(x: np.ndarray) -> np.ndarray:
    """Round float64 values to the nearest bf16 value (8 significant bits, ties-to-even).

    The fused cache is a bf16 object (BF16 serving stack; reading (t)).
    x = m * 2^e with m in [0.5, 1): keep 8 bits of m.  (bf16 subnormals do not occur here.)
    """
    x = np.asarray(x, dtype=np.float64)
    m, e = np.frexp(x)
    return np.ldexp(np.rint(m * 256.0) / 256.0, e)


def widen_bf16(bits: np.ndarray) -> np.ndarray:
    """bf16 bit patterns (uint16) -> float64 (exact)."""
    b = np.ascontiguousarray(bits, dtype=np.uint16)
    return (b.astype(np.uint32) << np.uint32(16)).view(np.float32).astype(np.float64)


# --------------------------------------------------------------------------- RoPE / Pi_i


def rope_angles(pos: np.ndarray, d: int, theta: float) -> np.ndarray:
    """phi[t, j] = pos_t * theta^(-2j/d), j in [0, d/2)  (reading (a))."""
    j = np.arange(d // 2, dtype=np.float64)
    inv_freq = np.power(np.float64(theta), -2.0 * j / np.float64(d))
    return np.asarray(pos, dtype=np.float64)[:, None] * inv_freq[None, :]


def rotate(x: np.ndarray, phi: np.ndarray) -> np.ndarray:
    """Rotate every half-split pair (x_j, x_{j+d/2}) of x[T, H, d] by phi[T, d/2]:
         out_j       = a cos(phi) - b sin(phi)
         out_{j+d/2} = b cos(phi) + a sin(phi)
    """
    d = x.shape[-1]
    a, b = x[..., : d // 2], x[..., d // 2:]
    c, s = np.cos(phi)[:, None, :], np.sin(phi)[:, None, :]
    return np.concatenate([a * c - b * s, b * c + a * s], axis=-1)


def rope(x: np.ndarray, pos: np.ndarray, theta: float) -> np.ndarray:
    """Plain RoPE of raw rows x[T, H, d] at positions pos[T]."""
    return rotate(x, rope_angles(pos, x.shape[-1], theta))


def reposition(k_pic: Sequence[np.ndarray], v_pic: Sequence[np.ndarray], theta: float,
               store_round: bool = True) -> Tuple[np.ndarray, np.ndarray]:
    """Eq. 4: KV^PIC(C) = [Pi_1(KV_1^PIC); ...; Pi_m(KV_m^PIC)].

    Chunk i sits at request offset off_i = sum_{j<i} |c_j|.  Its keys carry RoPE at chunk-local
    positions r = 0..|c_i|-1; Pi_i moves row r to request position off_i + r, i.e. rotates it by
    the angle of off_i (RoPE composes additively).  Values are stitched in the same token order.
    store_round=True rounds the re-positioned K to bf16 (reading (t)).
    Returns K'[N, Hkv, d], V'[N, Hkv, d].
    """
    ks, vs, off = [], [], 0
    for k_i, v_i in zip(k_pic, v_pic):
        ln, _, d = k_i.shape
        phi = rope_angles(np.full(ln, off, dtype=np.float64), d, theta)
        k_rot = rotate(np.asarray(k_i, dtype=np.float64), phi)
        ks.append(bf16_round(k_rot) if store_round else k_rot)
        vs.append(np.asarray(v_i, dtype=np.float64))
        off += ln
    return np.concatenate(ks, axis=0), np.concatenate(vs, axis=0)


def anchor_stitch(k_pic: Sequence[np.ndarray], v_pic: Sequence[np.ndarray],
                  anchor_idx: np.ndarray, anchor_ptr: np.ndarray, theta: float,
                  store_round: bool = True) -> Tuple[np.ndarray, np.ndarray, np.ndarray]:
    """Eq. 15-16: KV^A(C_A) = [Pi_1(KV_1^PIC[A_1]); ...].

    Only the anchor rows A_i of each chunk are kept, in order; each keeps its original request
    position off_i + a.  Returns K_A, V_A [|C_A|, Hkv, d] and pos[|C_A|].
    """
    ks, vs, ps, off = [], [], [], 0
    for i, (k_i, v_i) in enumerate(zip(k_pic, v_pic)):
        a = np.asarray(anchor_idx[anchor_ptr[i]: anchor_ptr[i + 1]], dtype=np.int64)
        ln, _, d = k_i.shape
        phi = rope_angles(np.full(len(a), off, dtype=np.float64), d, theta)
        k_rot = rotate(np.asarray(k_i, dtype=np.float64)[a], phi)
        ks.append(bf16_round(k_rot) if store_round else k_rot)
        vs.append(np.asarray(v_i, dtype=np.float64)[a])
        ps.append(off + a)
        off += ln
    return np.concatenate(ks, 0), np.concatenate(vs, 0), np.concatenate(ps, 0).astype(np.int64)


# --------------------------------------------------------------------------- Phase I: anchors (Eq. 14)


def n_anchor(chunk_len: int, r_a: float) -> int:
    """ceil(r_a |c_i|) (Eq. 14), evaluated in double with a 1e-6 guard against r_a * len landing a hair
    above an integer (0.1 * 512 = 51.2 -> 52; 0.25 * 64 = 16 exactly -> 16)."""
    return int(min(chunk_len, np.ceil(np.float64(r_a) * np.float64(chunk_len) - 1e-6)))


def anchor_scores(k_chunk: np.ndarray, rule: str) -> np.ndarray:
    """G_i(r) of Eq. 14 for the two key-statistics rules the paper names:
         'sink'  keeps tokens near the beginning of the chunk:  G(r) = -r
         'knorm' ranks positions by the norm of their key-cache rows.  The paper does not say which end is kept; the rule
                 it cites keeps LOW-norm keys, so G(r) = -||K_i[r]||_2 over all kv-heads and dims (reading (o')).
    k_chunk [len, Hkv, d] (one layer's PIC keys of the chunk; RoPE does not change the norm)."""
    ln = k_chunk.shape[0]
    if rule == "sink":
        return -np.arange(ln, dtype=np.float64)
    if rule == "knorm":
        return -np.sqrt(np.sum(np.square(np.asarray(k_chunk, dtype=np.float64).reshape(ln, -1)), axis=1))
    raise ValueError(rule)


def anchor_select(k_chunk: np.ndarray, r_a: float, rule: str) -> np.ndarray:
    """A_i = TopK(G_i, ceil(r_a |c_i|)) (Eq. 14), ties to the lower position, ascending chunk-local positions."""
    return select_topk(anchor_scores(k_chunk, rule), n_anchor(k_chunk.shape[0], r_a))


# --------------------------------------------------------------------------- score (Eq. 18, 20)


def softmax_rows(s: np.ndarray) -> np.ndarray:
    """p_t = exp(s_t - max_t s) / sum_t exp(s_t - max) along the last axis."""
    e = np.exp(s - s.max(axis=-1, keepdims=True))
    return e / e.sum(axis=-1, keepdims=True)


def score(q_probe: np.ndarray, k_ctx: np.ndarray, scale: float | None = None) -> np.ndarray:
    """Eq. 18 with Attn^l(.)_t as defined at PAPER.md:208:
    the user-query-to-context attention mass on context position t, aggregated over user-query
    tokens and heads.

      for q-head h (kv-head g = h // G), query token i:
          s_t = q[i, h] . K'[t, g] / sqrt(d)        t = 0..N-1 (context keys only, reading (c))
          p   = softmax_t(s)
          I(t) += p_t / (Hq * Lq)                   (mean, reading (b))

    q_probe [Lq, Hq, d], k_ctx [N, Hkv, d] (the stitched, re-positioned PIC keys, reading (e)).
    """
    lq, hq, d = q_probe.shape
    n, hkv, _ = k_ctx.shape
    g_sz = hq // hkv
    scale = 1.0 / np.sqrt(np.float64(d)) if scale is None else np.float64(scale)
    out = np.zeros(n, dtype=np.float64)
    for h in range(hq):
        g = h // g_sz
        s = (q_probe[:, h, :] @ k_ctx[:, g, :].T) * scale          # [Lq, N]
        out += softmax_rows(s).sum(axis=0)
    return out / np.float64(hq * lq)


def score_layers(q_probes: Sequence[np.ndarray], k_ctxs: Sequence[np.ndarray],
                 scale: float | None = None) -> np.ndarray:
    """Eq. 20: I_{L_k}(t) = sum_{l in L_k} Attn^l(Q_U^l(C_A), K_C^{PIC,l})_t."""
    total = np.zeros(k_ctxs[0].shape[0], dtype=np.float64)
    for q_l, k_l in zip(q_probes, k_ctxs):
        total += score(q_l, k_l, scale)
    return total


# --------------------------------------------------------------------------- top-k (Eq. 11)


def n_select(n_ctx: int, ratio: float) -> int:
    """|P| = floor(rho N) (Eq. 8), evaluated in double with a 1e-6 guard (reading (g))."""
    return int(np.floor(np.float64(ratio) * np.float64(n_ctx) + 1e-6))


def select_topk(scores: np.ndarray, k: int) -> np.ndarray:
    """Eq. 11: P = TopK(I(t), k) over all context positions (global, reading (i)).

    Order positions by (score descending, index ascending) — lower index wins ties (reading (h)) —
    take the first k, return them ascending.
    """
    s = np.asarray(scores)
    order = np.argsort(-s, kind="stable")        # stable: equal scores keep ascending index order
    return np.sort(order[:k]).astype(np.int64)


# --------------------------------------------------------------------------- fuse (Eq. 7) + attention


def fuse(k_ctx: np.ndarray, v_ctx: np.ndarray, sel: np.ndarray,
         k_new: np.ndarray, v_new: np.ndarray) -> Tuple[np.ndarray, np.ndarray]:
    """Eq. 7: KV^Fuse_p = KV^New_p if p in P else KV^PIC_p; the user query's own
    K/V are appended at positions N..N+Lq-1 (U is the online suffix).

    k_ctx/v_ctx [N, Hkv, d] from `reposition`; k_new/v_new [N+Lq, Hkv, d] indexed by request position.
    Returns K_f, V_f [N+Lq, Hkv, d].
    """
    n = k_ctx.shape[0]
    k_f = np.concatenate([k_ctx, k_new[n:]], axis=0).copy()
    v_f = np.concatenate([v_ctx, v_new[n:]], axis=0).copy()
    sel = np.asarray(sel, dtype=np.int64)
    k_f[sel] = k_new[sel]
    v_f[sel] = v_new[sel]
    return k_f, v_f


def recompute_attn(q_rows: np.ndarray, pos: np.ndarray, k_f: np.ndarray, v_f: np.ndarray,
                   scale: float | None = None, return_lse: bool = False):
    """each recomputed row at request position p reads prefix positions j <= p through
    the partially fused prefix cache (causal attention over K_f, V_f):

        o[r, h] = sum_{j <= p_r} softmax_j( q[r, h] . K_f[j, g] / sqrt(d) ) V_f[j, g]

    q_rows [n_R, Hq, d] with request positions pos[n_R]; all rows are independent given the fused
    cache (reading (k)).  Returns O [n_R, Hq, d] (float64, unrounded).
    """
    n_r, hq, d = q_rows.shape
    t, hkv, _ = k_f.shape
    g_sz = hq // hkv
    scale = 1.0 / np.sqrt(np.float64(d)) if scale is None else np.float64(scale)
    pos = np.asarray(pos, dtype=np.int64)
    out = np.zeros((n_r, hq, d), dtype=np.float64)
    lse = np.zeros((n_r, hq), dtype=np.float64)
    visible = np.arange(t)[None, :] <= pos[:, None]                  # [n_R, T]  j <= p
    for h in range(hq):
        g = h // g_sz
        s = (q_rows[:, h, :] @ k_f[:, g, :].T) * scale               # [n_R, T]
        s = np.where(visible, s, -np.inf)
        m = s.max(axis=-1, keepdims=True)
        e = np.exp(s - m)
        z = e.sum(axis=-1, keepdims=True)
        out[:, h, :] = (e / z) @ v_f[:, g, :]
        lse[:, h] = (m + np.log(z))[:, 0]
    return (out, lse) if return_lse else out


def full_prefill_attn(q: np.ndarray, k: np.ndarray, v: np.ndarray,
                      scale: float | None = None) -> np.ndarray:
    """Eq. 2 at one layer: dense causal GQA attention of all T rows over
    themselves — the rho = 1 reference."""
    return recompute_attn(q, np.arange(q.shape[0]), k, v, scale)


# --------------------------------------------------------------------------- the chained step


def layer_step(k_pic: Sequence[np.ndarray], v_pic: Sequence[np.ndarray], theta: float,
               q_probe: np.ndarray, ratio: float,
               q_new: np.ndarray, k_new: np.ndarray, v_new: np.ndarray,
               scale: float | None = None, sel: np.ndarray | None = None,
               prior_scores: np.ndarray | None = None) -> dict:
    """Fig. 9 / PAPER.md:337-344, one layer, one request:
       a1 reposition -> a2 score (critical layer) -> a3 top-k -> a4 fuse -> a5 recompute rows P u U.

    q_new/k_new/v_new are indexed by request position ([N+Lq, ...]).  If `sel` is given the
    selection stage is skipped (non-critical layer / teacher-forced parity).
    """
    k_ctx, v_ctx = reposition(k_pic, v_pic, theta)
    n = k_ctx.shape[0]
    lq = q_new.shape[0] - n
    out = {"k_ctx": k_ctx, "v_ctx": v_ctx}
    if sel is None:
        sc = score(q_probe, k_ctx, scale)
        if prior_scores is not None:
            sc = sc + prior_scores                                    # Eq. 20 running sum
        sel = select_topk(sc, n_select(n, ratio))
        out["scores"] = sc
    sel = np.asarray(sel, dtype=np.int64)
    k_f, v_f = fuse(k_ctx, v_ctx, sel, k_new, v_new)
    rows = np.concatenate([sel, np.arange(n, n + lq)])                # R = P u U, ascending
    o = recompute_attn(q_new[rows], rows, k_f, v_f, scale)
    out.update(sel=sel, rows=rows, k_fused=k_f, v_fused=v_f, out=o)
    return out
