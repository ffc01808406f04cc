"""Pins for oracle/qcf_stack_oracle.py (config 3): library routines, closed forms, invariants and special cases chosen
so that a dropped term, a wrong head mapping, a transposed weight or a mis-placed position fails one of them.
CPU only."""
import numpy as np
import pytest
import torch
import torch.nn.functional as F

from oracle import qcf_oracle as O
from oracle import qcf_stack_oracle as S
from paper_2606_05875_b200 import inputs


def _stack(name="s_small", n_layers=None):
    wl = inputs.make_stack_workload(name)
    sp = wl.spec
    cfg = S.StackConfig(n_layers or sp.n_layers, sp.hidden, sp.ffn, sp.n_q_heads, sp.n_kv_heads, sp.head_dim,
                        sp.rope_theta, sp.rms_eps)
    layers = [S.LayerWeights(**{k: O.widen_bf16(v) for k, v in lw.items()}) for lw in wl.layers[: cfg.n_layers]]
    emb = O.widen_bf16(wl.embed)
    return wl, cfg, layers, emb


def _small_request(wl, emb, n_chunks=3, chunk_len=24, lq=5):
    chunks = [emb[t[:chunk_len]] for t in wl.chunk_tokens[:n_chunks]]
    xq = emb[wl.query_tokens[:lq]]
    return chunks, xq


# ------------------------------------------------------------------------------------------- dense ops vs torch fp64

def test_dense_ops_match_torch_library_routines():
    rng = np.random.default_rng(0)
    x = rng.standard_normal((7, 48))
    g = 1 + 0.1 * rng.standard_normal(48)
    w = rng.standard_normal((20, 48))
    tx, tg, tw = map(torch.from_numpy, (x, g, w))
    np.testing.assert_allclose(S.rms_norm(x, g, 1e-6), F.rms_norm(tx, (48,), tg, 1e-6).numpy(), rtol=1e-13)
    np.testing.assert_allclose(S.linear(x, w), F.linear(tx, tw).numpy(), rtol=1e-12, atol=1e-13)
    np.testing.assert_allclose(S.silu(x), F.silu(tx).numpy(), rtol=1e-13)
    # eps matters for tiny rows, and the gain multiplies AFTER the normalisation
    tiny = np.full((1, 4), 1e-4)
    np.testing.assert_allclose(S.rms_norm(tiny, np.ones(4), 1e-6), tiny / np.sqrt(1e-8 + 1e-6), rtol=1e-12)


def test_layer_matches_torch_composition():
    """One decoder layer, dense causal: q/k/v head split, GQA head mapping, QK-norm before RoPE, residuals — against a
    composition of torch fp64 library routines (rms_norm, linear, SDPA with enable_gqa, silu)."""
    wl, cfg, layers, emb = _stack("s_small", 1)
    w = layers[0]
    x0 = emb[wl.chunk_tokens[0][:40]]
    x1, ks, vs = S.full_prefill(x0, layers, cfg)
    t = torch.from_numpy
    hq, hkv, d, n = cfg.n_q_heads, cfg.n_kv_heads, cfg.head_dim, 40
    h = F.rms_norm(t(x0), (cfg.hidden,), t(w.g_attn), cfg.rms_eps)
    q = F.rms_norm(F.linear(h, t(w.wq)).view(n, hq, d), (d,), t(w.g_q), cfg.rms_eps)
    k = F.rms_norm(F.linear(h, t(w.wk)).view(n, hkv, d), (d,), t(w.g_k), cfg.rms_eps)
    v = F.linear(h, t(w.wv)).view(n, hkv, d)
    # rotary in complex form (half-split pairs), independent of the oracle's rotate()
    inv = cfg.rope_theta ** (-2.0 * torch.arange(d // 2, dtype=torch.float64) / d)
    ang = torch.arange(n, dtype=torch.float64)[:, None] * inv[None, :]
    rot = torch.polar(torch.ones_like(ang), ang)[:, None, :]

    def rope(z):
        c = torch.complex(z[..., : d // 2], z[..., d // 2:]) * rot
        return torch.cat([c.real, c.imag], -1)

    q, k = rope(q), rope(k)
    k = t(O.bf16_round(k.numpy()))
    v = t(O.bf16_round(v.numpy()))
    np.testing.assert_array_equal(ks[0], k.numpy())
    np.testing.assert_array_equal(vs[0], v.numpy())
    a = F.scaled_dot_product_attention(q.transpose(0, 1)[None], k.transpose(0, 1)[None], v.transpose(0, 1)[None],
                                       is_causal=True, enable_gqa=True)[0].transpose(0, 1).reshape(n, hq * d)
    x = t(x0) + F.linear(a, t(w.wo))
    h2 = F.rms_norm(x, (cfg.hidden,), t(w.g_ffn), cfg.rms_eps)
    x = x + F.linear(F.silu(F.linear(h2, t(w.wg))) * F.linear(h2, t(w.wu)), t(w.wd))
    np.testing.assert_allclose(x1, x.numpy(), rtol=1e-9, atol=1e-11)


def test_zero_projections_special_cases():
    wl, cfg, layers, emb = _stack("s_small", 1)
    w = layers[0]
    x0 = emb[wl.chunk_tokens[1][:16]]
    import dataclasses
    w0 = dataclasses.replace(w, wo=np.zeros_like(w.wo), wd=np.zeros_like(w.wd))
    np.testing.assert_array_equal(S.full_prefill(x0, [w0], cfg)[0], x0)           # both residual branches vanish
    wg0 = dataclasses.replace(w, wg=np.zeros_like(w.wg))                           # silu(0) = 0: MLP branch vanishes
    wd0 = dataclasses.replace(w, wd=np.zeros_like(w.wd))
    np.testing.assert_allclose(S.full_prefill(x0, [wg0], cfg)[0], S.full_prefill(x0, [wd0], cfg)[0], rtol=0, atol=1e-15)
    # one row alone: softmax over a single key = 1, so attention returns v of that row
    q, k, v = S.layer_qkv(x0[:1], np.array([0]), w, cfg)
    a = O.recompute_attn(q, np.array([0]), k, v)
    g = cfg.n_q_heads // cfg.n_kv_heads
    np.testing.assert_allclose(a[0], np.repeat(v[0], g, axis=0), rtol=1e-14)


# ------------------------------------------------------------------------------------------- invariants

def test_causality_of_full_prefill():
    wl, cfg, layers, emb = _stack("s_small", 2)
    x0 = emb[wl.chunk_tokens[0][:32]].copy()
    a, ka, _ = S.full_prefill(x0, layers, cfg)
    x0[20] += 1.0
    b, kb, _ = S.full_prefill(x0, layers, cfg)
    np.testing.assert_array_equal(a[:20], b[:20])
    np.testing.assert_array_equal(ka[1][:20], kb[1][:20])
    assert np.abs(a[20:] - b[20:]).max() > 1e-3


def test_position_shift_ties_stack_rope_to_eq4():
    """Attention depends on relative positions only: prefill at positions D.. gives the same hidden states and V, and
    K caches that are the unshifted ones moved by Pi(D) (Eq. 4) — up to the bf16 rounding of K."""
    wl, cfg, layers, emb = _stack("s_small", 2)
    x0 = emb[wl.chunk_tokens[2][:24]]
    a, ka, va = S.full_prefill(x0, layers, cfg, 0)
    # the check needs unrounded caches on both sides: compare q.k logits instead of rounded K
    D = 777
    b, kb, vb = S.full_prefill(x0, layers, cfg, D)
    np.testing.assert_array_equal(va[0], vb[0])                                   # layer-0 V does not see positions
    half = cfg.head_dim // 2
    phi = O.rope_angles(np.full(24, D, dtype=np.float64), cfg.head_dim, cfg.rope_theta)
    for l in range(2):
        k_moved = O.rotate(ka[l], phi)
        # layer 0: both caches round the same real vector in two rotated frames, so they differ by at most one bf16
        # rounding of each frame, which is bounded by 2^-8 of the PAIR's norm (a rotation mixes the two elements);
        # layer 1 additionally sees the (tiny) difference of its inputs
        pair = np.hypot(k_moved[..., :half], k_moved[..., half:])
        bound = (2.0 ** -8) * np.concatenate([pair, pair], -1) * (2.0 if l == 0 else 6.0) + 1e-12
        assert np.all(np.abs(kb[l] - k_moved) <= bound)
    # hidden states agree to the level the bf16 cache rounding allows (rounding happens in rotated frames)
    assert np.max(np.abs(a - b)) < 5e-2 * max(1.0, np.abs(a).max())


# ------------------------------------------------------------------------------------------- fusion special cases

def test_single_chunk_fused_equals_full_prefill_every_layer():
    wl, cfg, layers, emb = _stack("s_small")
    chunks, xq = _small_request(wl, emb, n_chunks=1, chunk_len=40, lq=6)
    k_pic, v_pic = S.build_pic(chunks, layers, cfg)
    x_all = np.concatenate(chunks + [xq], 0)
    ref, _, _, hid = S.full_prefill(x_all, layers, cfg, return_hidden=True)
    sel = np.array([0, 3, 4, 17, 39])
    rows = np.concatenate([sel, np.arange(40, 46)])
    got, ghid = S.fuse_stage(x_all[rows], sel, 40, k_pic, v_pic, layers, cfg, return_hidden=True)
    for l in range(cfg.n_layers):
        np.testing.assert_allclose(ghid[l], hid[l][rows], rtol=1e-9, atol=1e-10)
    np.testing.assert_allclose(got, ref[rows], rtol=1e-9, atol=1e-10)


def test_rho1_multi_chunk_equals_full_prefill():
    wl, cfg, layers, emb = _stack("s_small")
    chunks, xq = _small_request(wl, emb)
    k_pic, v_pic = S.build_pic(chunks, layers, cfg)
    n = sum(c.shape[0] for c in chunks)
    x_all = np.concatenate(chunks + [xq], 0)
    ref, kf, vf = S.full_prefill(x_all, layers, cfg)
    got = S.fuse_stage(x_all, np.arange(n), n, k_pic, v_pic, layers, cfg)
    np.testing.assert_allclose(got, ref, rtol=1e-9, atol=1e-10)
    # and the PIC caches were irrelevant: garbage PIC gives the same result
    junk = [[np.full_like(k, 3.0) for k in kl] for kl in k_pic]
    np.testing.assert_allclose(S.fuse_stage(x_all, np.arange(n), n, junk, junk, layers, cfg), ref, rtol=1e-9, atol=1e-10)


def test_rho0_equals_probe_with_every_token_an_anchor():
    """Direct reuse (Eq. 5): the query over the stitched PIC cache.  The probe path (anchor_stitch) with A_i = all
    positions and the fuse path (reposition) with P = {} are two separate code paths for the same function."""
    wl, cfg, layers, emb = _stack("s_small")
    chunks, xq = _small_request(wl, emb)
    k_pic, v_pic = S.build_pic(chunks, layers, cfg)
    lens = [c.shape[0] for c in chunks]
    n = sum(lens)
    a_idx = np.concatenate([np.arange(ln) for ln in lens]).astype(np.int32)
    a_ptr = np.concatenate([[0], np.cumsum(lens)]).astype(np.int32)
    crit = [cfg.n_layers - 1]
    pr = S.probe_stage(xq, k_pic, v_pic, a_idx, a_ptr, layers, cfg, crit, 0.3, return_hidden=True)
    _, hid = S.fuse_stage(xq, np.empty(0, np.int64), n, k_pic, v_pic, layers, cfg, return_hidden=True)
    for l in range(cfg.n_layers):
        np.testing.assert_allclose(pr["hidden"][l], hid[l], rtol=1e-9, atol=1e-10)
    assert abs(pr["scores"].sum() - len(crit)) < 1e-9                              # Eq. 20: |L*| unit masses
    assert len(pr["sel"]) == O.n_select(n, 0.3)


def test_probe_uses_only_anchor_rows_and_original_positions():
    wl, cfg, layers, emb = _stack("s_small")
    chunks, xq = _small_request(wl, emb)
    k_pic, v_pic = S.build_pic(chunks, layers, cfg)
    a_idx = np.array([0, 1, 5, 0, 2, 23, 1, 7, 8], dtype=np.int32)
    a_ptr = np.array([0, 3, 6, 9], dtype=np.int32)
    crit = [1, 2]
    base = S.probe_stage(xq, k_pic, v_pic, a_idx, a_ptr, layers, cfg, crit, 0.25)
    # perturbing a NON-anchor PIC row of a non-critical layer (layer 0 here) changes nothing
    import copy
    kp = copy.deepcopy(k_pic); vp = copy.deepcopy(v_pic)
    kp[0][1][10] += 1.0; vp[0][1][10] += 1.0
    same = S.probe_stage(xq, kp, vp, a_idx, a_ptr, layers, cfg, crit, 0.25)
    np.testing.assert_array_equal(base["scores"], same["scores"])
    # perturbing an anchor row does
    kp[0][1][2] += 1.0
    diff = S.probe_stage(xq, kp, vp, a_idx, a_ptr, layers, cfg, crit, 0.25)
    assert np.abs(diff["scores"] - base["scores"]).max() > 0
    # the tapped query states sit at positions N..N+Lq-1: undo RoPE there and the per-head RMS is that of a QK-normed
    # vector (sqrt(mean(g_q^2 * xhat^2)) with unit-RMS xhat) — checks the tap is post-norm, post-RoPE
    n = sum(c.shape[0] for c in chunks)
    q = base["q_probe"][1]
    phi = O.rope_angles(np.arange(n, n + q.shape[0]), cfg.head_dim, cfg.rope_theta)
    q0 = O.rotate(q, -phi)
    xhat = q0 / layers[1].g_q
    np.testing.assert_allclose(np.sqrt(np.mean(xhat ** 2, -1)), 1.0, rtol=1e-4)


def test_first_token_matches_torch_and_argmax_ties():
    rng = np.random.default_rng(8)
    x = rng.standard_normal(48); g = 1 + 0.1 * rng.standard_normal(48); w = rng.standard_normal((33, 48))
    tok, logits = S.first_token(x, g, w, 1e-6)
    t = torch.from_numpy
    want = F.linear(F.rms_norm(t(x), (48,), t(g), 1e-6), t(w)).numpy()
    np.testing.assert_allclose(logits, want, rtol=1e-12, atol=1e-13)
    assert tok == int(np.argmax(want))
    w2 = w.copy(); w2[7] = w2[tok]                      # an exact tie: the lower id wins
    assert S.first_token(x, g, w2, 1e-6)[0] == min(7, tok)


# ------------------------------------------------------------------------------------------- decoding over KV^Fuse

def test_decode_step_equals_last_row_of_a_longer_full_prefill():
    """decode_step on the caches of a T-token prefill is, by the causal structure of Eq. 2, the (T+1)-th row of a
    (T+1)-token prefill: same hidden state, same appended K/V at row T, in every layer.  A wrong position, a cache row
    dropped or double-counted, or attention that does not include the token's own K/V fails this."""
    wl, cfg, layers, emb = _stack("s_small")
    toks = np.concatenate(wl.chunk_tokens)[:37]
    x_long, ks_long, vs_long = S.full_prefill(emb[toks], layers, cfg)
    _, ks, vs = S.full_prefill(emb[toks[:-1]], layers, cfg)
    x, k2, v2 = S.decode_step(emb[toks[-1]], len(toks) - 1, ks, vs, layers, cfg)
    np.testing.assert_allclose(x, x_long[-1], rtol=1e-9, atol=1e-11)
    for l in range(cfg.n_layers):
        assert k2[l].shape[0] == len(toks)
        np.testing.assert_array_equal(k2[l][:-1], ks[l])           # existing rows untouched
        np.testing.assert_allclose(k2[l], ks_long[l], rtol=0, atol=1e-12 + 2.0 ** -8 * 1e-6)
        np.testing.assert_allclose(v2[l], vs_long[l], rtol=0, atol=1e-12 + 2.0 ** -8 * 1e-6)
    # the inputs were not modified
    assert ks[0].shape[0] == len(toks) - 1


def test_decode_attention_is_single_row_sdpa():
    """The attention inside decode_step: one query row over [cache ; own K/V] == torch fp64 SDPA (no mask needed: the row
    is the last one), with GQA head mapping."""
    wl, cfg, layers, emb = _stack("s_small", 1)
    w = layers[0]
    toks = np.concatenate(wl.chunk_tokens)[:21]
    _, ks, vs = S.full_prefill(emb[toks[:-1]], layers, cfg)
    x_tok = emb[toks[-1]]
    pos = len(toks) - 1
    q, k_new, v_new = S.layer_qkv(x_tok[None], np.array([pos]), w, cfg)
    t = torch.from_numpy
    k_l, v_l = np.concatenate([ks[0], k_new]), np.concatenate([vs[0], v_new])
    a = F.scaled_dot_product_attention(t(q).transpose(0, 1)[None], t(k_l).transpose(0, 1)[None], t(v_l).transpose(0, 1)[None],
                                       enable_gqa=True)[0].transpose(0, 1).numpy()
    want = S.layer_finish(x_tok[None], a, w, cfg)[0]
    got, _, _ = S.decode_step(x_tok, pos, ks, vs, layers, cfg)
    np.testing.assert_allclose(got, want, rtol=1e-10, atol=1e-12)


def test_greedy_decode_equals_brute_force_reprefill():
    """greedy_decode == the definition of greedy generation written the slow way: re-run the full prefill on the whole
    growing sequence and take argmax of the last row's logits, token by token."""
    wl, cfg, layers, emb = _stack("s_small")
    rng = np.random.default_rng(4)
    g_final = 1 + 0.1 * rng.standard_normal(cfg.hidden)
    w_lm = rng.standard_normal((wl.spec.vocab, cfg.hidden)) * 0.05
    prompt = list(np.concatenate(wl.chunk_tokens)[:19])
    x, ks, vs = S.full_prefill(emb[prompt], layers, cfg)
    first, _ = S.first_token(x[-1], g_final, w_lm, cfg.rms_eps)
    toks, logs, k2, _ = S.greedy_decode(first, 5, emb, ks, vs, layers, cfg, g_final, w_lm)
    seq = prompt + [first]
    for i in range(5):
        xs, _, _ = S.full_prefill(emb[seq], layers, cfg)
        tok, lg = S.first_token(xs[-1], g_final, w_lm, cfg.rms_eps)
        np.testing.assert_allclose(logs[i], lg, rtol=1e-8, atol=1e-10)
        assert tok == toks[i]
        seq.append(tok)
    assert k2[0].shape[0] == len(prompt) + 5
