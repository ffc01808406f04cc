"""Pins for the fp64 oracle: what the paper and the mathematics fix (no GPU, no CUDA path).

Each test is chosen so that a plausible mistake in oracle/qcf_oracle.py (dropped term, wrong sign or
index, transposed operand, wrong head mapping, off-by-one in the causal limit) fails at least one.
Citations are PAPER.md line numbers.
"""
import os

import numpy as np
import pytest
import torch

from oracle import qcf_oracle as O

GOLDEN = os.path.join(os.path.dirname(__file__), "golden")


def _load(name):
    rows = []
    with open(os.path.join(GOLDEN, name)) as f:
        for line in f:
            line = line.strip()
            if line and not line.startswith("#"):
                rows.append(np.array([float(x) for x in line.split()]))
    return rows


def _rng(seed):
    return np.random.default_rng(seed)


# ------------------------------------------------------------------ bf16 rounding

def test_bf16_round_matches_torch_rne():
    x = _rng(0).standard_normal(20000) * np.array([1e-3, 1.0, 37.0, 1e4])[_rng(1).integers(0, 4, 20000)]
    x32 = x.astype(np.float32).astype(np.float64)     # exactly-fp32 inputs: torch's fp32->bf16 RNE applies
    want = torch.from_numpy(x32.astype(np.float32)).to(torch.bfloat16).to(torch.float64).numpy()
    assert np.array_equal(O.bf16_round(x32), want)


def test_bf16_round_ties_to_even_and_widen():
    # 1 + 2^-8 is exactly half-way between bf16 neighbours 1.0 and 1 + 2^-7 -> even mantissa -> 1.0
    assert O.bf16_round(np.array([1.0 + 2.0 ** -8]))[0] == 1.0
    assert O.bf16_round(np.array([1.0 + 3 * 2.0 ** -8]))[0] == 1.0 + 2.0 ** -6
    assert O.widen_bf16(np.array([0x3F80, 0xC000, 0x0000], dtype=np.uint16)).tolist() == [1.0, -2.0, 0.0]


# ------------------------------------------------------------------ a1: reposition (Eq. 4)

def test_reposition_golden_unit_angle():
    rows = _load("rope_unit_angle.txt")
    k1 = np.array([5., 6., 7., 8.]).reshape(1, 1, 4)
    k2 = np.array([1., 2., 3., 4.]).reshape(1, 1, 4)
    v1, v2 = k1 * 10, k2 * 10
    k, v = O.reposition([k1, k2], [v1, v2], theta=10000.0, store_round=False)
    np.testing.assert_allclose(k[0, 0], rows[0], rtol=0, atol=1e-14)
    np.testing.assert_allclose(k[1, 0], rows[1], rtol=0, atol=1e-14)
    assert np.array_equal(v[:, 0, :], np.array([[50., 60., 70., 80.], [10., 20., 30., 40.]]))


@pytest.mark.parametrize("d,theta", [(64, 1e6), (128, 1e6), (8, 1e4)])
def test_reposition_closed_form_equals_rope_at_global_position(d, theta):
    """north star: re-positioning a cached K equals recomputing K at the global position."""
    r = _rng(3)
    lens = [5, 1, 17, 64]
    raw = [r.standard_normal((ln, 2, d)) for ln in lens]
    pic = [O.rope(x, np.arange(len(x)), theta) for x in raw]               # local positions 0..len-1
    vs = [r.standard_normal((ln, 2, d)) for ln in lens]
    k, v = O.reposition(pic, vs, theta, store_round=False)
    want = O.rope(np.concatenate(raw), np.arange(sum(lens)), theta)         # global positions
    np.testing.assert_allclose(k, want, rtol=0, atol=1e-10)
    assert np.array_equal(v, np.concatenate(vs))
    # rounded variant: within one bf16 ulp (2^-8 relative) of the exact value
    kr, _ = O.reposition(pic, vs, theta, store_round=True)
    assert np.all(np.abs(kr - want) <= np.abs(want) * 2.0 ** -8 + 1e-30)
    assert np.array_equal(kr, O.bf16_round(kr))


def test_reposition_complex_restatement_and_norms():
    """Independent formulation: pair (x_j, x_{j+d/2}) as a complex number times exp(i*off*w_j)."""
    r = _rng(4)
    d, theta, lens = 16, 1e6, [3, 4, 2]
    pic = [r.standard_normal((ln, 3, d)) for ln in lens]
    k, _ = O.reposition(pic, pic, theta, store_round=False)
    off = 0
    w = theta ** (-2.0 * np.arange(d // 2) / d)
    for p in pic:
        z = (p[..., : d // 2] + 1j * p[..., d // 2:]) * np.exp(1j * off * w)
        got = k[off: off + len(p)]
        np.testing.assert_allclose(got[..., : d // 2], z.real, atol=1e-12)
        np.testing.assert_allclose(got[..., d // 2:], z.imag, atol=1e-12)
        # per-pair norm preserved
        np.testing.assert_allclose(got[..., : d // 2] ** 2 + got[..., d // 2:] ** 2, np.abs(z) ** 2, atol=1e-12)
        off += len(p)
    # off = 0 is the identity, bit for bit
    k0, _ = O.reposition(pic[:1], pic[:1], theta, store_round=False)
    assert np.array_equal(k0, pic[0])


def test_logits_depend_only_on_relative_position():
    """q at p, k at j: q.k depends only on p-j (the property Pi_i relies on)."""
    r = _rng(5)
    d, theta = 32, 1e6
    q_raw, k_raw = r.standard_normal((1, 1, d)), r.standard_normal((1, 1, d))
    base = (O.rope(q_raw, np.array([40]), theta) * O.rope(k_raw, np.array([7]), theta)).sum()
    for shift in (1, 100, 5000):
        s = (O.rope(q_raw, np.array([40 + shift]), theta) * O.rope(k_raw, np.array([7 + shift]), theta)).sum()
        assert abs(s - base) < 1e-9


def test_anchor_stitch_is_row_subset_of_reposition():
    """Eq. 15-16: anchors are rows of the stitched cache with original positions."""
    r = _rng(6)
    lens, d = [6, 9, 4], 8
    pic = [r.standard_normal((ln, 2, d)) for ln in lens]
    vs = [r.standard_normal((ln, 2, d)) for ln in lens]
    a_idx = np.array([0, 2, 5, 1, 8, 3], dtype=np.int32)
    a_ptr = np.array([0, 3, 5, 6], dtype=np.int32)
    ka, va, pos = O.anchor_stitch(pic, vs, a_idx, a_ptr, 1e4)
    k, v = O.reposition(pic, vs, 1e4)
    assert pos.tolist() == [0, 2, 5, 6 + 1, 6 + 8, 15 + 3]
    assert np.array_equal(ka, k[pos]) and np.array_equal(va, v[pos])


# ------------------------------------------------------------------ a2: score (Eq. 18 / 20)

def test_score_golden_log_keys():
    rows = _load("softmax_log_keys.txt")
    k = np.zeros((3, 1, 4)); k[:, 0, 0] = np.log([1., 2., 3.])
    q = np.zeros((1, 1, 4)); q[0, 0, 0] = 2.0
    np.testing.assert_allclose(O.score(q, k), rows[0], atol=1e-15)


def test_score_invariants():
    r = _rng(7)
    lq, hq, hkv, d, n = 5, 6, 2, 16, 37
    q, k = r.standard_normal((lq, hq, d)), r.standard_normal((n, hkv, d))
    s = O.score(q, k)
    assert abs(s.sum() - 1.0) < 1e-12 and np.all(s > 0)                  # reading (b): mean => sums to 1
    # identical keys => uniform
    ku = np.repeat(k[:1], n, axis=0)
    np.testing.assert_allclose(O.score(q, ku), np.full(n, 1.0 / n), atol=1e-14)
    # one key aligned with every query direction with a huge logit => its score -> 1
    kh = k.copy() * 1e-3
    kh[11] = 50.0 * np.stack([q[:, :3].mean((0, 1)), q[:, 3:].mean((0, 1))])   # arbitrary big key
    qh = np.abs(q) * np.sign(kh[11].repeat(3, axis=0))[None]                  # all logits positive & large
    assert O.score(qh, kh)[11] > 0.999
    # permuting context rows permutes scores
    perm = r.permutation(n)
    np.testing.assert_allclose(O.score(q, k[perm]), s[perm], atol=1e-15)
    # Eq. 20: plain sum over layers
    q2, k2 = r.standard_normal((lq, hq, d)), r.standard_normal((n, hkv, d))
    np.testing.assert_allclose(O.score_layers([q, q2], [k, k2]), s + O.score(q2, k2), atol=1e-15)


def test_score_equals_torch_softmax_column_mean_and_head_mapping():
    """Library pin: column mean of torch fp64 softmax(QK^T/sqrt d) with kv heads repeat_interleaved
    (q-head h -> kv-head h // G).  A transposed operand or h % Hkv mapping fails this."""
    r = _rng(8)
    lq, hq, hkv, d, n = 4, 8, 2, 32, 50
    q, k = r.standard_normal((lq, hq, d)), r.standard_normal((n, hkv, d))
    tq = torch.from_numpy(q).permute(1, 0, 2)                             # [Hq, Lq, d]
    tk = torch.from_numpy(k).permute(1, 0, 2).repeat_interleave(hq // hkv, dim=0)   # [Hq, N, d]
    p = torch.softmax(tq @ tk.transpose(1, 2) / d ** 0.5, dim=-1)         # [Hq, Lq, N]
    np.testing.assert_allclose(O.score(q, k), p.mean(dim=(0, 1)).numpy(), atol=1e-14)


# ------------------------------------------------------------------ a3: top-k (Eq. 11)

def test_n_select_pins():
    """floor(rho N) for every BASELINE config (38, 1536, 3072, 819/2457/4096, 4915)."""
    assert [O.n_select(128, .3), O.n_select(5120, .3), O.n_select(10240, .3)] == [38, 1536, 3072]
    assert [O.n_select(8192, x) for x in (.1, .3, .5)] == [819, 2457, 4096]
    assert O.n_select(32768, .15) == 4915
    assert O.n_select(10, 0.0) == 0 and O.n_select(10, 1.0) == 10


def test_topk_golden_ties():
    sc, k, want = _load("topk_ties.txt")
    assert O.select_topk(sc, int(k[0])).tolist() == [int(x) for x in want]


def test_topk_brute_force():
    r = _rng(9)
    for n in (1, 2, 7, 33, 200):
        s = np.round(r.standard_normal(n), 1)            # coarse => many ties
        for k in {0, 1, n // 3, n - 1 if n > 1 else 0, n}:
            brute = sorted(sorted(range(n), key=lambda i: (-s[i], i))[:k])
            assert O.select_topk(s, k).tolist() == brute
    assert O.select_topk(np.array([3., 1., 2.]), 0).size == 0
    assert O.select_topk(np.array([3., 1., 2.]), 3).tolist() == [0, 1, 2]


# ------------------------------------------------------------------ a4 + a5: fuse + recompute attention

def _sdpa(q, k, v, mask=None, causal=False):
    """torch CPU fp64 SDPA with GQA; q [T,Hq,d], k/v [S,Hkv,d] -> [T,Hq,d]."""
    tq = torch.from_numpy(q).permute(1, 0, 2)[None]
    tk = torch.from_numpy(k).permute(1, 0, 2)[None]
    tv = torch.from_numpy(v).permute(1, 0, 2)[None]
    o = torch.nn.functional.scaled_dot_product_attention(
        tq, tk, tv, attn_mask=mask, is_causal=causal, enable_gqa=True)
    return o[0].permute(1, 0, 2).numpy()


def _case(seed, lens=(7, 12, 5), lq=4, hq=6, hkv=2, d=16, theta=1e6):
    r = _rng(seed)
    pic_k = [r.standard_normal((ln, hkv, d)) for ln in lens]
    pic_v = [r.standard_normal((ln, hkv, d)) for ln in lens]
    n = sum(lens)
    q_new = r.standard_normal((n + lq, hq, d))
    k_new = r.standard_normal((n + lq, hkv, d))
    v_new = r.standard_normal((n + lq, hkv, d))
    q_probe = r.standard_normal((lq, hq, d))
    return pic_k, pic_v, q_probe, q_new, k_new, v_new, n, lq, theta


def test_attention_golden_log_keys():
    rows = _load("softmax_log_keys.txt")
    k = np.zeros((3, 1, 4)); k[:, 0, 0] = np.log([1., 2., 3.])
    v = np.array([[t + 1, 10 * (t + 1), 0, -1] for t in range(3)], dtype=np.float64).reshape(3, 1, 4)
    q = np.zeros((2, 1, 4)); q[:, 0, 0] = 2.0
    o = O.recompute_attn(q, np.array([2, 1]), k, v)
    np.testing.assert_allclose(o[0, 0], rows[1], atol=1e-14)
    np.testing.assert_allclose(o[1, 0], rows[2], atol=1e-14)


def test_rho1_reproduces_full_prefill_sdpa():
    """north star: r=1 reproduces full-prefill attention (PIC content irrelevant)."""
    pk, pv, qp, qn, kn, vn, n, lq, th = _case(10)
    res = O.layer_step(pk, pv, th, qp, 1.0, qn, kn, vn)
    assert res["sel"].tolist() == list(range(n))
    want = _sdpa(qn, kn, vn, causal=True)
    np.testing.assert_allclose(res["out"], want, atol=1e-12)
    np.testing.assert_allclose(O.full_prefill_attn(qn, kn, vn), want, atol=1e-12)
    assert np.array_equal(res["k_fused"], kn) and np.array_equal(res["v_fused"], vn)


def test_rho0_reproduces_direct_reuse():
    """north star: r=0 reproduces direct reuse: query rows over [K'; K_U] (Eq. 5 endpoint)."""
    pk, pv, qp, qn, kn, vn, n, lq, th = _case(11)
    res = O.layer_step(pk, pv, th, qp, 0.0, qn, kn, vn)
    assert res["sel"].size == 0 and res["rows"].tolist() == list(range(n, n + lq))
    kc, vc = O.reposition(pk, pv, th)
    kf, vf = np.concatenate([kc, kn[n:]]), np.concatenate([vc, vn[n:]])
    assert np.array_equal(res["k_fused"], kf) and np.array_equal(res["v_fused"], vf)
    mask = torch.ones(lq, n + lq, dtype=torch.bool)
    mask[:, n:] = torch.tril(torch.ones(lq, lq, dtype=torch.bool))
    np.testing.assert_allclose(res["out"], _sdpa(qn[n:], kf, vf, mask=mask), atol=1e-12)


@pytest.mark.parametrize("ratio", [0.0, 0.3, 0.55, 1.0])
def test_single_chunk_fused_equals_full_prefill(ratio):
    """north star: a single-chunk prompt fused equals full prefill: with one chunk at offset 0 the PIC
    entries ARE the full-prefill entries, so any rho gives the full-prefill rows."""
    r = _rng(12)
    n, lq, hq, hkv, d = 23, 3, 4, 2, 8
    qn, kn, vn = r.standard_normal((n + lq, hq, d)), r.standard_normal((n + lq, hkv, d)), \
        r.standard_normal((n + lq, hkv, d))
    kn[:n] = O.bf16_round(kn[:n])        # so that the bf16 store of K' is exact and fresh == PIC holds
    res = O.layer_step([kn[:n]], [vn[:n]], 1e6, r.standard_normal((lq, hq, d)), ratio, qn, kn, vn)
    full = _sdpa(qn, kn, vn, causal=True)
    np.testing.assert_allclose(res["out"], full[res["rows"]], atol=1e-12)


def test_mixed_rows_sdpa_with_explicit_mask_and_fuse_rule():
    """General rho: rows P u U over the fused cache == SDPA with mask j <= p on the same cache; the
    fused cache differs from the stitched PIC only at P (Eq. 7)."""
    pk, pv, qp, qn, kn, vn, n, lq, th = _case(13)
    res = O.layer_step(pk, pv, th, qp, 0.4, qn, kn, vn)
    sel, rows = res["sel"], res["rows"]
    assert len(sel) == O.n_select(n, 0.4) and np.all(np.diff(rows) > 0)
    kc, vc = O.reposition(pk, pv, th)
    changed = np.where(np.any(res["k_fused"][:n] != kc, axis=(1, 2)))[0]
    assert set(changed) <= set(sel.tolist())
    assert np.array_equal(res["k_fused"][sel], kn[sel]) and np.array_equal(res["v_fused"][sel], vn[sel])
    unsel = np.setdiff1d(np.arange(n), sel)
    assert np.array_equal(res["k_fused"][unsel], kc[unsel]) and np.array_equal(res["v_fused"][unsel], vc[unsel])
    mask = torch.from_numpy(np.arange(n + lq)[None, :] <= rows[:, None])
    np.testing.assert_allclose(res["out"], _sdpa(qn[rows], res["k_fused"], res["v_fused"], mask=mask), atol=1e-12)
    # top-k really is the top of the oracle's own scores
    sc = res["scores"]
    assert sc[sel].min() >= np.delete(sc, sel).max()


def test_future_rows_do_not_influence_a_row_and_lse():
    pk, pv, qp, qn, kn, vn, n, lq, th = _case(14)
    res = O.layer_step(pk, pv, th, qp, 0.3, qn, kn, vn)
    kf, vf, rows = res["k_fused"].copy(), res["v_fused"].copy(), res["rows"]
    r0 = 2
    p = rows[r0]
    kf[p + 1:] += 100.0
    vf[p + 1:] -= 55.0
    o2, lse = O.recompute_attn(qn[rows], rows, kf, vf, return_lse=True)
    np.testing.assert_allclose(o2[r0], res["out"][r0], atol=1e-13)
    # lse is the log of the softmax denominator: exp(s - lse) sums to 1 over the visible prefix
    s = (qn[rows[r0], 0] @ kf[: p + 1, 0].T) / np.sqrt(qn.shape[-1])
    assert abs(np.exp(s - lse[r0, 0]).sum() - 1.0) < 1e-12


# ----------------------------------------------------------------------------------------------- Phase I anchors (Eq. 14)

def test_anchor_count_is_ceil_eq14():
    # 20 chunks x ceil(0.1 * 512) = 1040 anchor rows; exact products are not bumped
    assert O.n_anchor(512, 0.1) == 52 and 20 * O.n_anchor(512, 0.1) == 1040
    assert O.n_anchor(64, 0.25) == 16 and O.n_anchor(10, 0.1) == 1 and O.n_anchor(7, 1.0) == 7 and O.n_anchor(5, 0.0) == 0
    assert O.n_anchor(131, 0.1) == 14


def test_anchor_rules_sink_and_knorm():
    rng = np.random.default_rng(4)
    k = rng.standard_normal((97, 2, 16))
    # sink: the first ceil(r_a len) positions
    assert np.array_equal(O.anchor_select(k, 0.1, "sink"), np.arange(10))
    # knorm: brute force over explicit norms (lowest norms kept), ascending output
    norms = np.array([np.linalg.norm(k[r]) for r in range(97)])
    want = np.sort(np.argsort(norms, kind="stable")[:10])
    assert np.array_equal(O.anchor_select(k, 0.1, "knorm"), want)
    # shrinking one row's key makes it an anchor; the norm ignores a rotation of the pairs (RoPE-invariant)
    k2 = k.copy(); k2[50] *= 1e-3
    assert 50 in O.anchor_select(k2, 0.1, "knorm")
    phi = O.rope_angles(np.arange(97) + 1234, 16, 1e4)
    assert np.array_equal(O.anchor_select(O.rotate(k, phi), 0.1, "knorm"), want)
    # ties go to the lower position
    k3 = np.ones((8, 1, 4))
    assert np.array_equal(O.anchor_select(k3, 0.5, "knorm"), np.arange(4))
