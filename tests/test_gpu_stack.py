"""GPU parity for config 3 (a1', a7, a8 and the two-stage pipeline) through the C ABI, against
oracle/qcf_stack_oracle.py on the same seeded bf16 weights and tokens.

Tolerances: values the GPU stores in bf16 after fp32 arithmetic on IDENTICAL inputs are within
max(2e-2, 1 bf16 ulp) of the fp64 oracle (north_star's 2e-2 for attention outputs and K/V, widened to one ulp where
|value| >= 4 makes a single ulp larger than 2e-2).  Hidden states that went through further bf16-rounded activations
(free-running) are compared relative to the row RMS, bound stated at each assert.
"""
import numpy as np
import pytest
import torch

from oracle import qcf_oracle as O
from oracle import qcf_stack_oracle as S
from paper_2606_05875_b200 import inputs

pytestmark = pytest.mark.gpu

# Free-running stage 1: stated bound on the relative score error after the probe went through bf16
# activations, and the selection overlap it allows on the reduced stacks (measured values are printed by the tests)
FREE_RUNNING_EPS = 1e-2          # measured 0.8e-3 .. 2.3e-3 on the reduced stacks: the north-star score bound holds
FREE_RUNNING_OVERLAP = 0.99      # measured 100 %
# free-running logits after every layer ran on bf16 activations: bound relative to the largest logit (measured values are
# printed by the test and recorded in DESIGN.md §5)
DECODE_LOGIT_TOL = 1e-2       # measured 1.2e-2 .. 2.2e-2 absolute on logits up to 5 (0.4 % of the largest logit)



def _bits(t):
    return t.detach().cpu().contiguous().view(torch.int16).numpy().view(np.uint16)


def _f64(t):
    return O.widen_bf16(_bits(t))


def _dev(bits):
    return torch.from_numpy(np.ascontiguousarray(bits).view(np.int16)).view(torch.bfloat16).cuda()


def _ulp(x):
    return np.ldexp(1.0, np.frexp(np.abs(x))[1] - 8)


def _close_bf16(got, want, extra=0.0):
    """|got - want| <= max(2e-2, 1 ulp_bf16(want)) (+ extra)."""
    return np.all(np.abs(got - want) <= np.maximum(2e-2, _ulp(want)) + extra)


def _binding():
    from paper_2606_05875_b200 import binding
    return binding


def _device_layers(wl):
    """Pack the seeded weights the way qcf_layer_weights wants them (layout plumbing only)."""
    out = []
    for lw in wl.layers:
        gu = np.empty((2 * lw["wg"].shape[0], lw["wg"].shape[1]), dtype=np.uint16)
        gu[0::2], gu[1::2] = lw["wg"], lw["wu"]
        out.append({"w_qkv": _dev(np.concatenate([lw["wq"], lw["wk"], lw["wv"]], 0)), "w_o": _dev(lw["wo"]),
                    "w_gate_up": _dev(gu), "w_down": _dev(lw["wd"]), "g_attn": _dev(lw["g_attn"]),
                    "g_ffn": _dev(lw["g_ffn"]), "g_q": _dev(lw["g_q"]), "g_k": _dev(lw["g_k"])})
    return out


def _oracle_stack(wl, n_layers=None):
    sp = wl.spec
    cfg = S.StackConfig(n_layers or sp.n_layers, sp.hidden, sp.ffn, sp.n_q_heads, sp.n_kv_heads, sp.head_dim,
                        sp.rope_theta, sp.rms_eps)
    layers = [S.LayerWeights(**{k: O.widen_bf16(v) for k, v in lw.items()}) for lw in wl.layers[: cfg.n_layers]]
    return cfg, layers


def _make(name, max_rows=None, extra_pos=0):
    binding = _binding()
    wl = inputs.make_stack_workload(name)
    sp = wl.spec
    t = sp.n_ctx + sp.n_query
    ctx = binding.Context(sp.n_q_heads, sp.n_kv_heads, sp.head_dim, sp.rope_theta, 1, max(sp.n_ctx, 1024), sp.n_query)
    dl = _device_layers(wl)
    emb = _dev(wl.embed)
    stack = binding.Stack(ctx, sp.n_layers, sp.hidden, sp.ffn, sp.vocab, sp.rms_eps, dl, emb, max_rows or t, t + extra_pos,
                          max_pool_rows=sp.n_ctx)
    return wl, ctx, stack


# ----------------------------------------------------------------------------------------------- qcf_linear

@pytest.mark.parametrize("mt", [0, 1, 2])
@pytest.mark.parametrize("M,N,K", [(200, 768, 512), (131, 1536, 384), (1, 512, 1536), (300, 264, 64), (515, 1032, 4096)])
def test_linear_store_and_residual(M, N, K, mt):
    binding = _binding()
    ctx = binding.Context(8, 2, 64, 1e6, 1, 1024, 8)
    ctx.qcf_debug_set(binding.QCF_DEBUG_GEMM_MT, mt)      # force the tile height the heuristic picks at other sizes
    rng = np.random.default_rng(M * 7 + N)
    a = inputs.f32_to_bf16_bits(rng.standard_normal((M, K), dtype=np.float32))
    w = inputs.f32_to_bf16_bits(rng.standard_normal((N, K), dtype=np.float32) * np.float32(K ** -0.5))
    r = inputs.f32_to_bf16_bits(rng.standard_normal((M, N), dtype=np.float32))
    exact = O.widen_bf16(a) @ O.widen_bf16(w).T
    da, dw = _dev(a), _dev(w)
    c = torch.full((M + 1, N), 7.0, dtype=torch.bfloat16, device="cuda")
    ctx.qcf_linear(da, dw, None, c, M, N, K, binding.QCF_EPI_STORE)
    torch.cuda.synchronize()
    got = _f64(c[:M])
    # one bf16 rounding of an fp32-accumulated sum: half an ulp + fp32 accumulation slack
    assert np.all(np.abs(got - exact) <= 0.5 * _ulp(exact) + 2e-5 * np.sqrt(K))
    assert torch.all(c[M] == 7.0), "rows past M are untouched"
    x = _dev(r)
    ctx.qcf_linear(da, dw, x, x, M, N, K, binding.QCF_EPI_ADD_RESIDUAL)          # in place
    torch.cuda.synchronize()
    want = O.widen_bf16(r) + exact
    assert np.all(np.abs(_f64(x) - want) <= 0.5 * _ulp(want) + 2e-5 * np.sqrt(K))


@pytest.mark.parametrize("M", [300, 1])
@pytest.mark.parametrize("mt", [0, 1, 2])
def test_linear_swiglu(mt, M):
    """M = 1 with the default heuristic takes the decode GEMV (a weight stream), any forced tile height the MMA kernel."""
    binding = _binding()
    ctx = binding.Context(8, 2, 64, 1e6, 1, 1024, 8)
    ctx.qcf_debug_set(binding.QCF_DEBUG_GEMM_MT, mt)
    F, K = 1160, 384
    rng = np.random.default_rng(9)
    a = inputs.f32_to_bf16_bits(rng.standard_normal((M, K), dtype=np.float32))
    wg = inputs.f32_to_bf16_bits(rng.standard_normal((F, K), dtype=np.float32) * np.float32(0.1))
    wu = inputs.f32_to_bf16_bits(rng.standard_normal((F, K), dtype=np.float32) * np.float32(0.1))
    gu = np.empty((2 * F, K), dtype=np.uint16)
    gu[0::2], gu[1::2] = wg, wu
    c = torch.zeros((M, F), dtype=torch.bfloat16, device="cuda")
    ctx.qcf_linear(_dev(a), _dev(gu), None, c, M, 2 * F, K, binding.QCF_EPI_SWIGLU)
    torch.cuda.synchronize()
    A = O.widen_bf16(a)
    want = S.silu(A @ O.widen_bf16(wg).T) * (A @ O.widen_bf16(wu).T)
    assert np.all(np.abs(_f64(c) - want) <= 0.5 * _ulp(want) + 1e-4 * (1 + np.abs(want)))


@pytest.mark.parametrize("M,N,K", [(1, 528, 1536), (64, 4096, 512), (100, 6160, 200), (128, 9472, 1536)])
def test_linear_skinny_tiles(M, N, K):
    """M <= 128 takes the 128 x 32 / 128 x 64 tile variants (32-wide while N / 32 <= the SM count) with a per-tile
    rotated K order; every epilogue, N and K tails."""
    binding = _binding()
    ctx = binding.Context(8, 2, 64, 1e6, 1, 1024, 8)
    rng = np.random.default_rng(M * 11 + N)
    a = inputs.f32_to_bf16_bits(rng.standard_normal((M, K), dtype=np.float32))
    w = inputs.f32_to_bf16_bits(rng.standard_normal((N, K), dtype=np.float32) * np.float32(K ** -0.5))
    r = inputs.f32_to_bf16_bits(rng.standard_normal((M, N), dtype=np.float32))
    A, W = O.widen_bf16(a), O.widen_bf16(w)
    exact = A @ W.T
    da, dw = _dev(a), _dev(w)
    c = torch.full((M + 1, N), 7.0, dtype=torch.bfloat16, device="cuda")
    ctx.qcf_linear(da, dw, None, c, M, N, K, binding.QCF_EPI_STORE)
    x = _dev(r)
    ctx.qcf_linear(da, dw, x, x, M, N, K, binding.QCF_EPI_ADD_RESIDUAL)
    g = torch.zeros((M, N // 2), dtype=torch.bfloat16, device="cuda")
    ctx.qcf_linear(da, dw, None, g, M, N, K, binding.QCF_EPI_SWIGLU)             # rows 2j / 2j+1 of w as (gate_j, up_j)
    torch.cuda.synchronize()
    assert np.all(np.abs(_f64(c[:M]) - exact) <= 0.5 * _ulp(exact) + 2e-5 * np.sqrt(K))
    assert torch.all(c[M] == 7.0), "rows past M are untouched"
    want = O.widen_bf16(r) + exact
    assert np.all(np.abs(_f64(x) - want) <= 0.5 * _ulp(want) + 2e-5 * np.sqrt(K))
    want = S.silu(exact[:, 0::2]) * exact[:, 1::2]
    assert np.all(np.abs(_f64(g) - want) <= 0.5 * _ulp(want) + 1e-4 * (1 + np.abs(want)))


# ----------------------------------------------------------------------------------------------- a1' anchor stitch

def test_anchor_stitch_parity():
    binding = _binding()
    wl = inputs.make_workload("t_ragged")
    cfg, r = wl.cfg, wl.requests[0]
    ctx = binding.Context(cfg.n_q_heads, cfg.n_kv_heads, cfg.head_dim, cfg.rope_theta, 1, 1024, 32)
    k_pic = [O.widen_bf16(wl.pool_k[i]) for i in r.chunk_ids]
    v_pic = [O.widen_bf16(wl.pool_v[i]) for i in r.chunk_ids]
    k_exact, v_want, pos = O.anchor_stitch(k_pic, v_pic, r.anchor_idx, r.anchor_ptr, cfg.rope_theta, store_round=False)
    # Phase-I artifact: the compact anchor pool (rows A_i of each chunk, chunk order)
    ak = np.concatenate([wl.pool_k[c][r.anchor_idx[r.anchor_ptr[i]: r.anchor_ptr[i + 1]]] for i, c in enumerate(r.chunk_ids)])
    av = np.concatenate([wl.pool_v[c][r.anchor_idx[r.anchor_ptr[i]: r.anchor_ptr[i + 1]]] for i, c in enumerate(r.chunk_ids)])
    n_a = np.diff(r.anchor_ptr)
    off = np.concatenate([[0], np.cumsum(r.chunk_len)[:-1]])
    pb = ctx.batch([n_a], [r.anchor_ptr[:-1]], [r.n_query], chunk_pos=[off])
    assert pb.n_ctx[0] == len(pos)
    kf = torch.full((1, pb.t_stride, cfg.n_kv_heads, cfg.head_dim), 3.0, dtype=torch.bfloat16, device="cuda")
    vf = torch.full_like(kf, -3.0)
    ctx.qcf_rope_reposition(pb, _dev(ak), _dev(av), kf, vf)
    torch.cuda.synchronize()
    got = _f64(kf[0, : len(pos)])
    half = cfg.head_dim // 2
    pair = np.hypot(k_exact[..., :half], k_exact[..., half:])
    assert np.all(np.abs(got - k_exact) <= 0.5 * _ulp(k_exact) + 1e-6 * np.concatenate([pair, pair], -1) + 1e-30)
    assert np.array_equal(_f64(vf[0, : len(pos)]), v_want)
    assert torch.all(kf[0, len(pos):] == 3.0)
    # K-only variant (scoring prefetch)
    kf2 = torch.zeros_like(kf)
    ctx.qcf_rope_reposition(pb, _dev(ak), None, kf2, None)
    torch.cuda.synchronize()
    assert torch.equal(kf2[0, : len(pos)], kf[0, : len(pos)])


# ----------------------------------------------------------------------------------------------- a7: one layer

def _rel_rms_err(got, want):
    """max over rows of |got - want|_max / max(1, rms(want row))."""
    rms = np.sqrt(np.mean(want ** 2, axis=-1, keepdims=True))
    return float(np.max(np.abs(got - want) / np.maximum(1.0, rms)))


@pytest.mark.parametrize("name,layer", [("s_small", 1), ("s_d128", 2), ("s_wide", 0)])
def test_stack_layer_teacher_forced(name, layer):
    """One layer of stage 2 on the GPU against oracle.fuse_layer fed the SAME layer input, the GPU's own stitched
    cache and the same P (teacher-forced): isolates a7 + a4 + a5 of one layer from everything
    upstream.  s_wide has the real config-3 widths (hidden 4096, FFN 12288, 32/8 heads)."""
    binding = _binding()
    wl, ctx, stack = _make(name)
    sp = wl.spec
    cfg, layers = _oracle_stack(wl)
    w = layers[layer]
    rng = np.random.default_rng(77)
    hkv, d, n, lq = sp.n_kv_heads, sp.head_dim, sp.n_ctx, sp.n_query
    # any bf16 K/V are legal PIC entries for a single layer: seeded normals, K RoPE'd nowhere in particular
    pool_k = inputs.f32_to_bf16_bits(rng.standard_normal((n, hkv, d), dtype=np.float32))
    pool_v = inputs.f32_to_bf16_bits(rng.standard_normal((n, hkv, d), dtype=np.float32))
    lens = [sp.chunk_len] * sp.n_chunks
    rows0 = [i * sp.chunk_len for i in range(sp.n_chunks)]
    mb = ctx.batch([lens], [rows0], [lq])
    k_sel = binding.qcf_n_select(n, sp.ratio)
    sel = np.sort(rng.choice(n, size=k_sel, replace=False)).astype(np.int32)
    rows = np.concatenate([sel, np.arange(n, n + lq)]).astype(np.int64)
    x_bits = inputs.f32_to_bf16_bits(rng.standard_normal((len(rows), sp.hidden), dtype=np.float32))
    kf = torch.zeros((1, mb.t_stride, hkv, d), dtype=torch.bfloat16, device="cuda")
    vf = torch.zeros_like(kf)
    ctx.qcf_rope_reposition(mb, _dev(pool_k), _dev(pool_v), kf, vf)
    torch.cuda.synchronize()
    k_ctx, v_ctx = _f64(kf[0, :n]), _f64(vf[0, :n])                      # the GPU's stitched cache feeds the oracle
    x = _dev(x_bits)
    d_sel = torch.from_numpy(sel).cuda()
    d_ns = torch.tensor([k_sel], dtype=torch.int32, device="cuda")
    q_tap = torch.zeros((len(rows), sp.n_q_heads, d), dtype=torch.bfloat16, device="cuda")
    stack.qcf_stack_layer(layer, mb, d_sel, d_ns, len(rows), x, kf, vf, q_tap=q_tap)
    torch.cuda.synchronize()
    ref = S.fuse_layer(O.widen_bf16(x_bits), rows, k_sel, k_ctx, v_ctx, w, cfg)
    # refreshed K/V rows and the query's own rows (Eq. 7): bf16 values from fp32 arithmetic on identical inputs
    assert _close_bf16(_f64(kf[0])[rows], ref["k_new"], extra=5e-3)
    assert _close_bf16(_f64(vf[0])[rows], ref["v_new"], extra=5e-3)
    untouched = np.setdiff1d(np.arange(n), sel)
    assert np.array_equal(_f64(kf[0])[untouched], k_ctx[untouched]), "unselected PIC entries are kept (Eq. 7)"
    assert _close_bf16(_f64(q_tap), ref["q"], extra=5e-3)
    # layer output: every intermediate activation is rounded to bf16 on the GPU (h, qkv, q/k/v, attention output,
    # the residual stream, the SwiGLU activation), each a relative 2^-9 perturbation; DESIGN.md §5 bounds the sum by
    # 3e-2 of max(1, row rms) for this block
    err = _rel_rms_err(_f64(x), ref["x"])
    assert err <= 3e-2, err


def test_stack_prefill_parity_small():
    """Eq. 2 / Eq. 3 free-running on the reduced stack: per-layer K/V caches and the final hidden states."""
    wl, ctx, stack = _make("s_small")
    sp = wl.spec
    cfg, layers = _oracle_stack(wl)
    emb = O.widen_bf16(wl.embed)
    toks = np.concatenate(wl.chunk_tokens[:2] + [wl.query_tokens]).astype(np.int32)      # 272 rows: 3 row tiles, ragged
    t = len(toks)
    b = ctx.batch([[t - sp.n_query]], [[0]], [sp.n_query])
    kc = [torch.zeros((t, sp.n_kv_heads, sp.head_dim), dtype=torch.bfloat16, device="cuda") for _ in range(sp.n_layers)]
    vc = [torch.zeros_like(k) for k in kc]
    hid = torch.zeros((t, sp.hidden), dtype=torch.bfloat16, device="cuda")
    stack.qcf_stack_prefill(b, torch.from_numpy(toks).cuda(), kc, vc, hid)
    torch.cuda.synchronize()
    ref, ks, vs = S.full_prefill(emb[toks], layers, cfg)
    assert _close_bf16(_f64(kc[0]), ks[0], extra=5e-3) and _close_bf16(_f64(vc[0]), vs[0], extra=5e-3)   # identical inputs
    for l in range(1, sp.n_layers):           # deeper layers see bf16-rounded residual streams: relative to the row rms
        assert _rel_rms_err(_f64(kc[l]).reshape(t, -1), ks[l].reshape(t, -1)) <= 5e-2
        assert _rel_rms_err(_f64(vc[l]).reshape(t, -1), vs[l].reshape(t, -1)) <= 5e-2
    assert _rel_rms_err(_f64(hid), ref) <= 5e-2


# ----------------------------------------------------------------------------------------------- the pipeline

def _pic_from_oracle(wl, cfg, layers):
    emb = O.widen_bf16(wl.embed)
    k_pic, v_pic = S.build_pic([emb[t] for t in wl.chunk_tokens], layers, cfg)
    return emb, k_pic, v_pic


def _to_bits(x):
    return inputs.f32_to_bf16_bits(x.astype(np.float32))          # values are already bf16: exact


@pytest.mark.parametrize("name", ["s_small", "s_d128"])
def test_stack_prefill_is_bit_identical_with_and_without_pdl(name):
    """The layer's kernels are chained with programmatic dependent launch (each one's prologue overlaps its
    predecessor's tail).  A stale or early read would change bits: the chained run must equal the serialised one
    (qcf_debug_set(QCF_DEBUG_PDL, 0)) exactly, every time."""
    binding = _binding()
    results = []
    for pdl in ("1", "0"):
        wl, ctx, stack = _make(name)
        ctx.qcf_debug_set(binding.QCF_DEBUG_PDL, int(pdl))
        sp = wl.spec
        t = sp.n_ctx + sp.n_query
        b = ctx.batch([[sp.chunk_len] * sp.n_chunks], [[i * sp.chunk_len for i in range(sp.n_chunks)]], [sp.n_query])
        toks = torch.from_numpy(np.concatenate(wl.chunk_tokens + [wl.query_tokens]).astype(np.int32)).cuda()
        for rep in range(3 if pdl == "1" else 1):
            kc = [torch.zeros((t, sp.n_kv_heads, sp.head_dim), dtype=torch.bfloat16, device="cuda") for _ in range(sp.n_layers)]
            vc = [torch.zeros_like(k) for k in kc]
            hid = torch.full((t, sp.hidden), 3.0, dtype=torch.bfloat16, device="cuda")
            stack.qcf_stack_prefill(b, toks, kc, vc, hid)
            torch.cuda.synchronize()
            results.append((hid, kc, vc))
    ref = results[-1]
    for hid, kc, vc in results[:-1]:
        assert torch.equal(hid, ref[0])
        assert all(torch.equal(x, y) for x, y in zip(kc, ref[1])) and all(torch.equal(x, y) for x, y in zip(vc, ref[2]))


def _check_free_running_selection(tag, got_sel, got_sc, want_sc, k, eps_bound):
    """Free-running stage 1: the GPU's probe queries went through bf16 activations of the layers below, so
    its scores differ from the oracle's by a relative eps.  north_star rule applied to the BAND: a position whose oracle
    score is above s_k (1+eps)/(1-eps) is certainly selected and one below s_{k+1} (1-eps)/(1+eps) certainly is not (any
    score moved by at most eps cannot cross the threshold); only positions inside the band may differ.  eps is the stated
    bound; the measured error and overlap are printed (pytest -s) and recorded in DESIGN.md §5."""
    n = len(want_sc)
    rel = float(np.max(np.abs(got_sc - want_sc) / np.maximum(want_sc, 1e-300)))
    want = O.select_topk(want_sc, k)
    inter = len(np.intersect1d(got_sel, want))
    srt = np.sort(want_sc)[::-1]
    gap = float((srt[k - 1] - srt[k]) / srt[k - 1]) if 0 < k < n else float("inf")
    hi = srt[k - 1] * (1 + eps_bound) / (1 - eps_bound) if 0 < k < n else -np.inf
    lo = srt[k] * (1 - eps_bound) / (1 + eps_bound) if 0 < k < n else np.inf
    sure_in = np.nonzero(want_sc > hi)[0]
    sure_out = np.nonzero(want_sc < lo)[0]
    band = n - len(sure_in) - len(sure_out)
    print("[free-running %s] max rel score err %.3e (bound %.1e), k/k+1 gap %.2e, overlap %d/%d = %.4f, band %d of %d positions"
          % (tag, rel, eps_bound, gap, inter, k, inter / max(k, 1), band, n))
    assert rel <= eps_bound
    assert np.all(np.isin(sure_in, got_sel)), "a position clearly above the threshold band was dropped"
    assert not np.any(np.isin(sure_out, got_sel)), "a position clearly below the threshold band was selected"
    return rel, inter / max(k, 1), band


@pytest.mark.parametrize("name", ["s_small", "s_d128"])
def test_stack_fuse_pipeline_free_running(name):
    """Fig. 9 end to end (stage 1 probe over the anchor cache, Eq. 20 scores, top-k, stage 2 with layer-ahead loading
    from pinned host pools) against the oracle on the same PIC caches (built by the oracle, so both sides start from
    identical bf16 Phase-I artifacts)."""
    binding = _binding()
    wl, ctx, stack = _make(name)
    sp = wl.spec
    cfg, layers = _oracle_stack(wl)
    emb, k_pic, v_pic = _pic_from_oracle(wl, cfg, layers)
    n, lq, L = sp.n_ctx, sp.n_query, sp.n_layers
    hkv, d = sp.n_kv_heads, sp.head_dim
    a_idx, a_ptr = wl.anchor_idx, wl.anchor_ptr
    # Phase-I artifacts in pinned host memory: PIC pools and compact anchor pools per layer
    pin = lambda bits: torch.from_numpy(np.ascontiguousarray(bits).view(np.int16)).view(torch.bfloat16).pin_memory()
    hk = [pin(_to_bits(np.concatenate(k_pic[l], 0))) for l in range(L)]
    hv = [pin(_to_bits(np.concatenate(v_pic[l], 0))) for l in range(L)]
    anchors = lambda pic: np.concatenate([c[a_idx[a_ptr[i]: a_ptr[i + 1]]] for i, c in enumerate(pic)], 0)
    ak = [pin(_to_bits(anchors(k_pic[l]))) for l in range(L)]
    av = [pin(_to_bits(anchors(v_pic[l]))) for l in range(L)]
    lens = [sp.chunk_len] * sp.n_chunks
    off = [i * sp.chunk_len for i in range(sp.n_chunks)]
    mb = ctx.batch([lens], [off], [lq])
    pb = ctx.batch([np.diff(a_ptr)], [a_ptr[:-1]], [lq], chunk_pos=[off])
    toks = torch.from_numpy(np.concatenate(wl.chunk_tokens + [wl.query_tokens]).astype(np.int32)).cuda()
    k_sel = binding.qcf_n_select(n, sp.ratio)
    n_r = k_sel + lq

    def run(overlap):
        kf = [torch.zeros((mb.t_stride, hkv, d), dtype=torch.bfloat16, device="cuda") for _ in range(L)]
        vf = [torch.zeros_like(k) for k in kf]
        scores = torch.zeros(n, device="cuda")
        sel = torch.zeros(n, dtype=torch.int32, device="cuda")
        n_sel = torch.zeros(1, dtype=torch.int32, device="cuda")
        hid = torch.zeros((n_r, sp.hidden), dtype=torch.bfloat16, device="cuda")
        stack.qcf_stack_fuse(mb, pb, k_pic=hk, v_pic=hv, pool_rows=n, k_anchor=ak, v_anchor=av, anchor_rows=int(a_ptr[-1]),
                             crit_layers=sp.crit_layers, ratio=sp.ratio, tokens=toks, k_fused=kf, v_fused=vf,
                             scores=scores, sel=sel, n_sel=n_sel, hidden_out=hid, overlap=overlap)
        torch.cuda.synchronize()
        return kf, vf, scores, sel, n_sel, hid

    kf, vf, scores, sel, n_sel, hid = run(True)
    kf2, vf2, scores2, sel2, _, hid2 = run(False)
    assert torch.equal(scores, scores2) and torch.equal(sel, sel2) and torch.equal(hid, hid2), "overlap changes no bit"
    assert all(torch.equal(a, b) for a, b in zip(kf, kf2))

    pr = S.probe_stage(emb[wl.query_tokens], k_pic, v_pic, a_idx, a_ptr, layers, cfg, sp.crit_layers, sp.ratio)
    got_sc = scores.cpu().numpy().astype(np.float64)
    assert abs(got_sc.sum() - len(sp.crit_layers)) < 1e-3                      # Eq. 20: one unit of mass per layer in L*
    assert int(n_sel[0]) == k_sel == len(pr["sel"])
    got_sel = sel[:k_sel].cpu().numpy().astype(np.int64)
    assert np.array_equal(got_sel, O.select_topk(scores.cpu().numpy(), k_sel))  # integer work: exact on its own scores
    _, overlap, band = _check_free_running_selection(name, got_sel, got_sc, pr["scores"], k_sel, FREE_RUNNING_EPS)
    assert overlap >= FREE_RUNNING_OVERLAP
    # stage 2 against the oracle run on the GPU's selection
    rows = np.concatenate([got_sel, np.arange(n, n + lq)])
    x0 = emb[np.concatenate(wl.chunk_tokens + [wl.query_tokens])[rows]]
    ref = S.fuse_stage(x0, got_sel, n, k_pic, v_pic, layers, cfg)
    assert _rel_rms_err(_f64(hid), ref) <= 6e-2
    # layer-0 fused cache is teacher-forced by construction (its input is the embedding rows)
    k_ctx, v_ctx = O.reposition(k_pic[0], v_pic[0], sp.rope_theta)
    l0 = S.fuse_layer(x0, rows, k_sel, k_ctx, v_ctx, layers[0], cfg)
    assert _close_bf16(_f64(kf[0])[: n + lq], l0["k_fused"], extra=5e-3)
    assert _close_bf16(_f64(vf[0])[: n + lq], l0["v_fused"], extra=5e-3)


def test_stack_prefill_builds_pic_like_the_oracle():
    """Eq. 3 on the GPU: one chunk alone at local positions — the Phase-I artifact the bench builds with the library."""
    wl, ctx, stack = _make("s_d128")
    sp = wl.spec
    cfg, layers = _oracle_stack(wl)
    emb = O.widen_bf16(wl.embed)
    toks = wl.chunk_tokens[1]
    b = ctx.batch([[len(toks)]], [[0]], [0])
    kc = [torch.zeros((len(toks), sp.n_kv_heads, sp.head_dim), dtype=torch.bfloat16, device="cuda") for _ in range(sp.n_layers)]
    vc = [torch.zeros_like(k) for k in kc]
    stack.qcf_stack_prefill(b, torch.from_numpy(toks).cuda(), kc, vc)
    torch.cuda.synchronize()
    _, ks, vs = S.full_prefill(emb[toks], layers, cfg)
    assert _close_bf16(_f64(kc[0]), ks[0], extra=5e-3) and _close_bf16(_f64(vc[0]), vs[0], extra=5e-3)
    for l in range(1, sp.n_layers):
        assert _rel_rms_err(_f64(kc[l]).reshape(len(toks), -1), ks[l].reshape(len(toks), -1)) <= 5e-2


# ----------------------------------------------------------------------------------------------- selector views (§8(f).1)

@pytest.mark.parametrize("view", ["fullview", "final"])
def test_stack_fuse_other_selector_views(view):
    """The compressed view is an argument of qcf_stack_fuse: full-view (every token an anchor, every layer scored:
    ProphetKV-style, Eq. 9-11) and query-only final-layer selection run on the same kernels and match the
    oracle's probe_stage given the same view; stage 1 and stage 2 issued separately reproduce the fused call bit for bit."""
    from paper_2606_05875_b200 import stack_device
    binding = _binding()
    wl = inputs.make_stack_workload("s_small")
    sp = wl.spec
    ctx = binding.Context(sp.n_q_heads, sp.n_kv_heads, sp.head_dim, sp.rope_theta, 1, max(sp.n_ctx, 1024), sp.n_query)
    run = stack_device.StackRun(wl, ctx, _device_layers(wl), _dev(wl.embed))
    cfg, layers = _oracle_stack(wl)
    emb, k_pic, v_pic = _pic_from_oracle(wl, cfg, layers)
    L, n = sp.n_layers, sp.n_ctx
    run.k_pic = [_dev(_to_bits(np.concatenate(k_pic[l], 0))) for l in range(L)]      # device-resident pools
    run.v_pic = [_dev(_to_bits(np.concatenate(v_pic[l], 0))) for l in range(L)]
    run.k_anchor, run.v_anchor = run.k_pic, run.v_pic                                  # replaced by use_selector
    run.use_selector(view)
    run.fuse()
    torch.cuda.synchronize()
    ref = [t.clone() for t in (run.scores, run.sel, run.hidden)] + [k.clone() for k in run.k_fused]
    if view == "fullview":
        lens = [sp.chunk_len] * sp.n_chunks
        a_idx = np.concatenate([np.arange(ln) for ln in lens]).astype(np.int32)
        a_ptr = np.concatenate([[0], np.cumsum(lens)]).astype(np.int32)
        crit = list(range(L))
    else:
        a_idx = np.empty(0, np.int32)
        a_ptr = np.zeros(sp.n_chunks + 1, np.int32)
        crit = [L - 1]
    pr = S.probe_stage(emb[wl.query_tokens], k_pic, v_pic, a_idx, a_ptr, layers, cfg, crit, sp.ratio)
    got = run.scores.cpu().numpy().astype(np.float64)
    assert abs(got.sum() - len(crit)) < 1e-3
    k_sel = run.k_sel
    got_sel = run.sel[:k_sel].cpu().numpy().astype(np.int64)
    assert np.array_equal(got_sel, O.select_topk(run.scores.cpu().numpy(), k_sel))
    _, overlap, band = _check_free_running_selection(view, got_sel, got, pr["scores"], k_sel, FREE_RUNNING_EPS)
    assert overlap >= FREE_RUNNING_OVERLAP
    # stages issued separately
    run.scores.zero_(); run.hidden.zero_()
    run.fuse(stages=1)
    torch.cuda.synchronize()
    assert torch.equal(run.scores, ref[0]) and torch.equal(run.sel[:k_sel], ref[1][:k_sel])
    assert torch.all(run.hidden == 0), "stage 1 alone recomputes nothing"
    run.fuse(stages=2)
    torch.cuda.synchronize()
    assert torch.equal(run.hidden, ref[2])
    assert all(torch.equal(a, b) for a, b in zip(run.k_fused, ref[3:]))
    # stage 2 alone with an external selection whose size is not floor(rho N): refused (every row count is host-derived)
    run.n_sel.fill_(k_sel - 1)
    with pytest.raises(binding.QcfError) as e:
        run.fuse(stages=2)
    assert e.value.status == binding.QCF_ERR_INVALID_ARG and "n_sel" in str(e.value)
    run.n_sel.fill_(k_sel)
    # bandwidth emulation changes timing only: same bits, and the call takes at least bytes / bandwidth
    import time
    kv_row = sp.n_kv_heads * sp.head_dim * 2
    bytes_min = 2 * kv_row * n * L                            # every PIC pool is loaded once
    gbps = 0.5
    t0 = time.perf_counter()
    run.fuse(load_gbps=gbps)
    torch.cuda.synchronize()
    dt = time.perf_counter() - t0
    assert torch.equal(run.hidden, ref[2]) and torch.equal(run.scores, ref[0])
    assert dt >= 0.9 * bytes_min / (gbps * 1e9)


# ----------------------------------------------------------------------------------------------- Phase I anchors (§8(f).2)

@pytest.mark.parametrize("rule", ["sink", "knorm"])
def test_anchor_rank_parity(rule):
    """Eq. 14 on the GPU: per-chunk anchor ranking (Sink / Knorm) + segmented top-ceil(r_a len) against the oracle."""
    binding = _binding()
    wl = inputs.make_workload("t_ragged")                      # chunk lengths 131 / 64 / 1 / 257 / 77
    cfg = wl.cfg
    lens = [k.shape[0] for k in wl.pool_k]
    starts = np.concatenate([[0], np.cumsum(lens)]).astype(np.int64)
    ctx = binding.Context(cfg.n_q_heads, cfg.n_kv_heads, cfg.head_dim, cfg.rope_theta, len(lens), 1024, 8)
    chunks = ctx.batch([[ln] for ln in lens], [[int(s)] for s in starts[:-1]], [0] * len(lens))
    pool = _dev(np.concatenate(wl.pool_k, 0))
    pool2 = _dev(np.concatenate(wl.pool_v, 0))                 # stands in for a second layer's keys
    B, Nn = len(lens), chunks.n_stride
    scores = torch.full((B, Nn), 7.0, device="cuda")
    idx = torch.full((B, Nn), -1, dtype=torch.int32, device="cuda")
    n_a = torch.zeros(B, dtype=torch.int32, device="cuda")
    r_a = 0.1
    code = binding.QCF_ANCHOR_SINK if rule == "sink" else binding.QCF_ANCHOR_KNORM
    ctx.qcf_anchor_rank(chunks, pool, code, r_a, scores, idx, n_a)
    torch.cuda.synchronize()
    for i, ln in enumerate(lens):
        want = O.anchor_select(O.widen_bf16(wl.pool_k[i]), r_a, rule)
        k = O.n_anchor(ln, r_a)
        assert int(n_a[i]) == k == len(want)
        got = idx[i, :k].cpu().numpy().astype(np.int64)
        g = scores[i, :ln].cpu().numpy()
        assert np.array_equal(got, O.select_topk(g, k)), "exact on the kernel's own scores"
        np.testing.assert_allclose(g, O.anchor_scores(O.widen_bf16(wl.pool_k[i]), rule), rtol=1e-5, atol=0)
        _check_sel = len(np.intersect1d(got, want))
        assert _check_sel >= np.ceil(0.99 * k)
        assert torch.all(idx[i, k:] == -1) and torch.all(scores[i, ln:] == 7.0)
    if rule == "knorm":                                        # norms summed over two layers, selection on the second call
        ctx.qcf_anchor_rank(chunks, pool, code, r_a, scores, idx, n_a, accumulate=False, select_now=False)
        ctx.qcf_anchor_rank(chunks, pool2, code, r_a, scores, idx, n_a, accumulate=True, select_now=True)
        torch.cuda.synchronize()
        for i, ln in enumerate(lens):
            g2 = O.anchor_scores(O.widen_bf16(wl.pool_k[i]), rule) + O.anchor_scores(O.widen_bf16(wl.pool_v[i]), rule)
            k = O.n_anchor(ln, r_a)
            got = idx[i, :k].cpu().numpy().astype(np.int64)
            assert len(np.intersect1d(got, O.select_topk(g2, k))) >= np.ceil(0.99 * k)


@pytest.mark.parametrize("rule", ["sink", "knorm"])
def test_phase1_rank_gather_stitch_through_the_c_abi(rule):
    """Phase I closed inside the library (Eq. 14 -> Eq. 16 -> Eq. 15): qcf_anchor_rank picks A_i per chunk, qcf_anchor_gather
    copies KV_i^PIC[A_i] into the compact anchor pool, qcf_rope_reposition on the chunk_pos batch stitches it.  Against the
    oracle's anchor_stitch on the GPU's own anchor lists: the gathered V rows byte for byte (a pure row gather), the gathered K
    rows byte for byte against the pool rows, and the stitched K within the a1 bound.  Rows past the last anchor untouched."""
    binding = _binding()
    wl = inputs.make_workload("t_ragged")                      # chunk lengths 131 / 64 / 1 / 257 / 77
    cfg, r = wl.cfg, wl.requests[0]
    ids = list(r.chunk_ids)
    lens = [wl.pool_k[c].shape[0] for c in ids]
    starts = np.concatenate([[0], np.cumsum(lens)]).astype(np.int64)
    ctx = binding.Context(cfg.n_q_heads, cfg.n_kv_heads, cfg.head_dim, cfg.rope_theta, len(lens), 1024, 32)
    chunks = ctx.batch([[ln] for ln in lens], [[int(x)] for x in starts[:-1]], [0] * len(lens))
    pool_k, pool_v = _dev(np.concatenate([wl.pool_k[c] for c in ids], 0)), _dev(np.concatenate([wl.pool_v[c] for c in ids], 0))
    B, Nn = len(lens), chunks.n_stride
    scores = torch.zeros((B, Nn), device="cuda")
    idx = torch.full((B, Nn), -1, dtype=torch.int32, device="cuda")
    n_a = torch.zeros(B, dtype=torch.int32, device="cuda")
    r_a = 0.1
    code = binding.QCF_ANCHOR_SINK if rule == "sink" else binding.QCF_ANCHOR_KNORM
    ctx.qcf_anchor_rank(chunks, pool_k, code, r_a, scores, idx, n_a)
    counts = [O.n_anchor(ln, r_a) for ln in lens]               # known on the host: sizes the anchor pool
    total = int(sum(counts))
    hkv, d = cfg.n_kv_heads, cfg.head_dim
    ak = torch.full((total + 3, hkv, d), 5.0, dtype=torch.bfloat16, device="cuda")
    av = torch.full_like(ak, -5.0)
    ctx.qcf_anchor_gather(chunks, pool_k, pool_v, idx, n_a, ak, av)
    torch.cuda.synchronize()
    assert n_a.cpu().tolist() == counts
    a_idx = np.concatenate([idx[i, :c].cpu().numpy() for i, c in enumerate(counts)]).astype(np.int64)
    a_ptr = np.concatenate([[0], np.cumsum(counts)]).astype(np.int64)
    k_pic = [O.widen_bf16(wl.pool_k[c]) for c in ids]
    v_pic = [O.widen_bf16(wl.pool_v[c]) for c in ids]
    k_exact, v_want, pos = O.anchor_stitch(k_pic, v_pic, a_idx, a_ptr, cfg.rope_theta, store_round=False)
    assert len(pos) == total
    assert np.array_equal(_f64(av[:total]), v_want)                                    # Eq. 16 on V: byte copy
    k_rows = np.concatenate([k_pic[i][a_idx[a_ptr[i]: a_ptr[i + 1]]] for i in range(B)])
    assert np.array_equal(_f64(ak[:total]), k_rows)                                    # Eq. 16 on K: byte copy (RoPE still local)
    assert torch.all(ak[total:] == 5.0) and torch.all(av[total:] == -5.0)
    # K-only and V-only calls write the same rows
    ak2, av2 = torch.zeros_like(ak), torch.zeros_like(av)
    ctx.qcf_anchor_gather(chunks, pool_k, None, idx, n_a, ak2, None)
    ctx.qcf_anchor_gather(chunks, None, pool_v, idx, n_a, None, av2)
    # Eq. 15: stitch the gathered pool at the chunks' ORIGINAL offsets
    off = starts[:-1]
    pb = ctx.batch([counts], [a_ptr[:-1]], [r.n_query], chunk_pos=[off])
    kf = torch.zeros((1, pb.t_stride, hkv, d), dtype=torch.bfloat16, device="cuda")
    vf = torch.zeros_like(kf)
    ctx.qcf_rope_reposition(pb, ak, av, kf, vf)
    torch.cuda.synchronize()
    assert torch.equal(ak2[:total], ak[:total]) and torch.equal(av2[:total], av[:total])
    half = d // 2
    pair = np.hypot(k_exact[..., :half], k_exact[..., half:])
    assert np.all(np.abs(_f64(kf[0, :total]) - k_exact) <= 0.5 * _ulp(k_exact) + 1e-6 * np.concatenate([pair, pair], -1) + 1e-30)
    assert np.array_equal(_f64(vf[0, :total]), v_want)
    with pytest.raises(binding.QcfError):
        ctx.qcf_anchor_gather(chunks, pool_k, None, idx, n_a, None, None)             # a pool without its destination


# ----------------------------------------------------------------------------------------------- config 3 at full size

def test_stack_layer_full_size_c3_sampled():
    """BASELINE configs[2] at its own sizes (N = 10240, Lq = 64, n_R = 3136, hidden 4096, FFN 12288, 32/8 heads), one
    layer, teacher-forced: refreshed K/V of ALL rows against the oracle, the layer output on a declared row sample (all
    query rows, first / last 32 selected rows, 64 seeded random rows) — rows are independent given the fused cache."""
    binding = _binding()
    wl = inputs.make_stack_workload("c3", n_layers=1)
    sp = wl.spec
    cfg, layers = _oracle_stack(wl)
    w = layers[0]
    n, lq, hkv, d = sp.n_ctx, sp.n_query, sp.n_kv_heads, sp.head_dim
    t = n + lq
    ctx = binding.Context(sp.n_q_heads, hkv, d, sp.rope_theta, 1, n, lq)
    stack = binding.Stack(ctx, 1, sp.hidden, sp.ffn, sp.vocab, sp.rms_eps, _device_layers(wl), _dev(wl.embed), t, t,
                          max_pool_rows=n)
    rng = np.random.default_rng(303)
    pool_k = inputs.f32_to_bf16_bits(rng.standard_normal((n, hkv, d), dtype=np.float32))
    pool_v = inputs.f32_to_bf16_bits(rng.standard_normal((n, hkv, d), dtype=np.float32))
    mb = ctx.batch([[sp.chunk_len] * sp.n_chunks], [[i * sp.chunk_len for i in range(sp.n_chunks)]], [lq])
    k_sel = binding.qcf_n_select(n, sp.ratio)
    assert k_sel == 3072
    sel = np.sort(rng.choice(n, size=k_sel, replace=False)).astype(np.int32)
    rows = np.concatenate([sel, np.arange(n, n + lq)]).astype(np.int64)
    x_bits = inputs.f32_to_bf16_bits(rng.standard_normal((len(rows), sp.hidden), dtype=np.float32))
    kf = torch.zeros((1, mb.t_stride, hkv, d), dtype=torch.bfloat16, device="cuda")
    vf = torch.zeros_like(kf)
    ctx.qcf_rope_reposition(mb, _dev(pool_k), _dev(pool_v), kf, vf)
    torch.cuda.synchronize()
    k_ctx, v_ctx = _f64(kf[0, :n]), _f64(vf[0, :n])
    x = _dev(x_bits)
    stack.qcf_stack_layer(0, mb, torch.from_numpy(sel).cuda(), torch.tensor([k_sel], dtype=torch.int32, device="cuda"),
                          len(rows), x, kf, vf)
    torch.cuda.synchronize()
    x_in = O.widen_bf16(x_bits)
    q, k_new, v_new = S.layer_qkv(x_in, rows, w, cfg)                     # all rows: the fused cache needs every refresh
    assert _close_bf16(_f64(kf[0])[rows], k_new, extra=5e-3)
    assert _close_bf16(_f64(vf[0])[rows], v_new, extra=5e-3)
    k_pos = np.zeros((t, hkv, d)); v_pos = np.zeros((t, hkv, d))
    k_pos[rows], v_pos[rows] = k_new, v_new
    k_f, v_f = O.fuse(k_ctx, v_ctx, sel.astype(np.int64), k_pos, v_pos)
    samp = np.unique(np.concatenate([np.arange(32), np.arange(k_sel - 32, k_sel), rng.choice(k_sel, 64, replace=False),
                                     np.arange(k_sel, k_sel + lq)]))
    a = O.recompute_attn(q[samp], rows[samp], k_f, v_f)
    want = S.layer_finish(x_in[samp], a, w, cfg)
    err = _rel_rms_err(_f64(x)[samp], want)
    assert err <= 3e-2, err


def test_first_token_parity():
    """End of TTFT: RMSNorm + LM head + argmax of the last query row against the oracle.  The decision is an integer taken
    from fp32 logits: exact where the oracle's top-2 gap exceeds the logit tolerance, else the chosen token must be within it."""
    binding = _binding()
    wl, ctx, stack = _make("s_d128")
    sp = wl.spec
    rng = np.random.default_rng(12)
    rows = 37
    hid_bits = inputs.f32_to_bf16_bits(rng.standard_normal((rows, sp.hidden), dtype=np.float32) * np.float32(3.0))
    g_bits = inputs.f32_to_bf16_bits(np.float32(1.0) + np.float32(0.1) * rng.standard_normal(sp.hidden, dtype=np.float32))
    w_bits = inputs.f32_to_bf16_bits(rng.standard_normal((sp.vocab, sp.hidden), dtype=np.float32) * np.float32(0.05))
    logits = torch.zeros(sp.vocab, device="cuda")
    token = torch.full((1,), -1, dtype=torch.int32, device="cuda")
    stack.qcf_stack_first_token(_dev(hid_bits), rows - 1, _dev(g_bits), _dev(w_bits), logits, token)
    torch.cuda.synchronize()
    tok, want = S.first_token(O.widen_bf16(hid_bits[rows - 1]), O.widen_bf16(g_bits), O.widen_bf16(w_bits), sp.rms_eps)
    got = logits.cpu().numpy().astype(np.float64)
    tol = 2e-2 * max(1.0, np.abs(want).max())               # h is rounded to bf16 on the GPU (2^-9 relative per term)
    assert np.max(np.abs(got - want)) <= tol
    t = int(token[0])
    assert t == int(np.argmax(logits.cpu().numpy())), "argmax of its own logits, ties to the lower id"
    top2 = np.sort(want)[-2:]
    if top2[1] - top2[0] > 2 * tol:
        assert t == tok
    else:
        assert want[t] >= top2[1] - 2 * tol


# ----------------------------------------------------------------------------------------------- decoding over KV^Fuse (§8(f).4)

@pytest.mark.parametrize("hq,hkv,d", [(4, 2, 64), (8, 2, 128), (32, 8, 128), (64, 8, 128), (16, 1, 64), (2, 2, 128)])
@pytest.mark.parametrize("n_keys", [1, 5, 127, 128, 129, 1000, 4100])
def test_decode_attn_parity(hq, hkv, d, n_keys):
    """qcf_decode_attn (one new token over a layer's cache) against the oracle's causal attention of a
    single row at position n_keys - 1: max-abs 2e-2 (north_star) plus the per-vector relative criterion, lse, rows past
    n_keys never read (poisoned with NaN), run-to-run bit identity (splits merged in split order)."""
    binding = _binding()
    ctx = binding.Context(hq, hkv, d, 1e6, 1, 8192, 8)
    rng = np.random.default_rng(n_keys * 131 + hq * 7 + d)
    q = inputs.f32_to_bf16_bits(rng.standard_normal((hq, d), dtype=np.float32))
    k = inputs.f32_to_bf16_bits(rng.standard_normal((n_keys, hkv, d), dtype=np.float32))
    v = inputs.f32_to_bf16_bits(rng.standard_normal((n_keys, hkv, d), dtype=np.float32))
    if n_keys > 100:                                              # a few heavy hitters: the softmax is not near-uniform
        k[rng.choice(n_keys, 5, replace=False)] = inputs.f32_to_bf16_bits(
            4 * rng.standard_normal((5, hkv, d), dtype=np.float32))
    pad = np.full((7, hkv, d), 0x7FC0, dtype=np.uint16)           # bf16 NaN rows behind the valid ones
    kc, vc = _dev(np.concatenate([k, pad])), _dev(np.concatenate([v, pad]))
    out = torch.full((hq, d), 9.0, dtype=torch.bfloat16, device="cuda")
    lse = torch.zeros(hq, device="cuda")
    ctx.qcf_decode_attn(_dev(q), kc, vc, n_keys, out, lse)
    torch.cuda.synchronize()
    want, want_lse = O.recompute_attn(O.widen_bf16(q)[None], np.array([n_keys - 1]), O.widen_bf16(k), O.widen_bf16(v),
                                      return_lse=True)
    got = _f64(out)
    assert np.all(np.isfinite(got))
    assert np.max(np.abs(got - want[0])) <= 2e-2
    num, den = np.linalg.norm(got - want[0], axis=-1), np.linalg.norm(want[0], axis=-1)
    assert np.all(num <= 2e-2 * den + 1e-3), float(np.max(num / den))
    np.testing.assert_allclose(lse.cpu().numpy(), want_lse[0], rtol=0, atol=2e-2)
    out2 = torch.zeros_like(out)
    ctx.qcf_decode_attn(_dev(q), kc, vc, n_keys, out2, None)
    torch.cuda.synchronize()
    assert torch.equal(out, out2)


@pytest.mark.parametrize("name", ["s_small", "s_d128"])
def test_stack_decode_over_kv_fuse(name):
    """Closes the TTFT -> generation loop: qcf_stack_fuse fills KV^Fuse, qcf_stack_first_token
    gives token 0, qcf_stack_decode generates 8 greedy tokens reading and extending those caches.  The oracle runs the same
    pipeline (stage 2 on the GPU's selection, as in test_stack_fuse_pipeline_free_running) and decodes from ITS caches.
    Logits within the stated free-running bound; token ids exact wherever the oracle's top-2 logit gap exceeds twice that
    bound (else the GPU's token must be within the bound of the best); the appended K/V rows against the oracle's."""
    binding = _binding()
    n_new = 8
    wl, ctx, stack = _make(name, extra_pos=n_new)
    sp = wl.spec
    cfg, layers = _oracle_stack(wl)
    emb, k_pic, v_pic = _pic_from_oracle(wl, cfg, layers)
    n, lq, L = sp.n_ctx, sp.n_query, sp.n_layers
    hkv, d = sp.n_kv_heads, sp.head_dim
    a_idx, a_ptr = wl.anchor_idx, wl.anchor_ptr
    hk = [_dev(_to_bits(np.concatenate(k_pic[l], 0))) for l in range(L)]
    hv = [_dev(_to_bits(np.concatenate(v_pic[l], 0))) for l in range(L)]
    anchors = lambda pic: np.concatenate([c[a_idx[a_ptr[i]: a_ptr[i + 1]]] for i, c in enumerate(pic)], 0)
    ak = [_dev(_to_bits(anchors(k_pic[l]))) for l in range(L)]
    av = [_dev(_to_bits(anchors(v_pic[l]))) for l in range(L)]
    lens = [sp.chunk_len] * sp.n_chunks
    off = [i * sp.chunk_len for i in range(sp.n_chunks)]
    mb = ctx.batch([lens], [off], [lq])
    pb = ctx.batch([np.diff(a_ptr)], [a_ptr[:-1]], [lq], chunk_pos=[off])
    toks = torch.from_numpy(np.concatenate(wl.chunk_tokens + [wl.query_tokens]).astype(np.int32)).cuda()
    k_sel = binding.qcf_n_select(n, sp.ratio)
    n_r = k_sel + lq
    t = n + lq
    kf = [torch.zeros((t + n_new, hkv, d), dtype=torch.bfloat16, device="cuda") for _ in range(L)]     # room for the new rows
    vf = [torch.zeros_like(x) for x in kf]
    scores = torch.zeros(n, device="cuda")
    sel = torch.zeros(n, dtype=torch.int32, device="cuda")
    n_sel = torch.zeros(1, dtype=torch.int32, device="cuda")
    hid = torch.zeros((n_r, sp.hidden), dtype=torch.bfloat16, device="cuda")
    stack.qcf_stack_fuse(mb, pb, k_pic=hk, v_pic=hv, pool_rows=n, k_anchor=ak, v_anchor=av, anchor_rows=int(a_ptr[-1]),
                         crit_layers=sp.crit_layers, ratio=sp.ratio, tokens=toks, k_fused=kf, v_fused=vf, scores=scores,
                         sel=sel, n_sel=n_sel, hidden_out=hid)
    rng = np.random.default_rng(77)
    g_bits = inputs.f32_to_bf16_bits(np.float32(1.0) + np.float32(0.1) * rng.standard_normal(sp.hidden, dtype=np.float32))
    w_bits = inputs.f32_to_bf16_bits(rng.standard_normal((sp.vocab, sp.hidden), dtype=np.float32) * np.float32(0.05))
    g_fin, w_lm = _dev(g_bits), _dev(w_bits)
    logits0 = torch.zeros(sp.vocab, device="cuda")
    tok0 = torch.zeros(1, dtype=torch.int32, device="cuda")
    stack.qcf_stack_first_token(hid, n_r - 1, g_fin, w_lm, logits0, tok0)
    logits = torch.zeros((n_new, sp.vocab), device="cuda")
    toks_out = torch.full((n_new,), -1, dtype=torch.int32, device="cuda")
    stack.qcf_stack_decode(tok0, t, n_new, kf, vf, g_fin, w_lm, logits, toks_out)
    torch.cuda.synchronize()

    # ---- oracle: stage 2 on the GPU's selection -> KV^Fuse per layer + final hidden -> first token -> greedy decode
    got_sel = sel[:k_sel].cpu().numpy().astype(np.int64)
    rows = np.concatenate([got_sel, np.arange(n, n + lq)])
    x = emb[np.concatenate(wl.chunk_tokens + [wl.query_tokens])[rows]]
    ks, vs = [], []
    for l in range(L):
        k_ctx, v_ctx = O.reposition(k_pic[l], v_pic[l], sp.rope_theta)
        r = S.fuse_layer(x, rows, k_sel, k_ctx, v_ctx, layers[l], cfg)
        x = r["x"]
        ks.append(r["k_fused"]); vs.append(r["v_fused"])
    G, W = O.widen_bf16(g_bits), O.widen_bf16(w_bits)
    first, lg0 = S.first_token(x[-1], G, W, sp.rms_eps)
    want_toks, want_logits, k2, v2 = S.greedy_decode(first, n_new, emb, ks, vs, layers, cfg, G, W)

    tol = DECODE_LOGIT_TOL * max(1.0, float(np.abs(want_logits).max()))
    def check_token(got_tok, got_lg, want_lg, tag):
        err = float(np.max(np.abs(got_lg - want_lg)))
        top2 = np.sort(want_lg)[-2:]
        print("[decode %s %s] max|logit err| %.3e (tol %.3e), oracle top-2 gap %.3e" % (name, tag, err, tol, top2[1] - top2[0]))
        assert err <= tol
        assert got_tok == int(np.argmax(got_lg)), "argmax of its own logits"
        if top2[1] - top2[0] > 2 * tol:
            assert got_tok == int(np.argmax(want_lg))
        else:
            assert want_lg[got_tok] >= top2[1] - 2 * tol
        return got_tok == int(np.argmax(want_lg))

    same = check_token(int(tok0[0]), logits0.cpu().numpy().astype(np.float64), lg0, "first")
    got_toks = toks_out.cpu().numpy()
    got_logits = logits.cpu().numpy().astype(np.float64)
    for i in range(n_new):
        if not same:
            break                       # a justified near-tie flip: the two sequences legitimately diverge from here
        same = check_token(int(got_toks[i]), got_logits[i], want_logits[i], "step %d" % i)
        # the K/V rows this token appended (free-running bound of DESIGN.md §5 for caches)
        for l in (0, L - 1):
            assert _rel_rms_err(_f64(kf[l][t + i])[None].reshape(1, -1), k2[l][t + i][None].reshape(1, -1)) <= 5e-2
            assert _rel_rms_err(_f64(vf[l][t + i])[None].reshape(1, -1), v2[l][t + i][None].reshape(1, -1)) <= 5e-2
    # KV^Fuse itself was not disturbed by decoding
    assert _rel_rms_err(_f64(kf[L - 1][:t]).reshape(t, -1), ks[L - 1].reshape(t, -1)) <= 5e-2
