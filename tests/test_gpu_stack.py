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


def _make(name, max_rows=None):
    binding = _binding()
    wl = inputs.make_stack_workload(name)
    sp = wl.spec
    t = sp.n_ctx + sp.n_query
    ctx = binding.Context(sp.n_q_heads, sp.n_kv_heads, sp.head_dim, sp.rope_theta, 1, max(sp.n_ctx, 1024), sp.n_query)
    dl = _device_layers(wl)
    emb = _dev(wl.embed)
    stack = binding.Stack(ctx, sp.n_layers, sp.hidden, sp.ffn, sp.vocab, sp.rms_eps, dl, emb, max_rows or t, t,
                          max_pool_rows=sp.n_ctx)
    return wl, ctx, stack


# ----------------------------------------------------------------------------------------------- qcf_linear

@pytest.mark.parametrize("mt", ["1", "2"])
@pytest.mark.parametrize("M,N,K", [(200, 768, 512), (131, 1536, 384), (1, 512, 1536), (300, 264, 64), (515, 1032, 4096)])
def test_linear_store_and_residual(M, N, K, mt, monkeypatch):
    monkeypatch.setenv("QCF_GEMM_MT", mt)
    binding = _binding()
    ctx = binding.Context(8, 2, 64, 1e6, 1, 1024, 8)
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


@pytest.mark.parametrize("mt", ["1", "2"])
def test_linear_swiglu(mt, monkeypatch):
    monkeypatch.setenv("QCF_GEMM_MT", mt)
    binding = _binding()
    ctx = binding.Context(8, 2, 64, 1e6, 1, 1024, 8)
    M, F, K = 300, 1160, 384
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
