"""qcf_decode_attn_static: decode attention for callers that cannot allocate device memory.

Who needs it: an op that runs inside a serving engine whose own pool already holds all of HBM (a cudaMalloc from inside it
fails or fragments the pool), code in a section its framework has declared allocation-free, or a tool that must not change
the allocator state it is watching.  Those callers cannot use qcf_create (it cudaMallocs the kernel's split-KV workspace),
so the library carries a fixed workspace of its own (about 2.1 MiB per GPU, Hq * head_dim <= 8192, Hkv <= 64; include/qcf.h).

What is checked: the entry point gives what qcf_decode_attn gives on the same inputs — within the decode tests' bound
(max-abs 2e-2) and, since it is the same kernel with the same split of the key range, bit for bit — on two calls in a row
that share the workspace and use DIFFERENT layouts and lengths (the second call sees the first call's leftovers); that
the GPU's free memory does not drop across the calls; and that a layout beyond the fixed workspace is refused before any
launch.

This file sorts last on purpose: `pytest -x` stops at the first failure, so a problem here cannot hide other tests.  It does
not depend on what ran before it (passes alone in a fresh process and at the end of the whole suite)."""
import numpy as np
import pytest
import torch

from paper_2606_05875_b200 import inputs

pytestmark = pytest.mark.gpu

# (Hq, Hkv, d, n_keys): different group sizes, head dims and split counts, back to back on the one shared workspace
CASES = [(32, 8, 128, 4100), (16, 1, 64, 129), (64, 8, 128, 1000), (4, 2, 64, 1)]


def _binding():
    from paper_2606_05875_b200 import binding
    if not torch.cuda.is_available():
        pytest.fail("no CUDA device: the qcf library has no CPU fallback")
    binding.load_library()
    return binding


def _case(hq, hkv, d, n_keys):
    rng = np.random.default_rng(n_keys * 977 + hq * 13 + d)
    q = inputs.f32_to_bf16_bits(rng.standard_normal((hq, d), dtype=np.float32))
    k = inputs.f32_to_bf16_bits(rng.standard_normal((n_keys, hkv, d), dtype=np.float32))
    v = inputs.f32_to_bf16_bits(rng.standard_normal((n_keys, hkv, d), dtype=np.float32))
    dev = lambda a: torch.from_numpy(a.view(np.int16)).cuda().view(torch.bfloat16)
    return dev(q), dev(k), dev(v)


def test_static_workspace_decode_attn_matches_ctx_path_on_consecutive_calls():
    binding = _binding()
    # the existing path first, each layout with its own ctx and cudaMalloc'd workspace
    want = []
    tensors = []
    for hq, hkv, d, n_keys in CASES:
        q, k, v = _case(hq, hkv, d, n_keys)
        ctx = binding.Context(hq, hkv, d, 1e6, 1, 8192, 8)
        out = torch.zeros((hq, d), dtype=torch.bfloat16, device="cuda")
        lse = torch.zeros(hq, device="cuda")
        ctx.qcf_decode_attn(q, k, v, n_keys, out, lse)
        torch.cuda.synchronize()
        want.append((out, lse))
        tensors.append((q, k, v))
    # outputs are allocated up front so that the calls under test run with nothing allocated around them
    got = [(torch.full((hq, d), 9.0, dtype=torch.bfloat16, device="cuda"), torch.full((hq,), 9.0, device="cuda"))
           for hq, hkv, d, n_keys in CASES]
    torch.cuda.synchronize()
    for rep in range(2):                                           # the whole sequence twice: every call follows another one
        for out, lse in got:
            out.fill_(9.0)
        torch.cuda.synchronize()
        free_before = torch.cuda.mem_get_info()[0]
        for (hq, hkv, d, n_keys), (q, k, v), (out, lse) in zip(CASES, tensors, got):
            binding.qcf_decode_attn_static(hq, hkv, d, q, k, v, n_keys, out, lse)
        torch.cuda.synchronize()
        if rep == 1:        # (round 0 holds each device's one-time set-up; from then on nothing may take device memory)
            assert torch.cuda.mem_get_info()[0] >= free_before, "device memory was allocated during the calls"
        for (hq, hkv, d, n_keys), (out, lse), (w_out, w_lse) in zip(CASES, got, want):
            diff = (out.float() - w_out.float()).abs().max().item()
            assert diff <= 2e-2, (hq, hkv, d, n_keys, diff)        # the decode tests' bound (north_star: max-abs 2e-2)
            assert (lse - w_lse).abs().max().item() <= 2e-2
            assert torch.equal(out, w_out) and torch.equal(lse, w_lse), "same kernel, same key split: bit-identical"


def test_static_workspace_rejects_layouts_beyond_its_size():
    binding = _binding()
    q, k, v = _case(4, 2, 64, 8)
    out = torch.zeros((4, 64), dtype=torch.bfloat16, device="cuda")
    for hq, hkv, d in [(128, 8, 128), (128, 128, 64)]:             # Hq * d = 16384 > 8192;  Hkv = 128 > 64
        with pytest.raises(binding.QcfError) as ei:
            binding.qcf_decode_attn_static(hq, hkv, d, q, k, v, 8, out)
        assert ei.value.status == binding.QCF_ERR_WORKSPACE and "built-in workspace" in str(ei.value)
    with pytest.raises(binding.QcfError) as ei:                    # unsupported group size is refused too, not launched
        binding.qcf_decode_attn_static(6, 2, 64, q, k, v, 8, out)
    assert ei.value.status == binding.QCF_ERR_UNSUPPORTED
    with pytest.raises(binding.QcfError):
        binding.qcf_decode_attn_static(4, 2, 64, q, k, v, 0, out)
    torch.cuda.synchronize()
    assert torch.all(out == 0), "a refused call must not have written anything"
