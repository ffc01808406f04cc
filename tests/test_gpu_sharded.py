"""GPU parity of the KV-head-sharded step (paper_2606_05875_b200/sharded.py) against
the fp64 oracle of the UNSHARDED layer.  One GPU: the ranks run one after the other (no kernel waits on another
rank), and the step's only exchange — the sum of the ranks' partial scores — is formed by qcf_score's own accumulate
path, which is the arithmetic an all-reduce(sum) performs.  A world-size-1 NCCL group covers the collective call itself.
Tolerances: BASELINE.json north_star's (see tests/test_gpu_parity.py).
"""
import os

import numpy as np
import pytest
import torch

from oracle import qcf_oracle as O
from paper_2606_05875_b200 import inputs

pytestmark = pytest.mark.gpu


def _mods():
    from paper_2606_05875_b200 import binding, device, sharded
    return binding, device, sharded


def _f64(t):
    return O.widen_bf16(t.detach().cpu().view(torch.int16).numpy().view(np.uint16))


def _check_selection(sel_g, scores_o, k):
    want = O.select_topk(scores_o, k)
    srt = np.sort(scores_o)[::-1]
    gap = (srt[k - 1] - srt[k]) / max(abs(srt[k - 1]), 1e-300) if 0 < k < len(scores_o) else 1.0
    if gap > 1e-3:
        assert np.array_equal(sel_g, want)                               # north_star: exact above the 1e-3 gap
    else:
        assert len(np.intersect1d(sel_g, want)) >= 0.99 * k


def _ranks(wl, world):
    _, device, sharded = _mods()
    cfg = wl.cfg
    steps, dws = [], []
    for rank in range(world):
        st = sharded.HeadShardedStep(cfg.n_q_heads, cfg.n_kv_heads, cfg.head_dim, cfg.rope_theta, max(cfg.batch, 1),
                                     max(cfg.n_ctx, 1024), max(cfg.n_query, 1), rank=rank, world=world)
        steps.append(st)
        dws.append(device.DeviceWorkload(inputs.shard_heads(wl, rank, world), st.ctx))
    return steps, dws


@pytest.mark.parametrize("exchange", ["accumulate", "fused"])
@pytest.mark.parametrize("name,world", [("t_mid", 2), ("t_mid", 4), ("t_batch", 2), ("t_ragged", 2), ("c1", 2)])
def test_head_sharded_step_matches_unsharded_oracle(name, world, exchange):
    """exchange = "accumulate": the sum over ranks formed by a2's own accumulate path (what an all-reduce computes);
    "fused": the exchange of include/qcf.h qcf_set_score_exchange — every rank's a2 stores its partial into every rank's
    exchange buffer and a3 sums the slots (here the "peers" are contexts of one process on one GPU, run one after the
    other, so no kernel waits on a flag that is still to be written)."""
    _, _, sharded = _mods()
    wl = inputs.make_workload(name)
    cfg = wl.cfg
    steps, dws = _ranks(wl, world)
    if exchange == "fused":
        slot = dws[0].batch.batch * dws[0].batch.n_stride
        bufs = [sharded.HeadShardedStep.alloc_exchange_buffer(world, slot) for _ in range(world)]
        for st in steps:
            st.enable_fused_exchange(bufs, slot)
        for st, dw in zip(steps, dws):                              # every rank its OWN scores array: nothing is shared but the slots
            dw.scores.fill_(7.0)
            st.score_phase(dw.batch, k_pool=dw.k_pool, v_pool=dw.v_pool, k_fused=dw.k_fused, v_fused=dw.v_fused,
                           q_probe=dw.q_probe, scores=dw.scores)
        for st, dw in zip(steps, dws):
            st.fuse_phase(dw.batch, scores=None, sel=dw.sel, n_sel=dw.n_sel, q_new=dw.q_new, k_new=dw.k_new, v_new=dw.v_new,
                          k_fused=dw.k_fused, v_fused=dw.v_fused, out=dw.out, lse=dw.lse, ratio=cfg.ratio)
        torch.cuda.synchronize()
        scores = steps[0].exchanged_scores(dws[0].batch)
        for st, dw in zip(steps[1:], dws[1:]):                      # every rank holds the same slots: bit-identical sums
            assert torch.equal(st.exchanged_scores(dw.batch), scores)
    else:
        scores = dws[0].scores                       # the array the all-reduce leaves on every rank
        scores.fill_(7.0)
        for rank, (st, dw) in enumerate(zip(steps, dws)):
            st.score_phase(dw.batch, k_pool=dw.k_pool, v_pool=dw.v_pool, k_fused=dw.k_fused, v_fused=dw.v_fused,
                           q_probe=dw.q_probe, scores=scores, accumulate=rank > 0)
        for st, dw in zip(steps, dws):
            st.fuse_phase(dw.batch, scores=scores, sel=dw.sel, n_sel=dw.n_sel, q_new=dw.q_new, k_new=dw.k_new, v_new=dw.v_new,
                          k_fused=dw.k_fused, v_fused=dw.v_fused, out=dw.out, lse=dw.lse, ratio=cfg.ratio)
        torch.cuda.synchronize()
    g = cfg.n_q_heads // cfg.n_kv_heads
    sc = scores.cpu().numpy()
    for b, r in enumerate(wl.requests):
        k_pic = [O.widen_bf16(wl.pool_k[i]) for i in r.chunk_ids]
        v_pic = [O.widen_bf16(wl.pool_v[i]) for i in r.chunk_ids]
        ref = O.layer_step(k_pic, v_pic, cfg.rope_theta, O.widen_bf16(r.q_probe), cfg.ratio, O.widen_bf16(r.q_new),
                           O.widen_bf16(r.k_new), O.widen_bf16(r.v_new))
        # a2: the summed partials are Eq. 18 over ALL heads of the layer
        np.testing.assert_allclose(sc[b, : r.n_ctx].astype(np.float64), ref["scores"], rtol=1e-2, atol=0)
        # a3: replicated selection, identical on every rank
        k = int(dws[0].n_sel[b])
        assert k == len(ref["sel"])
        sel0 = dws[0].sel[b, :k].cpu().numpy().astype(np.int64)
        for dw in dws[1:]:
            assert int(dw.n_sel[b]) == k and np.array_equal(dw.sel[b, :k].cpu().numpy(), sel0)
        _check_selection(sel0, ref["scores"], k)
        # a4 + a5: each rank's heads against the oracle run on the GPU's selection
        ref2 = O.layer_step(k_pic, v_pic, cfg.rope_theta, None, 0.0, O.widen_bf16(r.q_new), O.widen_bf16(r.k_new),
                            O.widen_bf16(r.v_new), sel=sel0)
        n_r = k + r.n_query
        per = cfg.n_kv_heads // world
        for rank, dw in enumerate(dws):
            qh = slice(rank * per * g, (rank + 1) * per * g)
            kv = slice(rank * per, (rank + 1) * per)
            got_o, want_o = _f64(dw.out[b, :n_r]), ref2["out"][:, qh]
            assert np.max(np.abs(got_o - want_o), initial=0.0) <= 2e-2                               # max-abs 2e-2
            num, den = np.linalg.norm(got_o - want_o, axis=-1), np.linalg.norm(want_o, axis=-1)
            assert np.all(num <= 2e-2 * den + 1e-3)                                                  # per-vector relative
            t = r.n_ctx + r.n_query
            assert np.array_equal(_f64(dw.v_fused[b, :t]), ref2["v_fused"][:, kv])
            kf, want = _f64(dw.k_fused[b, :t]), ref2["k_fused"][:, kv]
            ulp = np.ldexp(1.0, np.frexp(np.abs(want))[1] - 8)
            assert np.all(np.abs(kf - want) <= np.maximum(2e-2, ulp))
    if exchange == "fused":
        # a second step on the same buffers (a1 restores the stitched PIC keys): the epoch moves on — flags left from the
        # first step do not satisfy it — and the same selection comes out
        for st, dw in zip(steps, dws):
            st.score_phase(dw.batch, k_pool=dw.k_pool, v_pool=dw.v_pool, k_fused=dw.k_fused, v_fused=dw.v_fused,
                           q_probe=dw.q_probe, scores=dw.scores)
        sel_again = torch.zeros_like(dws[0].sel)
        steps[0].ctx.qcf_select_topk(dws[0].batch, None, cfg.ratio, sel_again, dws[0].n_sel)
        torch.cuda.synchronize()
        for b in range(dws[0].B):
            kb = int(dws[0].n_sel[b])
            assert torch.equal(sel_again[b, :kb], dws[0].sel[b, :kb])


def _swap_probe(wl):
    """Same requests with ANOTHER probe: the query rows of q_new stand in for q_probe (same shape, same positions)."""
    import copy
    wl2 = copy.copy(wl)
    wl2.requests = [copy.copy(r) for r in wl.requests]
    for r in wl2.requests:
        r.q_probe = np.ascontiguousarray(r.q_new[r.n_ctx: r.n_ctx + r.n_query])
    return wl2


@pytest.mark.parametrize("name", ["t_mid", "t_batch"])
def test_fused_exchange_rank_running_a_step_ahead(name):
    """The write-after-read case of the fused exchange (include/qcf.h, protocol invariant): rank A runs a1 + a2 of step i AND
    of step i + 1 (another probe, so other scores) before rank B has run a3 of step i.  With one slot per rank, A's second a2
    would overwrite what B is about to rank and the ranks would silently select different P.  With the slot sets indexed by
    epoch parity B still ranks step i's scores: B's P_i equals A's P_i and the oracle's on step-i inputs; both ranks then
    select the same P_{i+1}, the oracle's on step-(i+1) inputs.  A third step makes A's a2 pass the acknowledgement wait."""
    _, device, sharded = _mods()
    wl = inputs.make_workload(name)
    wl2 = _swap_probe(wl)
    cfg = wl.cfg
    world = 2
    steps, dws = _ranks(wl, world)
    dws2 = [device.DeviceWorkload(inputs.shard_heads(wl2, rank, world), st.ctx) for rank, st in enumerate(steps)]
    slot = dws[0].batch.batch * dws[0].batch.n_stride
    bufs = [sharded.HeadShardedStep.alloc_exchange_buffer(world, slot) for _ in range(world)]
    for st in steps:
        st.enable_fused_exchange(bufs, slot)
    A, B = 0, 1

    def score(rank, dw):
        steps[rank].score_phase(dw.batch, k_pool=dw.k_pool, v_pool=dw.v_pool, k_fused=dw.k_fused, v_fused=dw.v_fused,
                                q_probe=dw.q_probe, scores=dw.scores)

    def select(rank, dw):
        steps[rank].ctx.qcf_select_topk(dw.batch, None, cfg.ratio, dw.sel, dw.n_sel)

    score(A, dws[A]); score(B, dws[B])                 # step i on both ranks
    select(A, dws[A])                                  # A: a3 of step i ...
    score(A, dws2[A])                                  # ... and already a1 + a2 of step i + 1 (B has not selected yet)
    select(B, dws[B])                                  # B: a3 of step i — must still see step i's scores
    score(B, dws2[B])
    select(A, dws2[A]); select(B, dws2[B])             # step i + 1 on both
    score(A, dws[A])                                   # step i + 2: A's a2 waits for B's ack of step i (already there)
    score(B, dws[B])
    sel3 = torch.zeros_like(dws[A].sel)
    n3 = torch.zeros_like(dws[A].n_sel)
    steps[A].ctx.qcf_select_topk(dws[A].batch, None, cfg.ratio, sel3, n3)
    torch.cuda.synchronize()
    for step_wl, step_dws in ((wl, dws), (wl2, dws2)):
        for b, r in enumerate(step_wl.requests):
            k_pic = [O.widen_bf16(step_wl.pool_k[i]) for i in r.chunk_ids]
            ref = O.layer_step(k_pic, [O.widen_bf16(step_wl.pool_v[i]) for i in r.chunk_ids], cfg.rope_theta,
                               O.widen_bf16(r.q_probe), cfg.ratio, O.widen_bf16(r.q_new), O.widen_bf16(r.k_new),
                               O.widen_bf16(r.v_new))
            k = int(step_dws[A].n_sel[b])
            assert k == len(ref["sel"]) and int(step_dws[B].n_sel[b]) == k
            sel_a = step_dws[A].sel[b, :k].cpu().numpy().astype(np.int64)
            assert np.array_equal(step_dws[B].sel[b, :k].cpu().numpy(), sel_a), "the ranks selected different P"
            _check_selection(sel_a, ref["scores"], k)
    # the two probes really rank differently (else the test would pass with the hazard in place)
    assert any(not torch.equal(dws[A].sel[b, : int(dws[A].n_sel[b])], dws2[A].sel[b, : int(dws2[A].n_sel[b])])
               for b in range(dws[A].B))
    # step i + 2 repeats step i's inputs: same selection
    for b in range(dws[A].B):
        kb = int(n3[b])
        assert kb == int(dws[A].n_sel[b]) and torch.equal(sel3[b, :kb], dws[A].sel[b, :kb])


def test_head_sharded_full_size_c2_matches_the_unsharded_step():
    """BASELINE configs[1] at full size, two shards, against the UNSHARDED CUDA step on the same inputs (itself checked
    against the oracle in tests/test_gpu_parity.py): the summed partial scores agree to fp32 rounding, the selection is
    the same up to near-ties (north_star: >= 99 % overlap), and with the same selection forced on both sides every
    head's attention output and fused cache is bit-identical (same kernels, same per-kv-head tiles)."""
    binding, device, _ = _mods()
    wl = inputs.make_workload("c2")
    cfg = wl.cfg
    ctx = binding.Context(cfg.n_q_heads, cfg.n_kv_heads, cfg.head_dim, cfg.rope_theta, 1, cfg.n_ctx, cfg.n_query)
    ref = device.DeviceWorkload(wl, ctx)
    ctx.qcf_layer_step(ref.batch, ref.layer_args())
    torch.cuda.synchronize()
    steps, dws = _ranks(wl, 2)
    scores = dws[0].scores
    for rank, (st, dw) in enumerate(zip(steps, dws)):
        st.score_phase(dw.batch, k_pool=dw.k_pool, v_pool=dw.v_pool, k_fused=dw.k_fused, v_fused=dw.v_fused,
                       q_probe=dw.q_probe, scores=scores, accumulate=rank > 0)
    torch.cuda.synchronize()
    n = cfg.n_ctx
    np.testing.assert_allclose(scores[0, :n].cpu().numpy(), ref.scores[0, :n].cpu().numpy(), rtol=1e-5, atol=1e-12)
    k = int(ref.n_sel[0])
    steps[0].ctx.qcf_select_topk(dws[0].batch, scores, cfg.ratio, dws[0].sel, dws[0].n_sel)
    torch.cuda.synchronize()
    assert int(dws[0].n_sel[0]) == k
    assert len(np.intersect1d(dws[0].sel[0, :k].cpu().numpy(), ref.sel[0, :k].cpu().numpy())) >= 0.99 * k
    g = cfg.n_q_heads // cfg.n_kv_heads
    per = cfg.n_kv_heads // 2
    for rank, (st, dw) in enumerate(zip(steps, dws)):
        st.fuse_phase(dw.batch, scores=scores, sel=ref.sel, n_sel=ref.n_sel, q_new=dw.q_new, k_new=dw.k_new, v_new=dw.v_new,
                      k_fused=dw.k_fused, v_fused=dw.v_fused, out=dw.out, ratio=cfg.ratio, select_now=False)
        torch.cuda.synchronize()
        n_r = k + cfg.n_query
        assert torch.equal(dw.out[0, :n_r], ref.out[0, :n_r, rank * per * g:(rank + 1) * per * g])
        assert torch.equal(dw.k_fused[0], ref.k_fused[0][:, rank * per:(rank + 1) * per])
        assert torch.equal(dw.v_fused[0], ref.v_fused[0][:, rank * per:(rank + 1) * per])


def test_head_shards_restore_and_reject():
    binding, device, _ = _mods()
    wl = inputs.make_workload("t_mid")
    cfg = wl.cfg
    ctx = binding.Context(cfg.n_q_heads, cfg.n_kv_heads, cfg.head_dim, cfg.rope_theta, 1, 1024, cfg.n_query)
    dw = device.DeviceWorkload(wl, ctx)
    ctx.qcf_rope_reposition(dw.batch, dw.k_pool, dw.v_pool, dw.k_fused, dw.v_fused)
    ctx.qcf_score(dw.batch, dw.q_probe, dw.k_fused, dw.scores)
    s1 = dw.scores.clone()
    ctx.qcf_set_head_shards(4)
    ctx.qcf_score(dw.batch, dw.q_probe, dw.k_fused, dw.scores)
    assert torch.equal(dw.scores * 4, s1)                               # a power-of-two rescale is exact
    ctx.qcf_set_head_shards(1)
    ctx.qcf_score(dw.batch, dw.q_probe, dw.k_fused, dw.scores)
    assert torch.equal(dw.scores, s1)
    for bad in (0, -1, 65):
        with pytest.raises(binding.QcfError):
            ctx.qcf_set_head_shards(bad)


def test_layer_step_through_a_nccl_group_of_one():
    """The collective call itself (NCCL, one rank: the sum is the identity) inside the chained step."""
    import torch.distributed as dist
    _, device, sharded = _mods()
    wl = inputs.make_workload("t_mid")
    cfg = wl.cfg
    os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
    os.environ.setdefault("MASTER_PORT", "29617")
    created = not dist.is_initialized()
    if created:
        dist.init_process_group("nccl", rank=0, world_size=1)
    try:
        st = sharded.HeadShardedStep(cfg.n_q_heads, cfg.n_kv_heads, cfg.head_dim, cfg.rope_theta, 1, 1024, cfg.n_query)
        dw = device.DeviceWorkload(wl, st.ctx)
        st.layer_step(dw.batch, k_pool=dw.k_pool, v_pool=dw.v_pool, k_fused=dw.k_fused, v_fused=dw.v_fused,
                      q_probe=dw.q_probe, scores=dw.scores, sel=dw.sel, n_sel=dw.n_sel, q_new=dw.q_new, k_new=dw.k_new,
                      v_new=dw.v_new, out=dw.out, ratio=cfg.ratio)
        torch.cuda.synchronize()
        sel_a, out_a = dw.sel.clone(), dw.out.clone()
        dw2 = device.DeviceWorkload(wl, st.ctx)
        st.ctx.qcf_layer_step(dw2.batch, dw2.layer_args())
        torch.cuda.synchronize()
        assert torch.equal(sel_a, dw2.sel) and torch.equal(out_a, dw2.out)   # same kernels, same order: bit-identical
    finally:
        if created:
            dist.destroy_process_group()


# ----------------------------------------------------------------------------------------------- two processes, one GPU, CUDA IPC

def _ipc_rank(rank, world, name, port, q_res):
    """One rank of the fused-exchange step in its own PROCESS (own CUDA context).  Rendezvous exactly as production does it
    (sharded.share_exchange_buffers: CUDA IPC handles carried by torch.distributed, here a gloo group); phases are ordered on
    the host so that no kernel ever waits on a flag another process has not written yet (B200_PROFILING.md: ranks that
    spin on one another must not share a GPU)."""
    import torch
    import torch.distributed as dist
    from paper_2606_05875_b200 import device, inputs, sharded
    torch.cuda.set_device(0)
    dist.init_process_group("gloo", init_method="tcp://127.0.0.1:%d" % port, rank=rank, world_size=world)
    wl = inputs.make_workload(name)
    cfg = wl.cfg
    st = sharded.HeadShardedStep(cfg.n_q_heads, cfg.n_kv_heads, cfg.head_dim, cfg.rope_theta, max(cfg.batch, 1),
                                 max(cfg.n_ctx, 1024), max(cfg.n_query, 1), rank=rank, world=world)
    dw = device.DeviceWorkload(inputs.shard_heads(wl, rank, world), st.ctx)
    slot = dw.batch.batch * dw.batch.n_stride
    mine = sharded.HeadShardedStep.alloc_exchange_buffer(world, slot)
    st.enable_fused_exchange(sharded.share_exchange_buffers(mine, rank, world), slot)     # peers mapped with cudaIpc*
    dist.barrier()
    for turn in range(world):                     # a2 of one rank at a time (peer stores + flag release), host-ordered
        if turn == rank:
            st.score_phase(dw.batch, k_pool=dw.k_pool, v_pool=dw.v_pool, k_fused=dw.k_fused, v_fused=dw.v_fused,
                           q_probe=dw.q_probe, scores=dw.scores)
            torch.cuda.synchronize()
        dist.barrier()
    st.fuse_phase(dw.batch, scores=None, sel=dw.sel, n_sel=dw.n_sel, q_new=dw.q_new, k_new=dw.k_new, v_new=dw.v_new,
                  k_fused=dw.k_fused, v_fused=dw.v_fused, out=dw.out, ratio=cfg.ratio)      # a3 acquires flags already set
    torch.cuda.synchronize()
    q_res.put((rank, dw.n_sel.cpu().numpy(), dw.sel.cpu().numpy(), st.exchanged_scores(dw.batch).cpu().numpy(),
               dw.out.cpu().view(torch.int16).numpy()))
    dist.barrier()                                # keep the exported buffers alive until every peer is done
    dist.destroy_process_group()


def test_fused_exchange_two_processes_one_gpu_cuda_ipc():
    """the score exchange over PEER memory.  Two processes (two CUDA contexts) on the one GPU
    of this box map each other's exchange buffers through CUDA IPC handles; each rank's a2 stores its partial scores
    into both buffers and releases its flag; each rank's a3 acquires both flags and ranks the slot sum.  Checked against
    the oracle of the UNSHARDED layer: scores 1e-2 relative, the north-star selection rule, both ranks the same P."""
    import torch.multiprocessing as mp
    name, world = "t_mid", 2
    ctx = mp.get_context("spawn")
    q_res = ctx.Queue()
    procs = [ctx.Process(target=_ipc_rank, args=(r, world, name, 29747, q_res)) for r in range(world)]
    for p in procs:
        p.start()
    try:
        res = {}
        for _ in range(world):
            r, n_sel, sel, sc, out = q_res.get(timeout=300)
            res[r] = (n_sel, sel, sc, out)
    finally:
        for p in procs:
            p.join(timeout=60)
            if p.is_alive():
                p.kill()
    assert all(p.exitcode == 0 for p in procs)
    wl = inputs.make_workload(name)
    cfg = wl.cfg
    r0 = wl.requests[0]
    k_pic = [O.widen_bf16(wl.pool_k[i]) for i in r0.chunk_ids]
    v_pic = [O.widen_bf16(wl.pool_v[i]) for i in r0.chunk_ids]
    ref = O.layer_step(k_pic, v_pic, cfg.rope_theta, O.widen_bf16(r0.q_probe), cfg.ratio, O.widen_bf16(r0.q_new),
                       O.widen_bf16(r0.k_new), O.widen_bf16(r0.v_new))
    k = int(res[0][0][0])
    assert k == len(ref["sel"]) == int(res[1][0][0])
    assert np.array_equal(res[0][2], res[1][2]), "both ranks hold bit-identical slot sums"
    np.testing.assert_allclose(res[0][2][0, : r0.n_ctx].astype(np.float64), ref["scores"], rtol=1e-2, atol=0)
    sel0 = res[0][1][0, :k].astype(np.int64)
    assert np.array_equal(sel0, res[1][1][0, :k])
    _check_selection(sel0, ref["scores"], k)
    # a5 of each rank's heads against the oracle on that selection
    ref2 = O.layer_step(k_pic, v_pic, cfg.rope_theta, None, 0.0, O.widen_bf16(r0.q_new), O.widen_bf16(r0.k_new),
                        O.widen_bf16(r0.v_new), sel=sel0)
    g = cfg.n_q_heads // cfg.n_kv_heads
    per = cfg.n_kv_heads // world
    n_r = k + r0.n_query
    for rank in range(world):
        got = O.widen_bf16(res[rank][3].view(np.uint16))[0, :n_r]
        assert np.max(np.abs(got - ref2["out"][:, rank * per * g:(rank + 1) * per * g])) <= 2e-2
