"""Host side of the KV-head-sharded step (paper_2606_05875_b200/sharded.py) on CPU: the head partition, and — on a
two-rank gloo group — that the all-reduce of per-rank partial scores is Eq. 18 over all heads and leaves every rank
with the same selection.  The per-rank arithmetic here is the ORACLE's (tests may use it); the CUDA path is checked
against the same identities in tests/test_gpu_sharded.py.
"""
import numpy as np
import pytest

from oracle import qcf_oracle as O
from paper_2606_05875_b200 import inputs, sharded


def test_head_slice_partitions_the_heads():
    for hq, hkv, world in [(32, 8, 1), (32, 8, 2), (32, 8, 8), (64, 8, 4), (4, 2, 2)]:
        g = hq // hkv
        seen_q, seen_kv = [], []
        for rank in range(world):
            q, kv = sharded.head_slice(rank, world, hq, hkv)
            seen_q += list(range(hq))[q]
            seen_kv += list(range(hkv))[kv]
            assert all(h // g in range(hkv)[kv] for h in range(hq)[q])        # a rank owns the q heads of ITS kv-heads
        assert seen_q == list(range(hq)) and seen_kv == list(range(hkv))
    for bad in [(0, 3, 32, 8), (2, 2, 32, 8), (-1, 2, 32, 8)]:
        with pytest.raises(ValueError):
            sharded.head_slice(*bad)


def test_shard_heads_slices_every_tensor():
    wl = inputs.make_workload("t_mid")
    parts = [inputs.shard_heads(wl, r, 4) for r in range(4)]
    for r, p in enumerate(parts):
        assert p.cfg.n_kv_heads == wl.cfg.n_kv_heads // 4 and p.cfg.n_q_heads == wl.cfg.n_q_heads // 4
    for name in ("q_probe", "q_new", "k_new", "v_new"):
        assert np.array_equal(np.concatenate([getattr(p.requests[0], name) for p in parts], axis=1),
                              getattr(wl.requests[0], name))
    assert np.array_equal(np.concatenate([p.pool_k[1] for p in parts], axis=1), wl.pool_k[1])


def _worker(rank, world, port):
    import torch
    import torch.distributed as dist
    dist.init_process_group("gloo", init_method="tcp://127.0.0.1:%d" % port, rank=rank, world_size=world)
    wl = inputs.make_workload("t_mid")
    mine = inputs.shard_heads(wl, rank, world)
    r_all, r = wl.requests[0], mine.requests[0]
    k_ctx, _ = O.reposition([O.widen_bf16(mine.pool_k[i]) for i in r.chunk_ids],
                            [O.widen_bf16(mine.pool_v[i]) for i in r.chunk_ids], wl.cfg.rope_theta)
    # the rank's partial of Eq. 18: mean over ITS heads, weighted by its share of the layer's heads
    part = O.score(O.widen_bf16(r.q_probe), k_ctx) / world
    t = torch.from_numpy(part.copy())
    sharded.all_reduce_scores(t, world)
    k_full, _ = O.reposition([O.widen_bf16(wl.pool_k[i]) for i in r_all.chunk_ids],
                             [O.widen_bf16(wl.pool_v[i]) for i in r_all.chunk_ids], wl.cfg.rope_theta)
    want = O.score(O.widen_bf16(r_all.q_probe), k_full)
    np.testing.assert_allclose(t.numpy(), want, rtol=1e-12, atol=0)
    k = O.n_select(r_all.n_ctx, wl.cfg.ratio)
    sel = torch.from_numpy(O.select_topk(t.numpy(), k).astype(np.int64))
    gathered = [torch.zeros_like(sel) for _ in range(world)]
    dist.all_gather(gathered, sel)
    assert all(torch.equal(g, gathered[0]) for g in gathered)                # replicated a3: same P everywhere
    assert np.array_equal(sel.numpy(), O.select_topk(want, k))
    dist.barrier()
    dist.destroy_process_group()


def test_score_all_reduce_two_gloo_ranks():
    import torch.multiprocessing as mp
    mp.spawn(_worker, args=(2, 29741), nprocs=2, join=True)


def test_score_exchange_buffer_size_is_header_plus_slots():
    """include/qcf.h, qcf_score_exchange_bytes: 64 uint32 flags + 64 uint32 acks in front of TWO slot sets (epoch parity)
    of n_shards slots of slot_elems fp32 (pure host arithmetic, no device needed)."""
    from paper_2606_05875_b200 import binding
    assert binding.qcf_score_exchange_bytes(2, 1000) == 128 * 4 + 2 * 2 * 1000 * 4
    assert binding.qcf_score_exchange_bytes(8, 16 * 8192) == 512 + 2 * 8 * 16 * 8192 * 4
    assert binding.qcf_score_exchange_bytes(0, 10) == -1 and binding.qcf_score_exchange_bytes(65, 10) == -1
    assert binding.qcf_score_exchange_bytes(2, -1) == -1


def _bench_worker(rank, world, port):
    import torch.distributed as dist
    import bench
    dist.init_process_group("gloo", init_method="tcp://127.0.0.1:%d" % port, rank=rank, world_size=world)
    # the replica mode of bench.py (N > 1): every rank times its own replica, the line reports the MAX over ranks
    got = bench.max_over_ranks([10.0 + rank, 5.0 - rank, 7.0], dist, "cpu")
    assert got == [10.0 + world - 1, 5.0, 7.0]
    dist.barrier()
    dist.destroy_process_group()


def test_bench_takes_the_max_over_ranks_two_gloo_ranks():
    import torch.multiprocessing as mp
    mp.spawn(_bench_worker, args=(2, 29743), nprocs=2, join=True)
