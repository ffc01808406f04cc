"""KV-head-sharded layer step: one layer of the QCFuse step split over `world` ranks by
kv-head groups.  a1, a4 and a5 are independent per kv-head; a2 is a sum over heads (Eq. 18), so each
rank computes the partial of I(t) over ITS heads (qcf_set_head_shards makes qcf_score normalise by the whole layer's
Hq) and one all-reduce(sum) of scores[B][n_stride] fp32 — the only exchange of the step — gives every rank the same
I(t); a3 then runs replicated, so all ranks select the same P without a broadcast.

Plumbing only: the step's arithmetic is the C-ABI calls of include/qcf.h on the rank's head slices.  Two exchanges:
  * "fused" (enable_fused_exchange): a2's combine CTAs store the rank's partial straight into every peer's exchange
    buffer over peer memory (NVLink P2P or CUDA IPC mappings), a flag publishes the epoch, a3 acquires the flags and
    sums the slots in fixed order — no collective call, no host round trip (include/qcf.h, qcf_set_score_exchange);
  * "nccl" (default): torch.distributed.all_reduce on the caller's process group between the two launches — the
    baseline the fused path replaces.
torch.distributed is then only the rendezvous (exchanging the buffer handles).  With world == 1 nothing is exchanged.  Default deployments shard REQUESTS instead (replicas, no collective — DESIGN.md section 8); this module is
for a single long request that must be spread over GPUs.
"""
from __future__ import annotations

from typing import Optional, Sequence, Tuple

from . import binding


def head_slice(rank: int, world: int, n_q_heads: int, n_kv_heads: int) -> Tuple[slice, slice]:
    """(q-head slice, kv-head slice) owned by `rank`: contiguous kv-head groups, each with its G = Hq/Hkv q heads
    (q-head h reads kv-head h // G, include/qcf.h conventions)."""
    if world < 1 or not 0 <= rank < world:
        raise ValueError("rank %d outside world %d" % (rank, world))
    if n_kv_heads % world or n_q_heads % n_kv_heads:
        raise ValueError("Hkv = %d must be divisible by the number of head shards %d" % (n_kv_heads, world))
    per = n_kv_heads // world
    g = n_q_heads // n_kv_heads
    return slice(rank * per * g, (rank + 1) * per * g), slice(rank * per, (rank + 1) * per)


def all_reduce_scores(scores, world: int, group=None, stream=None):
    """The step's one exchange: element-wise sum of the ranks' partial scores, in place, ordered on `stream`.
    Skipped only when there is nothing to exchange with (world == 1 and no process group initialised)."""
    import torch
    import torch.distributed as dist
    if world == 1 and not dist.is_initialized():
        return
    if stream is not None and scores.is_cuda:
        with torch.cuda.stream(stream):
            dist.all_reduce(scores, op=dist.ReduceOp.SUM, group=group)
    else:
        dist.all_reduce(scores, op=dist.ReduceOp.SUM, group=group)


def share_exchange_buffers(mine, rank: int, world: int, group=None):
    """Rendezvous of the fused exchange across PROCESSES (one rank per GPU): every rank exports its exchange buffer as a
    CUDA IPC handle (torch.multiprocessing's reduce_tensor: cudaIpcGetMemHandle + offset inside the allocation),
    torch.distributed carries the handles (all_gather_object — the only thing the process group is used for), and each
    rank maps its peers' buffers (cudaIpcOpenMemHandle; over NVLink when the peers sit on other GPUs).  Returns the list
    peer_bufs for HeadShardedStep.enable_fused_exchange; `mine` must stay alive while any peer uses it."""
    import torch.distributed as dist
    from torch.multiprocessing.reductions import reduce_tensor
    if world == 1:
        return [mine]
    import torch
    torch.cuda.synchronize(mine.device)       # the zero fill of `mine` has run before any peer can store into it
    handles = [None] * world
    dist.all_gather_object(handles, (mine.device.index, reduce_tensor(mine)), group=group)
    peers = []
    for p in range(world):
        if p == rank:
            peers.append(mine)
            continue
        dev_p, (fn, args) = handles[p]
        if dev_p != mine.device.index:
            # the kernels dereference the peer's buffer directly: peer access must be on (NVLink / NVSwitch P2P)
            if not torch.cuda.can_device_access_peer(mine.device.index, dev_p):
                raise RuntimeError("GPU %d cannot access GPU %d: the fused score exchange needs peer access" %
                                   (mine.device.index, dev_p))
            err = torch.cuda.cudart().cudaDeviceEnablePeerAccess(dev_p, 0)
            if int(err) not in (0, 704):                      # 704: cudaErrorPeerAccessAlreadyEnabled
                raise RuntimeError("cudaDeviceEnablePeerAccess(%d) failed: %s" % (dev_p, err))
        peers.append(fn(*args))
    # nobody starts an exchanging call before every rank holds every mapping (include/qcf.h, rule (1))
    dist.barrier(group=group)
    return peers


class HeadShardedStep:
    """The rank-local half of a KV-head-sharded qcf_layer_step.  Every tensor argument is this rank's head slice
    ([...][Hq/world][d] or [...][Hkv/world][d], contiguous); scores / sel / n_sel are full-size and end up identical on
    all ranks."""

    def __init__(self, n_q_heads: int, n_kv_heads: int, head_dim: int, rope_theta: float, max_batch: int, max_ctx: int,
                 max_query: int, rank: int = 0, world: int = 1, group=None, softmax_scale: float = 0.0):
        self.q_heads, self.kv_heads = head_slice(rank, world, n_q_heads, n_kv_heads)
        self.rank, self.world, self.group = rank, world, group
        # the scale must be the layer's, not a function of the local head count (it is 1/sqrt(d) by default: unchanged)
        self.ctx = binding.Context(n_q_heads // world, n_kv_heads // world, head_dim, rope_theta, max_batch, max_ctx,
                                   max_query, softmax_scale)
        self.ctx.qcf_set_head_shards(world)
        self.fused = False

    # ---- fused exchange (include/qcf.h, qcf_set_score_exchange)
    @staticmethod
    def alloc_exchange_buffer(world: int, slot_elems: int, device="cuda"):
        """This rank's exchange buffer: [64 flags][64 acks][2 slot sets x world slots x slot_elems] fp32, zeroed (the
        library requires that and clears nothing itself).  Share it with the peers
        (same process: pass the tensor; other processes: send it through torch.multiprocessing, which maps it with CUDA
        IPC; other GPUs: enable peer access and pass the pointer)."""
        import torch
        n = binding.qcf_score_exchange_bytes(world, slot_elems) // 4
        return torch.zeros(n, dtype=torch.float32, device=device)

    def enable_fused_exchange(self, peer_bufs: Sequence, slot_elems: int):
        """peer_bufs[p] = rank p's exchange buffer as visible from this process (peer_bufs[self.rank] is this rank's own)."""
        if len(peer_bufs) != self.world:
            raise ValueError("need one exchange buffer per rank")
        self.fused = self.world > 1
        self._exch = list(peer_bufs)
        self.slot_elems = int(slot_elems)
        self._epoch = 0                                # mirrors the ctx's count of exchanging qcf_score calls
        if self.fused:
            self.ctx.qcf_set_score_exchange(self.rank, self.world, self._exch, slot_elems)

    def exchanged_scores(self, b: binding.Batch):
        """The summed scores [B][n_stride] this rank's a3 ranks (slot order), for inspection."""
        buf = self._exch[self.rank]
        first = 128 + (self._epoch & 1) * self.world * self.slot_elems      # slot set of the newest epoch's parity
        slots = buf[first: first + self.world * self.slot_elems].view(self.world, self.slot_elems)[:, : b.batch * b.n_stride]
        acc = slots[0].clone()
        for p in range(1, self.world):
            acc += slots[p]
        return acc.view(b.batch, b.n_stride)

    def batch(self, chunk_lens, chunk_rows, n_query, chunk_pos=None) -> binding.Batch:
        return self.ctx.batch(chunk_lens, chunk_rows, n_query, chunk_pos)

    def all_reduce_scores(self, scores, stream=None):
        all_reduce_scores(scores, self.world, self.group, stream)

    def score_phase(self, b: binding.Batch, *, k_pool, v_pool, k_fused, v_fused, q_probe, scores,
                    is_critical_layer: bool = True, accumulate: bool = False, stream=None):
        """a1 -> [a2: this rank's partial of Eq. 18 into (or, with accumulate, onto) `scores`]."""
        self.ctx.qcf_rope_reposition(b, k_pool, v_pool, k_fused, v_fused, stream)
        if is_critical_layer:
            self.ctx.qcf_score(b, q_probe, k_fused, scores, accumulate, stream)
            if self.fused and b.total_ctx > 0:
                self._epoch += 1

    def fuse_phase(self, b: binding.Batch, *, scores, sel, n_sel, q_new, k_new, v_new, k_fused, v_fused, out, lse=None,
                   ratio: float = 0.0, rows_by_position: bool = True, select_now: bool = True, stream=None):
        """[a3 replicated on the summed scores] -> a4 + a5 on this rank's heads."""
        if select_now:
            self.ctx.qcf_select_topk(b, scores, ratio, sel, n_sel, stream)
        self.ctx.qcf_recompute_attn(b, sel, n_sel, q_new, k_new, v_new, rows_by_position, k_fused, v_fused, out, lse,
                                    stream)

    def layer_step(self, b: binding.Batch, *, k_pool, v_pool, k_fused, v_fused, q_probe, scores, sel, n_sel, q_new, k_new,
                   v_new, out, lse=None, ratio: float = 0.0, rows_by_position: bool = True,
                   is_critical_layer: bool = True, accumulate: bool = False, select_now: bool = True, stream=None):
        """a1 -> [a2 partial] -> [all-reduce -> a3 replicated] -> a4 + a5, the order of qcf_layer_step (Fig. 9,
        PAPER.md:337-344).  With accumulate the all-reduce is deferred to the layer that selects: the sum over critical
        layers (Eq. 20) commutes with the sum over ranks, so one exchange per request suffices."""
        self.score_phase(b, k_pool=k_pool, v_pool=v_pool, k_fused=k_fused, v_fused=v_fused, q_probe=q_probe, scores=scores,
                         is_critical_layer=is_critical_layer, accumulate=accumulate, stream=stream)
        if select_now and not self.fused:
            self.all_reduce_scores(scores, stream)        # fused: a2 already stored into every peer's buffer
        self.fuse_phase(b, scores=scores, sel=sel, n_sel=n_sel, q_new=q_new, k_new=k_new, v_new=v_new, k_fused=k_fused,
                        v_fused=v_fused, out=out, lse=lse, ratio=ratio, rows_by_position=rows_by_position,
                        select_now=select_now, stream=stream)
