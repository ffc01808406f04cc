// a3 — Eq. 11: P = TopK(I(t), floor(rho N)) over all context positions of a request.
//
// Exact integer selection: the fp32 score is mapped to an order-preserving uint32 key, a 4-pass MSB-first 8-bit
// radix select finds the k-th largest key T and how many elements equal to T belong to the top-k, then one ordered
// sweep emits the selected positions in ascending order (ties at T go to the lowest positions — reading (h)).
// One CTA per request: N <= 32768 scores are 128 KB, L1/L2-resident after the first pass; the stage is latency-
// bound, not bandwidth-bound.
#include "qcf_internal.cuh"

namespace qcf {

namespace {

constexpr int kThreads = 1024;

__device__ __forceinline__ uint32_t order_key(float f) {
  uint32_t u = __float_as_uint(f);
  if (u == 0x80000000u) u = 0u;                                  // -0 == +0
  return (u & 0x80000000u) ? ~u : (u | 0x80000000u);             // ascending in the value
}

// Fused exchange of the KV-head-sharded step (include/qcf.h, qcf_set_score_exchange): the scores are the sum, in slot
// order, of `world` slots of this rank's exchange buffer, each written by one rank's a2; flag[p] >= epoch says rank p's
// slot is complete.
struct Exch {
  const float* buf;        // nullptr: plain scores; else this rank's exchange buffer (flags in front)
  const float* slots;      // slot 0 of the slot set of this epoch's parity
  int world;
  long long slot_elems;
  unsigned int epoch;
};

// EXCH is a template parameter so that the plain kernel's sweeps keep their simple loop bodies (with the slot path as a
// run-time branch inside them the plain top-k went 36 -> 54 us at N = 32768).
template <bool EXCH>
__global__ void __launch_bounds__(kThreads) topk_kernel(BatchDev bd, const float* __restrict__ scores, double ratio,
                                                        int32_t* __restrict__ sel, int32_t* __restrict__ n_sel, int n_cached, int ceil_mode,
                                                        Exch ex) {
  extern __shared__ uint32_t s_keys[];                           // order keys of the first n_cached scores
  __shared__ unsigned int hist[2][256];        // double-buffered: pass p + 1's bins are zeroed while pass p's are scanned
  __shared__ unsigned int s_prefix, s_remaining;
  __shared__ unsigned int warp_cnt[32], warp_cnt2[32];           // per-warp counts of keys > T and == T
  pdl_trigger();
  const int b = blockIdx.x;
  const int N = bd.n_ctx[b];
  pdl_wait();
  // floor(rho N + 1e-6) for the recompute set (Eq. 8, reading (g)); ceil(r_a N - 1e-6) for anchors (Eq. 14)
  const int k = ceil_mode ? min(N, static_cast<int>(ceil(ratio * static_cast<double>(N) - 1e-6)))
                          : static_cast<int>(floor(ratio * static_cast<double>(N) + 1e-6));
  const float* s = scores + static_cast<size_t>(b) * bd.n_stride;
  int32_t* out = sel + static_cast<size_t>(b) * bd.n_stride;
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  if (EXCH) {
    // acquire every rank's epoch (bounded: a peer that never arrives is a trap, not a hang)
    if (tid < ex.world) {
      const unsigned int* flag = reinterpret_cast<const unsigned int*>(ex.buf) + tid;
      const long long t0 = clock64();
      unsigned int v;
      do {
        asm volatile("ld.acquire.sys.global.u32 %0, [%1];" : "=r"(v) : "l"(flag) : "memory");
        if (static_cast<int>(v - ex.epoch) >= 0) break;
        if (clock64() - t0 > 4000000000LL) __trap();
      } while (true);
    }
    __syncthreads();
  }
  // score of position i: plain, or the slot sum in fixed order
  auto score_at = [&](int i) -> float {
    if (!EXCH) return __ldcg(s + i);
    const float* p = ex.slots + static_cast<size_t>(b) * bd.n_stride + i;
    float acc = __ldcg(p);
    for (int q = 1; q < ex.world; ++q) acc += __ldcg(p + static_cast<size_t>(q) * ex.slot_elems);
    return acc;
  };
  if (tid == 0) n_sel[b] = k;
  if (k <= 0) return;
  if (k >= N) {
    for (int i = tid; i < N; i += kThreads) out[i] = i;
    return;
  }

  // the five sweeps below read every score; one coalesced global read fills shared memory, the rest stay on chip
  const int n_sm_keys = min(N, n_cached);
  for (int i = tid; i < n_sm_keys; i += kThreads) s_keys[i] = order_key(score_at(i));
  auto key_of = [&](int i) -> uint32_t { return i < n_sm_keys ? s_keys[i] : order_key(score_at(i)); };
  if (tid < 256) hist[0][tid] = 0u;
  if (tid == 0) { s_prefix = 0u; s_remaining = static_cast<unsigned int>(k); }
  __syncthreads();

  // ---- radix select: after pass p the top 8(p+1) bits of the k-th largest key are known
#pragma unroll 1
  for (int pass = 0; pass < 4; ++pass) {
    const int shift = 24 - 8 * pass;
    unsigned int* h = hist[pass & 1];
    const uint32_t prefix = s_prefix;
    const uint32_t mask = pass == 0 ? 0u : (0xffffffffu << (shift + 8));
    for (int i = tid; i < N; i += kThreads) {
      const uint32_t key = key_of(i);
      // (warp-aggregating these atomics with match.any was measured: 12.6 -> 16.7 us on c2, 41 -> 63 us on c5)
      if ((key & mask) == prefix) atomicAdd(&h[(key >> shift) & 0xffu], 1u);
    }
    __syncthreads();
    if (warp >= 1 && warp <= 8) hist[(pass + 1) & 1][tid - 32] = 0u;        // the next pass's bins
    if (warp == 0) {
      // bins from the top: find the digit where the cumulative count reaches `remaining`
      const unsigned int remaining = s_remaining;
      unsigned int cnt[8], tot = 0;
#pragma unroll
      for (int j = 0; j < 8; ++j) { cnt[j] = h[255 - (lane * 8 + j)]; tot += cnt[j]; }
      unsigned int incl = tot;
#pragma unroll
      for (int o = 1; o < 32; o <<= 1) {
        const unsigned int v = __shfl_up_sync(0xffffffffu, incl, o);
        if (lane >= o) incl += v;
      }
      unsigned int run = incl - tot;                             // elements in higher bins than this lane's
      if (run < remaining && incl >= remaining) {
#pragma unroll
        for (int j = 0; j < 8; ++j) {
          if (run + cnt[j] >= remaining) {
            s_prefix = prefix | (static_cast<uint32_t>(255 - (lane * 8 + j)) << shift);
            s_remaining = remaining - run;
            break;
          }
          run += cnt[j];
        }
      }
    }
    __syncthreads();
  }
  const uint32_t T = s_prefix;
  const unsigned int need = s_remaining;                         // elements equal to T that are selected (>= 1)

  // ---- ordered emission: position of element i = #(key > T before i) + min(#(key == T before i), need).
  // Warp w owns the contiguous block [w * rows * 32, (w + 1) * rows * 32) and walks it in rows of 32 (lane = element, so
  // shared-memory and global accesses stay conflict-free / coalesced): a counting sweep, ONE block-level exchange of the
  // 32 warp totals, then an emitting sweep with running offsets.
  const int rows = ((N + 31) / 32 + 31) / 32;                    // rows of 32 elements per warp
  const int base = warp * rows * 32;
  unsigned int wg = 0, we = 0;
  for (int j = 0; j < rows; ++j) {
    const int i = base + j * 32 + lane;
    const uint32_t key = i < N ? key_of(i) : 0u;
    wg += __popc(__ballot_sync(0xffffffffu, i < N && key > T));
    we += __popc(__ballot_sync(0xffffffffu, i < N && key == T));
  }
  if (lane == 0) { warp_cnt[warp] = wg; warp_cnt2[warp] = we; }
  __syncthreads();
  unsigned int run_gt, run_eq;
  {
    const unsigned int vg = warp_cnt[lane], ve = warp_cnt2[lane];
    unsigned int ig = vg, ie = ve;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
      const unsigned int ug = __shfl_up_sync(0xffffffffu, ig, o), ue = __shfl_up_sync(0xffffffffu, ie, o);
      if (lane >= o) { ig += ug; ie += ue; }
    }
    run_gt = __shfl_sync(0xffffffffu, ig - vg, warp);
    run_eq = __shfl_sync(0xffffffffu, ie - ve, warp);
  }
  const unsigned int lt_mask = (1u << lane) - 1u;
  for (int j = 0; j < rows; ++j) {
    const int i = base + j * 32 + lane;
    const uint32_t key = i < N ? key_of(i) : 0u;
    const bool gt = i < N && key > T, eq = i < N && key == T;
    const unsigned int bg = __ballot_sync(0xffffffffu, gt), be = __ballot_sync(0xffffffffu, eq);
    const unsigned int gt_before = run_gt + __popc(bg & lt_mask), eq_before = run_eq + __popc(be & lt_mask);
    if (gt || (eq && eq_before < need)) out[gt_before + min(eq_before, need)] = i;
    run_gt += __popc(bg);
    run_eq += __popc(be);
  }
}

}  // namespace

cudaError_t launch_topk(const qcf_ctx* ctx, const qcf_batch* b, const float* scores, double ratio, int32_t* sel,
                        int32_t* n_sel, cudaStream_t stream, int ceil_mode) {
  if (b->batch == 0) return cudaSuccess;
  // up to 48 K keys (192 KB) are cached in shared memory; longer contexts read the remainder from L2
  const int n_cached = b->n_stride < 49152 ? b->n_stride : 49152;
  const size_t smem = static_cast<size_t>(n_cached) * sizeof(uint32_t);
  // per device / context, so set on every launch (as the other launchers do) rather than once per process
  cudaFuncSetAttribute(topk_kernel<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, 49152 * 4);
  cudaFuncSetAttribute(topk_kernel<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, 49152 * 4);
  Exch ex{nullptr, nullptr, 1, 0, 0u};
  if (ctx->exch_world > 1 && !ceil_mode) {     // (the anchor ranking of Phase I is never sharded)
    ex.buf = ctx->exch_peers_host[ctx->exch_rank];
    ex.world = ctx->exch_world;
    ex.slot_elems = ctx->exch_slot_elems;
    ex.epoch = ctx->exch_epoch;
    ex.slots = ex.buf + kExchHeaderElems + static_cast<size_t>(ex.epoch & 1u) * ex.world * ex.slot_elems;
    return launch_pdl(ctx->pdl, topk_kernel<true>, dim3(b->batch), dim3(kThreads), smem, stream, b->dev, scores, ratio, sel, n_sel, n_cached, ceil_mode, ex);
  }
  return launch_pdl(ctx->pdl, topk_kernel<false>, dim3(b->batch), dim3(kThreads), smem, stream, b->dev, scores, ratio, sel, n_sel, n_cached, ceil_mode, ex);
}

}  // namespace qcf
