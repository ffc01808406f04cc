// a5, persistent variant — PAPER.md:134: causal GQA attention of the recomputed rows R = P u U over the fused cache.
//
// Same tile math as recompute_attn_tc.cu (128 MMA rows = 128/G rows of R x G heads of one kv-head, 64-key tiles,
// S = Q K^T SS into double-buffered TMEM, O += P V TS, one softmax thread per row) but the grid is 2 CTAs per SM that
// WALK a device-built work list instead of one CTA per tile:
//   plan kernel   one CTA: per (request, row tile) the key-tile count, a split of heavy tiles into balanced key chunks
//                 (so that no unit is longer than ~half a CTA's fair share), units emitted heaviest first
//   warp 0        TMA producer, runs ahead across unit boundaries (K / V rings keep their phase)
//   warp 1        UMMA issuer
//   warps 2-5     softmax / correction / epilogue
//   warp 6        Q loader: gathers the NEXT unit's Q rows (cp.async) as soon as the last Q K^T of the current unit has
//                 completed, i.e. under the current unit's last softmax, P V and epilogue
// What this removes: the per-CTA prologue (TMEM allocation, barrier init, descriptor fetch, Q gather latency, pipeline
// fill) that every tile paid, the ~900 empty CTAs of a selective launch, and the 81-tile critical path of the heaviest
// tile.  Split units park (O, m, l) in a global workspace; the last chunk to arrive merges them in chunk order
// (deterministic).
//
// STATUS: opt-in (QCF_ATTN_IMPL=ptc), parity-green, but SLOWER than the one-CTA-per-tile kernel on every measured shape
// (c2 selective 150-170 us vs 112 us, c2 dense 290-320 us vs 254 us; static zig-zag or dynamic claiming, any split length;
// ncu: SMs active 91 % of the time but every pipe at about half the utilisation of recompute_attn_tc.cu, warps parked on
// mbarriers).  The cause is not understood yet; the default stays recompute_attn_tc.cu.
#include <cstdlib>

#include "qcf_internal.cuh"
#include "sm100_ptx.cuh"

namespace qcf {

namespace {

using namespace ptx;

constexpr int BM = 128;
constexpr int BN = 64;
constexpr int kStages = 2;
constexpr int kThreads = 224;       // producer, issuer, 4 softmax warps, Q loader
constexpr int kTmemCols = 256;
constexpr int kColO = 128;
constexpr int kMaxSplit = 4;
constexpr float kLog2e = 1.4426950408889634f;
constexpr float kLn2 = 0.6931471805599453f;
constexpr float kRescaleThreshold = 8.0f;

struct __align__(16) WorkUnit {
  int32_t b, g, tile, jt0;          // request, kv-head, row tile, first key tile
  int32_t n_kt, chunk, n_chunks;    // key tiles of this unit, chunk index / count of the item
  int32_t slot;                     // first partial slot of the item (split items), -1 otherwise
};

struct PlanOut {
  WorkUnit* units;
  int32_t* n_units;                 // device scalar
  unsigned int* next_unit;          // work counter of the attention kernel, reset here
  int max_units, max_slots;
};

__device__ __forceinline__ int row_pos(const BatchDev& bd, const int32_t* sel, int b, int N, int ns, int n_rows, int r) {
  if (r >= n_rows) return 0;
  if (!sel) return r;
  return r < ns ? __ldg(sel + static_cast<size_t>(b) * bd.n_stride + r) : N + (r - ns);
}

// One CTA.  Entry e = (tile descending, request): n_kt(e) key tiles.  S = chunk length such that a unit is at most about
// half of a resident CTA's fair share of the total; items longer than S are cut into ceil(n_kt / S) equal chunks.
__global__ void __launch_bounds__(1024) attn_plan_kernel(BatchDev bd, int hkv, int G, int max_tiles, int slots_resident, int split_div,
                                                         const int32_t* __restrict__ sel, const int32_t* __restrict__ n_sel,
                                                         PlanOut po) {
  __shared__ int s_red[32];
  __shared__ int s_total, s_S, s_off_units, s_off_slots;
  const int PT = BM / G;
  const int n_entries = max_tiles * bd.batch;
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  auto entry_kt = [&](int e) -> int {
    const int tile = max_tiles - 1 - e / bd.batch, b = e % bd.batch;
    const int N = bd.n_ctx[b], Lq = bd.n_query[b];
    const int ns = sel ? n_sel[b] : 0;
    const int n_rows = sel ? ns + Lq : N + Lq;
    if (tile * PT >= n_rows) return 0;
    const int p_max = row_pos(bd, sel, b, N, ns, n_rows, min(tile * PT + PT, n_rows) - 1);
    return p_max / BN + 1;
  };
  auto block_sum = [&](int v) -> int {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    if (lane == 0) s_red[warp] = v;
    __syncthreads();
    if (warp == 0) {
      int t = s_red[lane];
#pragma unroll
      for (int o = 16; o > 0; o >>= 1) t += __shfl_xor_sync(0xffffffffu, t, o);
      if (lane == 0) s_total = t;
    }
    __syncthreads();
    return s_total;
  };
  // key-tile counts of this thread's entries, kept in registers for the three passes (entries beyond 4096 are recomputed)
  int kt_reg[4];
#pragma unroll
  for (int k = 0; k < 4; ++k) kt_reg[k] = (tid + k * 1024 < n_entries) ? entry_kt(tid + k * 1024) : 0;
  auto kt_of = [&](int e) -> int {
    const int k = e >> 10;
    return k == 0 ? kt_reg[0] : (k == 1 ? kt_reg[1] : (k == 2 ? kt_reg[2] : (k == 3 ? kt_reg[3] : entry_kt(e))));
  };
  // ---- pass 1: total key-tile steps
  int my = 0;
  for (int e = tid; e < n_entries; e += blockDim.x) my += kt_of(e);
  const int total = block_sum(my) * hkv;
  if (tid == 0) {
    const int fair = (total + slots_resident - 1) / max(slots_resident, 1);
    s_S = max(8, (fair + split_div - 1) / split_div);
    s_off_units = 0;
    s_off_slots = 0;
  }
  __syncthreads();
  int S = s_S;
  // would the split need more partial slots than the workspace holds?  then do not split at all
  int need = 0;
  for (int e = tid; e < n_entries; e += blockDim.x) {
    const int kt = kt_of(e);
    const int nc = min(kMaxSplit, (kt + S - 1) / S);
    if (nc > 1) need += nc * hkv;
  }
  if (block_sum(need) > po.max_slots) S = 1 << 30;
  // ---- pass 2: emit units in entry order (heaviest tiles first); block-wide exclusive scan per sweep of 1024 entries
  for (int base = 0; base < n_entries; base += blockDim.x) {
    const int e = base + tid;
    const int kt = e < n_entries ? kt_of(e) : 0;
    const int nc = kt > 0 ? min(kMaxSplit, max(1, (kt + S - 1) / S)) : 0;
    const int n_u = nc * hkv, n_s = nc > 1 ? nc * hkv : 0;
    // inclusive scan of (n_u, n_s) packed in 64 bits
    unsigned long long v = (static_cast<unsigned long long>(n_u) << 32) | static_cast<unsigned int>(n_s);
    unsigned long long inc = v;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
      const unsigned long long t = __shfl_up_sync(0xffffffffu, inc, o);
      if (lane >= o) inc += t;
    }
    __shared__ unsigned long long s_w[32];
    if (lane == 31) s_w[warp] = inc;
    __syncthreads();
    if (warp == 0) {
      unsigned long long w = s_w[lane], wi = w;
#pragma unroll
      for (int o = 1; o < 32; o <<= 1) {
        const unsigned long long t = __shfl_up_sync(0xffffffffu, wi, o);
        if (lane >= o) wi += t;
      }
      s_w[lane] = wi - w;                                   // exclusive prefix of the warp totals
    }
    __syncthreads();
    const unsigned long long excl = s_w[warp] + inc - v;
    const int u0 = s_off_units + static_cast<int>(excl >> 32);
    const int s0 = s_off_slots + static_cast<int>(excl & 0xffffffffu);
    if (nc > 0 && u0 + n_u <= po.max_units) {
      const int tile = max_tiles - 1 - e / bd.batch, b = e % bd.batch;
      const int kb = kt / nc, kr = kt % nc;                 // chunk c has kb + (c < kr) key tiles
      for (int c = 0; c < nc; ++c)
        for (int g = 0; g < hkv; ++g) {
          WorkUnit w;
          w.b = b; w.g = g; w.tile = tile;
          w.jt0 = c * kb + min(c, kr);
          w.n_kt = kb + (c < kr ? 1 : 0);
          w.chunk = c; w.n_chunks = nc;
          w.slot = nc > 1 ? s0 + g * nc : -1;
          po.units[u0 + c * hkv + g] = w;
        }
    }
    __syncthreads();
    if (tid == blockDim.x - 1) {
      s_off_units += static_cast<int>((excl + v) >> 32);
      s_off_slots += static_cast<int>((excl + v) & 0xffffffffu);
    }
    __syncthreads();
  }
  if (tid == 0) {
    *po.n_units = min(s_off_units, po.max_units);
    *po.next_unit = 0u;
  }
}

template <int D>
struct Smem {
  static constexpr int kQBlk = BM * 128;
  static constexpr int kBlk = BN * 128;
  static constexpr int kQ = BM * D * 2;
  static constexpr int kTile = BN * D * 2;
  static constexpr int oQ = 0;
  static constexpr int oK = oQ + kQ;
  static constexpr int oV = oK + kStages * kTile;
  static constexpr int oBar = oV + kStages * kTile;
  static constexpr int kNumBar = 4 * kStages + 6 + 3 + 4;  // + q_full, q_empty, o_free, sched_full[2], sched_empty[2]
  static constexpr int oTmem = oBar + kNumBar * 8;
  static constexpr int oFlag = oTmem + 16;
  static constexpr int oSched = oFlag + 16;                 // unit ids published by the scheduler lane (2 slots)
  static constexpr int kBytes = oSched + 16;
};
enum { kFullK = 0, kEmptyK = kStages, kFullV = 2 * kStages, kEmptyV = 3 * kStages, kSFull = 4 * kStages,
       kPReady = 4 * kStages + 2, kODone = 4 * kStages + 4, kQFull = 4 * kStages + 6, kQEmpty = 4 * kStages + 7,
       kOFree = 4 * kStages + 8, kSchedFull = 4 * kStages + 9, kSchedEmpty = 4 * kStages + 11 };

struct AttnArgs {
  const WorkUnit* units;
  const int32_t* n_units;
  unsigned int* next_unit;    // global work counter, zeroed by the plan kernel
  int hq, hkv;
  float scale_log2;
  const int32_t* sel;
  const int32_t* n_sel;
  const __nv_bfloat16* q;
  int q_by_position;
  __nv_bfloat16* out;
  float* lse;
  float* part_o;              // [slot][D/4][BM] float4
  float* part_ml;             // [slot][2][BM]
  unsigned int* item_ctr;     // [max_tiles * hkv * B], zeroed, self-resetting
  int max_tiles;
};

template <int D>
__global__ void __launch_bounds__(kThreads, 2)
attn_ptc_kernel(const __grid_constant__ CUtensorMap tm_k, const __grid_constant__ CUtensorMap tm_v, BatchDev bd, AttnArgs a) {
  extern __shared__ unsigned char smem_raw[];
  unsigned char* smem = smem_raw + ((1024u - (smem_u32(smem_raw) & 1023u)) & 1023u);
  using S = Smem<D>;
  const int G = a.hq / a.hkv;
  const int PT = BM / G;
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const bool dense = a.sel == nullptr;
  const int n_units = __ldg(a.n_units);
  // Units are claimed dynamically from the heaviest-first list (greedy LPT): lane 0 of the Q-loader warp takes the next
  // index with one atomicAdd and publishes it through a 2-slot shared-memory ring; every other role reads it there.

  const uint32_t sbase = smem_u32(smem);
  const uint32_t sQ = sbase + S::oQ, sK = sbase + S::oK, sV = sbase + S::oV;
  auto bar = [&](int i) -> uint32_t { return sbase + S::oBar + 8 * i; };
  volatile uint32_t* tmem_slot = reinterpret_cast<volatile uint32_t*>(smem + S::oTmem);

  if (warp == 0) {
    if (lane == 0) {
      prefetch_tensormap(&tm_k);
      prefetch_tensormap(&tm_v);
      for (int i = 0; i < S::kNumBar; ++i)
        mbar_init(bar(i), (i == kPReady || i == kPReady + 1 || i == kOFree) ? 128
                          : ((i == kSchedEmpty || i == kSchedEmpty + 1) ? 130 : 1));
      fence_barrier_init();
    }
  } else if (warp == 1) {
    tmem_alloc<kTmemCols>(sbase + S::oTmem);
  }
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  const uint32_t tmem_base = *tmem_slot;
  const uint32_t tmem_o = tmem_base + kColO;

  volatile int* s_sched = reinterpret_cast<volatile int*>(smem + S::oSched);
  // consumer side of the ring: the i-th unit of this CTA (>= n_units: no more work)
  auto unit_of = [&](int i) -> int {
    mbar_wait(bar(kSchedFull + (i & 1)), (i >> 1) & 1);
    const int u = s_sched[i & 1];
    mbar_arrive(bar(kSchedEmpty + (i & 1)));
    return u;
  };
  struct Geo { int b, g, N, Lq, ns, n_rows, ridx0; };
  auto geo_of = [&](const WorkUnit& w) -> Geo {
    Geo r;
    r.b = w.b; r.g = w.g;
    r.N = bd.n_ctx[w.b]; r.Lq = bd.n_query[w.b];
    r.ns = dense ? 0 : a.n_sel[w.b];
    r.n_rows = dense ? r.N + r.Lq : r.ns + r.Lq;
    r.ridx0 = w.tile * PT;
    return r;
  };

  if (warp == 0) {
    // ===================================================================== TMA producer
    if (lane == 0) {
      int t = 0;
      for (int i = 0;; ++i) {
        const int u = unit_of(i);
        if (u >= n_units) break;
        const WorkUnit w = a.units[u];
        for (int j = 0; j < w.n_kt; ++j, ++t) {
          const int st = t % kStages;
          const uint32_t ph = (t / kStages) & 1;
          mbar_wait(bar(kEmptyK + st), ph ^ 1);
          mbar_arrive_expect_tx(bar(kFullK + st), S::kTile);
#pragma unroll
          for (int kb = 0; kb < D / 64; ++kb)
            tma_load_4d(sK + st * S::kTile + kb * S::kBlk, &tm_k, bar(kFullK + st), kb * 64, w.g, (w.jt0 + j) * BN, w.b);
          mbar_wait(bar(kEmptyV + st), ph ^ 1);
          mbar_arrive_expect_tx(bar(kFullV + st), S::kTile);
#pragma unroll
          for (int kb = 0; kb < D / 64; ++kb)
            tma_load_4d(sV + st * S::kTile + kb * S::kBlk, &tm_v, bar(kFullV + st), kb * 64, w.g, (w.jt0 + j) * BN, w.b);
        }
      }
    }
    __syncwarp();
  } else if (warp == 1) {
    // ===================================================================== UMMA issuer
    if (lane == 0) {
      constexpr uint32_t idesc_qk = umma_idesc_bf16(BM, BN, false, false);
      constexpr uint32_t idesc_pv = umma_idesc_bf16(BM, D, false, true);
      int t0 = 0;
      for (int i = 0;; ++i) {
        const int u = unit_of(i);
        if (u >= n_units) break;
        const int n_kt = a.units[u].n_kt;
        auto issue_qk = [&](int j) {
          const int t = t0 + j, st = t % kStages;
          mbar_wait(bar(kFullK + st), (t / kStages) & 1);
          tc_fence_after();
          const uint32_t d_tmem = tmem_base + (t & 1) * BN;
#pragma unroll
          for (int ks = 0; ks < D / 16; ++ks)
            umma_ss(d_tmem, umma_smem_desc_sw128(sQ + (ks >> 2) * S::kQBlk + (ks & 3) * 32, 16, 1024),
                    umma_smem_desc_sw128(sK + st * S::kTile + (ks >> 2) * S::kBlk + (ks & 3) * 32, 16, 1024), idesc_qk,
                    ks > 0 ? 1u : 0u);
          umma_commit(bar(kEmptyK + st));
          umma_commit(bar(kSFull + (t & 1)));
          if (j == n_kt - 1) umma_commit(bar(kQEmpty));          // every Q K^T of this unit done: Q may be replaced
        };
        mbar_wait(bar(kQFull), i & 1);
        tc_fence_after();
        issue_qk(0);
        for (int j = 0; j < n_kt; ++j) {
          if (j + 1 < n_kt) issue_qk(j + 1);
          const int t = t0 + j, st = t % kStages;
          mbar_wait(bar(kPReady + (t & 1)), (t >> 1) & 1);
          mbar_wait(bar(kFullV + st), (t / kStages) & 1);
          if (j == 0 && i > 0) mbar_wait(bar(kOFree), (i - 1) & 1);   // the previous unit's epilogue has read O
          tc_fence_after();
#pragma unroll
          for (int ks = 0; ks < BN / 16; ++ks)
            umma_ts(tmem_o, tmem_base + (t & 1) * BN + ks * 8,
                    umma_smem_desc_sw128(sV + st * S::kTile + ks * 2048, S::kBlk, 1024), idesc_pv,
                    (j > 0 || ks > 0) ? 1u : 0u);
          umma_commit(bar(kEmptyV + st));
          umma_commit(bar(kODone + (t & 1)));
        }
        t0 += n_kt;
      }
    }
    __syncwarp();
  } else if (warp == 6) {
    // ===================================================================== Q loader (next unit's rows, cp.async)
    for (int i = 0;; ++i) {
      int u = 0;
      if (lane == 0) {
        mbar_wait(bar(kSchedEmpty + (i & 1)), ((i >> 1) & 1) ^ 1);        // slot read by all 130 consumers two units ago
        u = static_cast<int>(atomicAdd(a.next_unit, 1u));
        s_sched[i & 1] = u;
        mbar_arrive(bar(kSchedFull + (i & 1)));
      }
      u = __shfl_sync(0xffffffffu, u, 0);
      if (u >= n_units) break;
      const WorkUnit w = a.units[u];
      const Geo ge = geo_of(w);
      if (lane == 0) mbar_wait(bar(kQEmpty), (i & 1) ^ 1);      // one lane polls; 31 spinning lanes would steal issue slots
      __syncwarp();
      // The source row of every tile position first (one load per lane, <= 4 positions per lane), then all cp.async
      // of the tile back to back with no dependent loads in between: 2 rows x 16 chunks per sweep for D = 128 (4 x 8 for
      // D = 64), i.e. 256-byte contiguous global segments.
      constexpr int kCh = D / 8;
      constexpr int kRowsPer = 32 / kCh;
      int src_of[4];
#pragma unroll
      for (int k = 0; k < 4; ++k) {
        const int pl = k * 32 + lane;
        const int ridx = ge.ridx0 + pl;
        src_of[k] = -1;
        if (pl < PT && ridx < ge.n_rows)
          src_of[k] = (dense || a.q_by_position) ? row_pos(bd, a.sel, ge.b, ge.N, ge.ns, ge.n_rows, ridx) : ridx;
      }
      const __nv_bfloat16* qb = a.q + (static_cast<size_t>(ge.b) * bd.t_stride * a.hq + ge.g * G) * D;
#pragma unroll
      for (int r0 = 0; r0 < BM; r0 += kRowsPer) {
        const int r = r0 + lane / kCh, c = lane % kCh;
        const int pl = r / G, hl = r % G;
        int src = __shfl_sync(0xffffffffu, src_of[0], pl & 31);
        if (PT > 32) {
          const int s1 = __shfl_sync(0xffffffffu, src_of[1], pl & 31), s2 = __shfl_sync(0xffffffffu, src_of[2], pl & 31);
          const int s3 = __shfl_sync(0xffffffffu, src_of[3], pl & 31);
          const int k = pl >> 5;
          src = k == 0 ? src : (k == 1 ? s1 : (k == 2 ? s2 : s3));
        }
        const uint32_t dst = sQ + (c >> 3) * S::kQBlk + r * 128 + (((c & 7) ^ (r & 7)) << 4);
        if (src >= 0) {
          cp_async16(dst, qb + (static_cast<size_t>(src) * a.hq + hl) * D + c * 8);
        } else {
          asm volatile("st.shared.v4.u32 [%0], {%1, %1, %1, %1};" ::"r"(dst), "r"(0u) : "memory");
        }
      }
      cp_async_commit();
      cp_async_wait<0>();
      fence_proxy_async_smem();
      __syncwarp();
      if (lane == 0) mbar_arrive(bar(kQFull));
    }
  } else {
    // ===================================================================== softmax / correction / epilogue
    const int quarter = warp & 3;
    const int r = quarter * 32 + lane;
    const uint32_t lane_addr = tmem_base + (static_cast<uint32_t>(quarter * 32) << 16);
    const int pl = r / G, hl = r % G;
    volatile int* s_flag = reinterpret_cast<volatile int*>(smem + S::oFlag);
    int t0 = 0;
    for (int i = 0;; ++i) {
      const int u = unit_of(i);
      if (u >= n_units) break;
      const WorkUnit w = a.units[u];
      const Geo ge = geo_of(w);
      const int ridx = ge.ridx0 + pl;
      const bool valid = ridx < ge.n_rows;
      const int pos = row_pos(bd, a.sel, ge.b, ge.N, ge.ns, ge.n_rows, ridx);
      const int p_min = row_pos(bd, a.sel, ge.b, ge.N, ge.ns, ge.n_rows, ge.ridx0);
      const int t_end = ge.N + ge.Lq;
      float m_used = -1e30f, l = 0.f;
      for (int j = 0; j < w.n_kt; ++j) {
        const int t = t0 + j;
        const int key0 = (w.jt0 + j) * BN;
        const bool need_mask = key0 + BN - 1 > p_min;
        const uint32_t s_addr = lane_addr + (t & 1) * BN;
        mbar_wait(bar(kSFull + (t & 1)), (t >> 1) & 1);
        tc_fence_after();
        uint32_t pk[BN / 2];
        float tile_max, tile_sum;
        auto sweep = [&](float m_ref) {
          float mx0 = -INFINITY, mx1 = -INFINITY, mx2 = -INFINITY, mx3 = -INFINITY;
          float l0 = 0.f, l1 = 0.f, l2 = 0.f, l3 = 0.f;
          uint32_t sa[32], sb[32];
          tmem_ld32(s_addr, sa);
          tmem_ld32(s_addr + 32, sb);
#pragma unroll
          for (int c = 0; c < BN / 32; ++c) {
            uint32_t(&cur)[32] = (c & 1) ? sb : sa;
            if (c == 0) tmem_wait_ld();
#pragma unroll
            for (int e = 0; e < 32; e += 4) {
              float v0 = __uint_as_float(cur[e]), v1 = __uint_as_float(cur[e + 1]);
              float v2 = __uint_as_float(cur[e + 2]), v3 = __uint_as_float(cur[e + 3]);
              if (need_mask) {
                const int k = key0 + c * 32 + e;
                if (k > pos) v0 = -INFINITY;
                if (k + 1 > pos) v1 = -INFINITY;
                if (k + 2 > pos) v2 = -INFINITY;
                if (k + 3 > pos) v3 = -INFINITY;
              }
              mx0 = fmaxf(mx0, v0); mx1 = fmaxf(mx1, v1); mx2 = fmaxf(mx2, v2); mx3 = fmaxf(mx3, v3);
              const float p0 = ex2(fmaf(v0, a.scale_log2, -m_ref));
              const float p1 = ex2(fmaf(v1, a.scale_log2, -m_ref));
              const float p2 = ex2(fmaf(v2, a.scale_log2, -m_ref));
              const float p3 = ex2_poly(fmaf(v3, a.scale_log2, -m_ref));
              l0 += p0; l1 += p1; l2 += p2; l3 += p3;
              pk[c * 16 + (e >> 1)] = pack_bf16(p0, p1);
              pk[c * 16 + (e >> 1) + 1] = pack_bf16(p2, p3);
            }
          }
          tile_max = fmaxf(fmaxf(mx0, mx1), fmaxf(mx2, mx3)) * a.scale_log2;
          tile_sum = (l0 + l1) + (l2 + l3);
        };
        if (j == 0) {
          // first tile of the unit: the reference is its own max, clamped finite (a row may see none of a later chunk's keys)
          float mx0 = -INFINITY, mx1 = -INFINITY;
#pragma unroll
          for (int c = 0; c < BN / 32; ++c) {
            uint32_t tt[32];
            tmem_ld32(s_addr + c * 32, tt);
            tmem_wait_ld();
#pragma unroll
            for (int e = 0; e < 32; e += 2) {
              float v0 = __uint_as_float(tt[e]), v1 = __uint_as_float(tt[e + 1]);
              if (need_mask) {
                if (key0 + c * 32 + e > pos) v0 = -INFINITY;
                if (key0 + c * 32 + e + 1 > pos) v1 = -INFINITY;
              }
              mx0 = fmaxf(mx0, v0); mx1 = fmaxf(mx1, v1);
            }
          }
          m_used = fmaxf(fmaxf(mx0, mx1) * a.scale_log2, -1e30f);
          sweep(m_used);
        } else {
          sweep(m_used);
          if (__any_sync(0xffffffffu, tile_max > m_used + kRescaleThreshold)) {
            mbar_wait(bar(kODone + ((t - 1) & 1)), ((t - 1) >> 1) & 1);
            tc_fence_after();
            const float m_t = fmaxf(m_used, tile_max);
            const float f = ex2(m_used - m_t);
            m_used = m_t;
            l *= f;
#pragma unroll
            for (int c = 0; c < D / 32; ++c) {
              uint32_t o[32];
              tmem_ld32(lane_addr + kColO + c * 32, o);
              tmem_wait_ld();
#pragma unroll
              for (int e = 0; e < 32; ++e) o[e] = __float_as_uint(__uint_as_float(o[e]) * f);
              tmem_st32(lane_addr + kColO + c * 32, o);
            }
            tmem_wait_st();
            sweep(m_used);
          }
        }
        l += tile_sum;
        tmem_st32(s_addr, pk);
        if (key0 + BN > t_end) {
          const int st = t % kStages;
          mbar_wait(bar(kFullV + st), (t / kStages) & 1);
          if (r < BN && key0 + r >= t_end) {
#pragma unroll
            for (int kb = 0; kb < D / 64; ++kb) {
              uint4* row = reinterpret_cast<uint4*>(smem + S::oV + st * S::kTile + kb * S::kBlk + r * 128);
#pragma unroll
              for (int c = 0; c < 8; ++c) row[c] = make_uint4(0u, 0u, 0u, 0u);
            }
          }
          fence_proxy_async_smem();
        }
        tmem_wait_st();
        tc_fence_before();
        mbar_arrive(bar(kPReady + (t & 1)));
      }
      t0 += w.n_kt;

      // ---- epilogue of the unit
      const int t_last = t0 - 1;
      mbar_wait(bar(kODone + (t_last & 1)), (t_last >> 1) & 1);
      tc_fence_after();
      __nv_bfloat16* dst = a.out + ((static_cast<size_t>(ge.b) * bd.t_stride + ridx) * a.hq + ge.g * G + hl) * D;
      float* lse_dst = a.lse ? a.lse + (static_cast<size_t>(ge.b) * bd.t_stride + ridx) * a.hq + ge.g * G + hl : nullptr;
      if (w.n_chunks == 1) {
        const float inv = 1.f / l;
#pragma unroll
        for (int c = 0; c < D / 32; ++c) {
          uint32_t o[32];
          tmem_ld32(lane_addr + kColO + c * 32, o);
          tmem_wait_ld();
          if (c == D / 32 - 1) {                           // O is in registers: the next unit may overwrite it
            tc_fence_before();
            mbar_arrive(bar(kOFree));
          }
          if (valid) {
#pragma unroll
            for (int v4 = 0; v4 < 4; ++v4) {
              uint4 ww;
              ww.x = pack_bf16(__uint_as_float(o[8 * v4 + 0]) * inv, __uint_as_float(o[8 * v4 + 1]) * inv);
              ww.y = pack_bf16(__uint_as_float(o[8 * v4 + 2]) * inv, __uint_as_float(o[8 * v4 + 3]) * inv);
              ww.z = pack_bf16(__uint_as_float(o[8 * v4 + 4]) * inv, __uint_as_float(o[8 * v4 + 5]) * inv);
              ww.w = pack_bf16(__uint_as_float(o[8 * v4 + 6]) * inv, __uint_as_float(o[8 * v4 + 7]) * inv);
              *reinterpret_cast<uint4*>(dst + c * 32 + v4 * 8) = ww;
            }
          }
        }
        if (valid && lse_dst) *lse_dst = (m_used + log2f(l)) * kLn2;
      } else {
        // split item: park the unnormalised partial (O relative to m_used, m_used, l); [D/4][BM] float4 keeps both the
        // stores here and the merge loads coalesced
        const size_t slot = static_cast<size_t>(w.slot + w.chunk);
        float4* po4 = reinterpret_cast<float4*>(a.part_o) + slot * (D / 4) * BM;
#pragma unroll
        for (int c = 0; c < D / 32; ++c) {
          uint32_t o[32];
          tmem_ld32(lane_addr + kColO + c * 32, o);
          tmem_wait_ld();
          if (c == D / 32 - 1) {
            tc_fence_before();
            mbar_arrive(bar(kOFree));
          }
#pragma unroll
          for (int v4 = 0; v4 < 8; ++v4)
            __stcg(po4 + (c * 8 + v4) * BM + r, make_float4(__uint_as_float(o[4 * v4]), __uint_as_float(o[4 * v4 + 1]),
                                                              __uint_as_float(o[4 * v4 + 2]), __uint_as_float(o[4 * v4 + 3])));
        }
        __stcg(a.part_ml + slot * 2 * BM + r, m_used);
        __stcg(a.part_ml + slot * 2 * BM + BM + r, l);
        __threadfence();
        asm volatile("bar.sync 1, 128;" ::: "memory");
        if (r == 0) {
          unsigned int* ctr = a.item_ctr + (static_cast<size_t>(w.b) * a.hkv + w.g) * a.max_tiles + w.tile;
          const unsigned int prev = atomicAdd(ctr, 1u);
          const int last = prev == static_cast<unsigned int>(w.n_chunks - 1);
          if (last) *ctr = 0u;
          *s_flag = last;
        }
        asm volatile("bar.sync 1, 128;" ::: "memory");
        if (*s_flag) {
          // last chunk to arrive merges all chunks of the item in chunk order (bit-reproducible)
          __threadfence();
          float mc[kMaxSplit], wc[kMaxSplit];
          float m_all = -1e30f, l_all = 0.f;
          const float* ml0 = a.part_ml + static_cast<size_t>(w.slot) * 2 * BM;
#pragma unroll
          for (int c = 0; c < kMaxSplit; ++c) {
            mc[c] = -1e30f;
            if (c < w.n_chunks) { mc[c] = __ldcg(ml0 + c * 2 * BM + r); m_all = fmaxf(m_all, mc[c]); }
          }
#pragma unroll
          for (int c = 0; c < kMaxSplit; ++c) {
            wc[c] = 0.f;
            if (c < w.n_chunks) { wc[c] = ex2(mc[c] - m_all); l_all += __ldcg(ml0 + c * 2 * BM + BM + r) * wc[c]; }
          }
          const float inv = 1.f / l_all;
          const float4* p0 = reinterpret_cast<const float4*>(a.part_o) + static_cast<size_t>(w.slot) * (D / 4) * BM;
#pragma unroll 1
          for (int cc = 0; cc < D / 8; ++cc) {             // 8 output elements per step
            float acc[8] = {0.f, 0.f, 0.f, 0.f, 0.f, 0.f, 0.f, 0.f};
#pragma unroll
            for (int c = 0; c < kMaxSplit; ++c) {
              if (c < w.n_chunks) {
                const float4* pc = p0 + static_cast<size_t>(c) * (D / 4) * BM;
                const float4 x0 = __ldcg(pc + (cc * 2) * BM + r), x1 = __ldcg(pc + (cc * 2 + 1) * BM + r);
                acc[0] = fmaf(x0.x, wc[c], acc[0]); acc[1] = fmaf(x0.y, wc[c], acc[1]);
                acc[2] = fmaf(x0.z, wc[c], acc[2]); acc[3] = fmaf(x0.w, wc[c], acc[3]);
                acc[4] = fmaf(x1.x, wc[c], acc[4]); acc[5] = fmaf(x1.y, wc[c], acc[5]);
                acc[6] = fmaf(x1.z, wc[c], acc[6]); acc[7] = fmaf(x1.w, wc[c], acc[7]);
              }
            }
            if (valid)
              *reinterpret_cast<uint4*>(dst + cc * 8) =
                  make_uint4(pack_bf16(acc[0] * inv, acc[1] * inv), pack_bf16(acc[2] * inv, acc[3] * inv),
                             pack_bf16(acc[4] * inv, acc[5] * inv), pack_bf16(acc[6] * inv, acc[7] * inv));
          }
          if (valid && lse_dst) *lse_dst = (m_all + log2f(l_all)) * kLn2;
        }
      }
    }
  }

  tc_fence_before();
  __syncthreads();
  if (warp == 1) {
    tc_fence_after();
    tmem_dealloc<kTmemCols>(tmem_base);
  }
}

using EncodeFn = CUresult (*)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*, const cuuint64_t*,
                              const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave, CUtensorMapSwizzle,
                              CUtensorMapL2promotion, CUtensorMapFloatOOBfill);
EncodeFn get_encode() {
  static EncodeFn fn = []() -> EncodeFn {
    void* p = nullptr;
    cudaDriverEntryPointQueryResult qres;
    if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &p, cudaEnableDefault, &qres) != cudaSuccess ||
        qres != cudaDriverEntryPointSuccess)
      return nullptr;
    return reinterpret_cast<EncodeFn>(p);
  }();
  return fn;
}
bool make_kv_map(CUtensorMap* m, const void* base, int batch, int t_stride, int hkv, int d) {
  EncodeFn enc = get_encode();
  if (!enc) return false;
  const cuuint64_t dims[4] = {static_cast<cuuint64_t>(d), static_cast<cuuint64_t>(hkv),
                              static_cast<cuuint64_t>(t_stride), static_cast<cuuint64_t>(batch)};
  const cuuint64_t strides[3] = {static_cast<cuuint64_t>(d) * 2, static_cast<cuuint64_t>(hkv) * d * 2,
                                 static_cast<cuuint64_t>(t_stride) * hkv * d * 2};
  const cuuint32_t box[4] = {64, 1, BN, 1};
  const cuuint32_t estr[4] = {1, 1, 1, 1};
  return enc(m, CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, 4, const_cast<void*>(base), dims, strides, box, estr,
             CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
             CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) == CUDA_SUCCESS;
}

}  // namespace

// Workspace of the persistent kernel, sized for the ctx limits (qcf_create).
size_t attn_ptc_units_bytes(const qcf_ctx* ctx) {
  const int PT = BM / ctx->lay.g;
  const size_t tiles = (static_cast<size_t>(ctx->max_ctx) + ctx->max_query + PT - 1) / PT;
  return tiles * ctx->max_batch * ctx->lay.hkv * kMaxSplit * sizeof(WorkUnit) + 64;
}
size_t attn_ptc_items(const qcf_ctx* ctx) {
  const int PT = BM / ctx->lay.g;
  const size_t tiles = (static_cast<size_t>(ctx->max_ctx) + ctx->max_query + PT - 1) / PT;
  return tiles * ctx->max_batch * ctx->lay.hkv;
}
int attn_ptc_slots(const qcf_ctx* ctx) {
  const size_t cap = attn_ptc_items(ctx) * kMaxSplit;
  return static_cast<int>(cap < 1024 ? cap : 1024);
}
size_t attn_ptc_slot_bytes(const qcf_ctx* ctx) { return static_cast<size_t>(BM) * ctx->lay.d * 4 + 2 * BM * 4; }

cudaError_t launch_attn_ptc(const qcf_ctx* ctx, const qcf_batch* b, const int32_t* sel, const int32_t* n_sel,
                            const __nv_bfloat16* q, int rows_by_position, const __nv_bfloat16* k_f,
                            const __nv_bfloat16* v_f, __nv_bfloat16* out, float* lse, cudaStream_t stream) {
  if (b->batch == 0 || b->t_stride == 0) return cudaSuccess;
  const Layout& L = ctx->lay;
  CUtensorMap tm_k, tm_v;
  if (!make_kv_map(&tm_k, k_f, b->batch, b->t_stride, L.hkv, L.d) ||
      !make_kv_map(&tm_v, v_f, b->batch, b->t_stride, L.hkv, L.d))
    return cudaErrorInvalidValue;
  const int PT = BM / L.g;
  const int max_tiles = (b->t_stride + PT - 1) / PT;
  const int n_cta = 2 * ctx->n_sm;
  PlanOut po;
  po.units = static_cast<WorkUnit*>(ctx->ptc_units);
  po.n_units = ctx->ptc_n_units;
  po.next_unit = reinterpret_cast<unsigned int*>(ctx->ptc_n_units) + 1;
  po.max_units = static_cast<int>((attn_ptc_units_bytes(ctx) - 64) / sizeof(WorkUnit));
  po.max_slots = attn_ptc_slots(ctx);
  static const int split_div = []() { const char* e = std::getenv("QCF_ATTN_SPLIT_DIV"); const int v = e ? std::atoi(e) : 3; return v >= 1 && v <= 16 ? v : 3; }();
  attn_plan_kernel<<<1, 1024, 0, stream>>>(b->dev, L.hkv, L.g, max_tiles, n_cta, split_div, sel, n_sel, po);
  cudaError_t e = cudaGetLastError();
  if (e != cudaSuccess) return e;
  AttnArgs a;
  a.units = po.units; a.n_units = po.n_units; a.next_unit = po.next_unit;
  a.hq = L.hq; a.hkv = L.hkv;
  a.scale_log2 = L.scale * kLog2e;
  a.sel = sel; a.n_sel = n_sel; a.q = q; a.q_by_position = rows_by_position;
  a.out = out; a.lse = lse;
  a.part_o = ctx->ptc_part_o; a.part_ml = ctx->ptc_part_ml; a.item_ctr = ctx->ptc_item_ctr;
  a.max_tiles = (ctx->max_ctx + ctx->max_query + PT - 1) / PT;       // counter stride: the ctx bound, >= this batch's
  if (L.d == 128) {
    auto kern = attn_ptc_kernel<128>;
    const int smem = Smem<128>::kBytes + 1024;
    cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, smem);
    kern<<<n_cta, kThreads, smem, stream>>>(tm_k, tm_v, b->dev, a);
  } else {
    auto kern = attn_ptc_kernel<64>;
    const int smem = Smem<64>::kBytes + 1024;
    cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, smem);
    kern<<<n_cta, kThreads, smem, stream>>>(tm_k, tm_v, b->dev, a);
  }
  return cudaGetLastError();
}

}  // namespace qcf
