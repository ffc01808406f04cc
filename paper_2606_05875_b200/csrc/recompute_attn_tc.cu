// a5 on the 5th-generation tensor cores — PAPER.md:134: causal GQA attention of the recomputed rows R = P u U over
// the fused cache, as a warp-specialised tcgen05 / TMEM / TMA kernel.
//
//   tile      : 128 MMA rows = 128/G consecutive rows of R (ascending positions) x the G query heads of one kv-head,
//               against key tiles of 64 positions of that kv-head (K/V fetched once serve all G heads)
//   warp 0    : TMA producer — K and V tiles (4-D tensor maps over [B][T][Hkv][d], 128-byte swizzle) into 2-stage rings
//   warp 1    : UMMA issuer  — S[j] = Q K_j^T (SS, fp32 in TMEM, double-buffered), O += P_j V_j (TS: P read from TMEM,
//               V as an MN-major smem operand); S[j+1] is issued before P_j V_j so the softmax of tile j overlaps it
//   warps 2-5 : softmax      — one thread per row (= TMEM lane): row max, exp2, bf16 P written back over S[j] in TMEM,
//               lazy rescale of O (only when the running max grows by more than 2^8), final normalisation + store
// The causal limit is monotone in the tile (rows ascending), so only key tiles reaching past the tile's first position
// are masked and the key loop stops at the tile's last position.  sel == nullptr is the dense comparator (Eq. 2).
//
// Split-KV over a thread-block cluster: when the problem is too small to balance (the heaviest tile is a large share
// of an SM's load) the key tiles of one work item are divided among the 1, 2 or 4 CTAs of a cluster.  Ranks > 0 park
// their unnormalised O (fp32) and (m, l) in their own shared memory (the drained K/V rings), rank 0 pulls them over
// distributed shared memory, merges in rank order (deterministic) and stores.  No global workspace, no atomics.
#include <cmath>

#include "qcf_internal.cuh"
#include "sm100_ptx.cuh"

namespace qcf {

namespace {

using namespace ptx;

constexpr int BM = 128;         // MMA rows per tile
constexpr int BN = 64;          // keys per tile
constexpr int kStages = 2;      // K and V ring depth
constexpr int kThreads = 192;
constexpr int kTmemCols = 256;  // S_0, S_1 (BN fp32 columns each; bf16 P_j aliases the first BN/2 of S_j) + O (up to 128)
constexpr int kColO = 128;
constexpr float kLog2e = 1.4426950408889634f;
constexpr float kLn2 = 0.6931471805599453f;
constexpr float kRescaleSum = 256.0f;         // rescale when a tile's row sum (relative to the reference max) exceeds 2^8
// Of every 4 exponential pairs, 3 take MUFU.EX2 and 1 the packed polynomial on the FMA pipe (MUFU and tensor pipe are both
// ~60 % busy; this unloads the tighter one).  What bounds the kernel and the arrangements measured and rejected: DESIGN.md §9.4.
constexpr int kMufuPairs = 3;

// Two CTAs are resident per SM (96 KB of shared memory, 256 TMEM columns and <= 168 registers each).  Inside a CTA
// S_{j+1} = Q K_{j+1}^T is issued before P_j V_j, so the softmax of tile j overlaps it; across the two CTAs the
// remaining bubbles (barrier round trips, TMA latency) are filled, and each SM sub-partition holds two softmax warps.
template <int D>
struct Smem {
  static constexpr int kQBlk = BM * 128;                   // one 64-column block of Q (128 rows x 128 B)
  static constexpr int kBlk = BN * 128;                    // one 64-column block of a K or V tile
  static constexpr int kQ = BM * D * 2;
  static constexpr int kTile = BN * D * 2;                 // bytes of one K or V tile
  static constexpr int oQ = 0;
  static constexpr int oK = oQ + kQ;
  static constexpr int oV = oK + kStages * kTile;
  static constexpr int oBar = oV + kStages * kTile;        // mbarriers (8 B each)
  static constexpr int kNumBar = 4 * kStages + 7;
  static constexpr int oTmem = oBar + kNumBar * 8;
  static constexpr int oStat = oTmem + 16;                 // split-KV: (m, l) of this CTA's 128 rows
  static constexpr int kBytes = oStat + 2 * BM * 4;
  static_assert(2 * kStages * kTile >= BM * D * 4, "the K/V rings must hold one fp32 O tile for the split-KV merge");
};
// (the kEmptyK / kEmptyV slots are unused: a K stage is free when S of its tile is signalled, a V stage when its P V is)
enum { kFullK = 0, kEmptyK = kStages, kFullV = 2 * kStages, kEmptyV = 3 * kStages, kSFull = 4 * kStages,
       kPReady = 4 * kStages + 2, kODone = 4 * kStages + 4, kQFull = 4 * kStages + 6 };

__device__ __forceinline__ uint32_t cluster_ctarank() {
  uint32_t r;
  asm volatile("mov.u32 %0, %%cluster_ctarank;" : "=r"(r));
  return r;
}
__device__ __forceinline__ uint32_t cluster_nctarank() {
  uint32_t r;
  asm volatile("mov.u32 %0, %%cluster_nctarank;" : "=r"(r));
  return r;
}
__device__ __forceinline__ void cluster_sync_all() {        // every thread of every CTA of the cluster
  asm volatile("barrier.cluster.arrive.release.aligned;\n\tbarrier.cluster.wait.acquire.aligned;" ::: "memory");
}
__device__ __forceinline__ uint32_t dsmem_addr(uint32_t local_smem_addr, uint32_t rank) {
  uint32_t r;
  asm volatile("mapa.shared::cluster.u32 %0, %1, %2;" : "=r"(r) : "r"(local_smem_addr), "r"(rank));
  return r;
}
__device__ __forceinline__ float ld_dsmem_f32(uint32_t addr) {
  float v;
  asm volatile("ld.shared::cluster.f32 %0, [%1];" : "=f"(v) : "r"(addr) : "memory");
  return v;
}
__device__ __forceinline__ float4 ld_dsmem_f32x4(uint32_t addr) {
  float4 v;
  asm volatile("ld.shared::cluster.v4.f32 {%0,%1,%2,%3}, [%4];" : "=f"(v.x), "=f"(v.y), "=f"(v.z), "=f"(v.w) : "r"(addr) : "memory");
  return v;
}

template <int D>
__global__ void __launch_bounds__(kThreads, 2)
attn_tc_kernel(const __grid_constant__ CUtensorMap tm_k, const __grid_constant__ CUtensorMap tm_v, BatchDev bd, int hq,
               int hkv, int tiles_hint, int unit_grp, float scale_log2, const int32_t* __restrict__ sel,
               const int32_t* __restrict__ n_sel, const __nv_bfloat16* q, int q_by_position,
               __nv_bfloat16* __restrict__ out, float* __restrict__ lse_out) {
  extern __shared__ unsigned char smem_raw[];
  // 128-byte-swizzle atoms need 1024-byte alignment; the launch reserves 1 KB of slack for this round-up
  unsigned char* smem = smem_raw + ((1024u - (smem_u32(smem_raw) & 1023u)) & 1023u);
  using S = Smem<D>;
  const int G = hq / hkv;
  const int PT = BM / G;
  // 1-D grid of work items (one 128-row tile of one (request, kv-head) "unit"); the CTAs of a cluster (consecutive block
  // ids) share one item and split its key tiles.  Order = L2 locality first, then heaviest first:
  //   section A: groups of `unit_grp` consecutive units whose K/V fit in a fraction of the L2; inside a group the tiles
  //              of all its units from the heaviest (last rows, longest causal extent) down — the CTAs resident at any
  //              time read the K/V of ONE group (at c4, 16 requests x 34 MB interleaved made every key tile an HBM read:
  //              18.8 GB of DRAM traffic for 0.55 GB of cache, profiles/r02_c4_base.md);
  //   section B: tiles past the host's row-count hint `tiles_hint` (the selection size lives on the device), all units —
  //              normally empty, they retire under the tail.
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const uint32_t sbase = smem_u32(smem);
  auto bar = [&](int i) -> uint32_t { return sbase + S::oBar + 8 * i; };
  pdl_trigger();
  // Everything that touches no predecessor data runs before the dependency wait, under the predecessor's tail: descriptor
  // prefetch and barrier init.  (The TMEM allocation stays behind the wait: CTAs that find no work below return early.)
  if (warp == 0 && lane == 0) {
    prefetch_tensormap(&tm_k);
    prefetch_tensormap(&tm_v);
    for (int i = 0; i < S::kNumBar; ++i) mbar_init(bar(i), (i == kPReady || i == kPReady + 1 || i == kQFull) ? 128 : 1);
    fence_barrier_init();
  }
  pdl_wait();          // n_sel / sel below are written by the predecessors
  const int ncl = static_cast<int>(cluster_nctarank());
  const int crank = static_cast<int>(cluster_ctarank());
  const int item = static_cast<int>(blockIdx.x) / ncl;
  const int n_units = hkv * bd.batch;
  const int n_groups = (n_units + unit_grp - 1) / unit_grp;
  const int items_a = n_groups * tiles_hint * unit_grp;
  int t_idx, unit;                                  // t_idx 0 = the unit's heaviest (last) row tile
  if (item < items_a) {
    const int grp = item / (tiles_hint * unit_grp), rem = item % (tiles_hint * unit_grp);
    t_idx = rem / unit_grp;
    unit = grp * unit_grp + rem % unit_grp;
    if (unit >= n_units) return;                    // the last group may be partial (same decision in every CTA of a cluster)
  } else {
    const int rem = item - items_a;
    t_idx = tiles_hint + rem / n_units;
    unit = rem % n_units;
  }
  const int b = unit / hkv, g = unit % hkv;
  const int N = bd.n_ctx[b], Lq = bd.n_query[b];
  const bool dense = sel == nullptr;
  const int ns = dense ? 0 : ld_ca_s32(n_sel + b);     // coherent loads for everything a predecessor wrote (PDL)
  const int n_rows = dense ? N + Lq : ns + Lq;
  const int n_tiles = (n_rows + PT - 1) / PT;
  // heaviest first RELATIVE TO THE REQUEST'S OWN tile count (the grid is sized for t_stride rows)
  if (t_idx >= n_tiles) return;
  const int tile = n_tiles - 1 - t_idx;
  const int ridx0 = tile * PT;
  const int* sel_b = dense ? nullptr : sel + static_cast<size_t>(b) * bd.n_stride;
  auto pos_of = [&](int r) -> int {          // request position of row r of R (padding rows: 0, never stored)
    if (r >= n_rows) return 0;
    return dense ? r : (r < ns ? ld_ca_s32(sel_b + r) : N + (r - ns));
  };
  const int p_min = pos_of(ridx0);
  const int p_max = pos_of(min(ridx0 + PT, n_rows) - 1);
  const int n_kt_all = p_max / BN + 1;
  // this CTA's key tiles: [jt0, jt0 + n_kt); rank 0 always has at least one, ranks > 0 none when n_kt_all < ncl
  const int kt_base = n_kt_all / ncl, kt_rem = n_kt_all % ncl;
  const int jt0 = crank * kt_base + min(crank, kt_rem);
  const int n_kt = kt_base + (crank < kt_rem ? 1 : 0);
  const int t_end = N + Lq;                  // rows >= t_end of the cache are padding

  const uint32_t sQ = sbase + S::oQ, sK = sbase + S::oK, sV = sbase + S::oV;
  volatile uint32_t* tmem_slot = reinterpret_cast<volatile uint32_t*>(smem + S::oTmem);

  if (warp == 1) tmem_alloc<kTmemCols>(sbase + S::oTmem);
  // Q tile: the gathered rows are requested from global memory BEFORE the CTA-wide sync and land in shared memory after
  // it, signalled on their own barrier, so the producer's first K / V TMA loads (issued right after the sync) and the
  // TMEM allocation overlap the gather latency instead of queueing behind it.
  uint4 qv[D / 8];
  if (warp >= 2) {
    const int r = (warp & 3) * 32 + lane;
    const int pl = r / G, hl = r % G;
    const int ridx = ridx0 + pl;
    const uint4* src = nullptr;
    if (ridx < n_rows) {
      const int src_row = (dense || q_by_position) ? pos_of(ridx) : ridx;
      src = reinterpret_cast<const uint4*>(q + ((static_cast<size_t>(b) * bd.t_stride + src_row) * hq + g * G + hl) * D);
    }
#pragma unroll
    // coherent loads: in the stack path q is written by a predecessor this kernel's lifetime overlaps (PDL)
    for (int c = 0; c < D / 8; ++c) qv[c] = src ? ld_na_v4(src + c) : make_uint4(0u, 0u, 0u, 0u);
  }
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  if (warp >= 2) {
    // K-major 128B-swizzle layout: row r at r*128 in each 64-column block, chunk c at c ^ (r & 7)
    const int r = (warp & 3) * 32 + lane;
#pragma unroll
    for (int c = 0; c < D / 8; ++c) {
      unsigned char* dst = smem + S::oQ + (c >> 3) * S::kQBlk + r * 128 + (((c & 7) ^ (r & 7)) << 4);
      *reinterpret_cast<uint4*>(dst) = qv[c];
    }
    fence_proxy_async_smem();
    mbar_arrive(bar(kQFull));
  }
  const uint32_t tmem_base = *tmem_slot;
  const uint32_t tmem_o = tmem_base + kColO;

  if (warp == 0) {
    // ===================================================================== TMA producer
    // The whole warp walks the loop converged and ONE ELECTED lane issues (elect.sync): inside a divergent `if (lane == 0)`
    // the compiler cannot prove uniformity and wraps every TMA / UMMA instruction (they take uniform registers) in a
    // per-lane ELECT / BRA.U.ANY loop with vector-to-uniform moves — ~40 SASS instructions per UMMA on the issuer's
    // critical path (traced: ~450 cycles to issue one tile's MMAs).
    for (int j = 0; j < n_kt; ++j) {
      const int st = j % kStages;
      const uint32_t ph = (j / kStages) & 1;
      // stage st is free once Q K_{j-2}^T has completed: that is the phase S_{j-2} was signalled on (no separate commit)
      if (j >= kStages) mbar_wait(bar(kSFull + st), ph ^ 1);
      if (elect_one()) {
        mbar_arrive_expect_tx(bar(kFullK + st), S::kTile);
#pragma unroll
        for (int kb = 0; kb < D / 64; ++kb)
          tma_load_4d(sK + st * S::kTile + kb * S::kBlk, &tm_k, bar(kFullK + st), kb * 64, g, (jt0 + j) * BN, b);
      }
      if (j >= kStages) mbar_wait(bar(kODone + st), ph ^ 1);     // P_{j-2} V_{j-2} has completed
      if (elect_one()) {
        mbar_arrive_expect_tx(bar(kFullV + st), S::kTile);
#pragma unroll
        for (int kb = 0; kb < D / 64; ++kb)
          tma_load_4d(sV + st * S::kTile + kb * S::kBlk, &tm_v, bar(kFullV + st), kb * 64, g, (jt0 + j) * BN, b);
      }
      __syncwarp();
    }
  } else if (warp == 1) {
    // ===================================================================== UMMA issuer
    {
      // converged warp, one elected lane issues (see the producer)
      constexpr uint32_t idesc_qk = umma_idesc_bf16(BM, BN, false, false);
      constexpr uint32_t idesc_pv = umma_idesc_bf16(BM, D, false, true);
      // base descriptors once; a tile's descriptors are base + (byte offset >> 4) (the start-address field is in 16-byte
      // units and shared memory is far below its 256 KB range, so the add never carries out of the field)
      const uint64_t dq = umma_smem_desc_sw128(sQ, 16, 1024), dk = umma_smem_desc_sw128(sK, 16, 1024);
      const uint64_t dv = umma_smem_desc_sw128(sV, S::kBlk, 1024);
      auto issue_qk = [&](int j) {
        const int st = j % kStages;
        mbar_wait(bar(kFullK + st), (j / kStages) & 1);
        tc_fence_after();
        // S_j overwrites the buffer of S_{j-2} / P_{j-2}: P_{j-2} V_{j-2} was issued earlier and UMMAs of one CTA
        // execute in issue order; the softmax warps finished reading S_{j-2} before they signalled P_{j-2}.
        const uint32_t d_tmem = tmem_base + (j & 1) * BN;
        if (elect_one()) {
          const uint64_t dk_st = dk + static_cast<uint64_t>((st * S::kTile) >> 4);
#pragma unroll
          for (int ks = 0; ks < D / 16; ++ks)
            umma_ss(d_tmem, dq + static_cast<uint64_t>(((ks >> 2) * S::kQBlk + (ks & 3) * 32) >> 4),
                    dk_st + static_cast<uint64_t>(((ks >> 2) * S::kBlk + (ks & 3) * 32) >> 4), idesc_qk, ks > 0 ? 1u : 0u);
          umma_commit(bar(kSFull + (j & 1)));
        }
        __syncwarp();
      };
      mbar_wait(bar(kQFull), 0);
      tc_fence_after();
      if (n_kt > 0) issue_qk(0);
      for (int j = 0; j < n_kt; ++j) {
        if (j + 1 < n_kt) issue_qk(j + 1);
        const int st = j % kStages;
        mbar_wait(bar(kPReady + (j & 1)), (j >> 1) & 1);
        mbar_wait(bar(kFullV + st), (j / kStages) & 1);
        tc_fence_after();
        if (elect_one()) {
          const uint64_t dv_st = dv + static_cast<uint64_t>((st * S::kTile) >> 4);
#pragma unroll
          for (int ks = 0; ks < BN / 16; ++ks)
            umma_ts(tmem_o, tmem_base + (j & 1) * BN + ks * 8, dv_st + static_cast<uint64_t>((ks * 2048) >> 4), idesc_pv,
                    (j > 0 || ks > 0) ? 1u : 0u);
          umma_commit(bar(kODone + (j & 1)));
        }
        __syncwarp();
      }
    }
  } else {
    // ===================================================================== softmax / correction / epilogue
    const int quarter = warp & 3;
    const int r = quarter * 32 + lane;
    const uint32_t lane_addr = tmem_base + (static_cast<uint32_t>(quarter * 32) << 16);
    const int pl = r / G, hl = r % G;
    const int ridx = ridx0 + pl;
    const bool valid = ridx < n_rows;
    const int pos = pos_of(ridx);
    float m_used = -INFINITY, l = 0.f;

    for (int j = 0; j < n_kt; ++j) {
      const int key0 = (jt0 + j) * BN;
      const bool need_mask = key0 + BN - 1 > p_min;     // tile reaches past the tile's first position
      const uint32_t s_addr = lane_addr + (j & 1) * BN;
      mbar_wait(bar(kSFull + (j & 1)), (j >> 1) & 1);
      tc_fence_after();

      uint32_t pk[BN / 2];      // P_j as bf16 pairs, kept in registers until the reference max is known to be valid
      float tile_sum;
      // max over this row's visible scores of the tile, in log2 units (only the first tile and the rare rescale need it)
      auto row_max = [&]() -> float {
        float mx0 = -INFINITY, mx1 = -INFINITY;
#pragma unroll
        for (int c = 0; c < BN / 32; ++c) {
          uint32_t t[32];
          tmem_ld32(s_addr + c * 32, t);
          tmem_wait_ld();
#pragma unroll
          for (int i = 0; i < 32; i += 2) {
            float v0 = __uint_as_float(t[i]), v1 = __uint_as_float(t[i + 1]);
            if (need_mask) {
              if (key0 + c * 32 + i > pos) v0 = -INFINITY;
              if (key0 + c * 32 + i + 1 > pos) v1 = -INFINITY;
            }
            mx0 = fmaxf(mx0, v0); mx1 = fmaxf(mx1, v1);
          }
        }
        return fmaxf(mx0, mx1) * scale_log2;
      };
      // One sweep over the S row: p = 2^(s*scale - m_ref) against the REFERENCE max of the previous tiles; returns whether
      // the reference max is stale (see the test at the end).  The sweep is issue-bound, so the unmasked tiles (all but the
      // diagonal ones) run on packed pairs: FFMA2 for scale-and-subtract, FADD2 for the row sum, MUFU.EX2 for the exponentials.
      auto sweep = [&](float m_ref) -> bool {
        uint32_t sa[32], sb[32];
        tmem_ld32(s_addr, sa);
        tmem_ld32(s_addr + 32, sb);
        if (!need_mask) {
          const uint64_t sc2 = f2_pack(scale_log2, scale_log2), nm2 = f2_pack(-m_ref, -m_ref);
          uint64_t l2a = 0ull, l2b = 0ull;
#pragma unroll
          for (int c = 0; c < BN / 32; ++c) {
            uint32_t(&cur)[32] = (c & 1) ? sb : sa;
            if (c == 0) tmem_wait_ld();
#pragma unroll
            for (int i = 0; i < 32; i += 8) {
              float p[8];
#pragma unroll
              for (int q = 0; q < 4; ++q) {
                const uint64_t t = f2_fma(f2_pack(__uint_as_float(cur[i + 2 * q]), __uint_as_float(cur[i + 2 * q + 1])), sc2, nm2);
                if (q < kMufuPairs) {
                  float t0, t1;
                  f2_unpack(t, t0, t1);
                  p[2 * q] = ex2(t0); p[2 * q + 1] = ex2(t1);
                } else {
                  ex2_poly2(t, p[2 * q], p[2 * q + 1]);
                }
              }
              l2a = f2_add(l2a, f2_add(f2_pack(p[0], p[1]), f2_pack(p[2], p[3])));
              l2b = f2_add(l2b, f2_add(f2_pack(p[4], p[5]), f2_pack(p[6], p[7])));
#pragma unroll
              for (int q = 0; q < 4; ++q) {
                const uint32_t w = pack_bf16(p[2 * q], p[2 * q + 1]);
                pk[c * 16 + (i >> 1) + q] = w;
              }
            }
          }
          float s0, s1;
          f2_unpack(f2_add(l2a, l2b), s0, s1);
          tile_sum = s0 + s1;
        } else {
          float l0 = 0.f, l1 = 0.f;
          tmem_wait_ld();
#pragma unroll
          for (int c = 0; c < BN / 32; ++c) {
            uint32_t(&cur)[32] = (c & 1) ? sb : sa;
#pragma unroll
            for (int i = 0; i < 32; i += 2) {
              float v0 = __uint_as_float(cur[i]), v1 = __uint_as_float(cur[i + 1]);
              const int k = key0 + c * 32 + i;
              if (k > pos) v0 = -INFINITY;
              if (k + 1 > pos) v1 = -INFINITY;
              const float p0 = ex2(fmaf(v0, scale_log2, -m_ref));
              const float p1 = ex2(fmaf(v1, scale_log2, -m_ref));
              l0 += p0; l1 += p1;
              const uint32_t w = pack_bf16(p0, p1);
              pk[c * 16 + (i >> 1)] = w;
            }
          }
          tile_sum = l0 + l1;
        }
        // Staleness test at no cost per element: any p > 2^8 (or an inf / NaN from an overflowed p) makes the row sum
        // exceed 2^8, and with an exact reference the sum is at most BN = 64, so P stays <= 2^8 as with a per-element
        // test (a 2^14 bound — BN * 2^8 — was tried and cost accuracy on the heavy-hitter config: 2.8e-2 vs <= 2e-2).
        return !(tile_sum <= kRescaleSum);
      };

      if (j == 0) {
        // first tile: the reference is its own max.  Key 0 is visible to every row, so it is finite on rank 0; on a
        // split-KV rank > 0 a row may see none of this CTA's keys: the clamp keeps the reference finite (p = 0, l = 0).
        m_used = fmaxf(row_max(), -1e30f);
        sweep(m_used);
      } else {
        const bool grow = sweep(m_used);
        if (__any_sync(0xffffffffu, grow)) {
          // lazy correction: O and l are relative to m_used; move the reference only when the max grew by > 2^8
          // P_{j-1} V_{j-1} has landed in O.  (Two alternating barriers: a warp may run one tile ahead of the
          // slowest warp, and a single barrier's parity would then alias two phases.)
          mbar_wait(bar(kODone + ((j - 1) & 1)), ((j - 1) >> 1) & 1);
          tc_fence_after();
          const float m_t = fmaxf(m_used, row_max());
          const float f = ex2(m_used - m_t);
          m_used = m_t;
          l *= f;
#pragma unroll
          for (int c = 0; c < D / 32; ++c) {
            uint32_t o[32];
            tmem_ld32(lane_addr + kColO + c * 32, o);
            tmem_wait_ld();
#pragma unroll
            for (int i = 0; i < 32; ++i) o[i] = __float_as_uint(__uint_as_float(o[i]) * f);
            tmem_st32(lane_addr + kColO + c * 32, o);
          }
          tmem_wait_st();
          sweep(m_used);                                 // S_j is still intact: P_j has not been stored yet
        }
      }
      l += tile_sum;
      tmem_st32(s_addr, pk);                             // P_j (BN/2 packed columns) over the first half of S_j
      if (key0 + BN > t_end) {
        // the last tile reaches into padding rows of the cache: their V must not poison O (0 * NaN)
        const int st = j % kStages;
        mbar_wait(bar(kFullV + st), (j / kStages) & 1);
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
      mbar_arrive(bar(kPReady + (j & 1)));
    }

    // epilogue: O / l -> bf16 -> global (each thread owns one (row, head) vector of D elements)
    if (n_kt > 0) {
      mbar_wait(bar(kODone + ((n_kt - 1) & 1)), ((n_kt - 1) >> 1) & 1);
      tc_fence_after();
    } else {
      m_used = -1e30f;                                       // no keys on this rank: neutral element of the merge
    }
    __nv_bfloat16* dst = out + ((static_cast<size_t>(b) * bd.t_stride + ridx) * hq + g * G + hl) * D;
    float w_own = 1.f, m_all = m_used;
    float w_rem[3] = {0.f, 0.f, 0.f};
    if (ncl > 1) {
      // ---- split-KV merge.  Ranks > 0 park (O, m, l) in their own shared memory: all of this CTA's TMA loads and
      // UMMAs have completed (o_done of the last tile), so the K/V rings are free.  O is laid out [D/4][128 rows] float4
      // so that both the local stores and rank 0's remote loads are conflict-free.
      float* s_stat = reinterpret_cast<float*>(smem + S::oStat);
      if (crank > 0) {
        float4* park = reinterpret_cast<float4*>(smem + S::oK);
#pragma unroll
        for (int c = 0; c < D / 32; ++c) {
          uint32_t o[32];
          if (n_kt > 0) {
            tmem_ld32(lane_addr + kColO + c * 32, o);
            tmem_wait_ld();
          } else {
#pragma unroll
            for (int i = 0; i < 32; ++i) o[i] = 0u;
          }
#pragma unroll
          for (int v4 = 0; v4 < 8; ++v4)
            park[(c * 8 + v4) * BM + r] = make_float4(__uint_as_float(o[4 * v4]), __uint_as_float(o[4 * v4 + 1]),
                                                      __uint_as_float(o[4 * v4 + 2]), __uint_as_float(o[4 * v4 + 3]));
        }
        s_stat[r] = m_used;
        s_stat[BM + r] = l;
      }
    }
    if (ncl > 1) {
      cluster_sync_all();                                    // parked partials are visible cluster-wide
      if (crank == 0) {
        float m_r[3] = {-1e30f, -1e30f, -1e30f}, l_r[3] = {0.f, 0.f, 0.f};
#pragma unroll
        for (int q = 1; q < 4; ++q) {
          if (q < ncl) {
            const uint32_t st_addr = dsmem_addr(sbase + S::oStat + r * 4, q);
            m_r[q - 1] = ld_dsmem_f32(st_addr);
            l_r[q - 1] = ld_dsmem_f32(st_addr + BM * 4);
            m_all = fmaxf(m_all, m_r[q - 1]);
          }
        }
        w_own = ex2(m_used - m_all);
        l *= w_own;
#pragma unroll
        for (int q = 1; q < 4; ++q) {                        // fixed rank order: bit-reproducible
          if (q < ncl) {
            w_rem[q - 1] = ex2(m_r[q - 1] - m_all);
            l += l_r[q - 1] * w_rem[q - 1];
          }
        }
      }
    }
    if (crank == 0) {
      const float inv = 1.f / l;
#pragma unroll
      for (int c = 0; c < D / 32; ++c) {
        uint32_t o[32];
        tmem_ld32(lane_addr + kColO + c * 32, o);
        tmem_wait_ld();
        if (ncl > 1) {
#pragma unroll
          for (int i = 0; i < 32; ++i) o[i] = __float_as_uint(__uint_as_float(o[i]) * w_own);
#pragma unroll
          for (int q = 1; q < 4; ++q) {
            if (q >= ncl) break;
            const uint32_t base = dsmem_addr(sK + (c * 8 * BM + r) * 16, q);
            const float w = w_rem[q - 1];
#pragma unroll
            for (int v4 = 0; v4 < 8; ++v4) {
              const float4 t = ld_dsmem_f32x4(base + v4 * BM * 16);
              o[4 * v4] = __float_as_uint(fmaf(t.x, w, __uint_as_float(o[4 * v4])));
              o[4 * v4 + 1] = __float_as_uint(fmaf(t.y, w, __uint_as_float(o[4 * v4 + 1])));
              o[4 * v4 + 2] = __float_as_uint(fmaf(t.z, w, __uint_as_float(o[4 * v4 + 2])));
              o[4 * v4 + 3] = __float_as_uint(fmaf(t.w, w, __uint_as_float(o[4 * v4 + 3])));
            }
          }
        }
        if (valid) {
#pragma unroll
          for (int v4 = 0; v4 < 4; ++v4) {
            uint4 w;
            w.x = pack_bf16(__uint_as_float(o[8 * v4 + 0]) * inv, __uint_as_float(o[8 * v4 + 1]) * inv);
            w.y = pack_bf16(__uint_as_float(o[8 * v4 + 2]) * inv, __uint_as_float(o[8 * v4 + 3]) * inv);
            w.z = pack_bf16(__uint_as_float(o[8 * v4 + 4]) * inv, __uint_as_float(o[8 * v4 + 5]) * inv);
            w.w = pack_bf16(__uint_as_float(o[8 * v4 + 6]) * inv, __uint_as_float(o[8 * v4 + 7]) * inv);
            *reinterpret_cast<uint4*>(dst + c * 32 + v4 * 8) = w;
          }
        }
      }
      if (valid && lse_out)
        lse_out[(static_cast<size_t>(b) * bd.t_stride + ridx) * hq + g * G + hl] = (m_all + log2f(l)) * kLn2;
    }
  }
  if (ncl > 1) {
    if (warp < 2) cluster_sync_all();                        // producer / issuer warps: pair the softmax warps' first sync
    cluster_sync_all();                                      // parked partials stay alive until rank 0 has merged them
  }

  tc_fence_before();
  __syncthreads();
  if (warp == 1) {
    tc_fence_after();
    tmem_dealloc<kTmemCols>(tmem_base);
  }
}

// ---------------------------------------------------------------------------------------------- host side
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

// [B][T][Hkv][d] bf16, box = 128 rows x 64 elements of one head, 128-byte swizzle, zero fill out of bounds
bool make_kv_map(CUtensorMap* m, const void* base, int batch, int t_stride, int hkv, int d) {
  EncodeFn enc = get_encode();
  if (!enc) return false;
  const cuuint64_t dims[4] = {static_cast<cuuint64_t>(d), static_cast<cuuint64_t>(hkv),
                              static_cast<cuuint64_t>(t_stride), static_cast<cuuint64_t>(batch)};
  const cuuint64_t strides[3] = {static_cast<cuuint64_t>(d) * 2, static_cast<cuuint64_t>(hkv) * d * 2,
                                 static_cast<cuuint64_t>(t_stride) * hkv * d * 2};
  const cuuint32_t box[4] = {64, 1, BN, 1};   // BN keys x 64 elements
  const cuuint32_t estr[4] = {1, 1, 1, 1};
  return enc(m, CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, 4, const_cast<void*>(base), dims, strides, box, estr,
             CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
             CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) == CUDA_SUCCESS;
}

}  // namespace

cudaError_t launch_attn(const qcf_ctx* ctx, const qcf_batch* b, const int32_t* sel, const int32_t* n_sel,
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
  // Split-KV width (cluster size).  Splitting costs a second prologue/epilogue per item and a cluster rendezvous, and
  // measured on c2 (400 items for 296 resident CTAs, where the SMs are throughput-bound) it loses to the unsplit launch,
  // so it is used only where the unsplit grid leaves most of the machine empty: few rows against a long cache
  // (rho ~ 0: the Lq query rows alone give Lq*G/128 items per kv-head).  A scheduling hint only — the selected rows
  // are device-side: rows ~ ratio_hint * N + Lq in selective mode.
  int ncl = ctx->attn_cluster;
  if (ncl == 0) {
    double items = 0.0;
    for (int i = 0; i < b->batch; ++i) {
      const int n = b->h_n_ctx[i], lq = b->h_n_query[i];
      const double rows = sel ? ctx->ratio_hint * n + lq : static_cast<double>(n + lq);
      items += std::ceil(rows / PT) * L.hkv;
    }
    const double slots = 2.0 * ctx->n_sm;
    const int kt_max = (b->t_stride + BN - 1) / BN;
    ncl = (kt_max >= 16 && items * 4 <= slots) ? 4 : ((kt_max >= 8 && items * 2 <= slots) ? 2 : 1);
  }
  // L2-locality groups (see the kernel's work decode): units whose K + V (t_stride rows of one kv-head each) fit in ~48 MB
  // of the 126 MB L2 — two consecutive groups overlap at their boundary; whole requests when more than one fits.
  const int n_units = L.hkv * b->batch;
  const double unit_bytes = static_cast<double>(b->t_stride) * L.d * 2.0 * 2.0;
  // (16 / 24 / 48 / 96 MB measured: a5 at c4 x 16 2.89 / 2.86 / 2.84 / 2.97 ms, c5 2.55 / 2.59 / 2.55 / 2.61 ms)
  int unit_grp = static_cast<int>(48.0 * 1024 * 1024 / unit_bytes);
  if (unit_grp >= L.hkv) unit_grp -= unit_grp % L.hkv;
  if (unit_grp < 1) unit_grp = 1;
  if (unit_grp > n_units) unit_grp = n_units;
  const int n_groups = (n_units + unit_grp - 1) / unit_grp;
  // row-count hint: |R_b| ~ ratio_hint * N_b + Lq_b in selective mode (the true count is device-side: tiles past the hint
  // are still covered, in section B of the grid)
  int tiles_hint = max_tiles;
  if (sel) {
    const double rows = ctx->ratio_hint * b->n_stride + b->q_stride;
    tiles_hint = static_cast<int>(std::ceil(rows / PT)) + 1;
    if (tiles_hint > max_tiles) tiles_hint = max_tiles;
    if (tiles_hint < 1) tiles_hint = 1;
  }
  const long long n_items = static_cast<long long>(n_groups) * tiles_hint * unit_grp +
                            static_cast<long long>(max_tiles - tiles_hint) * n_units;
  const dim3 grid(static_cast<unsigned>(n_items * ncl));
  const float scale_log2 = L.scale * kLog2e;
  cudaLaunchConfig_t cfg{};
  cfg.gridDim = grid;
  cfg.blockDim = dim3(kThreads);
  cfg.stream = stream;
  cudaLaunchAttribute attrs[2];
  attrs[1].id = cudaLaunchAttributeProgrammaticStreamSerialization;
  attrs[1].val.programmaticStreamSerializationAllowed = 1;
  attrs[0].id = cudaLaunchAttributeClusterDimension;
  attrs[0].val.clusterDim.x = static_cast<unsigned>(ncl);
  attrs[0].val.clusterDim.y = 1;
  attrs[0].val.clusterDim.z = 1;
  cfg.attrs = attrs;
  cfg.numAttrs = ctx->pdl ? 2 : 1;
  const BatchDev bd = b->dev;
  const int hq = L.hq, hkv = L.hkv;
  if (L.d == 128) {
    auto kern = attn_tc_kernel<128>;
    cfg.dynamicSmemBytes = Smem<128>::kBytes + 1024;
    cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, static_cast<int>(cfg.dynamicSmemBytes));
    return cudaLaunchKernelEx(&cfg, kern, tm_k, tm_v, bd, hq, hkv, tiles_hint, unit_grp, scale_log2, sel, n_sel, q,
                              rows_by_position, out, lse);
  }
  auto kern = attn_tc_kernel<64>;
  cfg.dynamicSmemBytes = Smem<64>::kBytes + 1024;
  cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, static_cast<int>(cfg.dynamicSmemBytes));
  return cudaLaunchKernelEx(&cfg, kern, tm_k, tm_v, bd, hq, hkv, tiles_hint, unit_grp, scale_log2, sel, n_sel, q,
                            rows_by_position, out, lse);
}

}  // namespace qcf
