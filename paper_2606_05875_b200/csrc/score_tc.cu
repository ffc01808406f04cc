// a2 on the 5th-generation tensor cores — Eq. 18 / 20:
//
//   I(t) = 1/(Hq Lq) sum_{i,h} exp(s_{i,h,t} - lse_{i,h}),   s = q_probe[i][h] . K'[t][h/G] * scale
//
// The row normaliser lse spans ALL context keys, so two sweeps are needed, and each wants its reduction to be local to a
// thread (= one TMEM lane):
//   pass 1 (stats)  : S   = Q_tile K_j^T   query rows on the lanes, key tiles streamed -> per-row (max, sum-exp)
//   pass 2 (colsum) : S^T = K_tile Q_j^T   KEYS on the lanes, query-row chunks streamed -> per-key sum_r 2^(s - lse_r)
// Both are the same warp-specialised skeleton: a fixed 128-row operand A and a 2-stage TMA ring of 128-row operands B
// (128-byte swizzle), S double-buffered in TMEM (2 x 128 fp32 columns), one UMMA-issuing thread, and 256 consumer
// threads: two per TMEM lane, each sweeping one 64-column half of the lane (a sweep is bound by MUFU / TMEM-load latency
// per warp, not by issue slots — ncu on the one-thread-per-lane version: 0.59 eligible warps per cycle and scheduler,
// XU pipe 68 % / 52 % busy — so twice the warps per SM sub-partition is what fills the pipe; nothing has to be agreed
// between the two halves inside the loop: each keeps its own lazy reference max / partial column sum).  GQA packing: a "query row" is (token i, head hl) of one kv-head,
// r = i * G + hl, loaded by TMA boxes {64 elements, G heads, 128/G tokens}.  The Hkv per-head partial column sums are
// combined in fixed order by the last CTA of each key tile (bit-reproducible scores, deterministic top-k).
#include <cmath>

#include "qcf_internal.cuh"
#include "sm100_ptx.cuh"

namespace qcf {

namespace {

using namespace ptx;

constexpr int BT = 128;            // rows of A, rows of one B tile, fp32 columns of one S buffer
constexpr int kThreads = 320;       // producer warp, issuer warp, 2 x 4 consumer warps
constexpr int kConsumers = 256;
constexpr int HC = BT / 2;          // S columns swept by one consumer thread
constexpr int kTmemCols = 256;
constexpr float kLog2e = 1.4426950408889634f;
constexpr float kStaleSum = 1099511627776.0f;      // 2^40
// Of every 4 pairs, how many take MUFU.EX2 (the rest: the packed polynomial on the FMA pipe).  Unlike attention (no P V, no
// P packing) these sweeps are MUFU-bound — 128 x 128 exponentials against a 256-cycle MMA per tile — so a quarter of them
// moves to the FMA pipe: a2 on c4 600 -> 530 us, c5 295 -> 262 us, c2 30.8 -> 29.1 us (a half: 570 / 273 / 29.6).
constexpr int kMufuPairs = 3;

template <int D>
struct Smem {
  static constexpr int kBlk = BT * 128;                 // one 64-column block (128 rows x 128 B)
  static constexpr int kTile = BT * D * 2;
  static constexpr int oA = 0;
  static constexpr int oB = kTile;
  static constexpr int oBar = oB + 2 * kTile;
  static constexpr int kNumBar = 10;
  static constexpr int oTmem = oBar + kNumBar * 8;
  static constexpr int oFlag = oTmem + 8;
  static constexpr int oLse = oFlag + 8;                // pass 2: -lse of ALL query rows of the (request, kv-head), then the upper
                                                        // halves' column sums [2][128] and the last-arriver flags [kt_per_cta]; size set at launch
  static constexpr int kBytes = oLse;
};
enum { kAFull = 0, kBFull = 1, kBEmpty = 3, kSFull = 5, kSEmpty = 7, kAEmpty = 9 };

struct ScoreArgs {
  float scale_log2;
  int hq, hkv, n_splits;
  int norm_heads;                                        // Hq of the WHOLE layer (Hq * head shards): Eq. 18's 1/(Hq Lq)
  int kt_per_cta;                                        // pass 2: key tiles walked by one CTA
  float* stats_m; float* stats_l; int stats_rows;        // [B][2 * n_splits][stats_rows]: a key split x a column half
  float* part; int part_stride;                          // [B][Hkv][part_stride]
  unsigned int* counters;
  float* scores; int accumulate;
  // fused exchange of the KV-head-sharded step: the combined value also goes to slot exch_rank of every rank's buffer
  // (slot set exch_parity = epoch & 1: the other set still holds the previous epoch, which a slower peer may be ranking)
  float* const* exch_peers; int exch_rank, exch_world, exch_parity; long long exch_slot_elems;
};

template <int D, int PASS>
__global__ void __launch_bounds__(kThreads, 2)
score_tc_kernel(const __grid_constant__ CUtensorMap tm_q, const __grid_constant__ CUtensorMap tm_k, BatchDev bd,
                ScoreArgs a) {
  extern __shared__ unsigned char smem_raw[];
  unsigned char* smem = smem_raw + ((1024u - (smem_u32(smem_raw) & 1023u)) & 1023u);
  using S = Smem<D>;
  const int G = a.hq / a.hkv;
  const int TPT = BT / G;                         // query tokens per 128-row tile
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;

  // ---- work decode
  int b, g, row_tile = 0, key_tile = 0, split = 0;
  if (PASS == 1) {
    split = blockIdx.x; row_tile = blockIdx.y; g = blockIdx.z % a.hkv; b = blockIdx.z / a.hkv;
  } else {
    key_tile = blockIdx.x * a.kt_per_cta; g = blockIdx.y; b = blockIdx.z;       // first key tile of this CTA
  }
  const int N = bd.n_ctx[b], Lq = bd.n_query[b];
  const int rows = Lq * G;
  int k_begin = 0, k_end = 0, n_j = 0, n_kt = 1;          // n_kt: A tiles this CTA walks (pass 2: key tiles)
  if (PASS == 1) {
    if (row_tile * BT >= rows) { pdl_trigger(); pdl_wait(); return; }   // every CTA waits: the grid never completes before its predecessor
    const int span = (((N + a.n_splits - 1) / a.n_splits + BT - 1) / BT) * BT;
    k_begin = split * span;
    k_end = min(N, k_begin + span);
    n_j = k_end > k_begin ? (k_end - k_begin + BT - 1) / BT : 0;
  } else {
    n_kt = min(a.kt_per_cta, (N + BT - 1) / BT - key_tile);
    if (n_kt <= 0) { pdl_trigger(); pdl_wait(); return; }
    n_j = (rows + BT - 1) / BT;
  }

  const uint32_t sbase = smem_u32(smem);
  const uint32_t sA = sbase + S::oA, sB = sbase + S::oB;
  auto bar = [&](int i) -> uint32_t { return sbase + S::oBar + 8 * i; };
  volatile uint32_t* tmem_slot = reinterpret_cast<volatile uint32_t*>(smem + S::oTmem);
  float* s_lse = reinterpret_cast<float*>(smem + S::oLse);

  if (warp == 0) {
    if (lane == 0) {
      prefetch_tensormap(&tm_q);
      prefetch_tensormap(&tm_k);
      mbar_init(bar(kAFull), 1);
      mbar_init(bar(kAEmpty), 1);
      for (int i = 0; i < 2; ++i) {
        mbar_init(bar(kBFull + i), 1);
        mbar_init(bar(kBEmpty + i), 1);
        mbar_init(bar(kSFull + i), 1);
        mbar_init(bar(kSEmpty + i), kConsumers);
      }
      fence_barrier_init();
    }
  } else if (warp == 1) {
    tmem_alloc<kTmemCols>(sbase + S::oTmem);
  }
  pdl_trigger();
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  const uint32_t tmem_base = *tmem_slot;
  pdl_wait();          // barrier init, TMEM allocation and descriptor prefetch above overlap the predecessor's tail

  // TMA coordinates of a 128-row tile of query rows / of keys
  auto load_q_tile = [&](uint32_t dst, uint32_t mbar, int tile) {
#pragma unroll
    for (int kb = 0; kb < D / 64; ++kb) tma_load_4d(dst + kb * S::kBlk, &tm_q, mbar, kb * 64, g * G, tile * TPT, b);
  };
  auto load_k_tile = [&](uint32_t dst, uint32_t mbar, int key0) {
#pragma unroll
    for (int kb = 0; kb < D / 64; ++kb) tma_load_4d(dst + kb * S::kBlk, &tm_k, mbar, kb * 64, g, key0, b);
  };

  if (warp == 0) {
    // ===================================================================== producer
    // converged warp, one ELECTED lane issues: a divergent `if (lane == 0)` makes the compiler wrap every TMA / UMMA
    // instruction (uniform-register operands) in a per-lane ELECT / BRA.U.ANY loop
    if (n_j > 0) {
      for (int kt = 0, it = 0; kt < n_kt; ++kt) {
        if (kt > 0) mbar_wait(bar(kAEmpty), (kt - 1) & 1);      // every MMA that read the previous A tile has completed
        if (elect_one()) {
          mbar_arrive_expect_tx(bar(kAFull), S::kTile);
          if (PASS == 1) load_q_tile(sA, bar(kAFull), row_tile); else load_k_tile(sA, bar(kAFull), (key_tile + kt) * BT);
        }
        __syncwarp();
        for (int j = 0; j < n_j; ++j, ++it) {
          const int st = it & 1;
          // stage st is free once the MMAs of step it - 2 have completed: the phase S of that step was signalled on
          if (it >= 2) mbar_wait(bar(kSFull + st), ((it >> 1) & 1) ^ 1);
          if (elect_one()) {
            mbar_arrive_expect_tx(bar(kBFull + st), S::kTile);
            if (PASS == 1) load_k_tile(sB + st * S::kTile, bar(kBFull + st), k_begin + j * BT);
            else load_q_tile(sB + st * S::kTile, bar(kBFull + st), j);
          }
          __syncwarp();
        }
      }
    }
  } else if (warp == 1) {
    // ===================================================================== UMMA issuer (converged warp, elected lane)
    if (n_j > 0) {
      constexpr uint32_t idesc = umma_idesc_bf16(BT, BT, false, false);
      // base descriptors once; a k-step's operands are base + (byte offset >> 4) (16-byte units, no carry out of the field)
      const uint64_t da0 = umma_smem_desc_sw128(sA, 16, 1024), db0 = umma_smem_desc_sw128(sB, 16, 1024);
      for (int kt = 0, it = 0; kt < n_kt; ++kt) {
        mbar_wait(bar(kAFull), kt & 1);
        for (int j = 0; j < n_j; ++j, ++it) {
          const int st = it & 1;
          const uint32_t ph = (it >> 1) & 1;
          mbar_wait(bar(kSEmpty + st), ph ^ 1);               // consumers have released the S buffer used two steps ago
          mbar_wait(bar(kBFull + st), ph);
          tc_fence_after();
          if (elect_one()) {
            const uint64_t db = db0 + static_cast<uint64_t>((st * S::kTile) >> 4);
#pragma unroll
            for (int ks = 0; ks < D / 16; ++ks) {
              const uint64_t koff = static_cast<uint64_t>(((ks >> 2) * S::kBlk + (ks & 3) * 32) >> 4);
              umma_ss(tmem_base + st * BT, da0 + koff, db + koff, idesc, ks > 0 ? 1u : 0u);
            }
            umma_commit(bar(kSFull + st));
            if (j == n_j - 1) umma_commit(bar(kAEmpty));
          }
          __syncwarp();
        }
      }
    }
  } else {
    // ===================================================================== consumers: two threads per TMEM lane
    const int quarter = warp & 3;                    // a warp may only touch TMEM lanes 32 * (warp % 4) ..
    const int half = (warp - 2) >> 2;                // which 64-column half of every S tile this thread sweeps
    const int r = quarter * 32 + lane;
    const uint32_t lane_addr = tmem_base + (static_cast<uint32_t>(quarter * 32) << 16) + half * HC;
    // One 64-column half of S[st]: sum over its columns of 2^(s * scale + z_c) with z_c = nz[c] (pass 2: -lse of the
    // chunk's rows, from shared memory) or one scalar (pass 1: -reference max).  Full tiles run on packed pairs (FFMA2 /
    // FADD2), kMufuPairs of every 4 pairs on MUFU.EX2 and the rest on the FMA pipe; 16-column TMEM loads, double-buffered.
    auto sweep_full = [&](uint32_t s_addr, const float4* z4, float zs, uint64_t& acc_a, uint64_t& acc_b) {
      const uint64_t sc2 = f2_pack(a.scale_log2, a.scale_log2);
      const uint64_t zs2 = f2_pack(zs, zs);
      uint32_t sa[16], sb[16];
      tmem_ld16(s_addr, sa);
#pragma unroll
      for (int c = 0; c < HC / 16; ++c) {
        uint32_t(&sv)[16] = (c & 1) ? sb : sa;
        tmem_wait_ld();
        if (c + 1 < HC / 16) tmem_ld16(s_addr + (c + 1) * 16, (c & 1) ? sa : sb);
#pragma unroll
        for (int i = 0; i < 16; i += 8) {
          uint64_t nz[4];
          if (z4) {
            const float4 za = z4[c * 4 + (i >> 2)], zb = z4[c * 4 + (i >> 2) + 1];   // same address in every lane: broadcast
            nz[0] = f2_pack(za.x, za.y); nz[1] = f2_pack(za.z, za.w); nz[2] = f2_pack(zb.x, zb.y); nz[3] = f2_pack(zb.z, zb.w);
          } else {
            nz[0] = nz[1] = nz[2] = nz[3] = zs2;
          }
          float p[8];
#pragma unroll
          for (int q = 0; q < 4; ++q) {
            const uint64_t t = f2_fma(f2_pack(__uint_as_float(sv[i + 2 * q]), __uint_as_float(sv[i + 2 * q + 1])), sc2, nz[q]);
            if (q < kMufuPairs) {
              float t0, t1;
              f2_unpack(t, t0, t1);
              p[2 * q] = ex2(t0); p[2 * q + 1] = ex2(t1);
            } else {
              ex2_poly2(t, p[2 * q], p[2 * q + 1]);
            }
          }
          acc_a = f2_add(acc_a, f2_add(f2_pack(p[0], p[1]), f2_pack(p[2], p[3])));
          acc_b = f2_add(acc_b, f2_add(f2_pack(p[4], p[5]), f2_pack(p[6], p[7])));
        }
      }
    };
    // the same over the first n_valid (< HC, possibly <= 0) columns only
    auto sweep_tail = [&](uint32_t s_addr, const float* z, float zs, int n_valid) -> float {
      float l0 = 0.f, l1 = 0.f;
#pragma unroll
      for (int c = 0; c < HC / 16; ++c) {
        uint32_t sv[16];
        tmem_ld16(s_addr + c * 16, sv);
        tmem_wait_ld();
#pragma unroll
        for (int i = 0; i < 16; i += 2) {
          const int col = c * 16 + i;
          const float z0 = z ? z[col] : zs, z1 = z ? z[col + 1] : zs;
          l0 += col < n_valid ? ex2(fmaf(__uint_as_float(sv[i]), a.scale_log2, z0)) : 0.f;
          l1 += col + 1 < n_valid ? ex2(fmaf(__uint_as_float(sv[i + 1]), a.scale_log2, z1)) : 0.f;
        }
      }
      return l0 + l1;
    };
    if (PASS == 1) {
      // lane = query row, this thread's key columns: online (max, sum-exp) over the streamed keys, reference max moved lazily
      float m_ref = -INFINITY, l = 0.f;
      for (int j = 0; j < n_j; ++j) {
        const int st = j & 1;
        const int key0 = k_begin + j * BT + half * HC;               // first key of my columns
        const int n_valid = k_end - key0;                            // >= HC: all my columns are keys of the range
        const uint32_t s_addr = lane_addr + st * BT;
        mbar_wait(bar(kSFull + st), (j >> 1) & 1);
        tc_fence_after();
        // max of this row's scores over my valid columns, log2 units (first tile and the rare rescale only)
        auto tile_rowmax = [&]() -> float {
          float mx0 = -INFINITY, mx1 = -INFINITY;
#pragma unroll
          for (int c = 0; c < HC / 16; ++c) {
            uint32_t sv[16];
            tmem_ld16(s_addr + c * 16, sv);
            tmem_wait_ld();
#pragma unroll
            for (int i = 0; i < 16; i += 2) {
              const int col = c * 16 + i;
              mx0 = fmaxf(mx0, col < n_valid ? __uint_as_float(sv[i]) : -INFINITY);
              mx1 = fmaxf(mx1, col + 1 < n_valid ? __uint_as_float(sv[i + 1]) : -INFINITY);
            }
          }
          return fmaxf(mx0, mx1) * a.scale_log2;
        };
        // no per-element max: a stale reference shows up as a huge (or inf) sum
        auto sweep_sum = [&](float ref) -> float {
          if (n_valid >= HC) {
            uint64_t la = 0ull, lb = 0ull;
            sweep_full(s_addr, nullptr, -ref, la, lb);
            float s0, s1;
            f2_unpack(f2_add(la, lb), s0, s1);
            return s0 + s1;
          }
          return sweep_tail(s_addr, nullptr, -ref, n_valid);
        };
        float tile_sum = 0.f;
        if (n_valid > 0) {
          if (m_ref == -INFINITY) {
            m_ref = tile_rowmax();                  // first tile with a valid column of mine: finite
            tile_sum = sweep_sum(m_ref);
          } else {
            tile_sum = sweep_sum(m_ref);
          }
        }
        // fp32 sums do not care how stale the reference is until they overflow: move it when a tile's sum passes 2^40
        if (__any_sync(0xffffffffu, !(tile_sum <= kStaleSum))) {
          const float m_t = fmaxf(m_ref, tile_rowmax());
          l *= ex2(m_ref - m_t);
          m_ref = m_t;
          tile_sum = sweep_sum(m_ref);
        }
        l += tile_sum;
        tc_fence_before();
        mbar_arrive(bar(kSEmpty + st));
      }
      // the two halves of a row are two more "splits" of the key range: partial (max, sum-exp), combined by pass 2
      const int row = row_tile * BT + r;
      if (row < rows) {
        const size_t o = (static_cast<size_t>(b) * (2 * a.n_splits) + 2 * split + half) * a.stats_rows + static_cast<size_t>(g) * rows + row;
        a.stats_m[o] = m_ref;                      // no valid key: (-inf, 0), neutral in the combine
        a.stats_l[o] = l;
      }
    } else {
      // lane = key, this thread's query-row columns: sum over the streamed rows of 2^(s * scale - lse_row).  The CTA walks
      // n_kt key tiles of one (request, kv-head); -lse of every query row is combined from the pass-1 partials ONCE
      // (log2 domain) and kept in shared memory.
      const int ctid = (warp - 2) * 32 + lane;               // 0..255
      const int n_parts = 2 * a.n_splits;
      for (int row = ctid; row < n_j * BT; row += kConsumers) {
        float lse = INFINITY;                                // rows past the end contribute 2^(-inf) = 0
        if (row < rows) {
          // partials are laid out [part][row]: for a fixed part consecutive threads read consecutive words
          const size_t o = static_cast<size_t>(b) * n_parts * a.stats_rows + static_cast<size_t>(g) * rows + row;
          float M = -INFINITY, L = 0.f;
          // sixteen parts at a time: all loads of a row are issued before the first is used — one L2 round trip per row
          // instead of one per few parts; the combine order is fixed, a missing part is the neutral (-inf, 0)
          for (int s0 = 0; s0 < n_parts; s0 += 16) {
            float ms[16], ls[16];
#pragma unroll
            for (int u = 0; u < 16; ++u) {
              const bool ok = s0 + u < n_parts;
              const size_t idx = o + static_cast<size_t>(ok ? s0 + u : 0) * a.stats_rows;
              ms[u] = __ldcg(a.stats_m + idx);
              ls[u] = __ldcg(a.stats_l + idx);
              if (!ok) { ms[u] = -INFINITY; ls[u] = 0.f; }
            }
#pragma unroll
            for (int u = 0; u < 16; ++u) {
              const float Mn = fmaxf(M, ms[u]);
              if (Mn > -INFINITY) L = L * ex2(M - Mn) + ls[u] * ex2(ms[u] - Mn);
              M = Mn;
            }
          }
          lse = M + log2f(L);
        }
        s_lse[row] = -lse;
      }
      asm volatile("bar.sync 1, 256;" ::: "memory");
      float* s_half = s_lse + n_j * BT;                      // [2][BT]: column sums of the upper halves, double-buffered
      int* s_last = reinterpret_cast<int*>(s_half + 2 * BT); // [n_kt]: this CTA was the last of the key tile's Hkv CTAs
      const int n_tiles_b = (bd.n_stride + BT - 1) / BT;
      for (int kt = 0, it = 0; kt < n_kt; ++kt) {
        uint64_t acc01 = 0ull, acc23 = 0ull;                 // packed fp32 pairs of partial column sums
        float acc_t = 0.f;
        for (int j = 0; j < n_j; ++j, ++it) {
          const int st = it & 1;
          mbar_wait(bar(kSFull + st), (it >> 1) & 1);
          tc_fence_after();
          const float* z = s_lse + j * BT + half * HC;       // -lse of my columns' rows
          const int n_valid = rows - (j * BT + half * HC);   // < HC only in the last chunk
          if (n_valid >= HC) sweep_full(lane_addr + st * BT, reinterpret_cast<const float4*>(z), 0.f, acc01, acc23);
          else acc_t += sweep_tail(lane_addr + st * BT, z, 0.f, n_valid);   // rows past the end hold whatever the buffer holds
          tc_fence_before();
          mbar_arrive(bar(kSEmpty + st));
        }
        const int kt_abs = key_tile + kt;
        const int key = kt_abs * BT + r;
        float a0, a1;
        f2_unpack(f2_add(acc01, acc23), a0, a1);
        const float tot = (a0 + a1) + acc_t;
        if (half == 1) s_half[(kt & 1) * BT + r] = tot;
        asm volatile("bar.sync 1, 256;" ::: "memory");
        if (half == 0 && key < N)
          a.part[(static_cast<size_t>(b) * a.hkv + g) * a.part_stride + key] = tot + s_half[(kt & 1) * BT + r];
      }
      // The last CTA of each key tile sums the Hkv partials in fixed order (deterministic).  ONE fence for all the tiles
      // this CTA walked (a device-scope fence inside the tile loop was 0.65 stall cycles per issue in the old kernel).
      __threadfence();
      asm volatile("bar.sync 1, 256;" ::: "memory");
      for (int kt = ctid; kt < n_kt; kt += kConsumers)
        s_last[kt] = atomicAdd(a.counters + static_cast<size_t>(b) * n_tiles_b + key_tile + kt, 1u) == static_cast<unsigned int>(a.hkv - 1);
      asm volatile("bar.sync 1, 256;" ::: "memory");
      __threadfence();
      for (int kt = half; kt < n_kt; kt += 2) {              // the two consumer groups take alternate tiles
        if (!s_last[kt]) continue;
        const int key = (key_tile + kt) * BT + r;
        if (key < N) {
          float sum = 0.f;
          for (int gg = 0; gg < a.hkv; ++gg) sum += __ldcg(a.part + (static_cast<size_t>(b) * a.hkv + gg) * a.part_stride + key);
          const float v = rows > 0 ? sum / static_cast<float>(a.norm_heads * Lq) : 0.f;
          float* dst = a.scores + static_cast<size_t>(b) * bd.n_stride + key;
          const float nv = a.accumulate ? *dst + v : v;
          *dst = nv;
          if (a.exch_world > 1) {
            // this rank's partial of Eq. 18, straight into every rank's exchange buffer (peer memory: NVLink / IPC)
            const size_t off = kExchHeaderElems + static_cast<size_t>(a.exch_parity * a.exch_world + a.exch_rank) * a.exch_slot_elems +
                               static_cast<size_t>(b) * bd.n_stride + key;
            for (int p = 0; p < a.exch_world; ++p) a.exch_peers[p][off] = nv;
          }
        }
        if (r == 0) a.counters[static_cast<size_t>(b) * n_tiles_b + key_tile + kt] = 0u;     // self-resetting
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
// [B][T][H][d] bf16; box = {64 elements, box_heads heads, box_rows rows}; 128-byte swizzle; zero fill out of bounds
bool make_map(CUtensorMap* m, const void* base, int batch, int t_stride, int heads, int d, int box_heads, int box_rows) {
  EncodeFn enc = get_encode();
  if (!enc) return false;
  const cuuint64_t dims[4] = {static_cast<cuuint64_t>(d), static_cast<cuuint64_t>(heads),
                              static_cast<cuuint64_t>(t_stride), static_cast<cuuint64_t>(batch)};
  const cuuint64_t strides[3] = {static_cast<cuuint64_t>(d) * 2, static_cast<cuuint64_t>(heads) * d * 2,
                                 static_cast<cuuint64_t>(t_stride) * heads * d * 2};
  const cuuint32_t box[4] = {64, static_cast<cuuint32_t>(box_heads), static_cast<cuuint32_t>(box_rows), 1};
  const cuuint32_t estr[4] = {1, 1, 1, 1};
  return enc(m, CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, 4, const_cast<void*>(base), dims, strides, box, estr,
             CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
             CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) == CUDA_SUCCESS;
}

template <int D>
cudaError_t launch(const qcf_ctx* ctx, const qcf_batch* b, const CUtensorMap& tm_q, const CUtensorMap& tm_k,
                   ScoreArgs a, int row_tiles, int key_tiles, cudaStream_t stream) {
  const int smem1 = Smem<D>::kBytes + 1024;
  // pass 2 keeps -lse of every query row of a (request, kv-head), 2 x 128 half sums and one flag per walked key tile
  const int smem = smem1 + row_tiles * BT * 4 + 2 * BT * 4 + a.kt_per_cta * 4;
  if (row_tiles > 0) {
    auto k1 = score_tc_kernel<D, 1>;
    cudaFuncSetAttribute(k1, cudaFuncAttributeMaxDynamicSharedMemorySize, smem1);
    cudaError_t e = launch_pdl(ctx->pdl, k1, dim3(a.n_splits, row_tiles, b->batch * a.hkv), dim3(kThreads), smem1, stream, tm_q, tm_k, b->dev, a);
    if (e != cudaSuccess) return e;
  }
  auto k2 = score_tc_kernel<D, 2>;
  cudaFuncSetAttribute(k2, cudaFuncAttributeMaxDynamicSharedMemorySize, smem);
  const int groups = (key_tiles + a.kt_per_cta - 1) / a.kt_per_cta;
  return launch_pdl(ctx->pdl, k2, dim3(groups, a.hkv, b->batch), dim3(kThreads), smem, stream, tm_q, tm_k, b->dev, a);
}

// One thread, launched behind pass 2 on the same stream: every score this rank stored into its peers' buffers has been
// performed when this kernel starts; the fence + system-scope release stores make them visible before the epoch is.
__global__ void exchange_flag_kernel(float* const* peers, int rank, int world, unsigned int epoch) {
  __threadfence_system();
  for (int p = 0; p < world; ++p) {
    unsigned int* flag = reinterpret_cast<unsigned int*>(peers[p]) + rank;
    asm volatile("st.release.sys.global.u32 [%0], %1;" ::"l"(flag), "r"(epoch) : "memory");
  }
}

// The reader's half of the protocol.  ack: one thread behind a3 on the same stream — every slot read of this rank's
// selection at `epoch` has been performed; tell every peer.  wait: one thread per peer in front of a2 — this rank is about
// to overwrite the slot set it last wrote two epochs ago, so every peer must have finished the selections that read it.
__global__ void exchange_ack_kernel(float* const* peers, int rank, int world, unsigned int epoch) {
  __threadfence_system();
  for (int p = 0; p < world; ++p) {
    unsigned int* ack = reinterpret_cast<unsigned int*>(peers[p]) + kExchAckOffset + rank;
    asm volatile("st.release.sys.global.u32 [%0], %1;" ::"l"(ack), "r"(epoch) : "memory");
  }
}

__global__ void exchange_wait_kernel(const float* own, int world, unsigned int need) {
  if (static_cast<int>(threadIdx.x) >= world) return;
  const unsigned int* ack = reinterpret_cast<const unsigned int*>(own) + kExchAckOffset + threadIdx.x;
  const long long t0 = clock64();
  unsigned int v;
  do {
    asm volatile("ld.acquire.sys.global.u32 %0, [%1];" : "=r"(v) : "l"(ack) : "memory");
    if (static_cast<int>(v - need) >= 0) break;
    if (clock64() - t0 > 4000000000LL) __trap();                  // a peer that never selects is a trap, not a hang
  } while (true);
}

}  // namespace

cudaError_t launch_exchange_flags(const qcf_ctx* ctx, cudaStream_t stream) {
  exchange_flag_kernel<<<1, 1, 0, stream>>>(ctx->exch_peers, ctx->exch_rank, ctx->exch_world, ctx->exch_epoch);
  return cudaGetLastError();
}

cudaError_t launch_exchange_ack(const qcf_ctx* ctx, cudaStream_t stream) {
  exchange_ack_kernel<<<1, 1, 0, stream>>>(ctx->exch_peers, ctx->exch_rank, ctx->exch_world, ctx->exch_epoch);
  return cudaGetLastError();
}

cudaError_t launch_exchange_wait(const qcf_ctx* ctx, unsigned int need, cudaStream_t stream) {
  exchange_wait_kernel<<<1, 64, 0, stream>>>(ctx->exch_peers_host[ctx->exch_rank], ctx->exch_world, need);
  return cudaGetLastError();
}

cudaError_t launch_score(const qcf_ctx* ctx, const qcf_batch* b, const __nv_bfloat16* q_probe,
                         const __nv_bfloat16* k_f, float* scores, int accumulate, cudaStream_t stream) {
  if (b->batch == 0 || b->max_ctx == 0) return cudaSuccess;
  const Layout& L = ctx->lay;
  const int max_rows = b->max_query * L.g;
  const int row_tiles = (max_rows + BT - 1) / BT;
  const int key_tiles = (b->max_ctx + BT - 1) / BT;
  if (row_tiles * BT * 4 > 32768) return cudaErrorInvalidValue;       // Lq * G <= 8192 query rows per kv-head (checked at qcf_create)
  const int slots = 2 * ctx->n_sm;                                     // resident CTAs (2 per SM)
  // pass 1: key splits.  Few CTAs: split until one resident wave is full.  More than a wave: the split count (<= 8) with
  // the best wave efficiency (512 CTAs on 296 slots is 2 waves at 86 %; 4 splits make it 7 waves at 99 %).
  int n_splits = 1;
  if (row_tiles > 0) {
    const int ctas = row_tiles * L.hkv * b->batch;
    if (ctas <= slots) {
      n_splits = slots / ctas;
    } else {
      double best = 0.0;
      for (int sp = 1; sp <= 8; ++sp) {
        const double w = static_cast<double>(ctas) * sp / slots;
        const double eff = w / std::ceil(w);
        if (eff > best + 0.02) { best = eff; n_splits = sp; }
      }
    }
    if (n_splits > key_tiles) n_splits = key_tiles;
    if (2 * n_splits > kScoreSplitsMax) n_splits = kScoreSplitsMax / 2;
    if (n_splits > 8) n_splits = 8;            // x 2 column halves = 16 partials per row: pass 2 combines them in one batch of loads
    if (n_splits < 1) n_splits = 1;
  }
  // pass 2: key tiles per CTA (kt).  Equal-sized CTAs run in rounds of `slots`; a launch wastes the empty part of its last
  // round and a fixed prologue per CTA (barriers, TMEM, combining the pass-1 partials into lse: ~0.3 of a tile walk).  Pick
  // the kt <= 32 with the best (fill of the last round) x kt / (kt + 0.3).  (Measurements behind it: DESIGN.md §9.4.)
  int kt_per_cta = 1;
  {
    const int pairs = L.hkv * b->batch;
    double best = -1.0;
    for (int kt = 1; kt <= 32 && kt <= key_tiles; ++kt) {
      const int groups = (key_tiles + kt - 1) / kt;
      const double rounds = static_cast<double>(groups) * pairs / slots;
      const double score = rounds / std::ceil(rounds) * kt / (kt + 0.3);
      if (score > best + 1e-9) { best = score; kt_per_cta = kt; }
    }
  }
  CUtensorMap tm_q, tm_k;
  // q_probe may be NULL when no request has query tokens: map a valid dummy address (never dereferenced: n_j == 0)
  const void* qbase = q_probe ? static_cast<const void*>(q_probe) : static_cast<const void*>(k_f);
  if (!make_map(&tm_q, qbase, b->batch, b->q_stride > 0 ? b->q_stride : 1, L.hq, L.d, L.g, BT / L.g) ||
      !make_map(&tm_k, k_f, b->batch, b->t_stride, L.hkv, L.d, 1, BT))
    return cudaErrorInvalidValue;
  ScoreArgs a;
  a.scale_log2 = L.scale * kLog2e;
  a.hq = L.hq; a.hkv = L.hkv; a.norm_heads = L.hq * ctx->head_shards; a.n_splits = n_splits; a.kt_per_cta = kt_per_cta;
  a.stats_m = ctx->stats_m; a.stats_l = ctx->stats_l; a.stats_rows = L.hq * ctx->max_query;
  a.part = ctx->score_part; a.part_stride = ctx->max_ctx;
  a.counters = ctx->counters;
  a.scores = scores; a.accumulate = accumulate;
  a.exch_peers = ctx->exch_peers; a.exch_rank = ctx->exch_rank; a.exch_world = ctx->exch_world; a.exch_slot_elems = ctx->exch_slot_elems;
  a.exch_parity = static_cast<int>(ctx->exch_epoch & 1u);
  return L.d == 128 ? launch<128>(ctx, b, tm_q, tm_k, a, row_tiles, key_tiles, stream)
                    : launch<64>(ctx, b, tm_q, tm_k, a, row_tiles, key_tiles, stream);
}

}  // namespace qcf
