// a2 on the 5th-generation tensor cores — Eq. 18 / 20:
//
//   I(t) = 1/(Hq Lq) sum_{i,h} exp(s_{i,h,t} - lse_{i,h}),   s = q_probe[i][h] . K'[t][h/G] * scale
//
// The row normaliser lse spans ALL context keys, so two sweeps are needed, and each wants its reduction to be local to a
// thread (= one TMEM lane):
//   pass 1 (stats)  : S   = Q_tile K_j^T   query rows on the lanes, key tiles streamed -> per-row (max, sum-exp)
//   pass 2 (colsum) : S^T = K_tile Q_j^T   KEYS on the lanes, query-row chunks streamed -> per-key sum_r 2^(s - lse_r)
// Both are the same warp-specialised skeleton: a fixed 128-row operand A and a 2-stage TMA ring of 128-row operands B
// (128-byte swizzle), S double-buffered in TMEM (2 x 128 fp32 columns), one UMMA-issuing thread, and 128 consumer
// threads that sweep their own TMEM lane.  GQA packing: a "query row" is (token i, head hl) of one kv-head,
// r = i * G + hl, loaded by TMA boxes {64 elements, G heads, 128/G tokens}.  The Hkv per-head partial column sums are
// combined in fixed order by the last CTA of each key tile (bit-reproducible scores, deterministic top-k).
#include <cmath>

#include "qcf_internal.cuh"
#include "sm100_ptx.cuh"

namespace qcf {

namespace {

using namespace ptx;

constexpr int BT = 128;            // rows of A, rows of one B tile, fp32 columns of one S buffer
constexpr int kThreads = 192;
constexpr int kTmemCols = 256;
constexpr float kLog2e = 1.4426950408889634f;
constexpr float kStaleSum = 1099511627776.0f;      // 2^40
#ifndef QCF_SCORE_MUFU_PAIRS
#define QCF_SCORE_MUFU_PAIRS 3
#endif
// Of every 4 pairs, how many take MUFU.EX2 (the rest: the packed polynomial on the FMA pipe).  Unlike attention (no P V, no
// P packing) these sweeps are MUFU-bound — 128 x 128 exponentials against a 256-cycle MMA per tile — so a quarter of them
// moves to the FMA pipe: a2 on c4 600 -> 530 us, c5 295 -> 262 us, c2 30.8 -> 29.1 us (a half: 570 / 273 / 29.6).
constexpr int kMufuPairs = QCF_SCORE_MUFU_PAIRS;

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
  static constexpr int oLse = oFlag + 8;                // pass 2: -lse of ALL query rows of the (request, kv-head), size set at launch
  static constexpr int kBytes = oLse;
};
enum { kAFull = 0, kBFull = 1, kBEmpty = 3, kSFull = 5, kSEmpty = 7, kAEmpty = 9 };

struct ScoreArgs {
  float scale_log2;
  int hq, hkv, n_splits;
  int norm_heads;                                        // Hq of the WHOLE layer (Hq * head shards): Eq. 18's 1/(Hq Lq)
  int kt_per_cta;                                        // pass 2: key tiles walked by one CTA
  float* stats_m; float* stats_l; int stats_rows;        // [B][n_splits][stats_rows]
  float* part; int part_stride;                          // [B][Hkv][part_stride]
  unsigned int* counters;
  float* scores; int accumulate;
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
        mbar_init(bar(kSEmpty + i), 128);
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
    // ===================================================================== consumers: one TMEM lane each
    const int quarter = warp & 3;
    const int r = quarter * 32 + lane;
    const uint32_t lane_addr = tmem_base + (static_cast<uint32_t>(quarter * 32) << 16);
    if (PASS == 1) {
      // lane = query row: online (max, sum-exp) over the streamed keys, reference max moved lazily
      float m_ref = -INFINITY, l = 0.f;
      for (int j = 0; j < n_j; ++j) {
        const int st = j & 1;
        const int key0 = k_begin + j * BT;
        const bool tail = key0 + BT > k_end;
        mbar_wait(bar(kSFull + st), (j >> 1) & 1);
        tc_fence_after();
        // max of this row's scores over the tile's valid keys, log2 units (first tile and the rare rescale only)
        auto tile_rowmax = [&]() -> float {
          float mx0 = -INFINITY, mx1 = -INFINITY;
#pragma unroll
          for (int c = 0; c < BT / 32; ++c) {
            uint32_t s[32];
            tmem_ld32(lane_addr + st * BT + c * 32, s);
            tmem_wait_ld();
#pragma unroll
            for (int i = 0; i < 32; i += 2) {
              float v0 = __uint_as_float(s[i]), v1 = __uint_as_float(s[i + 1]);
              if (tail) {
                const int k = key0 + c * 32 + i;
                if (k >= k_end) v0 = -INFINITY;
                if (k + 1 >= k_end) v1 = -INFINITY;
              }
              mx0 = fmaxf(mx0, v0); mx1 = fmaxf(mx1, v1);
            }
          }
          return fmaxf(mx0, mx1) * a.scale_log2;
        };
        // sum_k 2^(s_k * scale - ref) over the tile.  Issue-bound, so full tiles run on packed pairs (FFMA2 / FADD2) with
        // every exponential on the MUFU; no per-element max: a stale reference shows up as a huge (or inf) sum.
        auto sweep_sum = [&](float ref) -> float {
          float total;
          if (!tail) {
            const uint64_t sc2 = f2_pack(a.scale_log2, a.scale_log2), nr2 = f2_pack(-ref, -ref);
            uint64_t la = 0ull, lb = 0ull;
#pragma unroll
            uint32_t sa[32], sb[32];                   // chunk c + 1 is in flight while chunk c is processed
            tmem_ld32(lane_addr + st * BT, sa);
#pragma unroll
            for (int c = 0; c < BT / 32; ++c) {
              uint32_t(&s)[32] = (c & 1) ? sb : sa;
              tmem_wait_ld();
              if (c + 1 < BT / 32) tmem_ld32(lane_addr + st * BT + (c + 1) * 32, (c & 1) ? sa : sb);
#pragma unroll
              for (int i = 0; i < 32; i += 8) {
                float p[8];
#pragma unroll
                for (int q = 0; q < 4; ++q) {
                  const uint64_t t = f2_fma(f2_pack(__uint_as_float(s[i + 2 * q]), __uint_as_float(s[i + 2 * q + 1])), sc2, nr2);
                  if (q < kMufuPairs) {
                    float t0, t1;
                    f2_unpack(t, t0, t1);
                    p[2 * q] = ex2(t0); p[2 * q + 1] = ex2(t1);
                  } else {
                    ex2_poly2(t, p[2 * q], p[2 * q + 1]);
                  }
                }
                la = f2_add(la, f2_add(f2_pack(p[0], p[1]), f2_pack(p[2], p[3])));
                lb = f2_add(lb, f2_add(f2_pack(p[4], p[5]), f2_pack(p[6], p[7])));
              }
            }
            float s0, s1;
            f2_unpack(f2_add(la, lb), s0, s1);
            total = s0 + s1;
          } else {
            float l0 = 0.f, l1 = 0.f;
#pragma unroll
            for (int c = 0; c < BT / 32; ++c) {
              uint32_t s[32];
              tmem_ld32(lane_addr + st * BT + c * 32, s);
              tmem_wait_ld();
#pragma unroll
              for (int i = 0; i < 32; i += 2) {
                const int k = key0 + c * 32 + i;
                const float v0 = k < k_end ? __uint_as_float(s[i]) : -INFINITY;
                const float v1 = k + 1 < k_end ? __uint_as_float(s[i + 1]) : -INFINITY;
                l0 += ex2(fmaf(v0, a.scale_log2, -ref));
                l1 += ex2(fmaf(v1, a.scale_log2, -ref));
              }
            }
            total = l0 + l1;
          }
          return total;
        };
        float tile_sum;
        if (j == 0) {
          m_ref = tile_rowmax();                  // the first tile of a non-empty range has >= 1 valid key: finite
          tile_sum = sweep_sum(m_ref);
        } else {
          tile_sum = sweep_sum(m_ref);
          // fp32 sums do not care how stale the reference is until they overflow: move it when a tile's sum passes 2^40
          if (__any_sync(0xffffffffu, !(tile_sum <= kStaleSum))) {
            const float m_t = fmaxf(m_ref, tile_rowmax());
            l *= ex2(m_ref - m_t);
            m_ref = m_t;
            tile_sum = sweep_sum(m_ref);
          }
        }
        l += tile_sum;
        tc_fence_before();
        mbar_arrive(bar(kSEmpty + st));
      }
      const int row = row_tile * BT + r;
      if (row < rows) {
        const size_t o = (static_cast<size_t>(b) * a.n_splits + split) * a.stats_rows + static_cast<size_t>(g) * rows + row;
        a.stats_m[o] = m_ref;                      // empty key range: (-inf, 0), neutral in the combine
        a.stats_l[o] = l;
      }
    } else {
      // lane = key: sum over the streamed query rows of 2^(s * scale - lse_row).  The CTA walks n_kt key tiles of one
      // (request, kv-head); -lse of every query row is combined from the pass-1 partials ONCE (log2 domain) and kept
      // in shared memory.
      for (int row = r; row < n_j * BT; row += BT) {
        float lse = INFINITY;                                // rows past the end contribute 2^(-inf) = 0
        if (row < rows) {
          // partials are laid out [split][row]: for a fixed split the 128 threads read consecutive words
          const size_t o = static_cast<size_t>(b) * a.n_splits * a.stats_rows + static_cast<size_t>(g) * rows + row;
          float M = -INFINITY, L = 0.f;
          // sixteen splits at a time (the launcher asks for at most sixteen): all loads of a row are issued before the first
          // is used — one L2 round trip per row instead of one per few splits (this loop was 40 % of the kernel's samples at
          // c2); the combine order is unchanged, a missing split is the neutral (-inf, 0)
          for (int s0 = 0; s0 < a.n_splits; s0 += 16) {
            float ms[16], ls[16];
#pragma unroll
            for (int u = 0; u < 16; ++u) {
              const bool ok = s0 + u < a.n_splits;
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
      asm volatile("bar.sync 1, 128;" ::: "memory");
      volatile int* s_last = reinterpret_cast<volatile int*>(smem + S::oFlag);
      const int n_tiles_b = (bd.n_stride + BT - 1) / BT;
      for (int kt = 0, it = 0; kt < n_kt; ++kt) {
      uint64_t acc01 = 0ull, acc23 = 0ull;               // packed fp32 pairs of partial column sums
      for (int j = 0; j < n_j; ++j, ++it) {
        const int st = it & 1;
        mbar_wait(bar(kSFull + st), (it >> 1) & 1);
        tc_fence_after();
        const float4* lse4 = reinterpret_cast<const float4*>(s_lse + j * BT);       // -lse of the chunk's rows
        const int n_valid = rows - j * BT;                   // < BT only in the last chunk
        if (n_valid >= BT) {
          const uint64_t sc2 = f2_pack(a.scale_log2, a.scale_log2);
#pragma unroll
          uint32_t sa[32], sb[32];                     // chunk c + 1 is in flight while chunk c is processed
          tmem_ld32(lane_addr + st * BT, sa);
#pragma unroll
          for (int c = 0; c < BT / 32; ++c) {
            uint32_t(&s)[32] = (c & 1) ? sb : sa;
            tmem_wait_ld();
            if (c + 1 < BT / 32) tmem_ld32(lane_addr + st * BT + (c + 1) * 32, (c & 1) ? sa : sb);
#pragma unroll
            for (int i = 0; i < 32; i += 8) {
              const float4 za = lse4[c * 8 + (i >> 2)], zb = lse4[c * 8 + (i >> 2) + 1];   // same address in every lane: broadcast
              const uint64_t nz[4] = {f2_pack(za.x, za.y), f2_pack(za.z, za.w), f2_pack(zb.x, zb.y), f2_pack(zb.z, zb.w)};
              float p[8];
#pragma unroll
              for (int q = 0; q < 4; ++q) {
                const uint64_t t = f2_fma(f2_pack(__uint_as_float(s[i + 2 * q]), __uint_as_float(s[i + 2 * q + 1])), sc2, nz[q]);
                if (q < kMufuPairs) {
                  float t0, t1;
                  f2_unpack(t, t0, t1);
                  p[2 * q] = ex2(t0); p[2 * q + 1] = ex2(t1);
                } else {
                  ex2_poly2(t, p[2 * q], p[2 * q + 1]);
                }
              }
              acc01 = f2_add(acc01, f2_add(f2_pack(p[0], p[1]), f2_pack(p[2], p[3])));
              acc23 = f2_add(acc23, f2_add(f2_pack(p[4], p[5]), f2_pack(p[6], p[7])));
            }
          }
        } else {
#pragma unroll
          for (int c = 0; c < BT / 32; ++c) {
            uint32_t s[32];
            tmem_ld32(lane_addr + st * BT + c * 32, s);
            tmem_wait_ld();
#pragma unroll
            for (int i = 0; i < 32; i += 4) {
              const float4 z = lse4[c * 8 + (i >> 2)];
              const int col = c * 32 + i;                    // rows past the end hold whatever the buffer holds
              const float p0 = col < n_valid ? ex2(fmaf(__uint_as_float(s[i]), a.scale_log2, z.x)) : 0.f;
              const float p1 = col + 1 < n_valid ? ex2(fmaf(__uint_as_float(s[i + 1]), a.scale_log2, z.y)) : 0.f;
              const float p2 = col + 2 < n_valid ? ex2(fmaf(__uint_as_float(s[i + 2]), a.scale_log2, z.z)) : 0.f;
              const float p3 = col + 3 < n_valid ? ex2(fmaf(__uint_as_float(s[i + 3]), a.scale_log2, z.w)) : 0.f;
              acc01 = f2_add(acc01, f2_pack(p0, p1));
              acc23 = f2_add(acc23, f2_pack(p2, p3));
            }
          }
        }
        tc_fence_before();
        mbar_arrive(bar(kSEmpty + st));
      }
      const int kt_abs = key_tile + kt;
      const int key = kt_abs * BT + r;
      float a0, a1;
      f2_unpack(f2_add(acc01, acc23), a0, a1);
      if (key < N) a.part[(static_cast<size_t>(b) * a.hkv + g) * a.part_stride + key] = a0 + a1;
      // last CTA of this key tile sums the Hkv partials in fixed order (deterministic)
      __threadfence();
      asm volatile("bar.sync 1, 128;" ::: "memory");
      unsigned int* ctr = a.counters + static_cast<size_t>(b) * n_tiles_b + kt_abs;
      if (r == 0) *s_last = (atomicAdd(ctr, 1u) == static_cast<unsigned int>(a.hkv - 1));
      asm volatile("bar.sync 1, 128;" ::: "memory");
      if (*s_last) {
        __threadfence();
        if (key < N) {
          float sum = 0.f;
          for (int gg = 0; gg < a.hkv; ++gg) sum += __ldcg(a.part + (static_cast<size_t>(b) * a.hkv + gg) * a.part_stride + key);
          const float v = rows > 0 ? sum / static_cast<float>(a.norm_heads * Lq) : 0.f;
          float* dst = a.scores + static_cast<size_t>(b) * bd.n_stride + key;
          *dst = a.accumulate ? *dst + v : v;
        }
        if (r == 0) *ctr = 0u;
      }
      asm volatile("bar.sync 1, 128;" ::: "memory");           // s_last is rewritten by the next key tile
      }   // key tiles
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
  const int smem = smem1 + row_tiles * BT * 4;          // pass 2 keeps -lse of every query row of a (request, kv-head)
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

}  // namespace

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
    if (n_splits > kScoreSplitsMax) n_splits = kScoreSplitsMax;
    if (n_splits > 16) n_splits = 16;          // pass 2 combines the partials of a row in one batch of loads
    if (n_splits < 1) n_splits = 1;
  }
  // pass 2: key tiles per CTA.  A CTA per key tile is 4 tile steps under a full prologue at c4 (8192 CTAs): walk several.
  // Small problems: one resident wave; large ones: at most three waves' worth of CTAs.
  int kt_per_cta = 1;
  {
    const int pairs = L.hkv * b->batch;
    const int items = pairs * key_tiles;
    const int budget = items <= 3 * slots ? slots : 3 * slots;
    int per_pair = budget / pairs;
    if (per_pair < 1) per_pair = 1;
    kt_per_cta = (key_tiles + per_pair - 1) / per_pair;
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
  return L.d == 128 ? launch<128>(ctx, b, tm_q, tm_k, a, row_tiles, key_tiles, stream)
                    : launch<64>(ctx, b, tm_q, tm_k, a, row_tiles, key_tiles, stream);
}

}  // namespace qcf
