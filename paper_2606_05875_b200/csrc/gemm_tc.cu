// a7 — the row-wise dense projections of the recomputed rows ("full prefill computes Q/K/V
// projections and attention outputs for every context token"; cache fusion does so for the rows R = P u U only;
// BASELINE config 3 fixes the shapes):   C[M, N] = A[M, K] . W[N, K]^T   bf16 operands, fp32 accumulation.
//
// Persistent warp-specialised tcgen05 kernel, one CTA per SM:
//   warp 0      TMA producer: A tile (128*MT x 64) and W tile (256 x 64), 128-byte swizzle, kStages-deep mbarrier ring
//   warp 1      UMMA issuer : MT x (128 x 256 x 16) tcgen05.mma per 16-wide K step, fp32 accumulators in TMEM
//   warps 2-9   epilogue    : one TMEM lane (= output row) per thread, 32 columns at a time -> bf16 -> global
// MT = 1: 128 x 256 tiles, the two 256-column TMEM accumulators alternate, so the epilogue of tile i overlaps the
//         main loop of tile i+1 (best wave quantisation: M = 3136 gives 25 row blocks);
// MT = 2: 256 x 256 tiles, both accumulators belong to one tile (half the W re-reads from L2 per flop).
// M <= 128 (the 64-row probe GEMMs of stage 1, which only stream weights): 128 x 64 tiles and an 8-stage ring, so 4x as
//         many SMs pull weights and each UMMA is ~67 cycles instead of 128 (ncu, cold L2, M = 64: QKV 28.3 -> 19.8 us,
//         O 31.7 -> 24.6, gate/up 41.5 -> 52, down 75.8 -> 56; stage 1 of config 3 4.57 -> 3.95 ms).  These launches are
//         bound by the UMMA chain (4 MMAs + commit per 64-wide K block = 270-285 cycles, microbenchmarked) plus ~8 us of
//         fixed prologue / first-load / epilogue time per launch, not by the loads: removing every TMA load after the first
//         ring fill changes nothing, and an L2 prefetch 32 K blocks ahead of the ring made them slower.
// Tiles are walked row-block fastest, so the CTAs of one wave share a handful of W tiles: every weight is read from
// HBM once, A (<= 77 MB) stays in L2.
// Epilogues: store | + residual (in place allowed) | SwiGLU over interleaved (gate, up) output columns.
// (Tile shapes and split-K variants measured and dropped: DESIGN.md §9.4.)
#include "qcf_internal.cuh"
#include "sm100_ptx.cuh"

namespace qcf {

namespace {

using namespace ptx;

constexpr int BK = 64;
constexpr int kThreads = 320;           // producer warp, issuer warp, 8 epilogue warps
constexpr int kTmemCols = 512;

template <int MT, int BN>
struct GemmSmem {
  static constexpr int kStages = BN <= 64 ? 8 : (MT == 1 ? 4 : 3);
  static constexpr int kA = 128 * MT * BK * 2;
  static constexpr int kB = BN * BK * 2;
  static constexpr int kStage = kA + kB;
  static constexpr int oBar = kStages * kStage;
  static constexpr int kNumBar = 2 * kStages + 4;
  static constexpr int oTmem = oBar + kNumBar * 8;
  static constexpr int kBytes = oTmem + 16;
};

struct GemmArgs {
  int M, N, K;
  const __nv_bfloat16* residual;     // EPI 1: [M][N]
  __nv_bfloat16* c;                  // EPI 0/1: [M][N]; EPI 2: [M][N/2]
};

__device__ __forceinline__ float silu_f(float x) { return x / (1.f + __expf(-x)); }

template <int MT, int EPI, int BN>
__global__ void __launch_bounds__(kThreads, 1)
gemm_tc_kernel(const __grid_constant__ CUtensorMap tm_a, const __grid_constant__ CUtensorMap tm_w, GemmArgs g) {
  extern __shared__ unsigned char smem_raw[];
  unsigned char* smem = smem_raw + ((1024u - (smem_u32(smem_raw) & 1023u)) & 1023u);
  using S = GemmSmem<MT, BN>;
  constexpr int BM = 128 * MT;
  constexpr int kAccBufs = MT == 1 ? 2 : 1;
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int n_mblk = (g.M + BM - 1) / BM, n_nblk = (g.N + BN - 1) / BN;
  const int n_tiles = n_mblk * n_nblk;
  const int n_kb = (g.K + BK - 1) / BK;

  const uint32_t sbase = smem_u32(smem);
  auto bar = [&](int i) -> uint32_t { return sbase + S::oBar + 8 * i; };
  enum { kFull = 0, kEmpty = S::kStages, kAccFull = 2 * S::kStages, kAccEmpty = 2 * S::kStages + 2 };
  volatile uint32_t* tmem_slot = reinterpret_cast<volatile uint32_t*>(smem + S::oTmem);

  if (warp == 0) {
    if (lane == 0) {
      prefetch_tensormap(&tm_a);
      prefetch_tensormap(&tm_w);
      for (int i = 0; i < 2 * S::kStages + 2; ++i) mbar_init(bar(i), 1);
      mbar_init(bar(kAccEmpty), 8);
      mbar_init(bar(kAccEmpty + 1), 8);
      fence_barrier_init();
    }
  } else if (warp == 1) {
    tmem_alloc<kTmemCols>(sbase + S::oTmem);
  }
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  const uint32_t tmem_base = *tmem_slot;

  if (warp == 0) {
    // ===================================================================== TMA producer
    // Converged warp, one ELECTED lane issues (elect.sync): inside a divergent `if (lane == 0)` every TMA / UMMA instruction
    // (they take uniform registers) is wrapped in a per-lane ELECT / BRA.U.ANY loop with vector-to-uniform moves.
    {
      int it = 0;
      for (int t = blockIdx.x; t < n_tiles; t += gridDim.x) {
        const int m0 = (t % n_mblk) * BM, n0 = (t / n_mblk) * BN;
        // skinny tiles: every CTA reads the SAME A rows; start each tile at its own K block so that at any moment the
        // CTAs pull different lines of A instead of queueing on one L2 slice (the K order of the fp32 sum is per tile, fixed)
        const int rot = BN <= 64 ? (t * 5) % n_kb : 0;
        for (int kb = 0; kb < n_kb; ++kb, ++it) {
          const int st = it % S::kStages;
          const int kk = (kb + rot >= n_kb ? kb + rot - n_kb : kb + rot) * BK;
          mbar_wait(bar(kEmpty + st), ((it / S::kStages) & 1) ^ 1);
          if (elect_one()) {
            mbar_arrive_expect_tx(bar(kFull + st), S::kStage);
            const uint32_t sa = sbase + st * S::kStage;
#pragma unroll
            for (int mt = 0; mt < MT; ++mt) tma_load_2d(sa + mt * (128 * BK * 2), &tm_a, bar(kFull + st), kk, m0 + mt * 128);
            tma_load_2d(sa + S::kA, &tm_w, bar(kFull + st), kk, n0);
          }
          __syncwarp();
        }
      }
    }
  } else if (warp == 1) {
    // ===================================================================== UMMA issuer (converged warp, elected lane)
    {
      constexpr uint32_t idesc = umma_idesc_bf16(128, BN, false, false);
      // base descriptor once; a stage's operands are base + (byte offset >> 4) (16-byte units, no carry out of the field)
      const uint64_t d0 = umma_smem_desc_sw128(sbase, 16, 1024);
      int it = 0, tile_i = 0;
      for (int t = blockIdx.x; t < n_tiles; t += gridDim.x, ++tile_i) {
        const int buf = tile_i % kAccBufs;
        mbar_wait(bar(kAccEmpty + buf), ((tile_i / kAccBufs) & 1) ^ 1);      // epilogue has drained this accumulator
        tc_fence_after();
        for (int kb = 0; kb < n_kb; ++kb, ++it) {
          const int st = it % S::kStages;
          mbar_wait(bar(kFull + st), (it / S::kStages) & 1);
          tc_fence_after();
          if (elect_one()) {
            const uint64_t da = d0 + static_cast<uint64_t>((st * S::kStage) >> 4), db = da + static_cast<uint64_t>(S::kA >> 4);
#pragma unroll
            for (int mt = 0; mt < MT; ++mt) {
              const uint32_t d_tmem = tmem_base + (buf * MT + mt) * BN;
#pragma unroll
              for (int ks = 0; ks < BK / 16; ++ks)
                umma_ss(d_tmem, da + static_cast<uint64_t>((mt * (128 * BK * 2) + ks * 32) >> 4), db + static_cast<uint64_t>((ks * 32) >> 4),
                        idesc, (kb > 0 || ks > 0) ? 1u : 0u);
            }
            umma_commit(bar(kEmpty + st));
            if (kb == n_kb - 1) umma_commit(bar(kAccFull + buf));
          }
          __syncwarp();
        }
      }
    }
  } else {
    // ===================================================================== epilogue: thread = one output row
    const int ew = warp - 2;                        // 0..7
    const int quarter = warp & 3;                   // TMEM lane quarter this warp may read
    const int half = ew >> 2;                       // MT = 1: column half; MT = 2: accumulator (row half)
    int tile_i = 0;
    for (int t = blockIdx.x; t < n_tiles; t += gridDim.x, ++tile_i) {
      const int m0 = (t % n_mblk) * BM, n0 = (t / n_mblk) * BN;
      const int buf = tile_i % kAccBufs;
      mbar_wait(bar(kAccFull + buf), (tile_i / kAccBufs) & 1);
      tc_fence_after();
      const int row = m0 + (MT == 2 ? half * 128 : 0) + quarter * 32 + lane;
      // MT = 1: the two warps of a lane quarter split the columns (BN = 32: the second one has none and only hands back)
      constexpr int kCols = MT == 1 ? (BN >= 64 ? BN / 2 : BN) : BN;
      const int col_begin = MT == 1 ? half * kCols : 0;
      if (MT == 1 && BN < 64 && half == 1) {
        tc_fence_before();
        __syncwarp();
        if (lane == 0) mbar_arrive(bar(kAccEmpty + buf));
        continue;
      }
      const uint32_t taddr = tmem_base + (static_cast<uint32_t>(quarter * 32) << 16) +
                             (buf * MT + (MT == 2 ? half : 0)) * BN + col_begin;
      const bool row_ok = row < g.M;
#pragma unroll 1
      for (int c = 0; c < kCols; c += 32) {
        uint32_t v[32];
        tmem_ld32(taddr + c, v);
        tmem_wait_ld();
        if (c + 32 == kCols) {                      // accumulator fully read by this warp: hand it back early
          tc_fence_before();
          __syncwarp();
          if (lane == 0) mbar_arrive(bar(kAccEmpty + buf));
        }
        const int col = n0 + col_begin + c;
        if (!row_ok || col >= g.N) continue;
        if (EPI == 2) {
          // interleaved (gate, up) columns -> 16 outputs silu(gate) * up
          __nv_bfloat16* dst = g.c + static_cast<size_t>(row) * (g.N >> 1) + (col >> 1);
#pragma unroll
          for (int q = 0; q < 2; ++q) {
            if (col + 16 * q >= g.N) break;
            uint32_t w[4];
#pragma unroll
            for (int i = 0; i < 4; ++i) {
              const float g0 = __uint_as_float(v[16 * q + 4 * i]), u0 = __uint_as_float(v[16 * q + 4 * i + 1]);
              const float g1 = __uint_as_float(v[16 * q + 4 * i + 2]), u1 = __uint_as_float(v[16 * q + 4 * i + 3]);
              w[i] = pack_bf16(silu_f(g0) * u0, silu_f(g1) * u1);
            }
            *reinterpret_cast<uint4*>(dst + 8 * q) = make_uint4(w[0], w[1], w[2], w[3]);
          }
        } else {
          __nv_bfloat16* dst = g.c + static_cast<size_t>(row) * g.N + col;
          const __nv_bfloat16* res = EPI == 1 ? g.residual + static_cast<size_t>(row) * g.N + col : nullptr;
#pragma unroll
          for (int q = 0; q < 4; ++q) {
            if (col + 8 * q >= g.N) break;
            float f[8];
#pragma unroll
            for (int i = 0; i < 8; ++i) f[i] = __uint_as_float(v[8 * q + i]);
            if (EPI == 1) {
              const uint4 r = *reinterpret_cast<const uint4*>(res + 8 * q);
              f[0] += bf16lo(r.x); f[1] += bf16hi(r.x); f[2] += bf16lo(r.y); f[3] += bf16hi(r.y);
              f[4] += bf16lo(r.z); f[5] += bf16hi(r.z); f[6] += bf16lo(r.w); f[7] += bf16hi(r.w);
            }
            *reinterpret_cast<uint4*>(dst + 8 * q) =
                make_uint4(pack_bf16(f[0], f[1]), pack_bf16(f[2], f[3]), pack_bf16(f[4], f[5]), pack_bf16(f[6], f[7]));
          }
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

// row-major [rows][cols] bf16, box = box_rows x 64 columns, 128-byte swizzle, zero fill out of bounds
bool make_map_2d(CUtensorMap* m, const void* base, int rows, int cols, int box_rows) {
  EncodeFn enc = get_encode();
  if (!enc) return false;
  const cuuint64_t dims[2] = {static_cast<cuuint64_t>(cols), static_cast<cuuint64_t>(rows)};
  const cuuint64_t strides[1] = {static_cast<cuuint64_t>(cols) * 2};
  const cuuint32_t box[2] = {BK, static_cast<cuuint32_t>(box_rows)};
  const cuuint32_t estr[2] = {1, 1};
  return enc(m, CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, 2, const_cast<void*>(base), dims, strides, box, estr,
             CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
             CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) == CUDA_SUCCESS;
}

template <int MT, int EPI, int BN>
cudaError_t launch_one(const qcf_ctx* ctx, const CUtensorMap& tm_a, const CUtensorMap& tm_w, const GemmArgs& g,
                       cudaStream_t stream) {
  constexpr int BM = 128 * MT;
  const int n_tiles = ((g.M + BM - 1) / BM) * ((g.N + BN - 1) / BN);
  const int grid = n_tiles < ctx->n_sm ? n_tiles : ctx->n_sm;
  const int smem = GemmSmem<MT, BN>::kBytes + 1024;
  auto kern = gemm_tc_kernel<MT, EPI, BN>;
  cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, smem);
  kern<<<grid, kThreads, smem, stream>>>(tm_a, tm_w, g);
  return cudaGetLastError();
}

}  // namespace

cudaError_t launch_gemm(const qcf_ctx* ctx, const __nv_bfloat16* a, const __nv_bfloat16* w,
                        const __nv_bfloat16* residual, __nv_bfloat16* c, int M, int N, int K, int epilogue,
                        cudaStream_t stream) {
  if (M <= 0 || N <= 0) return cudaSuccess;
  // one row (decoding): a pure weight stream — the warp-per-row GEMV, not a 128-row MMA tile with 127 zero rows
  if (M == 1 && ctx->gemm_mt == 0 && N % 2 == 0 && K % 8 == 0 && K <= kGemvMaxK)
    return launch_gemv(ctx, a, w, nullptr, 0.f, residual, c, N, K, epilogue, stream);
  // Skinny problems (one row block: the 64-row probe GEMMs of stage 1) stream 34-200 MB of weights and are bound by how
  // many SMs pull them: 128 x 64 tiles give 4x the CTAs of 128 x 256 tiles and an 8-deep ring keeps ~100 KB in flight per SM.
  const bool skinny = M <= 128 && ctx->gemm_mt == 0;
  // 64-wide tiles, or 32-wide when that still leaves a single wave (N = 4096: 64 -> 128 CTAs; O 24.6 -> 20.8 us, down 56 -> 51)
  const int bn = skinny ? ((N + 31) / 32 <= ctx->n_sm ? 32 : 64) : 256;
  // tile height: 256-row tiles halve the W traffic per flop but quantise worse; take them when they cost no extra wave
  int mt = ctx->gemm_mt;
  if (mt == 0) {
    const int n_nblk = (N + bn - 1) / bn;
    const int w1 = (((M + 127) / 128) * n_nblk + ctx->n_sm - 1) / ctx->n_sm;       // waves of 128-row tiles
    const int w2 = (((M + 255) / 256) * n_nblk + ctx->n_sm - 1) / ctx->n_sm;       // waves of 256-row tiles (2x work)
    mt = (!skinny && 2 * w2 <= w1) ? 2 : 1;
  }
  CUtensorMap tm_a, tm_w;
  if (!make_map_2d(&tm_a, a, M, K, 128) || !make_map_2d(&tm_w, w, N, K, bn)) return cudaErrorInvalidValue;
  GemmArgs g{M, N, K, residual, c};
  if (skinny) {
    if (bn == 32) {
      if (epilogue == 0) return launch_one<1, 0, 32>(ctx, tm_a, tm_w, g, stream);
      if (epilogue == 1) return launch_one<1, 1, 32>(ctx, tm_a, tm_w, g, stream);
      return launch_one<1, 2, 32>(ctx, tm_a, tm_w, g, stream);
    }
    if (epilogue == 0) return launch_one<1, 0, 64>(ctx, tm_a, tm_w, g, stream);
    if (epilogue == 1) return launch_one<1, 1, 64>(ctx, tm_a, tm_w, g, stream);
    return launch_one<1, 2, 64>(ctx, tm_a, tm_w, g, stream);
  }
  if (mt == 1) {
    if (epilogue == 0) return launch_one<1, 0, 256>(ctx, tm_a, tm_w, g, stream);
    if (epilogue == 1) return launch_one<1, 1, 256>(ctx, tm_a, tm_w, g, stream);
    return launch_one<1, 2, 256>(ctx, tm_a, tm_w, g, stream);
  }
  if (epilogue == 0) return launch_one<2, 0, 256>(ctx, tm_a, tm_w, g, stream);
  if (epilogue == 1) return launch_one<2, 1, 256>(ctx, tm_a, tm_w, g, stream);
  return launch_one<2, 2, 256>(ctx, tm_a, tm_w, g, stream);
}

}  // namespace qcf
