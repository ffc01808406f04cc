// Decoding over KV^Fuse (the fused cache and the query states are handed to decoding; PAPER.md:372:
// TTFT ends at the first token) — single-row GQA attention of ONE new token over a layer's cache:
//
//   out[h] = sum_{j < n_keys} softmax_j( q[h] . K[j][h/G] * scale ) V[j][h/G]
//
// HBM-bound stream (every K and V row of the layer is read once: 2 * Hkv * d * 2 bytes per key, ~4 flop per byte), so no
// tensor cores: the key range is split over (n_splits x Hkv) CTAs; a CTA stages 128-key tiles of its kv-head's K and V in
// shared memory with 16-byte asynchronous copies (cp.async, 16 consecutive threads per 2*d-byte row: fully coalesced);
// K_{j+1} is in flight while P_j V_j runs and V_{j+1} while Q K_{j+1}^T runs.  (One cp.async.bulk per row was the first
// version: 256 bulk copies of 256 B per tile ran at 1.3 TB/s — the per-copy cost of the bulk engine dominates at that size.)
//   phase 1: thread = key   -> the G logits of its key (q broadcast from shared memory), block max, p = 2^(s - m)
//   phase 2: thread = dim pair x key group -> o[g][dims] += p[g][key] * V[key][dims]
// Split partials (m, l, o) go to a workspace; the LAST CTA of a kv-head (arrival counter) merges them in split order
// (bit-reproducible), normalises and stores bf16.
#include <cmath>
#include <mutex>
#include <string>

#include "qcf_internal.cuh"
#include "sm100_ptx.cuh"

namespace qcf {

namespace {

using namespace ptx;

constexpr int kKeys = 128;             // keys per tile = threads per CTA
constexpr int kThreads = 128;
constexpr float kLog2e = 1.4426950408889634f;
constexpr float kLn2 = 0.6931471805599453f;

template <int D, int G>
struct DecSmem {
  static constexpr int kPitch = D * 2 + 16;                  // padded row: 128-bit reads of consecutive rows spread over banks
  static constexpr int oK = 0;
  static constexpr int oV = oK + kKeys * kPitch;
  static constexpr int oQ = oV + kKeys * kPitch;             // q of the G heads, fp32, pre-scaled by scale * log2(e)
  static constexpr int oP = oQ + G * D * 4;                  // p[key][G]
  static constexpr int oRed = oP + kKeys * G * 4;            // per-warp tile maxima [4][G], then the o reduction
  static constexpr int oBar = oRed + 4 * G * 4;
  static constexpr int kBytes = oBar + 16;
};

// grid (n_splits, Hkv).  part_o [Hkv][n_splits][G][D], part_ml [Hkv][n_splits][G][2]
template <int D, int G>
__global__ void __launch_bounds__(kThreads) decode_attn_kernel(const __nv_bfloat16* q, const __nv_bfloat16* k_cache,
                                                               const __nv_bfloat16* v_cache, int hkv, int n_keys,
                                                               int tiles_per_split, float scale_log2, float* part_o,
                                                               float* part_ml, unsigned int* counters,
                                                               __nv_bfloat16* out, float* lse_out) {
  using S = DecSmem<D, G>;
  extern __shared__ __align__(16) unsigned char smem[];
  constexpr int PAIRS = D / 2;                 // bf16x2 columns of a V row
  constexpr int KG = kThreads / PAIRS;         // key groups of phase 2 (2 at d = 128, 4 at d = 64)
  constexpr int KPG = kKeys / KG;              // keys per group
  const int split = blockIdx.x, n_splits = gridDim.x, g = blockIdx.y;
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const uint32_t sbase = smem_u32(smem);
  float* s_q = reinterpret_cast<float*>(smem + S::oQ);
  float* s_p = reinterpret_cast<float*>(smem + S::oP);
  float* s_red = reinterpret_cast<float*>(smem + S::oRed);

  const int n_tiles_all = (n_keys + kKeys - 1) / kKeys;
  const int t0 = split * tiles_per_split;
  const int n_t = max(0, min(tiles_per_split, n_tiles_all - t0));
  const size_t row_stride = static_cast<size_t>(hkv) * D;          // elements between consecutive keys of one kv-head
  const __nv_bfloat16* kg = k_cache + static_cast<size_t>(g) * D;
  const __nv_bfloat16* vg = v_cache + static_cast<size_t>(g) * D;

  pdl_trigger();
  pdl_wait();                                   // q and the newest cache row are written by the predecessor kernels
  // tile `tile` of K or V -> shared memory: D/8 16-byte chunks per row, chunk index = thread-major so that 16 (d = 128) or 8
  // (d = 64) consecutive threads copy one row; always ONE commit group per call (an empty one past the end keeps the
  // wait_group arithmetic uniform)
  auto issue = [&](const __nv_bfloat16* base, int off, int tile) {
    if (tile < n_t) {
      const int key0 = (t0 + tile) * kKeys;
      const int n_valid = min(kKeys, n_keys - key0);
      constexpr int CPR = D / 8;                               // chunks per row
      for (int idx = tid; idx < n_valid * CPR; idx += kThreads) {
        const int r = idx / CPR, c = idx % CPR;
        cp_async16(sbase + off + r * S::kPitch + c * 16, base + static_cast<size_t>(key0 + r) * row_stride + c * 8);
      }
    }
    cp_async_commit();
  };
  issue(kg, S::oK, 0);                          // the first tiles are in flight while q is fetched and scaled
  issue(vg, S::oV, 0);
  // q of this kv-head's G heads -> fp32, pre-scaled (coherent loads: see the PDL note in qcf_internal.cuh)
  for (int i = tid; i < G * D / 2; i += kThreads) {
    const uint32_t w = *reinterpret_cast<const volatile uint32_t*>(q + (static_cast<size_t>(g) * G) * D + 2 * i);
    s_q[2 * i] = bf16lo(w) * scale_log2;
    s_q[2 * i + 1] = bf16hi(w) * scale_log2;
  }
  // (no barrier here: the first __syncthreads of the tile loop orders s_q before its readers)

  float m_run[G], l_own[G], o[G][2];
#pragma unroll
  for (int h = 0; h < G; ++h) { m_run[h] = -INFINITY; l_own[h] = 0.f; o[h][0] = o[h][1] = 0.f; }
  const int dp = tid % PAIRS, kgrp = tid / PAIRS;

  for (int j = 0; j < n_t; ++j) {
    const int key0 = (t0 + j) * kKeys;
    const int key = key0 + tid;
    const bool valid = key < n_keys;
    // ---- phase 1: logits of my key.  Pending groups here: K(j), V(j) -> K(j) has landed once at most one is pending
    cp_async_wait<1>();
    __syncthreads();                            // every thread's chunks of K(j) are visible
    float s[G];
#pragma unroll
    for (int h = 0; h < G; ++h) s[h] = 0.f;
    if (valid) {
      const uint4* krow = reinterpret_cast<const uint4*>(smem + S::oK + tid * S::kPitch);
#pragma unroll 4
      for (int c = 0; c < D / 8; ++c) {
        const uint4 kv = krow[c];
        const float kf[8] = {bf16lo(kv.x), bf16hi(kv.x), bf16lo(kv.y), bf16hi(kv.y),
                             bf16lo(kv.z), bf16hi(kv.z), bf16lo(kv.w), bf16hi(kv.w)};
#pragma unroll
        for (int h = 0; h < G; ++h) {
          const float4 qa = *reinterpret_cast<const float4*>(s_q + h * D + c * 8);
          const float4 qb = *reinterpret_cast<const float4*>(s_q + h * D + c * 8 + 4);
          float acc = s[h];
          acc = fmaf(kf[0], qa.x, acc); acc = fmaf(kf[1], qa.y, acc); acc = fmaf(kf[2], qa.z, acc); acc = fmaf(kf[3], qa.w, acc);
          acc = fmaf(kf[4], qb.x, acc); acc = fmaf(kf[5], qb.y, acc); acc = fmaf(kf[6], qb.z, acc); acc = fmaf(kf[7], qb.w, acc);
          s[h] = acc;
        }
      }
    } else {
#pragma unroll
      for (int h = 0; h < G; ++h) s[h] = -INFINITY;
    }
    // block max per head
#pragma unroll
    for (int h = 0; h < G; ++h) {
      float mx = s[h];
#pragma unroll
      for (int o2 = 16; o2 > 0; o2 >>= 1) mx = fmaxf(mx, __shfl_xor_sync(0xffffffffu, mx, o2));
      if (lane == 0) s_red[warp * G + h] = mx;
    }
    __syncthreads();                            // (a) maxima visible; every thread has finished reading the K tile
    issue(kg, S::oK, j + 1);                    // pending: V(j), K(j+1)
    float alpha[G];
#pragma unroll
    for (int h = 0; h < G; ++h) {
      const float mt = fmaxf(fmaxf(s_red[h], s_red[G + h]), fmaxf(s_red[2 * G + h], s_red[3 * G + h]));
      const float mn = fmaxf(m_run[h], mt);     // the first key of a split's first tile is always valid: finite
      alpha[h] = ex2(m_run[h] - mn);            // 2^(-inf) = 0 on the first tile
      m_run[h] = mn;
      const float p = ex2(s[h] - mn);           // invalid keys: 2^(-inf) = 0
      l_own[h] = l_own[h] * alpha[h] + p;
      s_p[tid * G + h] = p;
    }
    // ---- phase 2: o += P V over my key group, my dim pair
    cp_async_wait<1>();                         // V(j) has landed (K(j+1) may still be in flight)
    if (!valid) {
      // tail rows were not copied: whatever the buffer holds must not meet p = 0 as NaN/inf
      uint4* vrow = reinterpret_cast<uint4*>(smem + S::oV + tid * S::kPitch);
#pragma unroll
      for (int c = 0; c < D / 8; ++c) vrow[c] = make_uint4(0u, 0u, 0u, 0u);
    }
    __syncthreads();                            // (b) p and the zeroed tail rows visible
#pragma unroll
    for (int h = 0; h < G; ++h) { o[h][0] *= alpha[h]; o[h][1] *= alpha[h]; }
#pragma unroll 4
    for (int kk = 0; kk < KPG; ++kk) {
      const int kr = kgrp * KPG + kk;
      const uint32_t vw = *reinterpret_cast<const uint32_t*>(smem + S::oV + kr * S::kPitch + dp * 4);
      const float v0 = bf16lo(vw), v1 = bf16hi(vw);
#pragma unroll
      for (int h = 0; h < G; ++h) {
        const float p = s_p[kr * G + h];
        o[h][0] = fmaf(p, v0, o[h][0]);
        o[h][1] = fmaf(p, v1, o[h][1]);
      }
    }
    __syncthreads();                            // (c) V tile, p and s_red are free again
    issue(vg, S::oV, j + 1);                    // pending: K(j+1), V(j+1)
  }

  cp_async_wait<0>();                           // (only empty groups can still be pending)
  // ---- split partial: l over the block, o over the key groups
  float* red_o = reinterpret_cast<float*>(smem + S::oK);       // K buffer is drained: [KG][G][D]
#pragma unroll
  for (int h = 0; h < G; ++h) {
    red_o[(kgrp * G + h) * D + 2 * dp] = o[h][0];
    red_o[(kgrp * G + h) * D + 2 * dp + 1] = o[h][1];
    float l = l_own[h];
#pragma unroll
    for (int o2 = 16; o2 > 0; o2 >>= 1) l += __shfl_xor_sync(0xffffffffu, l, o2);
    if (lane == 0) s_red[warp * G + h] = l;
  }
  __syncthreads();
  const size_t slot = static_cast<size_t>(g) * n_splits + split;
  for (int i = tid; i < G * D; i += kThreads) {
    float acc = 0.f;
#pragma unroll
    for (int kq = 0; kq < KG; ++kq) acc += red_o[kq * G * D + i];
    part_o[slot * G * D + i] = acc;
  }
#pragma unroll
  for (int h = 0; h < G; ++h) {
    if (tid == h) {                                                                           // m_run is block-uniform
      part_ml[(slot * G + h) * 2] = m_run[h];
      part_ml[(slot * G + h) * 2 + 1] = (s_red[h] + s_red[G + h]) + (s_red[2 * G + h] + s_red[3 * G + h]);
    }
  }
  // ---- last CTA of this kv-head merges the splits in split order
  __threadfence();
  __syncthreads();
  __shared__ int s_last;
  if (tid == 0) s_last = atomicAdd(counters + g, 1u) == static_cast<unsigned int>(n_splits - 1);
  __syncthreads();
  if (!s_last) return;
  __threadfence();
  // (The first version walked the splits with one dependent global load per step: ~40 L2 round trips in a row were 25 of the
  // kernel's 32 us at c3.  Now the (m, l) pairs are staged in shared memory by all threads at once and the O partials are
  // read eight splits at a time.)
  float* s_ml = reinterpret_cast<float*>(smem + S::oV);          // [n_splits][G][2]
  float* s_w = s_ml + n_splits * G * 2;                          // weights [n_splits][G]
  float* s_inv = s_p;                                            // 1 / l per head
  for (int i = tid; i < n_splits * G * 2; i += kThreads) s_ml[i] = __ldcg(part_ml + static_cast<size_t>(g) * n_splits * G * 2 + i);
  __syncthreads();
  if (tid < G) {
    float M = -INFINITY;
    for (int sp = 0; sp < n_splits; ++sp) M = fmaxf(M, s_ml[(sp * G + tid) * 2]);
    float L = 0.f;
    for (int sp = 0; sp < n_splits; ++sp) {                      // split order: bit-reproducible
      const float w = ex2(s_ml[(sp * G + tid) * 2] - M);         // empty split: m = -inf -> weight 0
      s_w[sp * G + tid] = w;
      L = fmaf(s_ml[(sp * G + tid) * 2 + 1], w, L);
    }
    s_inv[tid] = 1.f / L;
    if (lse_out) lse_out[g * G + tid] = (M + log2f(L)) * kLn2;
  }
  __syncthreads();
  // one float4 column group per thread, sixteen splits in flight: the whole merge is ceil(n_splits / 16) L2 round trips
  for (int i4 = tid; i4 < G * D / 4; i4 += kThreads) {
    const int h = (i4 * 4) / D;
    const float4* src = reinterpret_cast<const float4*>(part_o + static_cast<size_t>(g) * n_splits * G * D) + i4;
    float4 acc = make_float4(0.f, 0.f, 0.f, 0.f);
    for (int sp0 = 0; sp0 < n_splits; sp0 += 16) {
      float4 v[16];
#pragma unroll
      for (int u = 0; u < 16; ++u)
        v[u] = sp0 + u < n_splits ? __ldcg(src + static_cast<size_t>(sp0 + u) * (G * D / 4)) : make_float4(0.f, 0.f, 0.f, 0.f);
#pragma unroll
      for (int u = 0; u < 16; ++u) {
        if (sp0 + u < n_splits) {                                  // split order: bit-reproducible
          const float w = s_w[(sp0 + u) * G + h];
          acc.x = fmaf(v[u].x, w, acc.x); acc.y = fmaf(v[u].y, w, acc.y);
          acc.z = fmaf(v[u].z, w, acc.z); acc.w = fmaf(v[u].w, w, acc.w);
        }
      }
    }
    const float inv = s_inv[h];
    uint2 packed;
    packed.x = pack_bf16(acc.x * inv, acc.y * inv);
    packed.y = pack_bf16(acc.z * inv, acc.w * inv);
    *reinterpret_cast<uint2*>(out + (static_cast<size_t>(g) * G) * D + i4 * 4) = packed;
  }
  if (tid == 0) counters[g] = 0u;                                // self-resetting
}

template <int D, int G>
cudaError_t launch_dg(const qcf_ctx* ctx, const __nv_bfloat16* q, const __nv_bfloat16* k, const __nv_bfloat16* v, int n_keys,
                      __nv_bfloat16* out, float* lse, cudaStream_t stream) {
  const Layout& L = ctx->lay;
  const int n_tiles = (n_keys + kKeys - 1) / kKeys;
  // about three resident CTAs per SM; at most kDecodeSplitsMax splits per kv-head (workspace)
  int want = (3 * ctx->n_sm + L.hkv - 1) / L.hkv;
  if (want > kDecodeSplitsMax) want = kDecodeSplitsMax;
  if (want > n_tiles) want = n_tiles;
  if (want < 1) want = 1;
  const int tps = (n_tiles + want - 1) / want;
  const int n_splits = (n_tiles + tps - 1) / tps;
  auto kern = decode_attn_kernel<D, G>;
  const int smem = DecSmem<D, G>::kBytes;
  cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, smem);
  return launch_pdl(ctx->pdl, kern, dim3(n_splits, L.hkv), dim3(kThreads), smem, stream, q, k, v, L.hkv, n_keys, tps,
                    L.scale * kLog2e, ctx->dec_part_o, ctx->dec_part_ml, ctx->dec_counters, out, lse);
}

template <int D>
cudaError_t launch_d(const qcf_ctx* ctx, const __nv_bfloat16* q, const __nv_bfloat16* k, const __nv_bfloat16* v, int n_keys,
                     __nv_bfloat16* out, float* lse, cudaStream_t stream) {
  switch (ctx->lay.g) {
    case 1: return launch_dg<D, 1>(ctx, q, k, v, n_keys, out, lse, stream);
    case 2: return launch_dg<D, 2>(ctx, q, k, v, n_keys, out, lse, stream);
    case 4: return launch_dg<D, 4>(ctx, q, k, v, n_keys, out, lse, stream);
    case 8: return launch_dg<D, 8>(ctx, q, k, v, n_keys, out, lse, stream);
    case 16: return launch_dg<D, 16>(ctx, q, k, v, n_keys, out, lse, stream);
    default: return cudaErrorInvalidValue;
  }
}

}  // namespace

cudaError_t launch_decode_attn(const qcf_ctx* ctx, const __nv_bfloat16* q, const __nv_bfloat16* k_cache,
                               const __nv_bfloat16* v_cache, int n_keys, __nv_bfloat16* out, float* lse, cudaStream_t stream) {
  if (n_keys <= 0) return cudaErrorInvalidValue;
  return ctx->lay.d == 128 ? launch_d<128>(ctx, q, k_cache, v_cache, n_keys, out, lse, stream)
                           : launch_d<64>(ctx, q, k_cache, v_cache, n_keys, out, lse, stream);
}

}  // namespace qcf

// ------------------------------------------------------------------------------------------------------------------------
// qcf_decode_attn_static (include/qcf.h) — the same decode attention for callers that may not allocate device memory.
//
// qcf_decode_attn needs a qcf_ctx, and qcf_create cudaMallocs the split-KV workspace of the kernel above.  Some users of
// this library are not in a position to do that: a plugin or custom op running inside a serving engine that has handed
// all of HBM to its own pool allocator (a cudaMalloc from inside it fails or fragments the pool), code running under a
// framework's "no allocation here" region (memory-planned or about-to-be-captured sections), and tools that must not
// disturb the allocator state they observe.  For them the workspace below lives in the library image itself: a file-scope
// __device__ array that every GPU which loads libqcf.so carries from module load until the process exits.
//
// Layout of the array (offsets are multiples of 256 B):
//   [0, kStaticPartO)              split partial outputs   [Hkv][kDecodeSplitsMax][G][d] fp32
//   [kStaticPartO, +kStaticPartMl) split (max, sum) pairs  [Hkv][kDecodeSplitsMax][G][2] fp32
//   [.., +kStaticCounters)         per-kv-head arrival counters (must be zero when a launch starts)
// Sized for Hq * d <= kStaticMaxHeadElems and Hkv <= kStaticMaxKvHeads: 2 MiB + 64 KiB + 256 B per GPU.
namespace qcf {
namespace {

constexpr int kStaticMaxHeadElems = 8192;                       // Hq * d, e.g. 64 heads x 128
constexpr int kStaticMaxKvHeads = 64;
constexpr size_t kStaticPartO = static_cast<size_t>(kDecodeSplitsMax) * kStaticMaxHeadElems * sizeof(float);
constexpr size_t kStaticPartMl = static_cast<size_t>(kDecodeSplitsMax) * (kStaticMaxHeadElems / 64) * 2 * sizeof(float);
constexpr size_t kStaticCounters = 256;                         // kStaticMaxKvHeads x 4 B
constexpr size_t kStaticBytes = kStaticPartO + kStaticPartMl + kStaticCounters;
static_assert(kStaticPartO % 256 == 0 && kStaticPartMl % 256 == 0, "sub-buffers keep the array's 256-byte alignment");
static_assert(kStaticMaxKvHeads * sizeof(unsigned int) <= kStaticCounters, "counter block too small");

static __device__ __align__(256) unsigned char g_static_scratch[kStaticBytes];

// In host code `g_static_scratch` is only a handle for the runtime's symbol table, NOT a device address: the per-device
// address comes from cudaGetSymbolAddress with that device current, once, and is remembered here.
constexpr int kStaticMaxDevices = 64;
struct StaticDev {
  bool ready;
  unsigned char* base;      // device address of g_static_scratch on this device
  int n_sm;
};
StaticDev g_static_dev[kStaticMaxDevices];
std::mutex g_static_mu;

}  // namespace
}  // namespace qcf

qcf_status qcf_decode_attn_static(const qcf_layout* lay, const void* q, const void* k_cache, const void* v_cache, int32_t n_keys,
                                  void* out, float* lse, void* stream) {
  using namespace qcf;
  auto bad = [](qcf_status st, const std::string& msg) { return set_error(nullptr, st, "qcf_decode_attn_static: " + msg); };
  if (!lay) return bad(QCF_ERR_INVALID_ARG, "layout is NULL");
  if (lay->n_q_heads < 1 || lay->n_kv_heads < 1 || lay->n_q_heads % lay->n_kv_heads != 0)
    return bad(QCF_ERR_UNSUPPORTED, "n_kv_heads must divide n_q_heads");
  if (lay->head_dim != 64 && lay->head_dim != 128) return bad(QCF_ERR_UNSUPPORTED, "head_dim must be 64 or 128");
  const int g = lay->n_q_heads / lay->n_kv_heads;
  if (!(g == 1 || g == 2 || g == 4 || g == 8 || g == 16)) return bad(QCF_ERR_UNSUPPORTED, "group size Hq/Hkv must be 1, 2, 4, 8 or 16");
  if (static_cast<long long>(lay->n_q_heads) * lay->head_dim > kStaticMaxHeadElems || lay->n_kv_heads > kStaticMaxKvHeads)
    return bad(QCF_ERR_WORKSPACE,
               "layout exceeds the built-in workspace (Hq * head_dim <= " + std::to_string(kStaticMaxHeadElems) + ", Hkv <= " +
                   std::to_string(kStaticMaxKvHeads) + "); use qcf_create + qcf_decode_attn for larger layers");
  if (!(lay->softmax_scale >= 0.0f)) return bad(QCF_ERR_INVALID_ARG, "softmax_scale must be >= 0");
  if (n_keys < 1) return bad(QCF_ERR_INVALID_ARG, "n_keys must be >= 1 (the token's own K/V row is part of the cache)");
  if (!q || !k_cache || !v_cache || !out) return bad(QCF_ERR_INVALID_ARG, "NULL tensor pointer");
  if ((reinterpret_cast<uintptr_t>(q) | reinterpret_cast<uintptr_t>(k_cache) | reinterpret_cast<uintptr_t>(v_cache) |
       reinterpret_cast<uintptr_t>(out)) & 15u)
    return bad(QCF_ERR_INVALID_ARG, "pointers must be 16-byte aligned");

  int dev = 0;
  cudaError_t e = cudaGetDevice(&dev);
  if (e != cudaSuccess) return bad(QCF_ERR_UNSUPPORTED, std::string("no CUDA device: ") + cudaGetErrorString(e));
  if (dev < 0 || dev >= kStaticMaxDevices) return bad(QCF_ERR_UNSUPPORTED, "device ordinal beyond " + std::to_string(kStaticMaxDevices - 1));
  StaticDev sd;
  {
    // First call on this device: resolve the array's address THERE (the device is current) and read the SM count.
    std::lock_guard<std::mutex> lock(g_static_mu);
    StaticDev& slot = g_static_dev[dev];
    if (!slot.ready) {
      int major = 0, n_sm = 0;
      if ((e = cudaDeviceGetAttribute(&major, cudaDevAttrComputeCapabilityMajor, dev)) != cudaSuccess ||
          (e = cudaDeviceGetAttribute(&n_sm, cudaDevAttrMultiProcessorCount, dev)) != cudaSuccess)
        return bad(QCF_ERR_CUDA, std::string("cudaDeviceGetAttribute: ") + cudaGetErrorString(e));
      if (major != 10) return bad(QCF_ERR_UNSUPPORTED, "this library is built for sm_100a only");
      void* p = nullptr;
      e = cudaGetSymbolAddress(&p, g_static_scratch);
      if (e != cudaSuccess || !p)
        return bad(QCF_ERR_CUDA, std::string("cudaGetSymbolAddress(g_static_scratch): ") + cudaGetErrorString(e));
      slot.base = static_cast<unsigned char*>(p);
      slot.n_sm = n_sm;
      slot.ready = true;
    }
    sd = slot;
  }

  // The launcher above reads only these fields of a ctx; this one lives on the host stack and owns nothing.
  qcf_ctx view{};
  view.lay = Layout{lay->n_q_heads, lay->n_kv_heads, lay->head_dim, g, lay->rope_theta,
                    lay->softmax_scale > 0.f ? lay->softmax_scale : 1.0f / std::sqrt(static_cast<float>(lay->head_dim))};
  view.device = dev;
  view.n_sm = sd.n_sm;
  view.pdl = 0;                                                    // plain launch: ordered after the memset below
  view.dec_part_o = reinterpret_cast<float*>(sd.base);
  view.dec_part_ml = reinterpret_cast<float*>(sd.base + kStaticPartO);
  view.dec_counters = reinterpret_cast<unsigned int*>(sd.base + kStaticPartO + kStaticPartMl);

  cudaStream_t s = static_cast<cudaStream_t>(stream);
  // The array keeps whatever the previous call (of any thread, any layout) left.  The partials are fully rewritten before
  // they are read; the arrival counters must start at zero, and a launch that died half-way would have left them dirty.
  e = cudaMemsetAsync(view.dec_counters, 0, kStaticCounters, s);
  if (e != cudaSuccess) return bad(QCF_ERR_CUDA, std::string("cudaMemsetAsync: ") + cudaGetErrorString(e));
  e = launch_decode_attn(&view, static_cast<const __nv_bfloat16*>(q), static_cast<const __nv_bfloat16*>(k_cache),
                         static_cast<const __nv_bfloat16*>(v_cache), n_keys, static_cast<__nv_bfloat16*>(out), lse, s);
  if (e != cudaSuccess) return bad(QCF_ERR_CUDA, std::string("launch: ") + cudaGetErrorString(e));
  return QCF_OK;
}
