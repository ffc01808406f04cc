// a2 — Eq. 18 / 20: user-query -> context attention mass per context position.
//
//   I(t) = 1/(Hq Lq) sum_{i,h} exp(s_{i,h,t} - lse_{i,h}),   s = q_probe[i][h] . K'[t][h/G] * scale
//
// The row normaliser lse_{i,h} spans ALL context keys, so the column sum cannot be formed in one sweep:
//   pass 1 (score_stats):  S = Q K^T with query rows on the MMA M axis; per-row online (max, sum-exp) over a key
//                          range; kScoreSplits partials per row.
//   pass 2 (score_colsum): S^T = K Q^T with KEYS on the M axis (each thread owns two keys), so the sum over query
//                          rows of exp2(s - lse_row) is a thread-local accumulation; one quad shuffle at the end.
//   The Hkv per-head partial column sums are combined in fixed order by the last CTA of each key tile, so the
//   score is bit-reproducible (no floating-point atomics), which keeps the top-k selection deterministic.
#include "qcf_internal.cuh"

namespace qcf {

namespace {

constexpr int kTile = 64;          // keys per tile (pass 1) / rows per chunk (pass 2); 4 warps x 16
constexpr float kLog2e = 1.4426950408889634f;

// A fragments (m16 x k=D) of two rows read straight from global memory (row pointers may be null -> zeros).
template <int D>
__device__ __forceinline__ void load_a_frags(uint32_t (&a)[D / 16][4], const __nv_bfloat16* r_lo,
                                             const __nv_bfloat16* r_hi, int tig) {
#pragma unroll
  for (int ks = 0; ks < D / 16; ++ks) {
    const int c = ks * 16 + 2 * tig;
    a[ks][0] = r_lo ? __ldg(reinterpret_cast<const uint32_t*>(r_lo + c)) : 0u;
    a[ks][1] = r_hi ? __ldg(reinterpret_cast<const uint32_t*>(r_hi + c)) : 0u;
    a[ks][2] = r_lo ? __ldg(reinterpret_cast<const uint32_t*>(r_lo + c + 8)) : 0u;
    a[ks][3] = r_hi ? __ldg(reinterpret_cast<const uint32_t*>(r_hi + c + 8)) : 0u;
  }
}

// C[16 x 64] = A(16 x D) * B^T where B is a swizzled smem tile [64 rows][D].
template <int D>
__device__ __forceinline__ void mma_tile(float (&c)[kTile / 8][4], const uint32_t (&a)[D / 16][4], uint32_t tile_base,
                                         int lane) {
#pragma unroll
  for (int nt = 0; nt < kTile / 8; ++nt) c[nt][0] = c[nt][1] = c[nt][2] = c[nt][3] = 0.f;
  const int lrow = ((lane >> 4) << 3) + (lane & 7);
  const int lchunk = (lane >> 3) & 1;
#pragma unroll
  for (int ks = 0; ks < D / 16; ++ks) {
#pragma unroll
    for (int np = 0; np < kTile / 16; ++np) {
      uint32_t bfr[4];
      ldmatrix_x4(bfr, tile_base + swz<D>(np * 16 + lrow, 2 * ks + lchunk));
      mma_bf16(c[2 * np], a[ks], bfr[0], bfr[1]);
      mma_bf16(c[2 * np + 1], a[ks], bfr[2], bfr[3]);
    }
  }
}

// ---------------------------------------------------------------------------------------------- pass 1
template <int D>
__global__ void __launch_bounds__(128) score_stats_kernel(BatchDev bd, int hq, int hkv, float scale_log2,
                                                          const __nv_bfloat16* __restrict__ q_probe,
                                                          const __nv_bfloat16* __restrict__ k_f,
                                                          float* __restrict__ stats_m, float* __restrict__ stats_l,
                                                          int stats_rows) {
  __shared__ __align__(128) unsigned char smem[2 * kTile * D * 2];
  const int G = hq / hkv;
  const int b = blockIdx.z / hkv, g = blockIdx.z % hkv;
  const int split = blockIdx.x;
  const int N = bd.n_ctx[b], Lq = bd.n_query[b];
  const int rows = Lq * G;
  const int row0 = blockIdx.y * kTile;
  if (row0 >= rows) return;
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31, gid = lane >> 2, tig = lane & 3;

  const int span = (((N + kScoreSplits - 1) / kScoreSplits + kTile - 1) / kTile) * kTile;
  const int k_begin = split * span;
  const int k_end = min(N, k_begin + span);

  const int r_lo = row0 + warp * 16 + gid, r_hi = r_lo + 8;
  float* m_out = stats_m + (static_cast<size_t>(b) * stats_rows + static_cast<size_t>(g) * rows) * kScoreSplits;
  float* l_out = stats_l + (static_cast<size_t>(b) * stats_rows + static_cast<size_t>(g) * rows) * kScoreSplits;
  if (k_begin >= k_end) {      // empty key range (short contexts): neutral partial
    if (tig == 0) {
      if (r_lo < rows) { m_out[r_lo * kScoreSplits + split] = -INFINITY; l_out[r_lo * kScoreSplits + split] = 0.f; }
      if (r_hi < rows) { m_out[r_hi * kScoreSplits + split] = -INFINITY; l_out[r_hi * kScoreSplits + split] = 0.f; }
    }
    return;
  }

  auto q_row = [&](int r) -> const __nv_bfloat16* {
    if (r >= rows) return nullptr;
    return q_probe + ((static_cast<size_t>(b) * bd.q_stride + r / G) * hq + g * G + r % G) * D;
  };
  uint32_t a[D / 16][4];
  load_a_frags<D>(a, q_row(r_lo), q_row(r_hi), tig);

  const __nv_bfloat16* kbase = k_f + (static_cast<size_t>(b) * bd.t_stride * hkv + g) * D;
  const size_t krow = static_cast<size_t>(hkv) * D;
  const uint32_t sbase = smem_u32(smem);
  auto load_tile = [&](int kt, int buf) {
    constexpr int kChunks = D / 8;
    for (int i = threadIdx.x; i < kTile * kChunks; i += 128) {
      const int r = i / kChunks, c = i % kChunks;
      const int key = min(kt + r, N - 1);
      cp_async16(sbase + buf * (kTile * D * 2) + swz<D>(r, c), kbase + key * krow + c * 8);
    }
    cp_async_commit();
  };

  float m0 = -INFINITY, m1 = -INFINITY, l0 = 0.f, l1 = 0.f;
  const int n_tiles = (k_end - k_begin + kTile - 1) / kTile;
  load_tile(k_begin, 0);
  for (int t = 0; t < n_tiles; ++t) {
    const int kt = k_begin + t * kTile;
    if (t + 1 < n_tiles) { load_tile(kt + kTile, (t + 1) & 1); cp_async_wait<1>(); } else { cp_async_wait<0>(); }
    __syncthreads();
    float c[kTile / 8][4];
    mma_tile<D>(c, a, sbase + (t & 1) * (kTile * D * 2), lane);
    float mx0 = -INFINITY, mx1 = -INFINITY;
#pragma unroll
    for (int nt = 0; nt < kTile / 8; ++nt) {
#pragma unroll
      for (int e = 0; e < 4; ++e) {
        const int key = kt + nt * 8 + 2 * tig + (e & 1);
        const float v = key < k_end ? c[nt][e] * scale_log2 : -INFINITY;
        c[nt][e] = v;
        if (e < 2) mx0 = fmaxf(mx0, v); else mx1 = fmaxf(mx1, v);
      }
    }
    // thread-local online update (the quad is merged once, at the end)
    const float mn0 = fmaxf(m0, mx0), mn1 = fmaxf(m1, mx1);
    float s0 = 0.f, s1 = 0.f;
    if (mn0 > -INFINITY) {
#pragma unroll
      for (int nt = 0; nt < kTile / 8; ++nt) s0 += exp2f(c[nt][0] - mn0) + exp2f(c[nt][1] - mn0);
      l0 = l0 * exp2f(m0 - mn0) + s0;
      m0 = mn0;
    }
    if (mn1 > -INFINITY) {
#pragma unroll
      for (int nt = 0; nt < kTile / 8; ++nt) s1 += exp2f(c[nt][2] - mn1) + exp2f(c[nt][3] - mn1);
      l1 = l1 * exp2f(m1 - mn1) + s1;
      m1 = mn1;
    }
    __syncthreads();
  }
  // merge the 4 lanes of the quad: (m, l) pairs
#pragma unroll
  for (int o = 1; o <= 2; o <<= 1) {
    const float om0 = __shfl_xor_sync(0xffffffffu, m0, o), ol0 = __shfl_xor_sync(0xffffffffu, l0, o);
    const float om1 = __shfl_xor_sync(0xffffffffu, m1, o), ol1 = __shfl_xor_sync(0xffffffffu, l1, o);
    const float n0 = fmaxf(m0, om0), n1 = fmaxf(m1, om1);
    l0 = (n0 > -INFINITY) ? l0 * exp2f(m0 - n0) + ol0 * exp2f(om0 - n0) : 0.f;
    l1 = (n1 > -INFINITY) ? l1 * exp2f(m1 - n1) + ol1 * exp2f(om1 - n1) : 0.f;
    m0 = n0; m1 = n1;
  }
  if (tig == 0) {
    if (r_lo < rows) { m_out[r_lo * kScoreSplits + split] = m0; l_out[r_lo * kScoreSplits + split] = l0; }
    if (r_hi < rows) { m_out[r_hi * kScoreSplits + split] = m1; l_out[r_hi * kScoreSplits + split] = l1; }
  }
}

// ---------------------------------------------------------------------------------------------- pass 2
template <int D>
__global__ void __launch_bounds__(128) score_colsum_kernel(BatchDev bd, int hq, int hkv, float scale_log2,
                                                           const __nv_bfloat16* __restrict__ q_probe,
                                                           const __nv_bfloat16* __restrict__ k_f,
                                                           const float* __restrict__ stats_m,
                                                           const float* __restrict__ stats_l, int stats_rows,
                                                           float* __restrict__ part, int part_stride, int norm_heads,
                                                           unsigned int* __restrict__ counters,
                                                           float* __restrict__ scores, int accumulate) {
  extern __shared__ __align__(128) unsigned char dsmem[];
  __shared__ int s_last;
  const int G = hq / hkv;
  const int b = blockIdx.z, g = blockIdx.y;
  const int N = bd.n_ctx[b], Lq = bd.n_query[b];
  const int key0 = blockIdx.x * kTile;
  if (key0 >= N) return;
  const int rows = Lq * G;
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31, gid = lane >> 2, tig = lane & 3;
  unsigned char* qbuf = dsmem;                                     // 2 x [64][D] bf16
  float* lse2 = reinterpret_cast<float*>(dsmem + 2 * kTile * D * 2);   // [rows]

  // combine the pass-1 partials: lse2[r] = log2 sum_t 2^(s_rt)
  {
    const float* m_in = stats_m + (static_cast<size_t>(b) * stats_rows + static_cast<size_t>(g) * rows) * kScoreSplits;
    const float* l_in = stats_l + (static_cast<size_t>(b) * stats_rows + static_cast<size_t>(g) * rows) * kScoreSplits;
    for (int r = threadIdx.x; r < rows; r += 128) {
      float mv[kScoreSplits], lv[kScoreSplits], M = -INFINITY;
#pragma unroll
      for (int s = 0; s < kScoreSplits; ++s) {
        mv[s] = m_in[r * kScoreSplits + s];
        lv[s] = l_in[r * kScoreSplits + s];
        M = fmaxf(M, mv[s]);
      }
      float L = 0.f;
#pragma unroll
      for (int s = 0; s < kScoreSplits; ++s) L += lv[s] * exp2f(mv[s] - M);
      lse2[r] = M + log2f(L);
    }
  }

  // this warp's 16 keys on the M axis
  const int k_lo = key0 + warp * 16 + gid, k_hi = k_lo + 8;
  const __nv_bfloat16* kbase = k_f + (static_cast<size_t>(b) * bd.t_stride * hkv + g) * D;
  const size_t krow = static_cast<size_t>(hkv) * D;
  uint32_t a[D / 16][4];
  load_a_frags<D>(a, kbase + min(k_lo, N - 1) * krow, kbase + min(k_hi, N - 1) * krow, tig);

  const uint32_t sbase = smem_u32(qbuf);
  auto load_rows = [&](int r0, int buf) {
    constexpr int kChunks = D / 8;
    for (int i = threadIdx.x; i < kTile * kChunks; i += 128) {
      const int rr = i / kChunks, c = i % kChunks;
      const int r = min(r0 + rr, rows - 1);
      const __nv_bfloat16* src = q_probe + ((static_cast<size_t>(b) * bd.q_stride + r / G) * hq + g * G + r % G) * D;
      cp_async16(sbase + buf * (kTile * D * 2) + swz<D>(rr, c), src + c * 8);
    }
    cp_async_commit();
  };

  float acc_lo = 0.f, acc_hi = 0.f;
  const int n_chunks = (rows + kTile - 1) / kTile;
  if (n_chunks > 0) load_rows(0, 0);
  for (int t = 0; t < n_chunks; ++t) {
    if (t + 1 < n_chunks) { load_rows((t + 1) * kTile, (t + 1) & 1); cp_async_wait<1>(); } else { cp_async_wait<0>(); }
    __syncthreads();      // also orders the lse2 writes before their first use
    float c[kTile / 8][4];
    mma_tile<D>(c, a, sbase + (t & 1) * (kTile * D * 2), lane);
#pragma unroll
    for (int nt = 0; nt < kTile / 8; ++nt) {
      const int r = t * kTile + nt * 8 + 2 * tig;
      if (r < rows) {
        const float z = lse2[r];
        acc_lo += exp2f(fmaf(c[nt][0], scale_log2, -z));
        acc_hi += exp2f(fmaf(c[nt][2], scale_log2, -z));
      }
      if (r + 1 < rows) {
        const float z = lse2[r + 1];
        acc_lo += exp2f(fmaf(c[nt][1], scale_log2, -z));
        acc_hi += exp2f(fmaf(c[nt][3], scale_log2, -z));
      }
    }
    __syncthreads();
  }
#pragma unroll
  for (int o = 1; o <= 2; o <<= 1) {
    acc_lo += __shfl_xor_sync(0xffffffffu, acc_lo, o);
    acc_hi += __shfl_xor_sync(0xffffffffu, acc_hi, o);
  }
  float* my_part = part + (static_cast<size_t>(b) * hkv + g) * part_stride;
  if (tig == 0) {
    if (k_lo < N) my_part[k_lo] = acc_lo;
    if (k_hi < N) my_part[k_hi] = acc_hi;
  }
  // last CTA of this key tile sums the Hkv partials in fixed order (deterministic)
  __threadfence();
  __syncthreads();
  const int n_tiles_b = (bd.n_stride + kTile - 1) / kTile;
  unsigned int* ctr = counters + static_cast<size_t>(b) * n_tiles_b + blockIdx.x;
  if (threadIdx.x == 0) s_last = (atomicAdd(ctr, 1u) == static_cast<unsigned int>(hkv - 1));
  __syncthreads();
  if (s_last) {
    __threadfence();
    if (threadIdx.x < kTile && key0 + threadIdx.x < N) {
      const int key = key0 + threadIdx.x;
      float sum = 0.f;
      for (int gg = 0; gg < hkv; ++gg) sum += __ldcg(part + (static_cast<size_t>(b) * hkv + gg) * part_stride + key);
      const float v = rows > 0 ? sum / static_cast<float>(norm_heads * Lq) : 0.f;
      float* dst = scores + static_cast<size_t>(b) * bd.n_stride + key;
      *dst = accumulate ? *dst + v : v;
    }
    if (threadIdx.x == 0) *ctr = 0u;
  }
}

}  // namespace

cudaError_t launch_score(const qcf_ctx* ctx, const qcf_batch* b, const __nv_bfloat16* q_probe,
                         const __nv_bfloat16* k_f, float* scores, int accumulate, cudaStream_t stream) {
  if (b->batch == 0 || b->max_ctx == 0) return cudaSuccess;
  if (ctx->score_impl == 1) return launch_score_tc(ctx, b, q_probe, k_f, scores, accumulate, stream);
  const Layout& L = ctx->lay;
  const float scale_log2 = L.scale * kLog2e;
  const int stats_rows = L.hq * ctx->max_query;
  const int max_rows = b->max_query * L.g;
  if (max_rows > 0) {
    dim3 g1(kScoreSplits, (max_rows + kTile - 1) / kTile, b->batch * L.hkv);
    if (L.d == 128)
      score_stats_kernel<128><<<g1, 128, 0, stream>>>(b->dev, L.hq, L.hkv, scale_log2, q_probe, k_f, ctx->stats_m,
                                                      ctx->stats_l, stats_rows);
    else
      score_stats_kernel<64><<<g1, 128, 0, stream>>>(b->dev, L.hq, L.hkv, scale_log2, q_probe, k_f, ctx->stats_m,
                                                     ctx->stats_l, stats_rows);
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return e;
  }
  dim3 g2((b->max_ctx + kTile - 1) / kTile, L.hkv, b->batch);
  const size_t smem = 2 * kTile * L.d * 2 + static_cast<size_t>(max_rows > 0 ? max_rows : 1) * sizeof(float);
  if (L.d == 128) {
    auto kern = score_colsum_kernel<128>;
    cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, static_cast<int>(smem));
    kern<<<g2, 128, smem, stream>>>(b->dev, L.hq, L.hkv, scale_log2, q_probe, k_f, ctx->stats_m, ctx->stats_l,
                                    stats_rows, ctx->score_part, ctx->max_ctx, L.hq * ctx->head_shards, ctx->counters, scores, accumulate);
  } else {
    auto kern = score_colsum_kernel<64>;
    cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, static_cast<int>(smem));
    kern<<<g2, 128, smem, stream>>>(b->dev, L.hq, L.hkv, scale_log2, q_probe, k_f, ctx->stats_m, ctx->stats_l,
                                    stats_rows, ctx->score_part, ctx->max_ctx, L.hq * ctx->head_shards, ctx->counters, scores, accumulate);
  }
  return cudaGetLastError();
}

}  // namespace qcf
