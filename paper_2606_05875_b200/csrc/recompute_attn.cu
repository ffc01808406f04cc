// a5 — PAPER.md:134: causal GQA attention of the recomputed rows R = P u U over the fused cache.
//
//   out[r][h] = sum_{j <= p_r} softmax_j(q[r][h] . K_f[j][h/G] * scale) V_f[j][h/G]
//
// Rows are gathered (sorted ascending by request position) and GQA-packed: one CTA tile is BM/G consecutive rows of
// R times the G query heads of one kv-head, so each K/V tile fetched from L2/HBM serves all G heads.  Because the
// rows of a tile are ascending, the causal limit is monotone: key tiles entirely below the tile's first position need
// no mask, and the key loop stops at the tile's last position.  Work per tile grows with position, so tiles are
// issued heaviest-first.  The same kernel in dense mode (sel == nullptr, rows 0..N+Lq-1) is the full-prefill
// comparator (Eq. 2).
#include "qcf_internal.cuh"

namespace qcf {

namespace {

constexpr int BM = 64;    // MMA rows per CTA (4 warps x 16)
constexpr int BN = 64;    // keys per tile
constexpr float kLog2e = 1.4426950408889634f;
constexpr float kLn2 = 0.6931471805599453f;

template <int D>
__global__ void __launch_bounds__(128) attn_kernel(BatchDev bd, int hq, int hkv, float scale_log2,
                                                   const int32_t* __restrict__ sel, const int32_t* __restrict__ n_sel,
                                                   const __nv_bfloat16* __restrict__ q, int q_by_position,
                                                   const __nv_bfloat16* __restrict__ k_f,
                                                   const __nv_bfloat16* __restrict__ v_f,
                                                   __nv_bfloat16* __restrict__ out, float* __restrict__ lse_out) {
  extern __shared__ __align__(128) unsigned char dsmem[];      // K[2][BN][D], V[2][BN][D]
  __shared__ int s_pos[BM];
  const int G = hq / hkv;
  const int PT = BM / G;                                       // positions (rows of R) per tile
  const int b = blockIdx.z, g = blockIdx.y;
  const int N = bd.n_ctx[b], Lq = bd.n_query[b];
  const bool dense = sel == nullptr;
  const int ns = dense ? 0 : n_sel[b];
  const int n_rows = dense ? N + Lq : ns + Lq;
  const int n_tiles = (n_rows + PT - 1) / PT;
  const int tile = static_cast<int>(gridDim.x) - 1 - static_cast<int>(blockIdx.x);     // heaviest first
  if (tile >= n_tiles) return;
  const int ridx0 = tile * PT;
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31, gid = lane >> 2, tig = lane & 3;

  if (threadIdx.x < PT) {
    const int r = ridx0 + threadIdx.x;
    int p = 0;                                                 // padding rows attend to key 0 only; never stored
    if (r < n_rows) p = dense ? r : (r < ns ? sel[static_cast<size_t>(b) * bd.n_stride + r] : N + (r - ns));
    s_pos[threadIdx.x] = p;
  }
  __syncthreads();
  const int last_valid = min(ridx0 + PT, n_rows) - 1 - ridx0;
  const int p_min = s_pos[0], p_max = s_pos[last_valid];
  const int n_key_tiles = p_max / BN + 1;

  // this thread's two MMA rows
  const int t_lo = warp * 16 + gid, t_hi = t_lo + 8;
  const int pl_lo = t_lo / G, pl_hi = t_hi / G;
  const int h_lo = g * G + t_lo % G, h_hi = g * G + t_hi % G;
  const bool ok_lo = ridx0 + pl_lo < n_rows, ok_hi = ridx0 + pl_hi < n_rows;
  const int pos_lo = s_pos[pl_lo], pos_hi = s_pos[pl_hi];
  const size_t rbase = static_cast<size_t>(b) * bd.t_stride;

  uint32_t a[D / 16][4];
  {
    const int src_lo = (dense || q_by_position) ? pos_lo : ridx0 + pl_lo;
    const int src_hi = (dense || q_by_position) ? pos_hi : ridx0 + pl_hi;
    const __nv_bfloat16* q_lo = ok_lo ? q + ((rbase + src_lo) * hq + h_lo) * D : nullptr;
    const __nv_bfloat16* q_hi = ok_hi ? q + ((rbase + src_hi) * hq + h_hi) * D : nullptr;
#pragma unroll
    for (int ks = 0; ks < D / 16; ++ks) {
      const int c = ks * 16 + 2 * tig;
      a[ks][0] = q_lo ? __ldg(reinterpret_cast<const uint32_t*>(q_lo + c)) : 0u;
      a[ks][1] = q_hi ? __ldg(reinterpret_cast<const uint32_t*>(q_hi + c)) : 0u;
      a[ks][2] = q_lo ? __ldg(reinterpret_cast<const uint32_t*>(q_lo + c + 8)) : 0u;
      a[ks][3] = q_hi ? __ldg(reinterpret_cast<const uint32_t*>(q_hi + c + 8)) : 0u;
    }
  }

  const __nv_bfloat16* kbase = k_f + (rbase * hkv + g) * D;
  const __nv_bfloat16* vbase = v_f + (rbase * hkv + g) * D;
  const size_t krow = static_cast<size_t>(hkv) * D;
  const uint32_t sK = smem_u32(dsmem), sV = sK + 2 * BN * D * 2;
  constexpr uint32_t kTileBytes = BN * D * 2;
  auto load_tile = [&](int kt, int buf) {
    constexpr int kChunks = D / 8;
    for (int i = threadIdx.x; i < BN * kChunks; i += 128) {
      const int r = i / kChunks, c = i % kChunks;
      const size_t key = static_cast<size_t>(min(kt * BN + r, p_max));       // rows past p_max are masked anyway
      cp_async16(sK + buf * kTileBytes + swz<D>(r, c), kbase + key * krow + c * 8);
      cp_async16(sV + buf * kTileBytes + swz<D>(r, c), vbase + key * krow + c * 8);
    }
    cp_async_commit();
  };

  float o[D / 8][4];
#pragma unroll
  for (int nt = 0; nt < D / 8; ++nt) o[nt][0] = o[nt][1] = o[nt][2] = o[nt][3] = 0.f;
  float m_lo = -INFINITY, m_hi = -INFINITY, l_lo = 0.f, l_hi = 0.f;

  const int lrow = ((lane >> 4) << 3) + (lane & 7);       // ldmatrix address pattern for the K (B, non-trans) operand
  const int lchunk = (lane >> 3) & 1;
  const int vrow = (((lane >> 3) & 1) << 3) + (lane & 7);  // ... and for the V (B, trans) operand
  const int vchunk = lane >> 4;

  load_tile(0, 0);
  for (int kt = 0; kt < n_key_tiles; ++kt) {
    if (kt + 1 < n_key_tiles) { load_tile(kt + 1, (kt + 1) & 1); cp_async_wait<1>(); } else { cp_async_wait<0>(); }
    __syncthreads();
    const uint32_t kb = sK + (kt & 1) * kTileBytes, vb = sV + (kt & 1) * kTileBytes;

    // S = Q K^T  (16 x BN per warp)
    float s[BN / 8][4];
#pragma unroll
    for (int nt = 0; nt < BN / 8; ++nt) s[nt][0] = s[nt][1] = s[nt][2] = s[nt][3] = 0.f;
#pragma unroll
    for (int ks = 0; ks < D / 16; ++ks) {
#pragma unroll
      for (int np = 0; np < BN / 16; ++np) {
        uint32_t bfr[4];
        ldmatrix_x4(bfr, kb + swz<D>(np * 16 + lrow, 2 * ks + lchunk));
        mma_bf16(s[2 * np], a[ks], bfr[0], bfr[1]);
        mma_bf16(s[2 * np + 1], a[ks], bfr[2], bfr[3]);
      }
    }
    // scale into the log2 domain; causal mask only where the tile reaches past the tile's first position
    const bool need_mask = kt * BN + BN - 1 > p_min;
    float mx_lo = -INFINITY, mx_hi = -INFINITY;
#pragma unroll
    for (int nt = 0; nt < BN / 8; ++nt) {
#pragma unroll
      for (int e = 0; e < 4; ++e) {
        float v = s[nt][e] * scale_log2;
        if (need_mask) {
          const int key = kt * BN + nt * 8 + 2 * tig + (e & 1);
          if (key > ((e < 2) ? pos_lo : pos_hi)) v = -INFINITY;
        }
        s[nt][e] = v;
        if (e < 2) mx_lo = fmaxf(mx_lo, v); else mx_hi = fmaxf(mx_hi, v);
      }
    }
#pragma unroll
    for (int off = 1; off <= 2; off <<= 1) {
      mx_lo = fmaxf(mx_lo, __shfl_xor_sync(0xffffffffu, mx_lo, off));
      mx_hi = fmaxf(mx_hi, __shfl_xor_sync(0xffffffffu, mx_hi, off));
    }
    // key 0 is visible to every row, so after the first tile the running max is finite
    const float mn_lo = fmaxf(m_lo, mx_lo), mn_hi = fmaxf(m_hi, mx_hi);
    const float corr_lo = exp2f(m_lo - mn_lo), corr_hi = exp2f(m_hi - mn_hi);
    m_lo = mn_lo; m_hi = mn_hi;
    l_lo *= corr_lo; l_hi *= corr_hi;
#pragma unroll
    for (int nt = 0; nt < D / 8; ++nt) { o[nt][0] *= corr_lo; o[nt][1] *= corr_lo; o[nt][2] *= corr_hi; o[nt][3] *= corr_hi; }
    uint32_t p[BN / 16][4];
#pragma unroll
    for (int kk = 0; kk < BN / 16; ++kk) {
      float e[2][4];
#pragma unroll
      for (int u = 0; u < 2; ++u) {
        e[u][0] = exp2f(s[2 * kk + u][0] - mn_lo); e[u][1] = exp2f(s[2 * kk + u][1] - mn_lo);
        e[u][2] = exp2f(s[2 * kk + u][2] - mn_hi); e[u][3] = exp2f(s[2 * kk + u][3] - mn_hi);
        l_lo += e[u][0] + e[u][1]; l_hi += e[u][2] + e[u][3];
      }
      p[kk][0] = pack_bf16(e[0][0], e[0][1]); p[kk][1] = pack_bf16(e[0][2], e[0][3]);
      p[kk][2] = pack_bf16(e[1][0], e[1][1]); p[kk][3] = pack_bf16(e[1][2], e[1][3]);
    }
    // O += P V
#pragma unroll
    for (int kk = 0; kk < BN / 16; ++kk) {
#pragma unroll
      for (int np = 0; np < D / 16; ++np) {
        uint32_t bfr[4];
        ldmatrix_x4_trans(bfr, vb + swz<D>(kk * 16 + vrow, 2 * np + vchunk));
        mma_bf16(o[2 * np], p[kk], bfr[0], bfr[1]);
        mma_bf16(o[2 * np + 1], p[kk], bfr[2], bfr[3]);
      }
    }
    __syncthreads();
  }

#pragma unroll
  for (int off = 1; off <= 2; off <<= 1) {
    l_lo += __shfl_xor_sync(0xffffffffu, l_lo, off);
    l_hi += __shfl_xor_sync(0xffffffffu, l_hi, off);
  }
  const float inv_lo = 1.f / l_lo, inv_hi = 1.f / l_hi;
  if (ok_lo) {
    __nv_bfloat16* dst = out + ((rbase + ridx0 + pl_lo) * hq + h_lo) * D;
#pragma unroll
    for (int nt = 0; nt < D / 8; ++nt)
      *reinterpret_cast<uint32_t*>(dst + nt * 8 + 2 * tig) = pack_bf16(o[nt][0] * inv_lo, o[nt][1] * inv_lo);
    if (lse_out && tig == 0) lse_out[(rbase + ridx0 + pl_lo) * hq + h_lo] = (m_lo + log2f(l_lo)) * kLn2;
  }
  if (ok_hi) {
    __nv_bfloat16* dst = out + ((rbase + ridx0 + pl_hi) * hq + h_hi) * D;
#pragma unroll
    for (int nt = 0; nt < D / 8; ++nt)
      *reinterpret_cast<uint32_t*>(dst + nt * 8 + 2 * tig) = pack_bf16(o[nt][2] * inv_hi, o[nt][3] * inv_hi);
    if (lse_out && tig == 0) lse_out[(rbase + ridx0 + pl_hi) * hq + h_hi] = (m_hi + log2f(l_hi)) * kLn2;
  }
}

}  // namespace

cudaError_t launch_attn(const qcf_ctx* ctx, const qcf_batch* b, const int32_t* sel, const int32_t* n_sel,
                        const __nv_bfloat16* q, int rows_by_position, const __nv_bfloat16* k_f,
                        const __nv_bfloat16* v_f, __nv_bfloat16* out, float* lse, cudaStream_t stream) {
  if (b->batch == 0 || b->t_stride == 0) return cudaSuccess;
  if (ctx->attn_impl == 2) return launch_attn_ptc(ctx, b, sel, n_sel, q, rows_by_position, k_f, v_f, out, lse, stream);
  if (ctx->attn_impl == 1) return launch_attn_tc(ctx, b, sel, n_sel, q, rows_by_position, k_f, v_f, out, lse, stream);
  const Layout& L = ctx->lay;
  const int PT = BM / L.g;
  const int max_tiles = (b->t_stride + PT - 1) / PT;            // |R_b| <= N_b + Lq_b <= t_stride
  const dim3 grid(max_tiles, L.hkv, b->batch);
  const size_t smem = 4 * static_cast<size_t>(BN) * L.d * 2;
  const float scale_log2 = L.scale * kLog2e;
  if (L.d == 128) {
    auto kern = attn_kernel<128>;
    cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, static_cast<int>(smem));
    kern<<<grid, 128, smem, stream>>>(b->dev, L.hq, L.hkv, scale_log2, sel, n_sel, q, rows_by_position, k_f, v_f, out,
                                      lse);
  } else {
    auto kern = attn_kernel<64>;
    cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, static_cast<int>(smem));
    kern<<<grid, 128, smem, stream>>>(b->dev, L.hq, L.hkv, scale_log2, sel, n_sel, q, rows_by_position, k_f, v_f, out,
                                      lse);
  }
  return cudaGetLastError();
}

}  // namespace qcf
