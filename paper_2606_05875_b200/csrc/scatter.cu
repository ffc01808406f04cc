// a4 — Eq. 7: write the refreshed K/V rows of the selected positions P into the fused cache at
// the same positions, and append the user query's own K/V rows at N..N+Lq-1 (U is the online suffix).
// Pure row gather/scatter: 2 * Hkv * d * 2 bytes read and written per refreshed row, 128-bit vectors.
#include "qcf_internal.cuh"

namespace qcf {

namespace {

// grid (row blocks, B); each warp moves whole rows (K then V) — a row is Hkv*d*2 bytes (2 KB at 8 x 128).
__global__ void __launch_bounds__(256) scatter_kernel(BatchDev bd, int row_vec, const int32_t* __restrict__ sel,
                                                      const int32_t* __restrict__ n_sel,
                                                      const uint4* __restrict__ k_new, const uint4* __restrict__ v_new,
                                                      int rows_by_position, uint4* __restrict__ k_f,
                                                      uint4* __restrict__ v_f) {
  pdl_trigger();
  const int b = blockIdx.y;
  const int N = bd.n_ctx[b], Lq = bd.n_query[b];
  pdl_wait();
  const int ns = __ldcg(n_sel + b);         // coherent loads: written by a predecessor this kernel may overlap (PDL)
  const int n_rows = ns + Lq;
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int warps = blockDim.x >> 5;
  const size_t base = static_cast<size_t>(b) * bd.t_stride;
  for (int r = blockIdx.x * warps + warp; r < n_rows; r += gridDim.x * warps) {
    const int p = r < ns ? __ldcg(sel + static_cast<size_t>(b) * bd.n_stride + r) : N + (r - ns);
    const size_t src = (base + (rows_by_position ? p : r)) * row_vec;
    const size_t dst = (base + p) * row_vec;
    for (int i = lane; i < row_vec; i += 128) {
      uint4 kk[4], vv[4];
#pragma unroll
      for (int u = 0; u < 4; ++u)
        if (i + 32 * u < row_vec) { kk[u] = ld_nc_v4(k_new + src + i + 32 * u); vv[u] = ld_nc_v4(v_new + src + i + 32 * u); }
#pragma unroll
      for (int u = 0; u < 4; ++u)
        if (i + 32 * u < row_vec) { k_f[dst + i + 32 * u] = kk[u]; v_f[dst + i + 32 * u] = vv[u]; }
    }
  }
}

}  // namespace

cudaError_t launch_scatter(const qcf_ctx* ctx, const qcf_batch* b, const int32_t* sel, const int32_t* n_sel,
                           const __nv_bfloat16* k_new, const __nv_bfloat16* v_new, int rows_by_position,
                           __nv_bfloat16* k_f, __nv_bfloat16* v_f, cudaStream_t stream) {
  if (b->batch == 0 || b->t_stride == 0) return cudaSuccess;
  const int row_vec = ctx->lay.hkv * ctx->lay.d / 8;
  const int max_rows = b->t_stride;                      // |R_b| <= N_b + Lq_b
  int blocks = (max_rows + 7) / 8;
  const int cap = ctx->n_sm * 8;
  if (blocks > cap) blocks = cap;
  return launch_pdl(ctx->pdl, scatter_kernel, dim3(blocks, b->batch), dim3(256), 0, stream,
      b->dev, row_vec, sel, n_sel, reinterpret_cast<const uint4*>(k_new), reinterpret_cast<const uint4*>(v_new),
      rows_by_position, reinterpret_cast<uint4*>(k_f), reinterpret_cast<uint4*>(v_f));
}

}  // namespace qcf
