// a4 — Eq. 7: write the refreshed K/V rows of the selected positions P into the fused cache at
// the same positions, and append the user query's own K/V rows at N..N+Lq-1 (U is the online suffix).
// Pure row gather/scatter: 2 * Hkv * d * 2 bytes read and written per refreshed row, 128-bit vectors.
#include "qcf_internal.cuh"
#include "sm100_ptx.cuh"

namespace qcf {

namespace {

// TMA-staged variant (the default whenever a row fits its 16 KB slot budget): a refreshed row is one contiguous
// Hkv*d*2-byte run at its source and at its destination, so it moves as ONE bulk async copy global -> shared
// (cp.async.bulk, completion on an mbarrier) and ONE bulk copy shared -> global, never through registers.  A CTA is a single
// warp whose lanes 0..15 each own a (row slot, K or V) pair with its own mbarrier: 8 rows x 2 tensors in flight per CTA,
// ~7 CTAs per SM.  Measured against the register-staged kernel below on c4 x 16: see DESIGN.md section 7.
constexpr int kScatterSlots = 16;

__global__ void __launch_bounds__(32) scatter_tma_kernel(BatchDev bd, uint32_t row_bytes, const int32_t* sel,
                                                         const int32_t* n_sel, const unsigned char* k_new,
                                                         const unsigned char* v_new, int rows_by_position,
                                                         unsigned char* k_f, unsigned char* v_f) {
  extern __shared__ __align__(128) unsigned char smem[];
  __shared__ __align__(8) unsigned long long s_bar[kScatterSlots];
  const int lane = threadIdx.x;
  const int b = blockIdx.y;
  const int N = bd.n_ctx[b], Lq = bd.n_query[b];
  if (lane < kScatterSlots) ptx::mbar_init(smem_u32(&s_bar[lane]), 1);
  ptx::fence_barrier_init();
  pdl_trigger();
  __syncwarp();
  pdl_wait();
  const int ns = __ldcg(n_sel + b);         // coherent loads: written by a predecessor this kernel may overlap (PDL)
  const int n_rows = ns + Lq;
  const int slot = lane >> 1, which = lane & 1;
  const size_t base = static_cast<size_t>(b) * bd.t_stride;
  const uint32_t bar = smem_u32(&s_bar[lane & (kScatterSlots - 1)]);
  const uint32_t buf = smem_u32(smem) + static_cast<uint32_t>(lane & (kScatterSlots - 1)) * row_bytes;
  uint32_t phase = 0;
  for (int r0 = blockIdx.x * 8; r0 < n_rows; r0 += gridDim.x * 8) {
    const int r = r0 + slot;
    if (lane < kScatterSlots && r < n_rows) {
      const int p = r < ns ? __ldcg(sel + static_cast<size_t>(b) * bd.n_stride + r) : N + (r - ns);
      const size_t src = (base + (rows_by_position ? p : r)) * row_bytes;
      const size_t dst = (base + p) * row_bytes;
      ptx::mbar_arrive_expect_tx(bar, row_bytes);
      asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
                   ::"r"(buf), "l"((which ? v_new : k_new) + src), "r"(row_bytes), "r"(bar) : "memory");
      ptx::mbar_wait(bar, phase);
      phase ^= 1u;
      asm volatile("cp.async.bulk.global.shared::cta.bulk_group [%0], [%1], %2;"
                   ::"l"((which ? v_f : k_f) + dst), "r"(buf), "r"(row_bytes) : "memory");
      asm volatile("cp.async.bulk.commit_group;" ::: "memory");
      asm volatile("cp.async.bulk.wait_group.read 0;" ::: "memory");     // the slot is reused by the next row
    }
  }
}

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
        if (i + 32 * u < row_vec) { kk[u] = ld_na_v4(k_new + src + i + 32 * u); vv[u] = ld_na_v4(v_new + src + i + 32 * u); }
#pragma unroll
      for (int u = 0; u < 4; ++u)
        if (i + 32 * u < row_vec) { k_f[dst + i + 32 * u] = kk[u]; v_f[dst + i + 32 * u] = vv[u]; }
    }
  }
}

// Zero-copy gather for the host-side step (qcf_layer_step_host): the position-indexed q_new lives in pinned, device-mapped
// HOST memory and only the rows of R are needed, so each row travels over PCIe as bulk async copies of <= 4 KB pieces
// (host -> shared -> device), landing COMPACT in R order (row r of the destination = position R_b[r] of the source) — the
// layout the attention kernel reads with q_by_position = 0.  Per-thread 16-byte loads from host memory reach ~12 GB/s
// (32-byte PCIe read requests); bulk copies reach the link rate (~50 GB/s, measured on a4 with host-resident k_new / v_new).
__global__ void __launch_bounds__(32) gather_rows_tma_kernel(BatchDev bd, uint32_t row_bytes, uint32_t piece_bytes,
                                                             const int32_t* sel, const int32_t* n_sel,
                                                             const unsigned char* src_by_pos, unsigned char* dst_compact) {
  extern __shared__ __align__(128) unsigned char smem[];
  __shared__ __align__(8) unsigned long long s_bar[kScatterSlots];
  const int lane = threadIdx.x;
  const int b = blockIdx.y;
  const int N = bd.n_ctx[b], Lq = bd.n_query[b];
  if (lane < kScatterSlots) ptx::mbar_init(smem_u32(&s_bar[lane]), 1);
  ptx::fence_barrier_init();
  pdl_trigger();
  __syncwarp();
  pdl_wait();
  const int ns = __ldcg(n_sel + b);
  const int pieces = static_cast<int>(row_bytes / piece_bytes);
  const long long n_items = static_cast<long long>(ns + Lq) * pieces;
  const size_t base = static_cast<size_t>(b) * bd.t_stride;
  const uint32_t bar = smem_u32(&s_bar[lane & (kScatterSlots - 1)]);
  const uint32_t buf = smem_u32(smem) + static_cast<uint32_t>(lane & (kScatterSlots - 1)) * piece_bytes;
  uint32_t phase = 0;
  for (long long w0 = static_cast<long long>(blockIdx.x) * kScatterSlots; w0 < n_items; w0 += static_cast<long long>(gridDim.x) * kScatterSlots) {
    const long long w = w0 + lane;
    if (lane < kScatterSlots && w < n_items) {
      const int r = static_cast<int>(w / pieces), piece = static_cast<int>(w % pieces);
      const int p = r < ns ? __ldcg(sel + static_cast<size_t>(b) * bd.n_stride + r) : N + (r - ns);
      const size_t off = static_cast<size_t>(piece) * piece_bytes;
      ptx::mbar_arrive_expect_tx(bar, piece_bytes);
      asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
                   ::"r"(buf), "l"(src_by_pos + (base + p) * row_bytes + off), "r"(piece_bytes), "r"(bar) : "memory");
      ptx::mbar_wait(bar, phase);
      phase ^= 1u;
      asm volatile("cp.async.bulk.global.shared::cta.bulk_group [%0], [%1], %2;"
                   ::"l"(dst_compact + (base + r) * row_bytes + off), "r"(buf), "r"(piece_bytes) : "memory");
      asm volatile("cp.async.bulk.commit_group;" ::: "memory");
      asm volatile("cp.async.bulk.wait_group.read 0;" ::: "memory");
    }
  }
}

}  // namespace

cudaError_t launch_gather_rows(const qcf_ctx* ctx, const qcf_batch* b, const int32_t* sel, const int32_t* n_sel,
                               const void* src_by_pos, void* dst_compact, int row_bytes, cudaStream_t stream) {
  if (b->batch == 0 || b->t_stride == 0) return cudaSuccess;
  uint32_t piece = 4096;
  while (row_bytes % piece) piece >>= 1;                  // row_bytes is a multiple of 16
  const long long max_items = static_cast<long long>(b->t_stride) * (row_bytes / piece);
  long long blocks = (max_items + kScatterSlots - 1) / kScatterSlots;
  if (blocks > ctx->n_sm * 16) blocks = ctx->n_sm * 16;
  const size_t smem = static_cast<size_t>(kScatterSlots) * piece;
  if (smem > 48 * 1024) cudaFuncSetAttribute(gather_rows_tma_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, static_cast<int>(smem));
  return launch_pdl(ctx->pdl, gather_rows_tma_kernel, dim3(static_cast<unsigned>(blocks), b->batch), dim3(32), smem, stream, b->dev,
                    static_cast<uint32_t>(row_bytes), piece, sel, n_sel, static_cast<const unsigned char*>(src_by_pos),
                    static_cast<unsigned char*>(dst_compact));
}

cudaError_t launch_scatter(const qcf_ctx* ctx, const qcf_batch* b, const int32_t* sel, const int32_t* n_sel,
                           const __nv_bfloat16* k_new, const __nv_bfloat16* v_new, int rows_by_position,
                           __nv_bfloat16* k_f, __nv_bfloat16* v_f, cudaStream_t stream) {
  if (b->batch == 0 || b->t_stride == 0) return cudaSuccess;
  const int row_vec = ctx->lay.hkv * ctx->lay.d / 8;
  const int max_rows = b->t_stride;                      // |R_b| <= N_b + Lq_b
  const uint32_t row_bytes = static_cast<uint32_t>(row_vec) * 16u;
  // Size-based choice, by measurement: the bulk-copy kernel moves a row as load -> wait -> store -> wait, a ~2.5 us chain
  // that wins once the launch is bandwidth-bound (c4 x 16, 170 MB: 68 -> 57 us = 0.91 of the HBM copy peak; rho = 0.5:
  // 0.96) and loses while it is latency-bound (c2, 6.5 MB: 8.5 -> 10.1 us); c5 (20 MB) is a tie.  The row count is a
  // host-side estimate (the selection size lives on the device).
  const double est_bytes = (ctx->ratio_hint * b->n_stride + b->q_stride) * static_cast<double>(b->batch) * row_bytes * 2.0;
  if (row_bytes <= 4096 && est_bytes >= 12.0 * 1024 * 1024) {     // 16 slots x row <= 64 KB per one-warp CTA
    int blocks = (max_rows + 7) / 8;
    const int cap = ctx->n_sm * 16;
    if (blocks > cap) blocks = cap;
    const size_t smem = static_cast<size_t>(kScatterSlots) * row_bytes;
    if (smem > 48 * 1024) cudaFuncSetAttribute(scatter_tma_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, static_cast<int>(smem));
    return launch_pdl(ctx->pdl, scatter_tma_kernel, dim3(blocks, b->batch), dim3(32), smem, stream, b->dev, row_bytes, sel, n_sel,
                      reinterpret_cast<const unsigned char*>(k_new), reinterpret_cast<const unsigned char*>(v_new),
                      rows_by_position, reinterpret_cast<unsigned char*>(k_f), reinterpret_cast<unsigned char*>(v_f));
  }
  int blocks = (max_rows + 7) / 8;
  const int cap = ctx->n_sm * 8;
  if (blocks > cap) blocks = cap;
  return launch_pdl(ctx->pdl, scatter_kernel, dim3(blocks, b->batch), dim3(256), 0, stream,
      b->dev, row_vec, sel, n_sel, reinterpret_cast<const uint4*>(k_new), reinterpret_cast<const uint4*>(v_new),
      rows_by_position, reinterpret_cast<uint4*>(k_f), reinterpret_cast<uint4*>(v_f));
}

}  // namespace qcf
