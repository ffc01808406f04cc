// a1 — Eq. 4: re-position per-chunk PIC keys to request positions and stitch K, V.
//
// HBM-bound stream: every K and V row is read once and written once (4 * Hkv * d * 2 bytes per context token).
// A thread owns one "pair slot" of a row — 8 consecutive pairs (j..j+7, j+d/2..j+d/2+7) of one kv-head, i.e. two
// 16-byte vectors — and keeps that slot's 8 (cos, sin) values of the chunk's rotation in registers while it walks
// the rows of its work item, so the only memory traffic in the loop is 128-bit coalesced K/V loads and stores.
#include "qcf_internal.cuh"
#include "sm100_ptx.cuh"

namespace qcf {

namespace {

__device__ __forceinline__ void rotate8(const uint4& a, const uint4& b, const float (&c)[8], const float (&s)[8],
                                        uint4& oa, uint4& ob) {
  const uint32_t aw[4] = {a.x, a.y, a.z, a.w};
  const uint32_t bw[4] = {b.x, b.y, b.z, b.w};
  uint32_t ow_a[4], ow_b[4];
#pragma unroll
  for (int i = 0; i < 4; ++i) {
    const float a0 = bf16lo(aw[i]), a1 = bf16hi(aw[i]);
    const float b0 = bf16lo(bw[i]), b1 = bf16hi(bw[i]);
    // out_j = a cos - b sin ; out_{j+d/2} = b cos + a sin     (fp32, one rounding to bf16 on store)
    const float ra0 = fmaf(a0, c[2 * i], -b0 * s[2 * i]);
    const float ra1 = fmaf(a1, c[2 * i + 1], -b1 * s[2 * i + 1]);
    const float rb0 = fmaf(b0, c[2 * i], a0 * s[2 * i]);
    const float rb1 = fmaf(b1, c[2 * i + 1], a1 * s[2 * i + 1]);
    ow_a[i] = pack_bf16(ra0, ra1);
    ow_b[i] = pack_bf16(rb0, rb1);
  }
  oa = make_uint4(ow_a[0], ow_a[1], ow_a[2], ow_a[3]);
  ob = make_uint4(ow_b[0], ow_b[1], ow_b[2], ow_b[3]);
}

// grid.x = number of work items (kRepoRows rows of one chunk); blockDim.x = slots * rows_per_pass where
// slots = Hkv * d / 16 pair slots per row.
template <int D>
__global__ void __launch_bounds__(512) reposition_kernel(BatchDev bd, int hkv, const __nv_bfloat16* __restrict__ k_pool,
                                                         const __nv_bfloat16* __restrict__ v_pool,
                                                         __nv_bfloat16* __restrict__ k_f,
                                                         __nv_bfloat16* __restrict__ v_f) {
  constexpr int kSlotsPerHead = D / 16;
  const int slots = hkv * kSlotsPerHead;
  const int row_elems = hkv * D;
  // this work item's flat record (RepoItem, qcf_internal.cuh): two 16-byte loads, no search
  const int4 w0 = __ldg(bd.repo_items + 2 * blockIdx.x), w1 = __ldg(bd.repo_items + 2 * blockIdx.x + 1);
  const size_t src_row = (static_cast<size_t>(static_cast<uint32_t>(w0.y)) << 32) | static_cast<uint32_t>(w0.x);
  const size_t dst_row = (static_cast<size_t>(static_cast<uint32_t>(w0.w)) << 32) | static_cast<uint32_t>(w0.z);
  const int rows = w1.x;
  const int c = w1.y;

  pdl_trigger();
  const int slot = threadIdx.x % slots;
  const int rsub = threadIdx.x / slots;
  const int rows_per_pass = blockDim.x / slots;
  const int head = slot / kSlotsPerHead;
  const int jc = slot % kSlotsPerHead;           // which group of 8 pairs
  const int e0 = head * D + jc * 8;              // first-half vector (elements), second half at + D/2

  // ---- K: rotate by the chunk's offset angle.  A rotation position of 0 is the identity and is copied bit-exactly.
  const __nv_bfloat16* ks = k_pool + src_row * row_elems;
  __nv_bfloat16* kd = k_f + dst_row * row_elems;
  const bool identity = w1.z != 0;
  pdl_wait();                          // before the first pool read / cache write (descriptor reads above are constant)
  // V rows of this work item (byte copy): the first sweep's loads are issued BEFORE the K section so that a thread has
  // all of its bytes (K pairs + V vectors, 128 B at 8 x 128) in flight at once — at c2 the whole 21 MB input is then
  // outstanding across the grid and the kernel is one HBM round trip plus the launch.
  const uint4* vs = v_pool ? reinterpret_cast<const uint4*>(v_pool + src_row * row_elems) : nullptr;
  const int n_vec = v_pool ? rows * (row_elems / 8) : 0;
  uint4 tv[4];
#pragma unroll
  for (int u = 0; u < 4; ++u)
    if (static_cast<int>(threadIdx.x + u * blockDim.x) < n_vec) tv[u] = ld_na_v4(vs + threadIdx.x + u * blockDim.x);
  if (k_pool == nullptr) {
    // V-only stitch (the K of a critical layer was re-positioned ahead of time for scoring)
  } else if (identity) {
    for (int r = rsub; r < rows; r += rows_per_pass) {
      const uint4 a = ld_na_v4(ks + static_cast<size_t>(r) * row_elems + e0);
      const uint4 b = ld_na_v4(ks + static_cast<size_t>(r) * row_elems + e0 + D / 2);
      st_na_v4(kd + static_cast<size_t>(r) * row_elems + e0, a);
      st_na_v4(kd + static_cast<size_t>(r) * row_elems + e0 + D / 2, b);
    }
  } else {
    float cs[8], sn[8];
    const float4* rt = reinterpret_cast<const float4*>(bd.rot + static_cast<size_t>(c) * (D / 2) + jc * 8);
#pragma unroll
    for (int i = 0; i < 4; ++i) {
      const float4 t = __ldg(rt + i);
      cs[2 * i] = t.x; sn[2 * i] = t.y; cs[2 * i + 1] = t.z; sn[2 * i + 1] = t.w;
    }
    // rows of this thread: rsub, rsub + rpp, ...  — at most kRepoRows / rpp, all loads issued before use
    constexpr int kMaxIter = kRepoRows;
    uint4 a[kMaxIter], b[kMaxIter];
    const int n_it = (rows - rsub + rows_per_pass - 1) / rows_per_pass;   // may be <= 0
#pragma unroll
    for (int it = 0; it < kMaxIter; ++it) {
      if (it < n_it) {
        const size_t r = rsub + it * rows_per_pass;
        a[it] = ld_na_v4(ks + r * row_elems + e0);
        b[it] = ld_na_v4(ks + r * row_elems + e0 + D / 2);
      }
    }
#pragma unroll
    for (int it = 0; it < kMaxIter; ++it) {
      if (it < n_it) {
        const size_t r = rsub + it * rows_per_pass;
        uint4 oa, ob;
        rotate8(a[it], b[it], cs, sn, oa, ob);
        st_na_v4(kd + r * row_elems + e0, oa);
        st_na_v4(kd + r * row_elems + e0 + D / 2, ob);
      }
    }
  }

  // ---- V: stitched in the same token order (byte copy); skipped for the K-only scoring prefetch
  if (v_pool == nullptr) return;
  uint4* vd = reinterpret_cast<uint4*>(v_f + dst_row * row_elems);
#pragma unroll
  for (int u = 0; u < 4; ++u)
    if (static_cast<int>(threadIdx.x + u * blockDim.x) < n_vec) st_na_v4(vd + threadIdx.x + u * blockDim.x, tv[u]);
  for (int i = threadIdx.x + blockDim.x * 4; i < n_vec; i += blockDim.x * 4) {
    uint4 t[4];
#pragma unroll
    for (int u = 0; u < 4; ++u)
      if (i + u * blockDim.x < n_vec) t[u] = ld_na_v4(vs + i + u * blockDim.x);
#pragma unroll
    for (int u = 0; u < 4; ++u)
      if (i + u * blockDim.x < n_vec) st_na_v4(vd + i + u * blockDim.x, t[u]);
  }
}

// ---- TMA-staged variant: the rows of a work item are contiguous in the pool (source) and in the fused cache
// (destination), so each tensor moves as ONE bulk async copy global -> shared (cp.async.bulk, completion on an mbarrier)
// and ONE bulk copy shared -> global; V never touches a register, K is rotated in place in shared memory in between.
__device__ __forceinline__ void bulk_g2s(uint32_t dst, const void* src, uint32_t bytes, uint32_t bar) {
  asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
               ::"r"(dst), "l"(src), "r"(bytes), "r"(bar) : "memory");
}
__device__ __forceinline__ void bulk_s2g(void* dst, uint32_t src, uint32_t bytes) {
  asm volatile("cp.async.bulk.global.shared::cta.bulk_group [%0], [%1], %2;" ::"l"(dst), "r"(src), "r"(bytes) : "memory");
}

template <int D>
__global__ void __launch_bounds__(256) reposition_tma_kernel(BatchDev bd, int hkv, const __nv_bfloat16* k_pool,
                                                             const __nv_bfloat16* v_pool, __nv_bfloat16* k_f,
                                                             __nv_bfloat16* v_f) {
  extern __shared__ __align__(128) unsigned char smem[];
  __shared__ __align__(8) unsigned long long s_bar;
  constexpr int kSlotsPerHead = D / 16;
  const int slots = hkv * kSlotsPerHead;
  const int row_elems = hkv * D;
  const uint32_t row_bytes = static_cast<uint32_t>(row_elems) * 2u;
  const int4 w0 = __ldg(bd.repo_items + 2 * blockIdx.x), w1 = __ldg(bd.repo_items + 2 * blockIdx.x + 1);
  const size_t src_row = (static_cast<size_t>(static_cast<uint32_t>(w0.y)) << 32) | static_cast<uint32_t>(w0.x);
  const size_t dst_row = (static_cast<size_t>(static_cast<uint32_t>(w0.w)) << 32) | static_cast<uint32_t>(w0.z);
  const int rows = w1.x;
  const int c = w1.y;
  const bool identity = w1.z != 0;
  const uint32_t bytes = static_cast<uint32_t>(rows) * row_bytes;
  const uint32_t sK = smem_u32(smem), sV = sK + (k_pool ? kRepoRows * row_bytes : 0u);
  const uint32_t bar = smem_u32(&s_bar);
  if (threadIdx.x == 0) {
    ptx::mbar_init(bar, 1);
    ptx::fence_barrier_init();
  }
  pdl_trigger();
  __syncthreads();
  pdl_wait();                          // before the first pool read / cache write
  if (threadIdx.x == 0) {
    ptx::mbar_arrive_expect_tx(bar, bytes * ((k_pool ? 1u : 0u) + (v_pool ? 1u : 0u)));
    if (k_pool) bulk_g2s(sK, k_pool + src_row * row_elems, bytes, bar);
    if (v_pool) bulk_g2s(sV, v_pool + src_row * row_elems, bytes, bar);
  }
  // the chunk's rotation for this thread's pair slot, fetched while the tiles are in flight
  const int slot = threadIdx.x % slots;
  const int rsub = threadIdx.x / slots;
  const int rows_per_pass = blockDim.x / slots;
  const int head = slot / kSlotsPerHead, jc = slot % kSlotsPerHead;
  const int e0 = head * D + jc * 8;
  float cs[8], sn[8];
  if (k_pool && !identity) {
    const float4* rt = reinterpret_cast<const float4*>(bd.rot + static_cast<size_t>(c) * (D / 2) + jc * 8);
#pragma unroll
    for (int i = 0; i < 4; ++i) {
      const float4 t = __ldg(rt + i);
      cs[2 * i] = t.x; sn[2 * i] = t.y; cs[2 * i + 1] = t.z; sn[2 * i + 1] = t.w;
    }
  }
  ptx::mbar_wait(bar, 0);
  if (k_pool && !identity) {
    for (int r = rsub; r < rows; r += rows_per_pass) {
      uint4* pa = reinterpret_cast<uint4*>(smem + static_cast<size_t>(r) * row_bytes + e0 * 2);
      uint4* pb = reinterpret_cast<uint4*>(smem + static_cast<size_t>(r) * row_bytes + (e0 + D / 2) * 2);
      uint4 oa, ob;
      rotate8(*pa, *pb, cs, sn, oa, ob);
      *pa = oa;
      *pb = ob;
    }
    ptx::fence_proxy_async_smem();      // the rotated rows (generic-proxy writes) are read by the bulk store (async proxy)
  }
  __syncthreads();
  if (threadIdx.x == 0) {
    if (k_pool) bulk_s2g(k_f + dst_row * row_elems, sK, bytes);
    if (v_pool) bulk_s2g(v_f + dst_row * row_elems, sV, bytes);
    asm volatile("cp.async.bulk.commit_group;" ::: "memory");
    asm volatile("cp.async.bulk.wait_group.read 0;" ::: "memory");     // shared memory may be released once it has been read
  }
}

}  // namespace

cudaError_t launch_reposition(const qcf_ctx* ctx, const qcf_batch* b, const __nv_bfloat16* k_pool,
                              const __nv_bfloat16* v_pool, __nv_bfloat16* k_f, __nv_bfloat16* v_f,
                              cudaStream_t stream) {
  if (b->repo_blocks == 0) return cudaSuccess;
  const int slots = ctx->lay.hkv * ctx->lay.d / 16;
  int rpp = 256 / slots;
  if (rpp < 1) rpp = 1;
  if (rpp > kRepoRows) rpp = kRepoRows;
  const int threads = slots * rpp;     // slots <= 512 is enforced at qcf_create
  {   // bulk-copy staged kernel whenever its work item fits shared memory; the register-staged kernel otherwise
    const size_t row_bytes = static_cast<size_t>(ctx->lay.hkv) * ctx->lay.d * 2;
    const size_t smem = kRepoRows * row_bytes * ((k_pool ? 1 : 0) + (v_pool ? 1 : 0));
    if (threads <= 256 && smem <= 200 * 1024) {
      if (ctx->lay.d == 128) {
        auto kern = reposition_tma_kernel<128>;
        if (smem > 48 * 1024) cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, static_cast<int>(smem));
        return launch_pdl(ctx->pdl, kern, dim3(b->repo_blocks), dim3(threads), smem, stream, b->dev, ctx->lay.hkv, k_pool, v_pool, k_f, v_f);
      }
      auto kern = reposition_tma_kernel<64>;
      if (smem > 48 * 1024) cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, static_cast<int>(smem));
      return launch_pdl(ctx->pdl, kern, dim3(b->repo_blocks), dim3(threads), smem, stream, b->dev, ctx->lay.hkv, k_pool, v_pool, k_f, v_f);
    }
  }
  if (ctx->lay.d == 128)
    return launch_pdl(ctx->pdl, reposition_kernel<128>, dim3(b->repo_blocks), dim3(threads), 0, stream, b->dev, ctx->lay.hkv, k_pool, v_pool, k_f, v_f);
  return launch_pdl(ctx->pdl, reposition_kernel<64>, dim3(b->repo_blocks), dim3(threads), 0, stream, b->dev, ctx->lay.hkv, k_pool, v_pool, k_f, v_f);
}

}  // namespace qcf
