// Internal declarations shared by the qcf translation units (not part of the C ABI).
#pragma once

#include <cuda_bf16.h>
#include <cuda_runtime.h>
#include <stdint.h>

#include <string>

#include "qcf.h"

namespace qcf {

// Device-resident description of a batch (arrays live in one allocation owned by qcf_batch).
struct BatchDev {
  int32_t batch;
  int32_t n_chunks;        // total over the batch
  int32_t t_stride;        // rows per request in fused caches / fresh rows / outputs
  int32_t n_stride;        // entries per request in scores / sel
  int32_t q_stride;        // rows per request in q_probe
  // per request [batch]
  const int32_t* n_ctx;    // N_b
  const int32_t* n_query;  // Lq_b
  // per chunk [n_chunks]
  const int32_t* chunk_req;    // owning request
  const int32_t* chunk_off;    // off_i: first row of the chunk in the request's fused cache
  const int32_t* chunk_rot;    // position the chunk is rotated by (= chunk_off unless qcf_request.chunk_pos is given)
  const int32_t* chunk_len;
  const int64_t* chunk_row;    // first row in the PIC pool
  const int32_t* chunk_blk;    // [n_chunks+1] exclusive prefix of ceil(len / kRepoRows): reposition work list
  const float2* rot;           // [n_chunks][d/2] (cos, sin)(off_i * theta^(-2j/d))
  const int4* repo_items;      // [repo_blocks][2]: one flat record per reposition work item (RepoItem)
};

// One reposition work item (kRepoRows rows of one chunk), 32 bytes: everything a CTA needs in ONE load, so that its pool
// reads are one dependent round trip behind the launch instead of five (binary search over chunk_blk, then the fields).
struct RepoItem {
  int64_t src_row;   // first pool row
  int64_t dst_row;   // first row in the fused cache (request * t_stride + off + row0)
  int32_t rows;      // <= kRepoRows
  int32_t chunk;     // index into rot
  int32_t identity;  // != 0: rotation position 0, K is copied bit-exactly
  int32_t pad;
};

struct Layout {
  int hq, hkv, d, g;
  float theta;
  float scale;        // softmax scale
};

constexpr int kRepoRows = 8;        // rows per reposition work item

}  // namespace qcf

struct qcf_ctx {
  qcf::Layout lay;
  int device;
  int n_sm;
  int max_batch, max_ctx, max_query;
  // test-only knobs, set through qcf_debug_set (never read from the environment)
  int pdl;               // 1: chain the step's kernels with programmatic dependent launch (default); 0: plain launches
  int gemm_mt;           // GEMM tile height in units of 128 rows: 0 = heuristic, else 1 / 2
  int attn_cluster;      // split-KV cluster size of the attention kernel: 0 = heuristic, else 1 / 2 / 4
  int head_shards;       // this ctx holds 1/head_shards of the layer's heads (qcf_set_head_shards); scores divide by Hq*shards
  double ratio_hint;     // rho of the most recent qcf_select_topk on this ctx (scheduling hint only; 0.3 until then)
  // fused score exchange of the KV-head-sharded step (qcf_set_score_exchange): rank r of exch_world; exch_peers (device
  // array [exch_world] of pointers, mirrored on the host) = every rank's exchange buffer as mapped into THIS process
  int exch_rank, exch_world;
  long long exch_slot_elems;
  float* exch_peers_host[64];
  float** exch_peers;          // device copy
  unsigned int exch_epoch;     // incremented by every exchanging qcf_score; the flag value peers wait for
  unsigned int exch_sel_epoch[2];  // the two most recent distinct epochs an exchanging qcf_select_topk ran at ([0] newest)
  // workspace (device)
  float* stats_m;        // score pass-1 partial row max      [max_batch][Hq*max_query][kScoreSplits]
  float* stats_l;        // score pass-1 partial row sum-exp
  float* score_lse;      // log2-sum-exp per probe row [max_batch][Hq*max_query]
  unsigned int* score_row_ctr;   // pass-1 arrival counters per (request, kv-head, row tile), self-resetting
  float* score_part;     // score pass-2 per-kv-head partial column sums [max_batch][Hkv][max_ctx]
  unsigned int* counters;  // tile counters (zeroed, self-resetting)
  size_t n_counters;
  // decode attention: split-KV partials [Hkv][kDecodeSplitsMax][G][d] fp32, (m, l) pairs, per-kv-head arrival counters
  float* dec_part_o;
  float* dec_part_ml;
  unsigned int* dec_counters;
  // host staging for qcf_layer_step_host
  struct HostStage* stage;
  // profiling
  int profiling;
  static constexpr int kEvRing = 512;   // profiled steps kept between two qcf_get_stage_ms calls
  cudaEvent_t (*ev_ring)[6];            // [kEvRing][6], created by qcf_set_profiling(1)
  int ev_count;                         // sets recorded since the last qcf_get_stage_ms
  cudaEvent_t* ev;                      // set being recorded by the current qcf_layer_step (or nullptr)
  bool ev_valid;
  mutable std::string err;
};

struct qcf_batch {
  qcf_ctx* ctx;
  qcf::BatchDev dev;       // pointers into `blob`
  void* blob;              // one device allocation
  // host copies for validation / grid sizing
  int32_t batch;
  int32_t n_chunks;
  int32_t t_stride, n_stride, q_stride;
  int32_t max_ctx, max_query;
  int64_t total_ctx;
  int32_t repo_blocks;     // total reposition work items
  int64_t pool_row_end;    // max over chunks of chunk_row + chunk_len: rows of the pool the batch reads (host-side validation)
  int64_t* h_pool_iv;      // [2 * n_pool_iv] merged (first row, row count) intervals of the pool rows the batch reads
  int32_t n_pool_iv;
  int64_t pool_rows_touched;   // sum of the interval lengths
  int32_t* h_n_ctx;        // [batch]
  int32_t* h_n_query;      // [batch]
};

namespace qcf {

constexpr int kDecodeSplitsMax = 64; // upper bound of the key splits of the decode attention kernel (sizes its workspace)
constexpr int kScoreSplitsMax = 32; // upper bound of the tcgen05 pass-1 key splits (sizes the statistics workspace)

// Records `msg` as the last error of ctx (or of this thread's failed qcf_create when ctx == nullptr); returns st.
qcf_status set_error(const qcf_ctx* ctx, qcf_status st, const std::string& msg);

// Stage launchers (each validates nothing: arguments were checked by the API layer). Return cudaGetLastError().
cudaError_t launch_reposition(const qcf_ctx*, const qcf_batch*, const __nv_bfloat16* k_pool,
                              const __nv_bfloat16* v_pool, __nv_bfloat16* k_f, __nv_bfloat16* v_f, cudaStream_t);
cudaError_t launch_score(const qcf_ctx*, const qcf_batch*, const __nv_bfloat16* q_probe, const __nv_bfloat16* k_f,
                         float* scores, int accumulate, cudaStream_t);
cudaError_t launch_topk(const qcf_ctx*, const qcf_batch*, const float* scores, double ratio, int32_t* sel,
                        int32_t* n_sel, cudaStream_t, int ceil_mode = 0);
// Exchange buffer of a rank (include/qcf.h, qcf_set_score_exchange):
//   words [0, 64)    flag[p]: newest epoch whose scores rank p has stored into THIS buffer     (written by p's a2 tail)
//   words [64, 128)  ack[p] : newest epoch at which rank p has finished a selection (a3)      (written by p's a3 tail)
//   then 2 slot sets (epoch parity) x n_shards slots x slot_elems fp32
constexpr int kExchHeaderElems = 128;
constexpr int kExchAckOffset = 64;
// after a2 on an exchanging ctx: publish `epoch` in flag[rank] of every peer's exchange buffer (system-scope release)
cudaError_t launch_exchange_flags(const qcf_ctx*, cudaStream_t);
// before a2: wait until every peer's ack in this rank's own buffer has reached `need` (bounded spin, then trap)
cudaError_t launch_exchange_wait(const qcf_ctx*, unsigned int need, cudaStream_t);
// after a3: publish `epoch` in ack[rank] of every peer's exchange buffer (system-scope release)
cudaError_t launch_exchange_ack(const qcf_ctx*, cudaStream_t);
// G_i(r) of Eq. 14 for every chunk row of the batch (rule 0: sink, 1: knorm) into scores[B][n_stride]
cudaError_t launch_anchor_scores(const qcf_ctx*, const qcf_batch*, const __nv_bfloat16* k_pool, int rule, int accumulate,
                                 float* scores, cudaStream_t);
// Eq. 16: rows chunk_row + anchor_idx[b][r] of the PIC pool -> compact anchor pool (chunk order); K and / or V
cudaError_t launch_anchor_gather(const qcf_ctx*, const qcf_batch*, const __nv_bfloat16* k_pool, const __nv_bfloat16* v_pool,
                                 const int32_t* anchor_idx, const int32_t* n_anchor, __nv_bfloat16* k_anchor,
                                 __nv_bfloat16* v_anchor, cudaStream_t);
cudaError_t launch_scatter(const qcf_ctx*, const qcf_batch*, const int32_t* sel, const int32_t* n_sel,
                           const __nv_bfloat16* k_new, const __nv_bfloat16* v_new, int rows_by_position,
                           __nv_bfloat16* k_f, __nv_bfloat16* v_f, cudaStream_t);
// rows R_b of a position-indexed source (may be device-mapped host memory) -> compact rows in R order
cudaError_t launch_gather_rows(const qcf_ctx*, const qcf_batch*, const int32_t* sel, const int32_t* n_sel,
                               const void* src_by_pos, void* dst_compact, int row_bytes, cudaStream_t);
// sel == nullptr: dense mode (rows 0..N+Lq-1 at their own positions, q indexed by position).
cudaError_t launch_attn(const qcf_ctx*, const qcf_batch*, const int32_t* sel, const int32_t* n_sel,
                        const __nv_bfloat16* q, int rows_by_position, const __nv_bfloat16* k_f,
                        const __nv_bfloat16* v_f, __nv_bfloat16* out, float* lse, cudaStream_t);

// single-row GQA attention of one new token over rows [0, n_keys) of a layer's cache [.][Hkv][d]
cudaError_t launch_decode_attn(const qcf_ctx*, const __nv_bfloat16* q, const __nv_bfloat16* k_cache, const __nv_bfloat16* v_cache,
                               int n_keys, __nv_bfloat16* out, float* lse, cudaStream_t);
cudaError_t launch_gemm(const qcf_ctx*, const __nv_bfloat16* a, const __nv_bfloat16* w, const __nv_bfloat16* residual,
                        __nv_bfloat16* c, int M, int N, int K, int epilogue, cudaStream_t);
constexpr int kGemvMaxK = 113 * 1024;   // x[K] bf16 must fit the 227 KB of shared memory a CTA can have
// one row: c[N] = epilogue(x[K] . w[N][K]^T), N even, K % 8 == 0, K <= kGemvMaxK (cudaErrorInvalidValue otherwise); gain != nullptr: x is RMS-normalised with that gain first (rounded to bf16)
cudaError_t launch_gemv(const qcf_ctx*, const __nv_bfloat16* x, const __nv_bfloat16* w, const __nv_bfloat16* gain, float eps,
                        const __nv_bfloat16* residual, __nv_bfloat16* c, int N, int K, int epilogue, cudaStream_t);
cudaError_t launch_lm_head(const qcf_ctx*, const __nv_bfloat16* w_lm, const __nv_bfloat16* h, int vocab, int hidden, float* logits,
                           int32_t* token, cudaStream_t);
cudaError_t launch_stamp(unsigned long long* t0, cudaStream_t);
cudaError_t launch_hold(const unsigned long long* t0, unsigned long long budget_ns, cudaStream_t);
cudaError_t launch_rope_table(float2* table, int n_pos, int d, double theta, cudaStream_t);
cudaError_t launch_embed_gather(const __nv_bfloat16* embed, const int32_t* tokens, const int32_t* sel, const int32_t* n_sel,
                                int n_ctx, int pos_off, int n_rows, int hidden, __nv_bfloat16* x, cudaStream_t);
cudaError_t launch_rmsnorm(const __nv_bfloat16* x, const __nv_bfloat16* gain, float eps, int n_rows, int hidden,
                           __nv_bfloat16* y, cudaStream_t);
// rows r < n_rows of one request; sel == nullptr: position pos_off + r; else sel[r] / query rows at n_ctx + (r - n_sel)
cudaError_t launch_qknorm_rope(const qcf_ctx*, const __nv_bfloat16* qkv, const __nv_bfloat16* g_q, const __nv_bfloat16* g_k,
                               const float2* table, const int32_t* sel, const int32_t* n_sel, int n_ctx, int pos_off,
                               float eps, int n_rows, __nv_bfloat16* q_out, __nv_bfloat16* k_out, __nv_bfloat16* v_out,
                               cudaStream_t);

// ------------------------------------------------------------------------------------------- device helpers
#ifdef __CUDACC__

// Host: launch `kern` with the programmatic-stream-serialization attribute when `pdl` is set (plain launch otherwise).
template <typename... KArgs, typename... Args>
inline cudaError_t launch_pdl(int pdl, void (*kern)(KArgs...), dim3 grid, dim3 block, size_t smem, cudaStream_t stream,
                              Args&&... args) {
  cudaLaunchConfig_t cfg{};
  cfg.gridDim = grid; cfg.blockDim = block; cfg.dynamicSmemBytes = smem; cfg.stream = stream;
  cudaLaunchAttribute at[1];
  at[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
  at[0].val.programmaticStreamSerializationAllowed = 1;
  cfg.attrs = at;
  cfg.numAttrs = pdl ? 1 : 0;
  return cudaLaunchKernelEx(&cfg, kern, KArgs(args)...);
}

// Programmatic dependent launch (PDL): a kernel launched with launch_pdl may start while its predecessor in the stream
// is still draining.  pdl_trigger() lets the NEXT kernel's CTAs be scheduled as soon as every CTA of this grid has
// called it; pdl_wait() blocks until every predecessor grid has completed and its writes are visible — it must precede
// the first access to anything a predecessor wrote OR still reads (the step reuses its buffers every layer).
// A PDL kernel's lifetime overlaps its predecessor's, so data the predecessor writes is NOT read-only for it: such data
// must be read with coherent loads (plain / __ldcg / TMA), never ld.global.nc / __ldg / const __restrict__ promotion.
__device__ __forceinline__ void pdl_trigger() { asm volatile("griddepcontrol.launch_dependents;" ::: "memory"); }
__device__ __forceinline__ void pdl_wait() { asm volatile("griddepcontrol.wait;" ::: "memory"); }

// coherent, L1-cached 32-bit load (never promoted to the non-coherent path, see the PDL note above)
__device__ __forceinline__ int ld_ca_s32(const int32_t* p) {
  int v;
  asm volatile("ld.global.ca.s32 %0, [%1];" : "=r"(v) : "l"(p));
  return v;
}
// coherent 128-bit load that does not allocate in L1 ("na"; NOT the non-coherent .nc path, see the PDL note above)
__device__ __forceinline__ uint4 ld_na_v4(const void* p) {
  uint4 r;
  asm volatile("ld.global.L1::no_allocate.v4.u32 {%0,%1,%2,%3}, [%4];"
               : "=r"(r.x), "=r"(r.y), "=r"(r.z), "=r"(r.w)
               : "l"(p));
  return r;
}
__device__ __forceinline__ void st_na_v4(void* p, const uint4& v) {
  asm volatile("st.global.L1::no_allocate.v4.u32 [%0], {%1,%2,%3,%4};" ::"l"(p), "r"(v.x), "r"(v.y), "r"(v.z),
               "r"(v.w)
               : "memory");
}
__device__ __forceinline__ float bf16lo(uint32_t w) { return __uint_as_float(w << 16); }
__device__ __forceinline__ float bf16hi(uint32_t w) { return __uint_as_float(w & 0xffff0000u); }
// pack two fp32 -> bf16x2 (RNE), lo in the low half
__device__ __forceinline__ uint32_t pack_bf16(float lo, float hi) {
  uint32_t r;
  asm("cvt.rn.bf16x2.f32 %0, %1, %2;" : "=r"(r) : "f"(hi), "f"(lo));
  return r;
}
__device__ __forceinline__ uint32_t smem_u32(const void* p) {
  return static_cast<uint32_t>(__cvta_generic_to_shared(p));
}
__device__ __forceinline__ void cp_async16(uint32_t dst, const void* src) {
  asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(dst), "l"(src) : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
template <int N>
__device__ __forceinline__ void cp_async_wait() {
  asm volatile("cp.async.wait_group %0;" ::"n"(N) : "memory");
}

#endif  // __CUDACC__

}  // namespace qcf
