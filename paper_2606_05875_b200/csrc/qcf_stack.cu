// Config 3 (BASELINE.json configs[2]): the decoder stack around the layer step — a7 (row-wise dense ops of the rows
// R = P u U), a8 (layer-ahead KV loading on a second stream) and the two-stage online pipeline of Fig. 9
// (PAPER.md:329-344).  Host-side orchestration only: every tensor operation is a kernel of the sibling files.
#include <algorithm>
#include <new>
#include <string>
#include <vector>

#include "qcf_internal.cuh"

using namespace qcf;

struct qcf_stack {
  qcf_ctx* ctx;
  qcf_stack_dims dims;
  std::vector<qcf_layer_weights> layers;
  const __nv_bfloat16* embed;
  int max_rows, max_pos;
  int64_t max_pool_rows;
  // activation workspace (device, bf16)
  __nv_bfloat16 *x, *h, *qkv, *q_new, *k_new, *v_new, *attn, *act;
  float2* rope_table;
  // qcf_stack_fuse: staging ring for the loaded pools, probe caches, loader stream, events
  static constexpr int kRing = 2;
  __nv_bfloat16* stage_k[kRing];
  __nv_bfloat16* stage_v[kRing];
  __nv_bfloat16* probe_k[2];
  __nv_bfloat16* probe_v[2];
  size_t probe_rows;
  cudaStream_t loader;
  cudaStream_t loader2;                            // stage 1: K of the critical layers, issued at t = 0
  __nv_bfloat16* stage_k2[2];                      // its staging ring
  static constexpr int kArena = 2;                 // anchor arena: kArena x max_pool_rows rows of K and of V
  __nv_bfloat16 *arena_k, *arena_v;                // stage 1, two-stream mode: anchor pools copied ahead of their stitch
  std::vector<cudaEvent_t> ev_copy;                // per probe layer: its anchor rows are in the arena
  std::vector<cudaEvent_t> ev_ready, ev_done;      // per pipeline slot
  cudaEvent_t ev_fork, ev_join;
  unsigned long long* load_t0;                     // device stamp of the bandwidth emulation (load_gbps)
  int32_t* zero_i32;                               // device zeros: the probe stage's empty selection
};

namespace {

#define STK_CUDA(ctx, call)                                                                             \
  do {                                                                                                  \
    cudaError_t e__ = (call);                                                                           \
    if (e__ != cudaSuccess) return set_error(ctx, QCF_ERR_CUDA, std::string(#call) + ": " + cudaGetErrorString(e__)); \
  } while (0)
#define STK_REQUIRE(ctx, cond, msg)                                          \
  do {                                                                       \
    if (!(cond)) return set_error(ctx, QCF_ERR_INVALID_ARG, std::string(msg)); \
  } while (0)

inline bool aligned16(const void* p) { return (reinterpret_cast<uintptr_t>(p) & 15u) == 0; }

template <class T>
cudaError_t dalloc(T** p, size_t n) { return cudaMalloc(reinterpret_cast<void**>(p), n * sizeof(T) + 16); }

// (Chaining the GEMMs, RMSNorm and QK-norm kernels with programmatic dependent launch as well was measured: bit-identical
// results, config-3 pipeline 53.1 ms serialised vs 53.6 ms chained — the ~2 us per launch it hides is below the run-to-run
// noise of 1.2 ms layers, so these launches stay plain; the attention and scatter kernels keep their PDL chain.)
// The block of DESIGN.md §7 for rows 0..n_rows-1 of `x` (in place).  sel == nullptr: dense (K/V go straight into
// k_fused / v_fused, rows are positions pos0..); else a4 + a5 through qcf_recompute_attn on compact fresh rows.
qcf_status run_layer(qcf_stack* s, int l, const qcf_batch* b, const int32_t* sel, const int32_t* n_sel, int n_rows,
                     int query_pos0, __nv_bfloat16* x, void* k_fused, void* v_fused, void* q_tap, cudaStream_t st) {
  qcf_ctx* ctx = s->ctx;
  const Layout& L = ctx->lay;
  const qcf_layer_weights& w = s->layers[l];
  const int hid = s->dims.hidden, ffn = s->dims.ffn;
  const int qkv_n = (L.hq + 2 * L.hkv) * L.d;
  const bool dense = sel == nullptr;
  auto bf = [](const void* p) { return static_cast<const __nv_bfloat16*>(p); };
  STK_CUDA(ctx, launch_rmsnorm(x, bf(w.g_attn), s->dims.rms_eps, n_rows, hid, s->h, st));
  STK_CUDA(ctx, launch_gemm(ctx, s->h, bf(w.w_qkv), nullptr, s->qkv, n_rows, qkv_n, hid, QCF_EPI_STORE, st));
  __nv_bfloat16* q_dst = q_tap ? static_cast<__nv_bfloat16*>(q_tap) : s->q_new;
  const int n_ctx = b->h_n_ctx[0];
  if (dense) {
    STK_CUDA(ctx, launch_qknorm_rope(ctx, s->qkv, bf(w.g_q), bf(w.g_k), s->rope_table, nullptr, nullptr, n_ctx, 0,
                                     s->dims.rms_eps, n_rows, q_dst, static_cast<__nv_bfloat16*>(k_fused),
                                     static_cast<__nv_bfloat16*>(v_fused), st));
    if (qcf_status e = qcf_full_prefill_attn(ctx, b, q_dst, k_fused, v_fused, s->attn, nullptr, st)) return e;
  } else {
    const int qp0 = query_pos0 >= 0 ? query_pos0 : n_ctx;
    STK_CUDA(ctx, launch_qknorm_rope(ctx, s->qkv, bf(w.g_q), bf(w.g_k), s->rope_table, sel, n_sel, qp0, 0,
                                     s->dims.rms_eps, n_rows, q_dst, s->k_new, s->v_new, st));
    if (qcf_status e = qcf_recompute_attn(ctx, b, sel, n_sel, q_dst, s->k_new, s->v_new, 0, k_fused, v_fused, s->attn,
                                          nullptr, st))
      return e;
  }
  STK_CUDA(ctx, launch_gemm(ctx, s->attn, bf(w.w_o), x, x, n_rows, hid, L.hq * L.d, QCF_EPI_ADD_RESIDUAL, st));
  STK_CUDA(ctx, launch_rmsnorm(x, bf(w.g_ffn), s->dims.rms_eps, n_rows, hid, s->h, st));
  STK_CUDA(ctx, launch_gemm(ctx, s->h, bf(w.w_gate_up), nullptr, s->act, n_rows, 2 * ffn, hid, QCF_EPI_SWIGLU, st));
  STK_CUDA(ctx, launch_gemm(ctx, s->act, bf(w.w_down), x, x, n_rows, hid, ffn, QCF_EPI_ADD_RESIDUAL, st));
  return QCF_OK;
}

qcf_status check_stack_batch(qcf_stack* s, const qcf_batch* b, const char* who) {
  if (!s) return set_error(nullptr, QCF_ERR_INVALID_ARG, std::string(who) + ": stack is NULL");
  qcf_ctx* ctx = s->ctx;
  STK_REQUIRE(ctx, b != nullptr && b->ctx == ctx, std::string(who) + ": batch is NULL or from another ctx");
  STK_REQUIRE(ctx, b->batch == 1, std::string(who) + ": the stack calls take single-request batches (B = 1)");
  return QCF_OK;
}

}  // namespace

extern "C" {

qcf_status qcf_linear(qcf_ctx* ctx, const void* a, const void* w, const void* residual, void* c, int32_t M, int32_t N,
                      int32_t K, int32_t epilogue, void* stream) {
  if (!ctx) return set_error(nullptr, QCF_ERR_INVALID_ARG, "ctx is NULL");
  STK_REQUIRE(ctx, M >= 0 && N >= 0 && K > 0, "qcf_linear: M, N must be >= 0 and K > 0");
  if (M == 0 || N == 0) return QCF_OK;
  STK_REQUIRE(ctx, epilogue >= 0 && epilogue <= 2, "qcf_linear: unknown epilogue");
  STK_REQUIRE(ctx, a && w && c, "qcf_linear: NULL tensor pointer");
  STK_REQUIRE(ctx, epilogue != QCF_EPI_ADD_RESIDUAL || residual, "qcf_linear: residual is NULL");
  STK_REQUIRE(ctx, aligned16(a) && aligned16(w) && aligned16(c) && aligned16(residual), "qcf_linear: pointers must be 16-byte aligned");
  STK_REQUIRE(ctx, K % 8 == 0 && N % 8 == 0 && (epilogue != QCF_EPI_SWIGLU || N % 16 == 0),
              "qcf_linear: K and N must be multiples of 8 (N of 16 for SWIGLU)");
  STK_CUDA(ctx, launch_gemm(ctx, static_cast<const __nv_bfloat16*>(a), static_cast<const __nv_bfloat16*>(w),
                            static_cast<const __nv_bfloat16*>(residual), static_cast<__nv_bfloat16*>(c), M, N, K, epilogue,
                            static_cast<cudaStream_t>(stream)));
  return QCF_OK;
}

qcf_status qcf_stack_create(qcf_ctx* ctx, const qcf_stack_dims* dims, const qcf_layer_weights* layers, const void* embed,
                            int32_t max_rows, int32_t max_pos, int64_t max_pool_rows, qcf_stack** out) {
  if (!ctx) return set_error(nullptr, QCF_ERR_INVALID_ARG, "ctx is NULL");
  STK_REQUIRE(ctx, out != nullptr, "qcf_stack_create: out is NULL");
  *out = nullptr;
  STK_REQUIRE(ctx, dims && layers && embed, "qcf_stack_create: NULL argument");
  STK_REQUIRE(ctx, dims->n_layers >= 1 && dims->hidden >= 8 && dims->ffn >= 8 && dims->vocab >= 1,
              "qcf_stack_create: n_layers, hidden, ffn, vocab must be positive");
  STK_REQUIRE(ctx, dims->hidden % 8 == 0 && dims->ffn % 8 == 0, "qcf_stack_create: hidden and ffn must be multiples of 8");
  STK_REQUIRE(ctx, max_rows >= 1 && max_pos >= 1 && max_pool_rows >= 0, "qcf_stack_create: bad limits");
  for (int l = 0; l < dims->n_layers; ++l) {
    const qcf_layer_weights& w = layers[l];
    STK_REQUIRE(ctx, w.w_qkv && w.w_o && w.w_gate_up && w.w_down && w.g_attn && w.g_ffn && w.g_q && w.g_k,
                "qcf_stack_create: NULL weight pointer");
    STK_REQUIRE(ctx, aligned16(w.w_qkv) && aligned16(w.w_o) && aligned16(w.w_gate_up) && aligned16(w.w_down) &&
                         aligned16(w.g_attn) && aligned16(w.g_ffn),
                "qcf_stack_create: weight pointers must be 16-byte aligned");
  }
  qcf_stack* s = new (std::nothrow) qcf_stack();
  if (!s) return set_error(ctx, QCF_ERR_WORKSPACE, "out of host memory");
  s->ctx = ctx; s->dims = *dims;
  s->layers.assign(layers, layers + dims->n_layers);
  s->embed = static_cast<const __nv_bfloat16*>(embed);
  s->max_rows = max_rows; s->max_pos = max_pos; s->max_pool_rows = max_pool_rows;
  const Layout& L = ctx->lay;
  const size_t R = max_rows, kv = static_cast<size_t>(L.hkv) * L.d, qd = static_cast<size_t>(L.hq) * L.d;
  s->x = s->h = s->qkv = s->q_new = s->k_new = s->v_new = s->attn = s->act = nullptr;
  s->rope_table = nullptr;
  for (int i = 0; i < qcf_stack::kRing; ++i) s->stage_k[i] = s->stage_v[i] = nullptr;
  s->probe_k[0] = s->probe_k[1] = s->probe_v[0] = s->probe_v[1] = nullptr;
  s->loader = s->loader2 = nullptr; s->ev_fork = s->ev_join = nullptr; s->zero_i32 = nullptr;
  s->stage_k2[0] = s->stage_k2[1] = nullptr;
  s->arena_k = s->arena_v = nullptr;
  s->probe_rows = static_cast<size_t>(max_pool_rows) + ctx->max_query;
  bool ok = dalloc(&s->x, R * dims->hidden) == cudaSuccess && dalloc(&s->h, R * dims->hidden) == cudaSuccess &&
            dalloc(&s->qkv, R * (qd + 2 * kv)) == cudaSuccess && dalloc(&s->q_new, R * qd) == cudaSuccess &&
            dalloc(&s->k_new, R * kv) == cudaSuccess && dalloc(&s->v_new, R * kv) == cudaSuccess &&
            dalloc(&s->attn, R * qd) == cudaSuccess && dalloc(&s->act, R * dims->ffn) == cudaSuccess &&
            dalloc(&s->rope_table, static_cast<size_t>(max_pos) * (L.d / 2)) == cudaSuccess;
  if (ok && max_pool_rows > 0) {
    for (int i = 0; i < qcf_stack::kRing && ok; ++i)
      ok = dalloc(&s->stage_k[i], static_cast<size_t>(max_pool_rows) * kv) == cudaSuccess &&
           dalloc(&s->stage_v[i], static_cast<size_t>(max_pool_rows) * kv) == cudaSuccess;
    for (int i = 0; i < 2 && ok; ++i)
      ok = dalloc(&s->probe_k[i], s->probe_rows * kv) == cudaSuccess && dalloc(&s->probe_v[i], s->probe_rows * kv) == cudaSuccess &&
           dalloc(&s->stage_k2[i], static_cast<size_t>(max_pool_rows) * kv) == cudaSuccess;
    ok = ok && dalloc(&s->arena_k, qcf_stack::kArena * static_cast<size_t>(max_pool_rows) * kv) == cudaSuccess &&
         dalloc(&s->arena_v, qcf_stack::kArena * static_cast<size_t>(max_pool_rows) * kv) == cudaSuccess;
  }
  s->load_t0 = nullptr;
  ok = ok && dalloc(&s->load_t0, 2) == cudaSuccess;
  ok = ok && dalloc(&s->zero_i32, 4) == cudaSuccess && cudaMemset(s->zero_i32, 0, 16) == cudaSuccess;
  ok = ok && cudaStreamCreateWithFlags(&s->loader, cudaStreamNonBlocking) == cudaSuccess &&
       cudaStreamCreateWithFlags(&s->loader2, cudaStreamNonBlocking) == cudaSuccess &&
       cudaEventCreateWithFlags(&s->ev_fork, cudaEventDisableTiming) == cudaSuccess &&
       cudaEventCreateWithFlags(&s->ev_join, cudaEventDisableTiming) == cudaSuccess;
  const int n_slots = 2 * dims->n_layers + 4;
  s->ev_ready.assign(n_slots, nullptr);
  s->ev_done.assign(n_slots, nullptr);
  s->ev_copy.assign(n_slots, nullptr);
  for (int i = 0; i < n_slots && ok; ++i)
    ok = cudaEventCreateWithFlags(&s->ev_copy[i], cudaEventDisableTiming) == cudaSuccess &&
         cudaEventCreateWithFlags(&s->ev_ready[i], cudaEventDisableTiming) == cudaSuccess &&
         cudaEventCreateWithFlags(&s->ev_done[i], cudaEventDisableTiming) == cudaSuccess;
  ok = ok && launch_rope_table(s->rope_table, max_pos, L.d, static_cast<double>(L.theta), nullptr) == cudaSuccess &&
       cudaDeviceSynchronize() == cudaSuccess;
  if (!ok) {
    const cudaError_t le = cudaGetLastError();
    qcf_stack_destroy(s);
    return set_error(ctx, QCF_ERR_WORKSPACE, std::string("qcf_stack_create: allocation failed: ") + cudaGetErrorString(le));
  }
  *out = s;
  return QCF_OK;
}

void qcf_stack_destroy(qcf_stack* s) {
  if (!s) return;
  for (void* p : {static_cast<void*>(s->x), static_cast<void*>(s->h), static_cast<void*>(s->qkv), static_cast<void*>(s->q_new),
                  static_cast<void*>(s->k_new), static_cast<void*>(s->v_new), static_cast<void*>(s->attn),
                  static_cast<void*>(s->act), static_cast<void*>(s->rope_table)})
    if (p) cudaFree(p);
  for (int i = 0; i < qcf_stack::kRing; ++i) { if (s->stage_k[i]) cudaFree(s->stage_k[i]); if (s->stage_v[i]) cudaFree(s->stage_v[i]); }
  for (int i = 0; i < 2; ++i) { if (s->probe_k[i]) cudaFree(s->probe_k[i]); if (s->probe_v[i]) cudaFree(s->probe_v[i]); if (s->stage_k2[i]) cudaFree(s->stage_k2[i]); }
  for (cudaEvent_t e : s->ev_ready) if (e) cudaEventDestroy(e);
  for (cudaEvent_t e : s->ev_done) if (e) cudaEventDestroy(e);
  for (cudaEvent_t e : s->ev_copy) if (e) cudaEventDestroy(e);
  if (s->arena_k) cudaFree(s->arena_k);
  if (s->arena_v) cudaFree(s->arena_v);
  if (s->ev_fork) cudaEventDestroy(s->ev_fork);
  if (s->ev_join) cudaEventDestroy(s->ev_join);
  if (s->load_t0) cudaFree(s->load_t0);
  if (s->zero_i32) cudaFree(s->zero_i32);
  if (s->loader) cudaStreamDestroy(s->loader);
  if (s->loader2) cudaStreamDestroy(s->loader2);
  delete s;
}

qcf_status qcf_stack_layer(qcf_stack* s, int32_t layer, const qcf_batch* b, const int32_t* sel, const int32_t* n_sel,
                           int32_t n_rows, int32_t query_pos0, void* x, void* k_fused, void* v_fused, void* q_tap,
                           void* stream) {
  if (qcf_status e = check_stack_batch(s, b, "qcf_stack_layer")) return e;
  qcf_ctx* ctx = s->ctx;
  STK_REQUIRE(ctx, layer >= 0 && layer < s->dims.n_layers, "qcf_stack_layer: layer out of range");
  STK_REQUIRE(ctx, n_rows >= 0 && n_rows <= s->max_rows, "qcf_stack_layer: n_rows exceeds max_rows of qcf_stack_create");
  STK_REQUIRE(ctx, x && k_fused && v_fused, "qcf_stack_layer: NULL tensor pointer");
  STK_REQUIRE(ctx, (sel == nullptr) || n_sel, "qcf_stack_layer: n_sel is NULL");
  STK_REQUIRE(ctx, sel != nullptr || n_rows == b->h_n_ctx[0] + b->h_n_query[0], "qcf_stack_layer: dense mode takes all N + Lq rows");
  const int top = sel ? (query_pos0 >= 0 ? query_pos0 : b->h_n_ctx[0]) + b->h_n_query[0] : n_rows;
  STK_REQUIRE(ctx, top <= s->max_pos, "qcf_stack_layer: positions exceed max_pos of qcf_stack_create");
  if (n_rows == 0) return QCF_OK;
  return run_layer(s, layer, b, sel, n_sel, n_rows, query_pos0, static_cast<__nv_bfloat16*>(x), k_fused, v_fused, q_tap,
                   static_cast<cudaStream_t>(stream));
}

qcf_status qcf_stack_first_token(qcf_stack* s, const void* hidden, int32_t row, const void* g_final, const void* w_lm,
                                 float* logits, int32_t* token, void* stream) {
  if (!s) return set_error(nullptr, QCF_ERR_INVALID_ARG, "qcf_stack_first_token: stack is NULL");
  qcf_ctx* ctx = s->ctx;
  STK_REQUIRE(ctx, hidden && g_final && w_lm && logits && token, "qcf_stack_first_token: NULL argument");
  STK_REQUIRE(ctx, row >= 0, "qcf_stack_first_token: row must be >= 0");
  STK_REQUIRE(ctx, aligned16(hidden) && aligned16(g_final) && aligned16(w_lm), "qcf_stack_first_token: pointers must be 16-byte aligned");
  cudaStream_t st = static_cast<cudaStream_t>(stream);
  const int hid = s->dims.hidden;
  const __nv_bfloat16* x = static_cast<const __nv_bfloat16*>(hidden) + static_cast<size_t>(row) * hid;
  STK_CUDA(ctx, launch_rmsnorm(x, static_cast<const __nv_bfloat16*>(g_final), s->dims.rms_eps, 1, hid, s->h, st));
  STK_CUDA(ctx, launch_lm_head(ctx, static_cast<const __nv_bfloat16*>(w_lm), s->h, s->dims.vocab, hid, logits, token, st));
  return QCF_OK;
}

qcf_status qcf_stack_decode(qcf_stack* s, const int32_t* token_in, int32_t pos0, int32_t n_new, void* const* k_cache,
                            void* const* v_cache, const void* g_final, const void* w_lm, float* logits, int32_t* tokens_out,
                            void* stream) {
  if (!s) return set_error(nullptr, QCF_ERR_INVALID_ARG, "qcf_stack_decode: stack is NULL");
  qcf_ctx* ctx = s->ctx;
  const Layout& L = ctx->lay;
  STK_REQUIRE(ctx, token_in && k_cache && v_cache && g_final && w_lm && logits && tokens_out, "qcf_stack_decode: NULL argument");
  STK_REQUIRE(ctx, pos0 >= 0 && n_new >= 0, "qcf_stack_decode: pos0 and n_new must be >= 0");
  STK_REQUIRE(ctx, static_cast<int64_t>(pos0) + n_new <= s->max_pos, "qcf_stack_decode: positions exceed max_pos of qcf_stack_create");
  STK_REQUIRE(ctx, aligned16(g_final) && aligned16(w_lm), "qcf_stack_decode: pointers must be 16-byte aligned");
  for (int l = 0; l < s->dims.n_layers; ++l)
    STK_REQUIRE(ctx, k_cache[l] && v_cache[l] && aligned16(k_cache[l]) && aligned16(v_cache[l]),
                "qcf_stack_decode: NULL or misaligned cache pointer");
  cudaStream_t st = static_cast<cudaStream_t>(stream);
  const int hid = s->dims.hidden, ffn = s->dims.ffn, vocab = s->dims.vocab;
  const int qkv_n = (L.hq + 2 * L.hkv) * L.d;
  // the decode layer is four weight-streaming GEMVs that keep their input row in shared memory
  if (hid > kGemvMaxK || ffn > kGemvMaxK || L.hq * L.d > kGemvMaxK)
    return set_error(ctx, QCF_ERR_UNSUPPORTED, "qcf_stack_decode: hidden, ffn and Hq * head_dim must be <= " + std::to_string(kGemvMaxK));
  const size_t kv_row = static_cast<size_t>(L.hkv) * L.d;
  auto bf = [](const void* p) { return static_cast<const __nv_bfloat16*>(p); };
  for (int i = 0; i < n_new; ++i) {
    const int pos = pos0 + i;
    const int32_t* tok = i == 0 ? token_in : tokens_out + (i - 1);
    STK_CUDA(ctx, launch_embed_gather(s->embed, tok, nullptr, nullptr, 0, 0, 1, hid, s->x, st));
    for (int l = 0; l < s->dims.n_layers; ++l) {
      const qcf_layer_weights& w = s->layers[l];
      __nv_bfloat16* kc = static_cast<__nv_bfloat16*>(k_cache[l]);
      __nv_bfloat16* vc = static_cast<__nv_bfloat16*>(v_cache[l]);
      // one row: weight-streaming GEMVs with the RMSNorm folded into their prologue (6 launches per layer, PDL-chained)
      STK_CUDA(ctx, launch_gemv(ctx, s->x, bf(w.w_qkv), bf(w.g_attn), s->dims.rms_eps, nullptr, s->qkv, qkv_n, hid, QCF_EPI_STORE, st));
      // QK-norm + RoPE at position pos; the token's K/V land in cache row pos
      STK_CUDA(ctx, launch_qknorm_rope(ctx, s->qkv, bf(w.g_q), bf(w.g_k), s->rope_table, nullptr, nullptr, 0, pos,
                                       s->dims.rms_eps, 1, s->q_new, kc + pos * kv_row, vc + pos * kv_row, st));
      STK_CUDA(ctx, launch_decode_attn(ctx, s->q_new, kc, vc, pos + 1, s->attn, nullptr, st));
      STK_CUDA(ctx, launch_gemv(ctx, s->attn, bf(w.w_o), nullptr, 0.f, s->x, s->x, hid, L.hq * L.d, QCF_EPI_ADD_RESIDUAL, st));
      STK_CUDA(ctx, launch_gemv(ctx, s->x, bf(w.w_gate_up), bf(w.g_ffn), s->dims.rms_eps, nullptr, s->act, 2 * ffn, hid, QCF_EPI_SWIGLU, st));
      STK_CUDA(ctx, launch_gemv(ctx, s->act, bf(w.w_down), nullptr, 0.f, s->x, s->x, hid, ffn, QCF_EPI_ADD_RESIDUAL, st));
    }
    STK_CUDA(ctx, launch_rmsnorm(s->x, bf(g_final), s->dims.rms_eps, 1, hid, s->h, st));
    STK_CUDA(ctx, launch_lm_head(ctx, bf(w_lm), s->h, vocab, hid, logits + static_cast<size_t>(i) * vocab, tokens_out + i, st));
  }
  return QCF_OK;
}

qcf_status qcf_stack_prefill(qcf_stack* s, const qcf_batch* b, const int32_t* tokens, void* const* k_cache,
                             void* const* v_cache, void* hidden_out, void* stream) {
  if (qcf_status e = check_stack_batch(s, b, "qcf_stack_prefill")) return e;
  qcf_ctx* ctx = s->ctx;
  const int T = b->h_n_ctx[0] + b->h_n_query[0];
  STK_REQUIRE(ctx, tokens && k_cache && v_cache, "qcf_stack_prefill: NULL argument");
  STK_REQUIRE(ctx, T <= s->max_rows && T <= s->max_pos, "qcf_stack_prefill: request exceeds max_rows / max_pos");
  if (T == 0) return QCF_OK;
  cudaStream_t st = static_cast<cudaStream_t>(stream);
  STK_CUDA(ctx, launch_embed_gather(s->embed, tokens, nullptr, nullptr, 0, 0, T, s->dims.hidden, s->x, st));
  for (int l = 0; l < s->dims.n_layers; ++l) {
    STK_REQUIRE(ctx, k_cache[l] && v_cache[l], "qcf_stack_prefill: NULL cache pointer");
    if (qcf_status e = run_layer(s, l, b, nullptr, nullptr, T, -1, s->x, k_cache[l], v_cache[l], nullptr, st)) return e;
  }
  if (hidden_out)
    STK_CUDA(ctx, cudaMemcpyAsync(hidden_out, s->x, static_cast<size_t>(T) * s->dims.hidden * 2, cudaMemcpyDeviceToDevice, st));
  return QCF_OK;
}

qcf_status qcf_stack_fuse(qcf_stack* s, const qcf_batch* mb, const qcf_batch* pb, const qcf_fuse_args* a, void* stream) {
  if (qcf_status e = check_stack_batch(s, mb, "qcf_stack_fuse")) return e;
  if (qcf_status e = check_stack_batch(s, pb, "qcf_stack_fuse")) return e;
  qcf_ctx* ctx = s->ctx;
  const Layout& L = ctx->lay;
  const int n_l = s->dims.n_layers;
  STK_REQUIRE(ctx, a != nullptr, "qcf_stack_fuse: args is NULL");
  STK_REQUIRE(ctx, a->k_pic && a->v_pic && a->k_anchor && a->v_anchor && a->k_fused && a->v_fused && a->tokens &&
                       a->scores && a->sel && a->n_sel,
              "qcf_stack_fuse: NULL argument");
  STK_REQUIRE(ctx, a->ratio >= 0.0 && a->ratio <= 1.0, "qcf_stack_fuse: ratio must be in [0, 1]");
  STK_REQUIRE(ctx, a->n_crit >= 1 && a->crit_layers, "qcf_stack_fuse: at least one critical layer is needed");
  for (int i = 0; i < a->n_crit; ++i)
    STK_REQUIRE(ctx, a->crit_layers[i] >= 0 && a->crit_layers[i] < n_l && (i == 0 || a->crit_layers[i] > a->crit_layers[i - 1]),
                "qcf_stack_fuse: crit_layers must be ascending layer indices");
  const int N = mb->h_n_ctx[0], Lq = mb->h_n_query[0];
  STK_REQUIRE(ctx, pb->h_n_query[0] == Lq, "qcf_stack_fuse: probe batch must carry the same query length");
  STK_REQUIRE(ctx, a->pool_rows >= 0 && a->anchor_rows >= 0 && a->pool_rows <= s->max_pool_rows &&
                       a->anchor_rows <= s->max_pool_rows && static_cast<size_t>(pb->t_stride) <= s->probe_rows,
              "qcf_stack_fuse: pools exceed max_pool_rows of qcf_stack_create");
  STK_REQUIRE(ctx, mb->pool_row_end <= a->pool_rows, "qcf_stack_fuse: a chunk of the main batch lies outside pool_rows");
  STK_REQUIRE(ctx, pb->pool_row_end <= a->anchor_rows, "qcf_stack_fuse: a chunk of the probe batch lies outside anchor_rows");
  // |P| is fixed on the host: floor(rho N).  With stages == 2 the caller's sel / n_sel must hold exactly that many rows
  // (include/qcf.h); the row count of every stage-2 kernel is derived from it.
  const int k_sel = qcf_n_select(N, a->ratio);
  const int n_rows = k_sel + Lq;
  STK_REQUIRE(ctx, n_rows <= s->max_rows && Lq <= s->max_rows && N + Lq <= s->max_pos,
              "qcf_stack_fuse: request exceeds max_rows / max_pos of qcf_stack_create");
  const int l_max = a->crit_layers[a->n_crit - 1];
  STK_REQUIRE(ctx, a->stages >= 0 && a->stages <= 3, "qcf_stack_fuse: stages must be 0..3");
  const bool do1 = a->stages == 0 || (a->stages & 1), do2 = a->stages == 0 || (a->stages & 2);
  cudaStream_t cs = static_cast<cudaStream_t>(stream);
  cudaStream_t ls = a->overlap ? s->loader : cs;
  // K of the critical layers (the only FULL-context tensors stage 1 needs, Eq. 18) travels on its own stream from t = 0:
  // on the main loader it would queue behind anchor jobs that are gated on the probe's progress and arrive at the very
  // end of stage 1 with nothing left to hide it.  (With the bandwidth emulation the link is one serial resource.)
  cudaStream_t ls2 = (a->overlap && !(a->load_gbps > 0.0)) ? s->loader2 : ls;
  const size_t kv_row = static_cast<size_t>(L.hkv) * L.d * 2;
  auto is_crit = [&](int l) { return std::find(a->crit_layers, a->crit_layers + a->n_crit, l) != a->crit_layers + a->n_crit; };
  const int slot_pic0 = l_max + 1;                       // event slot of PIC layer l = slot_pic0 + l; anchor layer l = l
  int ring = 0;

  STK_CUDA(ctx, cudaEventRecord(s->ev_fork, cs));
  if (ls != cs) STK_CUDA(ctx, cudaStreamWaitEvent(ls, s->ev_fork, 0));
  if (ls2 != ls) STK_CUDA(ctx, cudaStreamWaitEvent(ls2, s->ev_fork, 0));

  // Loader jobs, in the order the pipeline consumes them.  The staging buffer of a job is read by the stitch kernel
  // issued right behind it on the same stream, so ring reuse needs no cross-stream wait; destinations are per layer.
  STK_REQUIRE(ctx, a->load_gbps >= 0.0, "qcf_stack_fuse: load_gbps must be >= 0");
  // bandwidth emulation (load_gbps > 0): stamp before a job's copies, hold the loader until bytes / load_gbps have passed
  auto throttle_begin = [&]() -> cudaError_t { return a->load_gbps > 0.0 ? launch_stamp(s->load_t0, ls) : cudaSuccess; };
  auto throttle_end = [&](size_t bytes) -> cudaError_t {
    if (!(a->load_gbps > 0.0)) return cudaSuccess;
    return launch_hold(s->load_t0, static_cast<unsigned long long>(static_cast<double>(bytes) / a->load_gbps), ls);   // B / (GB/s) = ns
  };
  auto load_pic = [&](int l) -> qcf_status {
    STK_REQUIRE(ctx, a->k_pic[l] && a->v_pic[l] && a->k_fused[l] && a->v_fused[l], "qcf_stack_fuse: NULL pool / cache pointer");
    __nv_bfloat16 *sk = s->stage_k[ring], *sv = s->stage_v[ring];
    ring = (ring + 1) % qcf_stack::kRing;
    STK_CUDA(ctx, throttle_begin());
    STK_CUDA(ctx, cudaMemcpyAsync(sk, a->k_pic[l], a->pool_rows * kv_row, cudaMemcpyDefault, ls));
    STK_CUDA(ctx, cudaMemcpyAsync(sv, a->v_pic[l], a->pool_rows * kv_row, cudaMemcpyDefault, ls));
    STK_CUDA(ctx, throttle_end(2 * a->pool_rows * kv_row));
    if (qcf_status e = qcf_rope_reposition(ctx, mb, sk, sv, a->k_fused[l], a->v_fused[l], ls)) return e;      // a1
    STK_CUDA(ctx, cudaEventRecord(s->ev_ready[slot_pic0 + l], ls));
    return QCF_OK;
  };
  // Critical layers: K alone in stage 1 (scoring reads no V), V stitched later by the stage-2 loader
  int ring2 = 0;
  auto load_pic_k = [&](int l, cudaStream_t st) -> qcf_status {
    STK_REQUIRE(ctx, a->k_pic[l] && a->k_fused[l], "qcf_stack_fuse: NULL pool / cache pointer");
    __nv_bfloat16* sk = st == ls ? s->stage_k[ring] : s->stage_k2[ring2];
    if (st == ls) ring = (ring + 1) % qcf_stack::kRing; else ring2 ^= 1;
    if (st == ls) STK_CUDA(ctx, throttle_begin());
    STK_CUDA(ctx, cudaMemcpyAsync(sk, a->k_pic[l], a->pool_rows * kv_row, cudaMemcpyDefault, st));
    if (st == ls) STK_CUDA(ctx, throttle_end(a->pool_rows * kv_row));
    if (qcf_status e = qcf_rope_reposition(ctx, mb, sk, nullptr, a->k_fused[l], nullptr, st)) return e;         // a1, K only
    STK_CUDA(ctx, cudaEventRecord(s->ev_ready[slot_pic0 + l], st));
    return QCF_OK;
  };
  auto load_pic_v = [&](int l) -> qcf_status {
    STK_REQUIRE(ctx, a->v_pic[l] && a->v_fused[l], "qcf_stack_fuse: NULL pool / cache pointer");
    __nv_bfloat16* sv = s->stage_v[ring];
    ring = (ring + 1) % qcf_stack::kRing;
    STK_CUDA(ctx, throttle_begin());
    STK_CUDA(ctx, cudaMemcpyAsync(sv, a->v_pic[l], a->pool_rows * kv_row, cudaMemcpyDefault, ls));
    STK_CUDA(ctx, throttle_end(a->pool_rows * kv_row));
    if (qcf_status e = qcf_rope_reposition(ctx, mb, nullptr, sv, nullptr, a->v_fused[l], ls)) return e;         // V stitch
    STK_CUDA(ctx, cudaEventRecord(s->ev_ready[slot_pic0 + l], ls));      // re-recorded: stage 2 waits for K (earlier) and V
    return QCF_OK;
  };
  // Two-stream mode: the transfer stream ls2 carries pure copies, in the order stage 1 consumes them and never gated by
  // the probe's progress except through arena space: anchor rows of layer j land in arena slot j % n_aslots (its previous
  // tenant, layer j - n_aslots, must have been stitched), K of a critical layer follows its anchors.  The stitches stay
  // on ls, gated by the copy and by the probe cache they write.
  const int n_aslots = a->anchor_rows > 0
                           ? static_cast<int>(std::min<int64_t>(l_max + 1, qcf_stack::kArena * s->max_pool_rows / a->anchor_rows))
                           : l_max + 1;
  int next_copy = 0;
  auto issue_copies = [&](int upto) -> qcf_status {          // anchor (and critical-K) transfers of layers < = upto
    for (; ls2 != ls && next_copy <= std::min(upto, l_max); ++next_copy) {
      const int j = next_copy;
      STK_REQUIRE(ctx, a->k_anchor[j] && a->v_anchor[j], "qcf_stack_fuse: NULL anchor pool pointer");
      if (j >= n_aslots) STK_CUDA(ctx, cudaStreamWaitEvent(ls2, s->ev_ready[j - n_aslots], 0));   // that stitch was enqueued earlier
      const size_t off = static_cast<size_t>(j % n_aslots) * a->anchor_rows * kv_row;
      if (a->anchor_rows > 0) {
        STK_CUDA(ctx, cudaMemcpyAsync(reinterpret_cast<char*>(s->arena_k) + off, a->k_anchor[j], a->anchor_rows * kv_row, cudaMemcpyDefault, ls2));
        STK_CUDA(ctx, cudaMemcpyAsync(reinterpret_cast<char*>(s->arena_v) + off, a->v_anchor[j], a->anchor_rows * kv_row, cudaMemcpyDefault, ls2));
      }
      STK_CUDA(ctx, cudaEventRecord(s->ev_copy[j], ls2));
      if (is_crit(j)) if (qcf_status e = load_pic_k(j, ls2)) return e;
    }
    return QCF_OK;
  };
  auto load_anchor = [&](int l) -> qcf_status {
    STK_REQUIRE(ctx, a->k_anchor[l] && a->v_anchor[l], "qcf_stack_fuse: NULL anchor pool pointer");
    if (ls2 != ls) {
      // stitch(l) is enqueued here, so the copies that may overwrite slots stitched up to l can go out now
      const size_t off = static_cast<size_t>(l % n_aslots) * a->anchor_rows * kv_row;
      STK_CUDA(ctx, cudaStreamWaitEvent(ls, s->ev_copy[l], 0));
      if (l >= 2) STK_CUDA(ctx, cudaStreamWaitEvent(ls, s->ev_done[l - 2], 0));                    // probe cache l&1 is free again
      if (qcf_status e = qcf_rope_reposition(ctx, pb, reinterpret_cast<char*>(s->arena_k) + off, reinterpret_cast<char*>(s->arena_v) + off,
                                             s->probe_k[l & 1], s->probe_v[l & 1], ls))
        return e;                                                                                  // a1'
      STK_CUDA(ctx, cudaEventRecord(s->ev_ready[l], ls));
      return issue_copies(l + n_aslots);
    }
    __nv_bfloat16 *sk = s->stage_k[ring], *sv = s->stage_v[ring];
    ring = (ring + 1) % qcf_stack::kRing;
    STK_CUDA(ctx, throttle_begin());
    STK_CUDA(ctx, cudaMemcpyAsync(sk, a->k_anchor[l], a->anchor_rows * kv_row, cudaMemcpyDefault, ls));
    STK_CUDA(ctx, cudaMemcpyAsync(sv, a->v_anchor[l], a->anchor_rows * kv_row, cudaMemcpyDefault, ls));
    STK_CUDA(ctx, throttle_end(2 * a->anchor_rows * kv_row));
    if (l >= 2 && ls != cs) STK_CUDA(ctx, cudaStreamWaitEvent(ls, s->ev_done[l - 2], 0));   // probe cache l&1 is free again
    if (qcf_status e = qcf_rope_reposition(ctx, pb, sk, sv, s->probe_k[l & 1], s->probe_v[l & 1], ls)) return e;   // a1'
    STK_CUDA(ctx, cudaEventRecord(s->ev_ready[l], ls));
    return QCF_OK;
  };

  // ---- stage 1: selective token localization.  Loads are issued one layer ahead of their consumer.
  auto issue_stage1_loads = [&](int l) -> qcf_status {
    if (qcf_status e = load_anchor(l)) return e;
    if (is_crit(l) && ls2 == ls) if (qcf_status e = load_pic_k(l, ls)) return e;
    return QCF_OK;
  };
  if (do1) {
  if (qcf_status e = issue_copies(n_aslots - 1)) return e;
  if (qcf_status e = issue_stage1_loads(0)) return e;
  STK_CUDA(ctx, launch_embed_gather(s->embed, a->tokens, nullptr, nullptr, 0, N, Lq, s->dims.hidden, s->x, cs));
  bool first = true;
  for (int l = 0; l <= l_max; ++l) {
    if (l + 1 <= l_max) if (qcf_status e = issue_stage1_loads(l + 1)) return e;
    if (ls != cs) STK_CUDA(ctx, cudaStreamWaitEvent(cs, s->ev_ready[l], 0));
    if (qcf_status e = run_layer(s, l, pb, s->zero_i32, s->zero_i32, Lq, N, s->x, s->probe_k[l & 1], s->probe_v[l & 1], nullptr, cs))
      return e;
    if (is_crit(l)) {
      if (ls != cs) STK_CUDA(ctx, cudaStreamWaitEvent(cs, s->ev_ready[slot_pic0 + l], 0));
      if (qcf_status e = qcf_score(ctx, mb, s->q_new, a->k_fused[l], a->scores, first ? 0 : 1, cs)) return e;   // Eq. 18 / 20
      first = false;
    }
    STK_CUDA(ctx, cudaEventRecord(s->ev_done[l], cs));
  }
  if (qcf_status e = qcf_select_topk(ctx, mb, a->scores, a->ratio, a->sel, a->n_sel, cs)) return e;               // Eq. 11
  }
  if (!do2) return QCF_OK;
  if (!do1) {
    // stage 2 alone: sel / n_sel come from the caller.  Every row count below is derived from floor(rho N) on the host, so
    // the caller's |P| must match it (not a hot-path mode: one read-back and synchronisation)
    int32_t h_n_sel = -1;
    STK_CUDA(ctx, cudaMemcpyAsync(&h_n_sel, a->n_sel, sizeof(int32_t), cudaMemcpyDeviceToHost, cs));
    STK_CUDA(ctx, cudaStreamSynchronize(cs));
    STK_REQUIRE(ctx, h_n_sel == k_sel, "qcf_stack_fuse: stages == 2 needs n_sel[0] == qcf_n_select(N, ratio)");
  }

  // ---- stage 2: pipeline cache fusion.  The loader runs ahead through all remaining layers
  // (every layer has its own destination cache); the compute stream consumes them in order.
  for (int l = 0; l < n_l; ++l)
    if (qcf_status e = (!do1 || !is_crit(l)) ? load_pic(l) : load_pic_v(l)) return e;   // critical layers: K is in place since stage 1
  STK_CUDA(ctx, launch_embed_gather(s->embed, a->tokens, a->sel, a->n_sel, N, 0, n_rows, s->dims.hidden, s->x, cs));
  for (int l = 0; l < n_l; ++l) {
    if (ls != cs) STK_CUDA(ctx, cudaStreamWaitEvent(cs, s->ev_ready[slot_pic0 + l], 0));
    if (qcf_status e = run_layer(s, l, mb, a->sel, a->n_sel, n_rows, -1, s->x, a->k_fused[l], a->v_fused[l], nullptr, cs)) return e;
  }
  if (a->hidden_out)
    STK_CUDA(ctx, cudaMemcpyAsync(a->hidden_out, s->x, static_cast<size_t>(n_rows) * s->dims.hidden * 2, cudaMemcpyDeviceToDevice, cs));
  return QCF_OK;
}

}  // extern "C"
