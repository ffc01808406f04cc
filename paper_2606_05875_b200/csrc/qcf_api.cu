// C ABI of libqcf (include/qcf.h): context / batch lifetime, host-side argument validation, stage chaining.
// Everything that touches tensor data runs in the CUDA kernels of the sibling translation units.
#include <algorithm>
#include <cmath>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <new>
#include <string>
#include <vector>

#include "qcf_internal.cuh"

using namespace qcf;

namespace {

thread_local std::string g_create_err;

struct DevBuf {
  void* p = nullptr;
  size_t bytes = 0;
  cudaError_t reserve(size_t n) {
    if (n <= bytes) return cudaSuccess;
    if (p) cudaFree(p);
    p = nullptr; bytes = 0;
    cudaError_t e = cudaMalloc(&p, n);
    if (e == cudaSuccess) bytes = n;
    return e;
  }
  void release() { if (p) cudaFree(p); p = nullptr; bytes = 0; }
};

}  // namespace

namespace qcf {
qcf_status set_error(const qcf_ctx* ctx, qcf_status st, const std::string& msg) {
  if (ctx) ctx->err = msg; else g_create_err = msg;
  return st;
}
}  // namespace qcf

// Device staging buffers of qcf_layer_step_host (allocated on first use, kept by the ctx).
struct HostStage {
  DevBuf k_pool, v_pool, k_f, v_f, q_probe, scores, sel, n_sel, q_new, k_new, v_new, out, lse;
  void release_all() {
    for (DevBuf* d : {&k_pool, &v_pool, &k_f, &v_f, &q_probe, &scores, &sel, &n_sel, &q_new, &k_new, &v_new, &out, &lse})
      d->release();
  }
};

namespace {

qcf_status fail(const qcf_ctx* ctx, qcf_status st, const std::string& msg) { return qcf::set_error(ctx, st, msg); }
qcf_status cuda_fail(const qcf_ctx* ctx, cudaError_t e, const char* what) {
  return fail(ctx, QCF_ERR_CUDA, std::string(what) + ": " + cudaGetErrorString(e));
}

#define QCF_CUDA(ctx, call)                                       \
  do {                                                            \
    cudaError_t e__ = (call);                                     \
    if (e__ != cudaSuccess) return cuda_fail(ctx, e__, #call);    \
  } while (0)

#define QCF_REQUIRE(ctx, cond, msg)                                      \
  do {                                                                   \
    if (!(cond)) return fail(ctx, QCF_ERR_INVALID_ARG, std::string(msg)); \
  } while (0)

inline bool aligned16(const void* p) { return (reinterpret_cast<uintptr_t>(p) & 15u) == 0; }

qcf_status check_ctx_batch(qcf_ctx* ctx, const qcf_batch* b) {
  if (!ctx) return fail(nullptr, QCF_ERR_INVALID_ARG, "ctx is NULL");
  QCF_REQUIRE(ctx, b != nullptr, "batch is NULL");
  QCF_REQUIRE(ctx, b->ctx == ctx, "batch was created on a different ctx");
  return QCF_OK;
}

}  // namespace

extern "C" {

const char* qcf_version(void) { return "qcf 0.1 (sm_100a)"; }

const char* qcf_last_error(const qcf_ctx* ctx) { return ctx ? ctx->err.c_str() : g_create_err.c_str(); }

int32_t qcf_n_select(int32_t n_ctx, double ratio) {
  if (n_ctx < 0 || !(ratio >= 0.0) || !(ratio <= 1.0)) return -1;
  return static_cast<int32_t>(std::floor(ratio * static_cast<double>(n_ctx) + 1e-6));
}

qcf_status qcf_create(qcf_ctx** out, const qcf_layout* lay, int32_t max_batch, int32_t max_ctx, int32_t max_query) {
  if (!out) return fail(nullptr, QCF_ERR_INVALID_ARG, "out is NULL");
  *out = nullptr;
  if (!lay) return fail(nullptr, QCF_ERR_INVALID_ARG, "layout is NULL");
  if (max_batch < 1 || max_ctx < 1 || max_query < 0)
    return fail(nullptr, QCF_ERR_INVALID_ARG, "max_batch, max_ctx must be >= 1 and max_query >= 0");
  if (lay->n_q_heads < 1 || lay->n_kv_heads < 1 || lay->n_q_heads % lay->n_kv_heads != 0)
    return fail(nullptr, QCF_ERR_UNSUPPORTED, "n_kv_heads must divide n_q_heads");
  if (lay->head_dim != 64 && lay->head_dim != 128)
    return fail(nullptr, QCF_ERR_UNSUPPORTED, "head_dim must be 64 or 128");
  const int g = lay->n_q_heads / lay->n_kv_heads;
  if (!(g == 1 || g == 2 || g == 4 || g == 8 || g == 16))
    return fail(nullptr, QCF_ERR_UNSUPPORTED, "group size Hq/Hkv must be 1, 2, 4, 8 or 16");
  if (lay->n_kv_heads * lay->head_dim > 8192)
    return fail(nullptr, QCF_ERR_UNSUPPORTED, "Hkv * head_dim must be <= 8192");
  if (static_cast<long long>(max_query) * g > 8192)
    return fail(nullptr, QCF_ERR_UNSUPPORTED, "max_query * (Hq / Hkv) must be <= 8192 (query rows per kv-head kept in shared memory by qcf_score)");
  if (!(lay->rope_theta > 1.0f)) return fail(nullptr, QCF_ERR_INVALID_ARG, "rope_theta must be > 1");
  if (!(lay->softmax_scale >= 0.0f)) return fail(nullptr, QCF_ERR_INVALID_ARG, "softmax_scale must be >= 0");

  int dev = 0;
  cudaError_t e = cudaGetDevice(&dev);
  if (e != cudaSuccess) return fail(nullptr, QCF_ERR_UNSUPPORTED, std::string("no CUDA device: ") + cudaGetErrorString(e));
  cudaDeviceProp prop;
  e = cudaGetDeviceProperties(&prop, dev);
  if (e != cudaSuccess) return cuda_fail(nullptr, e, "cudaGetDeviceProperties");
  if (prop.major != 10)
    return fail(nullptr, QCF_ERR_UNSUPPORTED,
                "device is sm_" + std::to_string(prop.major * 10 + prop.minor) + "; this library is built for sm_100a only");

  qcf_ctx* c = new (std::nothrow) qcf_ctx();
  if (!c) return fail(nullptr, QCF_ERR_WORKSPACE, "out of host memory");
  c->lay = Layout{lay->n_q_heads, lay->n_kv_heads, lay->head_dim, g, lay->rope_theta,
                  lay->softmax_scale > 0.f ? lay->softmax_scale : 1.0f / std::sqrt(static_cast<float>(lay->head_dim))};
  c->device = dev;
  c->n_sm = prop.multiProcessorCount;
  c->max_batch = max_batch; c->max_ctx = max_ctx; c->max_query = max_query;
  c->stats_m = c->stats_l = c->score_part = c->score_lse = nullptr;
  c->score_row_ctr = nullptr;
  c->counters = nullptr;
  c->dec_part_o = c->dec_part_ml = nullptr; c->dec_counters = nullptr;
  c->stage = nullptr;
  c->pdl = 1; c->gemm_mt = 0; c->attn_cluster = 0;
  c->exch_rank = 0; c->exch_world = 1; c->exch_slot_elems = 0; c->exch_peers = nullptr; c->exch_epoch = 0;
  c->exch_sel_epoch[0] = c->exch_sel_epoch[1] = 0;
  c->ratio_hint = 0.3;
  c->head_shards = 1;
  c->profiling = 0; c->ev_valid = false;
  c->ev_ring = nullptr; c->ev_count = 0; c->ev = nullptr;

  const size_t stats_n = static_cast<size_t>(max_batch) * lay->n_q_heads * (max_query > 0 ? max_query : 1) * kScoreSplitsMax;
  const size_t part_n = static_cast<size_t>(max_batch) * lay->n_kv_heads * max_ctx;
  const size_t row_ctr_n = static_cast<size_t>(max_batch) * lay->n_kv_heads * ((static_cast<size_t>(max_query) * g + 127) / 128 + 1);
  c->n_counters = static_cast<size_t>(max_batch) * ((max_ctx + 63) / 64) + 64;
  bool ok = cudaMalloc(&c->stats_m, stats_n * sizeof(float)) == cudaSuccess &&
            cudaMalloc(&c->stats_l, stats_n * sizeof(float)) == cudaSuccess &&
            cudaMalloc(&c->score_part, part_n * sizeof(float)) == cudaSuccess &&
            cudaMalloc(&c->score_lse, stats_n / kScoreSplitsMax * sizeof(float)) == cudaSuccess &&
            cudaMalloc(&c->score_row_ctr, row_ctr_n * sizeof(unsigned int)) == cudaSuccess &&
            cudaMemset(c->score_row_ctr, 0, row_ctr_n * sizeof(unsigned int)) == cudaSuccess &&
            cudaMalloc(&c->counters, c->n_counters * sizeof(unsigned int)) == cudaSuccess &&
            cudaMemset(c->counters, 0, c->n_counters * sizeof(unsigned int)) == cudaSuccess &&
            cudaMalloc(&c->dec_part_o, static_cast<size_t>(lay->n_q_heads) * kDecodeSplitsMax * lay->head_dim * sizeof(float)) == cudaSuccess &&
            cudaMalloc(&c->dec_part_ml, static_cast<size_t>(lay->n_q_heads) * kDecodeSplitsMax * 2 * sizeof(float)) == cudaSuccess &&
            cudaMalloc(&c->dec_counters, static_cast<size_t>(lay->n_kv_heads) * sizeof(unsigned int)) == cudaSuccess &&
            cudaMemset(c->dec_counters, 0, static_cast<size_t>(lay->n_kv_heads) * sizeof(unsigned int)) == cudaSuccess;
  if (!ok) {
    const cudaError_t le = cudaGetLastError();
    qcf_destroy(c);
    return fail(nullptr, QCF_ERR_WORKSPACE, std::string("workspace allocation failed: ") + cudaGetErrorString(le));
  }
  *out = c;
  return QCF_OK;
}

void qcf_destroy(qcf_ctx* c) {
  if (!c) return;
  cudaFree(c->stats_m); cudaFree(c->stats_l); cudaFree(c->score_part); cudaFree(c->counters);
  cudaFree(c->score_lse); cudaFree(c->score_row_ctr);
  cudaFree(c->dec_part_o); cudaFree(c->dec_part_ml); cudaFree(c->dec_counters);
  cudaFree(c->exch_peers);
  if (c->ev_ring) {
    for (int i = 0; i < qcf_ctx::kEvRing; ++i)
      for (int j = 0; j < 6; ++j) if (c->ev_ring[i][j]) cudaEventDestroy(c->ev_ring[i][j]);
    delete[] c->ev_ring;
  }
  if (c->stage) { c->stage->release_all(); delete c->stage; }
  delete c;
}

qcf_status qcf_batch_create(qcf_ctx* ctx, const qcf_request* reqs, int32_t batch, qcf_batch** out) {
  if (!ctx) return fail(nullptr, QCF_ERR_INVALID_ARG, "ctx is NULL");
  QCF_REQUIRE(ctx, out != nullptr, "out is NULL");
  *out = nullptr;
  QCF_REQUIRE(ctx, batch >= 0, "batch must be >= 0");
  QCF_REQUIRE(ctx, batch == 0 || reqs != nullptr, "reqs is NULL");
  if (batch > ctx->max_batch) return fail(ctx, QCF_ERR_WORKSPACE, "batch exceeds max_batch of qcf_create");

  const int half = ctx->lay.d / 2;
  std::vector<int32_t> n_ctx(batch), n_query(batch), c_req, c_off, c_rot, c_len, c_blk;
  std::vector<int64_t> c_row;
  std::vector<float> rot;      // (cos, sin) interleaved
  int64_t total_ctx = 0, pool_row_end = 0;
  int32_t t_stride = 0, n_stride = 0, q_stride = 0;
  // inv_freq_j = theta^(-2j/d) in double (reading (a))
  std::vector<double> inv_freq(half);
  for (int j = 0; j < half; ++j)
    inv_freq[j] = std::pow(static_cast<double>(ctx->lay.theta), -2.0 * j / static_cast<double>(ctx->lay.d));
  c_blk.push_back(0);
  for (int b = 0; b < batch; ++b) {
    const qcf_request& r = reqs[b];
    QCF_REQUIRE(ctx, r.n_chunks >= 0 && r.n_query >= 0, "n_chunks and n_query must be >= 0");
    QCF_REQUIRE(ctx, r.n_chunks == 0 || (r.chunk_len && r.chunk_row), "chunk_len / chunk_row is NULL");
    int64_t off = 0;
    for (int i = 0; i < r.n_chunks; ++i) {
      QCF_REQUIRE(ctx, r.chunk_len[i] >= 0, "chunk_len must be >= 0");
      QCF_REQUIRE(ctx, r.chunk_row[i] >= 0, "chunk_row must be >= 0");
      QCF_REQUIRE(ctx, !r.chunk_pos || r.chunk_pos[i] >= 0, "chunk_pos must be >= 0");
      if (off + r.chunk_len[i] > ctx->max_ctx) return fail(ctx, QCF_ERR_WORKSPACE, "context length exceeds max_ctx of qcf_create");
      if (r.chunk_len[i] == 0) continue;
      c_req.push_back(b);
      c_off.push_back(static_cast<int32_t>(off));
      const int64_t rot_pos = r.chunk_pos ? r.chunk_pos[i] : off;     // Eq. 4 (off_i) or Eq. 15-16 (anchors keep off_i of c_i)
      c_rot.push_back(static_cast<int32_t>(rot_pos));
      c_len.push_back(r.chunk_len[i]);
      c_row.push_back(r.chunk_row[i]);
      pool_row_end = std::max<int64_t>(pool_row_end, r.chunk_row[i] + r.chunk_len[i]);
      c_blk.push_back(c_blk.back() + (r.chunk_len[i] + kRepoRows - 1) / kRepoRows);
      for (int j = 0; j < half; ++j) {
        const double phi = static_cast<double>(rot_pos) * inv_freq[j];
        rot.push_back(static_cast<float>(std::cos(phi)));
        rot.push_back(static_cast<float>(std::sin(phi)));
      }
      off += r.chunk_len[i];
    }
    if (r.n_query > ctx->max_query) return fail(ctx, QCF_ERR_WORKSPACE, "query length exceeds max_query of qcf_create");
    n_ctx[b] = static_cast<int32_t>(off);
    n_query[b] = r.n_query;
    total_ctx += off;
    t_stride = std::max<int32_t>(t_stride, static_cast<int32_t>(off) + r.n_query);
    n_stride = std::max<int32_t>(n_stride, static_cast<int32_t>(off));
    q_stride = std::max<int32_t>(q_stride, r.n_query);
  }
  const int n_chunks = static_cast<int>(c_req.size());

  qcf_batch* qb = new (std::nothrow) qcf_batch();
  if (!qb) return fail(ctx, QCF_ERR_WORKSPACE, "out of host memory");
  qb->ctx = ctx; qb->blob = nullptr; qb->h_pool_iv = nullptr; qb->n_pool_iv = 0; qb->pool_rows_touched = 0;
  qb->batch = batch; qb->n_chunks = n_chunks;
  qb->t_stride = t_stride; qb->n_stride = n_stride; qb->q_stride = q_stride;
  qb->max_ctx = n_stride; qb->max_query = q_stride; qb->total_ctx = total_ctx;
  qb->repo_blocks = c_blk.back();
  qb->pool_row_end = pool_row_end;
  // union of the pool row ranges the batch reads (chunks shared by requests or adjacent in the pool merge): what a host-side
  // step has to upload
  {
    std::vector<std::pair<int64_t, int64_t>> iv;
    for (int c = 0; c < n_chunks; ++c) iv.emplace_back(c_row[c], c_row[c] + c_len[c]);
    std::sort(iv.begin(), iv.end());
    std::vector<int64_t> flat;
    int64_t touched = 0;
    for (size_t i = 0; i < iv.size();) {
      int64_t lo = iv[i].first, hi = iv[i].second;
      size_t j = i + 1;
      while (j < iv.size() && iv[j].first <= hi) { hi = std::max(hi, iv[j].second); ++j; }
      flat.push_back(lo); flat.push_back(hi - lo);
      touched += hi - lo;
      i = j;
    }
    qb->n_pool_iv = static_cast<int32_t>(flat.size() / 2);
    qb->pool_rows_touched = touched;
    qb->h_pool_iv = static_cast<int64_t*>(std::malloc(sizeof(int64_t) * (flat.empty() ? 1 : flat.size())));
    if (!qb->h_pool_iv) { qcf_batch_destroy(qb); return fail(ctx, QCF_ERR_WORKSPACE, "qcf_batch_create: out of host memory"); }
    if (!flat.empty()) std::memcpy(qb->h_pool_iv, flat.data(), sizeof(int64_t) * flat.size());
  }
  qb->h_n_ctx = static_cast<int32_t*>(std::malloc(sizeof(int32_t) * (batch > 0 ? batch : 1)));
  qb->h_n_query = static_cast<int32_t*>(std::malloc(sizeof(int32_t) * (batch > 0 ? batch : 1)));
  if (!qb->h_n_ctx || !qb->h_n_query) { qcf_batch_destroy(qb); return fail(ctx, QCF_ERR_WORKSPACE, "qcf_batch_create: out of host memory"); }
  if (batch > 0) {
    std::memcpy(qb->h_n_ctx, n_ctx.data(), sizeof(int32_t) * batch);
    std::memcpy(qb->h_n_query, n_query.data(), sizeof(int32_t) * batch);
  }

  // one device blob: [n_ctx | n_query | chunk_req | chunk_off | chunk_len | chunk_blk | pad | chunk_row | rot | chunk_rot]
  auto up = [](size_t x, size_t a) { return (x + a - 1) / a * a; };
  size_t o_nctx = 0, o_nq = up(o_nctx + sizeof(int32_t) * batch, 16);
  size_t o_req = up(o_nq + sizeof(int32_t) * batch, 16), o_off = up(o_req + sizeof(int32_t) * n_chunks, 16);
  size_t o_len = up(o_off + sizeof(int32_t) * n_chunks, 16), o_blk = up(o_len + sizeof(int32_t) * n_chunks, 16);
  size_t o_row = up(o_blk + sizeof(int32_t) * (n_chunks + 1), 16), o_rot = up(o_row + sizeof(int64_t) * n_chunks, 16);
  size_t o_crot = up(o_rot + sizeof(float) * rot.size(), 16);
  size_t o_item = up(o_crot + sizeof(int32_t) * n_chunks, 32);
  std::vector<RepoItem> items;
  items.reserve(c_blk.back());
  for (int c = 0; c < n_chunks; ++c)
    for (int r0 = 0; r0 < c_len[c]; r0 += kRepoRows)
      items.push_back(RepoItem{c_row[c] + r0, static_cast<int64_t>(c_req[c]) * t_stride + c_off[c] + r0,
                               std::min<int32_t>(kRepoRows, c_len[c] - r0), c, c_rot[c] == 0 ? 1 : 0, 0});
  size_t total = up(o_item + sizeof(RepoItem) * items.size(), 16) + 16;
  std::vector<unsigned char> host(total, 0);
  if (batch > 0) {
    std::memcpy(host.data() + o_nctx, n_ctx.data(), sizeof(int32_t) * batch);
    std::memcpy(host.data() + o_nq, n_query.data(), sizeof(int32_t) * batch);
  }
  if (n_chunks > 0) {
    std::memcpy(host.data() + o_req, c_req.data(), sizeof(int32_t) * n_chunks);
    std::memcpy(host.data() + o_off, c_off.data(), sizeof(int32_t) * n_chunks);
    std::memcpy(host.data() + o_len, c_len.data(), sizeof(int32_t) * n_chunks);
    std::memcpy(host.data() + o_row, c_row.data(), sizeof(int64_t) * n_chunks);
    std::memcpy(host.data() + o_rot, rot.data(), sizeof(float) * rot.size());
    std::memcpy(host.data() + o_crot, c_rot.data(), sizeof(int32_t) * n_chunks);
  }
  std::memcpy(host.data() + o_blk, c_blk.data(), sizeof(int32_t) * (n_chunks + 1));
  if (!items.empty()) std::memcpy(host.data() + o_item, items.data(), sizeof(RepoItem) * items.size());
  cudaError_t e = cudaMalloc(&qb->blob, total);
  if (e == cudaSuccess) e = cudaMemcpy(qb->blob, host.data(), total, cudaMemcpyHostToDevice);
  if (e != cudaSuccess) {
    qcf_batch_destroy(qb);
    return cuda_fail(ctx, e, "batch upload");
  }
  unsigned char* d = static_cast<unsigned char*>(qb->blob);
  BatchDev& bd = qb->dev;
  bd.batch = batch; bd.n_chunks = n_chunks;
  bd.t_stride = t_stride; bd.n_stride = n_stride; bd.q_stride = q_stride;
  bd.n_ctx = reinterpret_cast<const int32_t*>(d + o_nctx);
  bd.n_query = reinterpret_cast<const int32_t*>(d + o_nq);
  bd.chunk_req = reinterpret_cast<const int32_t*>(d + o_req);
  bd.chunk_off = reinterpret_cast<const int32_t*>(d + o_off);
  bd.chunk_len = reinterpret_cast<const int32_t*>(d + o_len);
  bd.chunk_blk = reinterpret_cast<const int32_t*>(d + o_blk);
  bd.chunk_row = reinterpret_cast<const int64_t*>(d + o_row);
  bd.rot = reinterpret_cast<const float2*>(d + o_rot);
  bd.chunk_rot = reinterpret_cast<const int32_t*>(d + o_crot);
  bd.repo_items = reinterpret_cast<const int4*>(d + o_item);
  *out = qb;
  return QCF_OK;
}

void qcf_batch_destroy(qcf_batch* b) {
  if (!b) return;
  if (b->blob) cudaFree(b->blob);
  std::free(b->h_n_ctx);
  std::free(b->h_n_query);
  std::free(b->h_pool_iv);
  delete b;
}

qcf_status qcf_batch_get_info(const qcf_batch* b, qcf_batch_info* info) {
  if (!b || !info) return QCF_ERR_INVALID_ARG;
  info->batch = b->batch; info->t_stride = b->t_stride; info->n_stride = b->n_stride; info->q_stride = b->q_stride;
  info->total_ctx = b->total_ctx;
  info->pool_rows_touched = b->pool_rows_touched;
  return QCF_OK;
}

// ------------------------------------------------------------------------------------------------ stages

qcf_status qcf_rope_reposition(qcf_ctx* ctx, const qcf_batch* b, const void* k_pool, const void* v_pool, void* k_fused,
                               void* v_fused, void* stream) {
  if (qcf_status st = check_ctx_batch(ctx, b)) return st;
  if (b->total_ctx == 0) return QCF_OK;
  QCF_REQUIRE(ctx, (k_pool && k_fused) || (v_pool && v_fused), "qcf_rope_reposition: NULL tensor pointer");
  QCF_REQUIRE(ctx, (v_pool == nullptr) == (v_fused == nullptr) && (k_pool == nullptr) == (k_fused == nullptr),
              "qcf_rope_reposition: a pool and its cache must both be given or both be NULL");
  QCF_REQUIRE(ctx, aligned16(k_pool) && aligned16(v_pool) && aligned16(k_fused) && aligned16(v_fused),
              "qcf_rope_reposition: pointers must be 16-byte aligned");
  QCF_CUDA(ctx, launch_reposition(ctx, b, static_cast<const __nv_bfloat16*>(k_pool),
                                  static_cast<const __nv_bfloat16*>(v_pool), static_cast<__nv_bfloat16*>(k_fused),
                                  static_cast<__nv_bfloat16*>(v_fused), static_cast<cudaStream_t>(stream)));
  return QCF_OK;
}

qcf_status qcf_score(qcf_ctx* ctx, const qcf_batch* b, const void* q_probe, const void* k_fused, float* scores,
                     int32_t accumulate, void* stream) {
  if (qcf_status st = check_ctx_batch(ctx, b)) return st;
  if (b->total_ctx == 0) return QCF_OK;
  QCF_REQUIRE(ctx, k_fused && scores, "qcf_score: NULL tensor pointer");
  QCF_REQUIRE(ctx, q_probe || b->q_stride == 0, "qcf_score: q_probe is NULL");
  QCF_REQUIRE(ctx, aligned16(q_probe) && aligned16(k_fused), "qcf_score: pointers must be 16-byte aligned");
  cudaStream_t s = static_cast<cudaStream_t>(stream);
  if (ctx->exch_world > 1) {
    QCF_REQUIRE(ctx, static_cast<long long>(b->batch) * b->n_stride <= ctx->exch_slot_elems,
                "qcf_score: the batch does not fit a slot of the score exchange buffers");
    // This call is epoch e = exch_epoch + 1 and overwrites the slot set of epoch e - 2.  Every peer must have finished the
    // selections that read it: the newest selection epoch <= e - 2 of the (common) call sequence must be acknowledged.
    const unsigned int e = ctx->exch_epoch + 1;
    const unsigned int need = ctx->exch_sel_epoch[0] + 2 <= e ? ctx->exch_sel_epoch[0] : ctx->exch_sel_epoch[1];
    if (need > 0) QCF_CUDA(ctx, launch_exchange_wait(ctx, need, s));
    ctx->exch_epoch = e;                       // read by the two launches below; taken back if either fails
  }
  cudaError_t err = launch_score(ctx, b, static_cast<const __nv_bfloat16*>(q_probe), static_cast<const __nv_bfloat16*>(k_fused),
                                 scores, accumulate != 0, s);
  if (err == cudaSuccess && ctx->exch_world > 1) err = launch_exchange_flags(ctx, s);
  if (err != cudaSuccess) {
    if (ctx->exch_world > 1) ctx->exch_epoch--;
    return cuda_fail(ctx, err, "qcf_score");
  }
  return QCF_OK;
}

qcf_status qcf_select_topk(qcf_ctx* ctx, const qcf_batch* b, const float* scores, double ratio, int32_t* sel,
                           int32_t* n_sel, void* stream) {
  if (qcf_status st = check_ctx_batch(ctx, b)) return st;
  QCF_REQUIRE(ctx, ratio >= 0.0 && ratio <= 1.0, "qcf_select_topk: ratio must be in [0, 1]");
  if (b->batch == 0) return QCF_OK;
  QCF_REQUIRE(ctx, n_sel != nullptr, "qcf_select_topk: n_sel is NULL");
  QCF_REQUIRE(ctx, ((scores || ctx->exch_world > 1) && sel) || b->n_stride == 0, "qcf_select_topk: NULL tensor pointer");
  ctx->ratio_hint = ratio;
  QCF_CUDA(ctx, launch_topk(ctx, b, scores, ratio, sel, n_sel, static_cast<cudaStream_t>(stream)));
  if (ctx->exch_world > 1) {
    // tell the peers that this rank is done reading the slots of this epoch (they may overwrite them two epochs on)
    QCF_CUDA(ctx, launch_exchange_ack(ctx, static_cast<cudaStream_t>(stream)));
    if (ctx->exch_sel_epoch[0] != ctx->exch_epoch) {
      ctx->exch_sel_epoch[1] = ctx->exch_sel_epoch[0];
      ctx->exch_sel_epoch[0] = ctx->exch_epoch;
    }
  }
  return QCF_OK;
}

qcf_status qcf_anchor_rank(qcf_ctx* ctx, const qcf_batch* b, const void* k_pool, int32_t rule, double r_a, float* scores,
                           int32_t accumulate, int32_t select_now, int32_t* anchor_idx, int32_t* n_anchor, void* stream) {
  if (qcf_status st = check_ctx_batch(ctx, b)) return st;
  QCF_REQUIRE(ctx, rule == QCF_ANCHOR_SINK || rule == QCF_ANCHOR_KNORM, "qcf_anchor_rank: unknown rule");
  QCF_REQUIRE(ctx, r_a >= 0.0 && r_a <= 1.0, "qcf_anchor_rank: r_a must be in [0, 1]");
  QCF_REQUIRE(ctx, b->n_chunks <= b->batch && b->q_stride == 0, "qcf_anchor_rank: the batch must list one chunk per request and no query");
  if (b->batch == 0) return QCF_OK;
  QCF_REQUIRE(ctx, scores || b->n_stride == 0, "qcf_anchor_rank: scores is NULL");
  QCF_REQUIRE(ctx, rule == QCF_ANCHOR_SINK || k_pool, "qcf_anchor_rank: k_pool is NULL");
  QCF_REQUIRE(ctx, aligned16(k_pool), "qcf_anchor_rank: k_pool must be 16-byte aligned");
  cudaStream_t s = static_cast<cudaStream_t>(stream);
  QCF_CUDA(ctx, launch_anchor_scores(ctx, b, static_cast<const __nv_bfloat16*>(k_pool), rule, accumulate != 0, scores, s));
  if (select_now) {
    QCF_REQUIRE(ctx, n_anchor && (anchor_idx || b->n_stride == 0), "qcf_anchor_rank: NULL output pointer");
    QCF_CUDA(ctx, launch_topk(ctx, b, scores, r_a, anchor_idx, n_anchor, s, /*ceil_mode=*/1));
  }
  return QCF_OK;
}

qcf_status qcf_anchor_gather(qcf_ctx* ctx, const qcf_batch* b, const void* k_pool, const void* v_pool, const int32_t* anchor_idx,
                             const int32_t* n_anchor, void* k_anchor, void* v_anchor, void* stream) {
  if (qcf_status st = check_ctx_batch(ctx, b)) return st;
  QCF_REQUIRE(ctx, b->n_chunks <= b->batch && b->q_stride == 0, "qcf_anchor_gather: the batch must list one chunk per request and no query");
  if (b->batch == 0 || b->n_stride == 0) return QCF_OK;
  QCF_REQUIRE(ctx, anchor_idx && n_anchor, "qcf_anchor_gather: anchor_idx / n_anchor is NULL");
  QCF_REQUIRE(ctx, (k_pool != nullptr) == (k_anchor != nullptr) && (v_pool != nullptr) == (v_anchor != nullptr),
              "qcf_anchor_gather: a pool and its anchor pool must both be given or both be NULL");
  QCF_REQUIRE(ctx, k_pool || v_pool, "qcf_anchor_gather: nothing to gather");
  QCF_REQUIRE(ctx, aligned16(k_pool) && aligned16(v_pool) && aligned16(k_anchor) && aligned16(v_anchor),
              "qcf_anchor_gather: pointers must be 16-byte aligned");
  QCF_CUDA(ctx, launch_anchor_gather(ctx, b, static_cast<const __nv_bfloat16*>(k_pool), static_cast<const __nv_bfloat16*>(v_pool),
                                     anchor_idx, n_anchor, static_cast<__nv_bfloat16*>(k_anchor),
                                     static_cast<__nv_bfloat16*>(v_anchor), static_cast<cudaStream_t>(stream)));
  return QCF_OK;
}

namespace {

// a4 + a5.  q_gather_src != nullptr (the zero-copy host step only): q_new is position-indexed in device-mapped HOST memory;
// its rows R are first gathered into the compact device buffer q_gather_dst, which a5 then reads.
qcf_status recompute_attn_impl(qcf_ctx* ctx, const qcf_batch* b, const int32_t* sel, const int32_t* n_sel,
                               const void* q_new, const void* k_new, const void* v_new, int32_t rows_by_position,
                               void* k_fused, void* v_fused, void* out, float* lse, const void* q_gather_src,
                               void* q_gather_dst, void* stream) {
  if (qcf_status st = check_ctx_batch(ctx, b)) return st;
  if (b->batch == 0 || b->t_stride == 0) return QCF_OK;
  QCF_REQUIRE(ctx, n_sel != nullptr, "qcf_recompute_attn: n_sel is NULL");
  QCF_REQUIRE(ctx, sel || b->n_stride == 0, "qcf_recompute_attn: sel is NULL");
  QCF_REQUIRE(ctx, q_new && k_new && v_new && k_fused && v_fused && out, "qcf_recompute_attn: NULL tensor pointer");
  QCF_REQUIRE(ctx, aligned16(q_new) && aligned16(k_new) && aligned16(v_new) && aligned16(k_fused) &&
                       aligned16(v_fused) && aligned16(out),
              "qcf_recompute_attn: pointers must be 16-byte aligned");
  cudaStream_t s = static_cast<cudaStream_t>(stream);
  static const int32_t kDummy = 0;
  const int32_t* sel_nn = sel ? sel : &kDummy;     // n_stride == 0: never dereferenced (n_sel == 0), must be non-null
  QCF_CUDA(ctx, launch_scatter(ctx, b, sel_nn, n_sel, static_cast<const __nv_bfloat16*>(k_new),
                               static_cast<const __nv_bfloat16*>(v_new), rows_by_position != 0,
                               static_cast<__nv_bfloat16*>(k_fused), static_cast<__nv_bfloat16*>(v_fused), s));
  int q_by_position = rows_by_position != 0;
  if (q_gather_src) {
    // zero-copy host step: the rows R of the host-resident q_new are gathered (bulk copies over PCIe) into a compact device
    // buffer; a5 then reads q compactly while a4 above read k_new / v_new by position
    QCF_CUDA(ctx, launch_gather_rows(ctx, b, sel_nn, n_sel, q_gather_src, q_gather_dst, ctx->lay.hq * ctx->lay.d * 2, s));
    q_new = q_gather_dst;
    q_by_position = 0;
  }
  if (ctx->profiling && ctx->ev_valid) cudaEventRecord(ctx->ev[4], s);
  QCF_CUDA(ctx, launch_attn(ctx, b, sel_nn, n_sel, static_cast<const __nv_bfloat16*>(q_new), q_by_position,
                            static_cast<const __nv_bfloat16*>(k_fused), static_cast<const __nv_bfloat16*>(v_fused),
                            static_cast<__nv_bfloat16*>(out), lse, s));
  return QCF_OK;
}

}  // namespace

qcf_status qcf_recompute_attn(qcf_ctx* ctx, const qcf_batch* b, const int32_t* sel, const int32_t* n_sel,
                              const void* q_new, const void* k_new, const void* v_new, int32_t rows_by_position,
                              void* k_fused, void* v_fused, void* out, float* lse, void* stream) {
  return recompute_attn_impl(ctx, b, sel, n_sel, q_new, k_new, v_new, rows_by_position, k_fused, v_fused, out, lse, nullptr,
                             nullptr, stream);
}

qcf_status qcf_full_prefill_attn(qcf_ctx* ctx, const qcf_batch* b, const void* q, const void* k, const void* v,
                                 void* out, float* lse, void* stream) {
  if (qcf_status st = check_ctx_batch(ctx, b)) return st;
  if (b->batch == 0 || b->t_stride == 0) return QCF_OK;
  QCF_REQUIRE(ctx, q && k && v && out, "qcf_full_prefill_attn: NULL tensor pointer");
  QCF_REQUIRE(ctx, aligned16(q) && aligned16(k) && aligned16(v) && aligned16(out),
              "qcf_full_prefill_attn: pointers must be 16-byte aligned");
  QCF_CUDA(ctx, launch_attn(ctx, b, nullptr, nullptr, static_cast<const __nv_bfloat16*>(q), 1,
                            static_cast<const __nv_bfloat16*>(k), static_cast<const __nv_bfloat16*>(v),
                            static_cast<__nv_bfloat16*>(out), lse, static_cast<cudaStream_t>(stream)));
  return QCF_OK;
}

qcf_status qcf_decode_attn(qcf_ctx* ctx, const void* q, const void* k_cache, const void* v_cache, int32_t n_keys, void* out,
                           float* lse, void* stream) {
  if (!ctx) return fail(nullptr, QCF_ERR_INVALID_ARG, "ctx is NULL");
  QCF_REQUIRE(ctx, n_keys >= 1, "qcf_decode_attn: n_keys must be >= 1 (the token's own K/V row is part of the cache)");
  QCF_REQUIRE(ctx, q && k_cache && v_cache && out, "qcf_decode_attn: NULL tensor pointer");
  QCF_REQUIRE(ctx, aligned16(q) && aligned16(k_cache) && aligned16(v_cache) && aligned16(out),
              "qcf_decode_attn: pointers must be 16-byte aligned");
  QCF_CUDA(ctx, launch_decode_attn(ctx, static_cast<const __nv_bfloat16*>(q), static_cast<const __nv_bfloat16*>(k_cache),
                                   static_cast<const __nv_bfloat16*>(v_cache), n_keys, static_cast<__nv_bfloat16*>(out), lse,
                                   static_cast<cudaStream_t>(stream)));
  return QCF_OK;
}

namespace {

qcf_status layer_step_impl(qcf_ctx* ctx, const qcf_batch* b, const qcf_layer_args* a, const void* q_gather_src,
                           void* q_gather_dst, void* stream) {
  if (qcf_status st = check_ctx_batch(ctx, b)) return st;
  QCF_REQUIRE(ctx, a != nullptr, "qcf_layer_step: args is NULL");
  if (a->select_now) QCF_REQUIRE(ctx, a->ratio >= 0.0 && a->ratio <= 1.0, "qcf_layer_step: ratio must be in [0, 1]");
  cudaStream_t s = static_cast<cudaStream_t>(stream);
  const bool prof = ctx->profiling != 0 && ctx->ev_ring && ctx->ev_count < qcf_ctx::kEvRing;
  ctx->ev_valid = false;
  ctx->ev = prof ? ctx->ev_ring[ctx->ev_count] : nullptr;
  if (prof) cudaEventRecord(ctx->ev[0], s);
  if (qcf_status st = qcf_rope_reposition(ctx, b, a->k_pool, a->v_pool, a->k_fused, a->v_fused, stream)) return st;
  if (prof) cudaEventRecord(ctx->ev[1], s);
  if (a->is_critical_layer)
    if (qcf_status st = qcf_score(ctx, b, a->q_probe, a->k_fused, a->scores, a->accumulate, stream)) return st;
  if (prof) cudaEventRecord(ctx->ev[2], s);
  if (a->select_now)
    if (qcf_status st = qcf_select_topk(ctx, b, a->scores, a->ratio, a->sel, a->n_sel, stream)) return st;
  if (prof) cudaEventRecord(ctx->ev[3], s);
  ctx->ev_valid = prof;      // lets qcf_recompute_attn record ev[4] between a4 and a5
  qcf_status st = recompute_attn_impl(ctx, b, a->sel, a->n_sel, a->q_new, a->k_new, a->v_new, a->rows_by_position,
                                      a->k_fused, a->v_fused, a->out, a->lse, q_gather_src, q_gather_dst, stream);
  if (st) { ctx->ev_valid = false; return st; }
  if (prof) {
    if (b->batch == 0 || b->t_stride == 0) cudaEventRecord(ctx->ev[4], s);
    cudaEventRecord(ctx->ev[5], s);
    ctx->ev_count++;
  }
  ctx->ev_valid = false;
  return QCF_OK;
}

}  // namespace

qcf_status qcf_layer_step(qcf_ctx* ctx, const qcf_batch* b, const qcf_layer_args* a, void* stream) {
  return layer_step_impl(ctx, b, a, nullptr, nullptr, stream);
}

qcf_status qcf_set_head_shards(qcf_ctx* ctx, int32_t n_shards) {
  if (!ctx) return QCF_ERR_INVALID_ARG;
  if (n_shards < 1 || n_shards > 64) return fail(ctx, QCF_ERR_INVALID_ARG, "n_shards must be in [1, 64]");
  ctx->head_shards = n_shards;
  return QCF_OK;
}

qcf_status qcf_debug_set(qcf_ctx* ctx, int32_t knob, int32_t value) {
  if (!ctx) return QCF_ERR_INVALID_ARG;
  switch (knob) {
    case QCF_DEBUG_PDL:
      ctx->pdl = value != 0;
      return QCF_OK;
    case QCF_DEBUG_ATTN_CLUSTER:
      if (!(value == 0 || value == 1 || value == 2 || value == 4)) return fail(ctx, QCF_ERR_INVALID_ARG, "attention cluster size must be 0, 1, 2 or 4");
      ctx->attn_cluster = value;
      return QCF_OK;
    case QCF_DEBUG_GEMM_MT:
      if (value < 0 || value > 2) return fail(ctx, QCF_ERR_INVALID_ARG, "GEMM tile height must be 0, 1 or 2");
      ctx->gemm_mt = value;
      return QCF_OK;
    default:
      return fail(ctx, QCF_ERR_INVALID_ARG, "qcf_debug_set: unknown knob");
  }
}

int64_t qcf_score_exchange_bytes(int32_t n_shards, int64_t slot_elems) {
  if (n_shards < 1 || n_shards > 64 || slot_elems < 0) return -1;
  return static_cast<int64_t>(kExchHeaderElems) * 4 + 2 * static_cast<int64_t>(n_shards) * slot_elems * 4;
}

qcf_status qcf_set_score_exchange(qcf_ctx* ctx, int32_t rank, int32_t n_shards, void* const* peer_bufs, int64_t slot_elems) {
  if (!ctx) return QCF_ERR_INVALID_ARG;
  if (n_shards == 1 || peer_bufs == nullptr) {                  // off
    ctx->exch_world = 1; ctx->exch_rank = 0; ctx->exch_slot_elems = 0;
    return QCF_OK;
  }
  QCF_REQUIRE(ctx, n_shards >= 2 && n_shards <= 64 && rank >= 0 && rank < n_shards, "qcf_set_score_exchange: rank / n_shards out of range");
  QCF_REQUIRE(ctx, slot_elems >= 1, "qcf_set_score_exchange: slot_elems must be >= 1");
  for (int p = 0; p < n_shards; ++p)
    QCF_REQUIRE(ctx, peer_bufs[p] != nullptr && aligned16(peer_bufs[p]), "qcf_set_score_exchange: NULL or misaligned peer buffer");
  if (!ctx->exch_peers) QCF_CUDA(ctx, cudaMalloc(&ctx->exch_peers, 64 * sizeof(float*)));
  for (int p = 0; p < 64; ++p) ctx->exch_peers_host[p] = p < n_shards ? static_cast<float*>(peer_bufs[p]) : nullptr;
  QCF_CUDA(ctx, cudaMemcpy(ctx->exch_peers, ctx->exch_peers_host, 64 * sizeof(float*), cudaMemcpyHostToDevice));
  ctx->exch_rank = rank; ctx->exch_world = n_shards; ctx->exch_slot_elems = slot_elems;
  // Epochs count from 1 and the caller hands over ZEROED buffers: nothing is cleared here, because a faster peer may
  // already have published its first epoch into this rank's buffer by the time this rank gets to this call.
  ctx->exch_epoch = 0;
  ctx->exch_sel_epoch[0] = ctx->exch_sel_epoch[1] = 0;
  return QCF_OK;
}

qcf_status qcf_set_profiling(qcf_ctx* ctx, int32_t enable) {
  if (!ctx) return QCF_ERR_INVALID_ARG;
  if (enable && !ctx->ev_ring) {
    ctx->ev_ring = new (std::nothrow) cudaEvent_t[qcf_ctx::kEvRing][6]();
    if (!ctx->ev_ring) return fail(ctx, QCF_ERR_WORKSPACE, "out of host memory");
    for (int i = 0; i < qcf_ctx::kEvRing; ++i)
      for (int j = 0; j < 6; ++j) QCF_CUDA(ctx, cudaEventCreate(&ctx->ev_ring[i][j]));
  }
  ctx->profiling = enable != 0;
  ctx->ev_count = 0;
  ctx->ev_valid = false;
  return QCF_OK;
}

qcf_status qcf_get_stage_ms(qcf_ctx* ctx, float* ms5) {
  if (!ctx) return QCF_ERR_INVALID_ARG;
  QCF_REQUIRE(ctx, ms5 != nullptr, "ms5 is NULL");
  QCF_REQUIRE(ctx, ctx->ev_ring && ctx->ev_count > 0, "no profiled qcf_layer_step has been issued");
  const int n = ctx->ev_count;
  QCF_CUDA(ctx, cudaEventSynchronize(ctx->ev_ring[n - 1][5]));
  double acc[5] = {0, 0, 0, 0, 0};
  for (int k = 0; k < n; ++k)
    for (int i = 0; i < 5; ++i) {
      float ms = 0.f;
      QCF_CUDA(ctx, cudaEventElapsedTime(&ms, ctx->ev_ring[k][i], ctx->ev_ring[k][i + 1]));
      acc[i] += ms;
    }
  for (int i = 0; i < 5; ++i) ms5[i] = static_cast<float>(acc[i] / n);
  ctx->ev_count = 0;
  return QCF_OK;
}

qcf_status qcf_layer_step_host(qcf_ctx* ctx, const qcf_batch* b, const qcf_layer_args* h, int64_t pool_rows,
                               void* stream) {
  if (qcf_status st = check_ctx_batch(ctx, b)) return st;
  QCF_REQUIRE(ctx, h != nullptr, "qcf_layer_step_host: args is NULL");
  QCF_REQUIRE(ctx, pool_rows >= 0, "qcf_layer_step_host: pool_rows must be >= 0");
  QCF_REQUIRE(ctx, b->pool_row_end <= pool_rows, "qcf_layer_step_host: a chunk of the batch lies outside the pool_rows rows of k_pool / v_pool");
  QCF_REQUIRE(ctx, h->k_pool && h->v_pool && h->q_new && h->k_new && h->v_new && h->out && h->sel && h->n_sel,
              "qcf_layer_step_host: NULL tensor pointer");
  QCF_REQUIRE(ctx, !h->is_critical_layer || h->q_probe, "qcf_layer_step_host: q_probe is NULL on a critical layer");
  if (b->batch == 0) return QCF_OK;
  if (!ctx->stage) ctx->stage = new (std::nothrow) HostStage();
  if (!ctx->stage) return fail(ctx, QCF_ERR_WORKSPACE, "out of host memory");
  HostStage& S = *ctx->stage;
  cudaStream_t s = static_cast<cudaStream_t>(stream);
  const Layout& L = ctx->lay;
  const size_t B = b->batch;
  const size_t kv_row = static_cast<size_t>(L.hkv) * L.d * 2, q_row = static_cast<size_t>(L.hq) * L.d * 2;
  const size_t pool_bytes = static_cast<size_t>(pool_rows) * kv_row;
  const size_t fused_bytes = B * b->t_stride * kv_row;
  const size_t qnew_bytes = B * b->t_stride * q_row;
  const size_t probe_bytes = B * b->q_stride * q_row;
  const size_t score_bytes = B * b->n_stride * sizeof(float);
  const size_t sel_bytes = B * b->n_stride * sizeof(int32_t);
  QCF_CUDA(ctx, S.k_pool.reserve(pool_bytes + 16)); QCF_CUDA(ctx, S.v_pool.reserve(pool_bytes + 16));
  QCF_CUDA(ctx, S.k_f.reserve(fused_bytes + 16)); QCF_CUDA(ctx, S.v_f.reserve(fused_bytes + 16));
  QCF_CUDA(ctx, S.q_probe.reserve(probe_bytes + 16)); QCF_CUDA(ctx, S.scores.reserve(score_bytes + 16));
  QCF_CUDA(ctx, S.sel.reserve(sel_bytes + 16)); QCF_CUDA(ctx, S.n_sel.reserve(B * sizeof(int32_t)));
  // Position-indexed fresh rows: only the rows in R = P u U (~rho of them) are ever read, but P is decided on the device by
  // a3, so a staged upload has to move ALL of q_new / k_new / v_new (60 % of the step's H2D bytes at config 4).  When the three
  // host buffers are pinned AND mapped into the device's address space (cudaHostAlloc / cudaHostRegister under unified
  // addressing — what torch.pin_memory gives), the a4 and a5 kernels read the rows they need straight from host memory
  // over PCIe instead: zero-copy gather, only |R| rows cross the bus.
  const void *zq = nullptr, *zk = nullptr, *zv = nullptr;
  bool zero_copy = h->rows_by_position != 0;
  if (zero_copy) {
    const void* hp[3] = {h->q_new, h->k_new, h->v_new};
    const void** zp[3] = {&zq, &zk, &zv};
    for (int i = 0; i < 3 && zero_copy; ++i) {
      cudaPointerAttributes at{};
      if (cudaPointerGetAttributes(&at, hp[i]) != cudaSuccess || at.type != cudaMemoryTypeHost || at.devicePointer == nullptr) {
        cudaGetLastError();                        // pageable memory: not an error, just the staged path
        zero_copy = false;
      } else {
        *zp[i] = at.devicePointer;
      }
    }
  }
  QCF_CUDA(ctx, S.q_new.reserve(qnew_bytes + 16));                 // staged copy, or the compact gather destination
  if (!zero_copy) {
    QCF_CUDA(ctx, S.k_new.reserve(fused_bytes + 16));
    QCF_CUDA(ctx, S.v_new.reserve(fused_bytes + 16));
  }
  QCF_CUDA(ctx, S.out.reserve(qnew_bytes + 16));
  if (h->lse) QCF_CUDA(ctx, S.lse.reserve(B * b->t_stride * L.hq * sizeof(float) + 16));

  // uploads: the PIC pool rows the batch READS (merged intervals: chunks no request references stay on the host — at config 4
  // the 16 requests touch ~100 of the pool's 256 chunks), probe, fresh rows; scores / sel when the caller carries them across
  // layers.  One cudaMemcpyAsync per interval and tensor.
  for (int i = 0; i < b->n_pool_iv; ++i) {
    const size_t off = static_cast<size_t>(b->h_pool_iv[2 * i]) * kv_row, len = static_cast<size_t>(b->h_pool_iv[2 * i + 1]) * kv_row;
    QCF_CUDA(ctx, cudaMemcpyAsync(static_cast<char*>(S.k_pool.p) + off, static_cast<const char*>(h->k_pool) + off, len, cudaMemcpyHostToDevice, s));
    QCF_CUDA(ctx, cudaMemcpyAsync(static_cast<char*>(S.v_pool.p) + off, static_cast<const char*>(h->v_pool) + off, len, cudaMemcpyHostToDevice, s));
  }
  if (h->is_critical_layer) QCF_CUDA(ctx, cudaMemcpyAsync(S.q_probe.p, h->q_probe, probe_bytes, cudaMemcpyHostToDevice, s));
  if (h->is_critical_layer && h->accumulate) {
    QCF_REQUIRE(ctx, h->scores != nullptr, "qcf_layer_step_host: scores is NULL with accumulate");
    QCF_CUDA(ctx, cudaMemcpyAsync(S.scores.p, h->scores, score_bytes, cudaMemcpyHostToDevice, s));
  }
  if (!h->select_now) {
    QCF_CUDA(ctx, cudaMemcpyAsync(S.sel.p, h->sel, sel_bytes, cudaMemcpyHostToDevice, s));
    QCF_CUDA(ctx, cudaMemcpyAsync(S.n_sel.p, h->n_sel, B * sizeof(int32_t), cudaMemcpyHostToDevice, s));
  }
  if (!zero_copy) {
    QCF_CUDA(ctx, cudaMemcpyAsync(S.q_new.p, h->q_new, qnew_bytes, cudaMemcpyHostToDevice, s));
    QCF_CUDA(ctx, cudaMemcpyAsync(S.k_new.p, h->k_new, fused_bytes, cudaMemcpyHostToDevice, s));
    QCF_CUDA(ctx, cudaMemcpyAsync(S.v_new.p, h->v_new, fused_bytes, cudaMemcpyHostToDevice, s));
  }

  qcf_layer_args d = *h;
  d.k_pool = S.k_pool.p; d.v_pool = S.v_pool.p; d.k_fused = S.k_f.p; d.v_fused = S.v_f.p;
  d.q_probe = S.q_probe.p; d.scores = static_cast<float*>(S.scores.p);
  d.sel = static_cast<int32_t*>(S.sel.p); d.n_sel = static_cast<int32_t*>(S.n_sel.p);
  d.q_new = zero_copy ? zq : S.q_new.p; d.k_new = zero_copy ? zk : S.k_new.p; d.v_new = zero_copy ? zv : S.v_new.p;
  d.out = S.out.p;
  d.lse = h->lse ? static_cast<float*>(S.lse.p) : nullptr;
  if (qcf_status st_step = layer_step_impl(ctx, b, &d, zero_copy ? zq : nullptr, S.q_new.p, stream)) return st_step;

  // only the |R_b| = k_b + Lq_b rows the step wrote are read back (k_b is known on the host: floor(rho N_b) when the step
  // selects, the caller's n_sel otherwise)
  for (int i = 0; i < b->batch; ++i) {
    const int k_b = h->select_now ? qcf_n_select(b->h_n_ctx[i], h->ratio) : h->n_sel[i];
    const size_t rows_b = static_cast<size_t>(k_b < 0 ? 0 : k_b) + b->h_n_query[i];
    const size_t off = static_cast<size_t>(i) * b->t_stride * q_row;
    if (rows_b > 0)
      QCF_CUDA(ctx, cudaMemcpyAsync(static_cast<char*>(h->out) + off, static_cast<const char*>(S.out.p) + off,
                                    std::min(rows_b, static_cast<size_t>(b->t_stride)) * q_row, cudaMemcpyDeviceToHost, s));
  }
  QCF_CUDA(ctx, cudaMemcpyAsync(h->sel, S.sel.p, sel_bytes, cudaMemcpyDeviceToHost, s));
  QCF_CUDA(ctx, cudaMemcpyAsync(h->n_sel, S.n_sel.p, B * sizeof(int32_t), cudaMemcpyDeviceToHost, s));
  if (h->scores && h->is_critical_layer)
    QCF_CUDA(ctx, cudaMemcpyAsync(h->scores, S.scores.p, score_bytes, cudaMemcpyDeviceToHost, s));
  if (h->k_fused) QCF_CUDA(ctx, cudaMemcpyAsync(h->k_fused, S.k_f.p, fused_bytes, cudaMemcpyDeviceToHost, s));
  if (h->v_fused) QCF_CUDA(ctx, cudaMemcpyAsync(h->v_fused, S.v_f.p, fused_bytes, cudaMemcpyDeviceToHost, s));
  if (h->lse) QCF_CUDA(ctx, cudaMemcpyAsync(h->lse, S.lse.p, B * b->t_stride * L.hq * sizeof(float), cudaMemcpyDeviceToHost, s));
  QCF_CUDA(ctx, cudaStreamSynchronize(s));
  return QCF_OK;
}

}  // extern "C"
