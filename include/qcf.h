/* qcf.h — C ABI of the B200-native QCFuse selective-recompute layer step.
 *
 * What the library computes is defined by arxiv 2606.05875 (cited below as PAPER.md:<line>, the text
 * under /root/reference/PAPER.md, plus section / equation).  One call of `qcf_layer_step` is one layer of the
 * "pipeline cache fusion" stage of Fig. 9 for a batch of independent RAG requests
 * C = [c_1..c_m] + U (Eq. 1):
 *
 *   a1  qcf_rope_reposition   Eq. 4   re-position per-chunk PIC K caches (RoPE at chunk-local positions)
 *                                     to request positions, stitch K and V
 *   a2  qcf_score             Eq. 18/20 user-query -> context attention mass per context position,
 *                                     aggregated over query tokens and heads
 *   a3  qcf_select_topk       Eq. 11  P = TopK(I(t), floor(rho N))
 *   a4+a5 qcf_recompute_attn  Eq. 7   scatter refreshed K/V of rows P (+ the query's own K/V) into the fused
 *                                     cache, then causal GQA attention of rows P u U over the fused cache
 *
 *       qcf_full_prefill_attn Eq. 2   dense causal GQA over all N+Lq rows: the rho = 1 comparator
 *
 *
 * Conventions (every entry point):
 *   - All tensors are bf16 unless stated, token-major: caches [T][Hkv][d], queries/outputs [T][Hq][d];
 *     q-head h reads kv-head g = h / (Hq/Hkv).  RoPE pairs are half-split (j, j+d/2), angle
 *     pos * theta^(-2j/d) (reading (a)).
 *   - "dev" = device pointer (16-byte aligned), "host" = host pointer.  The caller owns every buffer; the
 *     library allocates only in qcf_create / qcf_batch_create and never on the hot path.
 *   - Hot-path calls are asynchronous on `stream` (a cudaStream_t passed as void*), launch kernels only, do
 *     no host<->device copies and no synchronisation; they may be captured in a CUDA graph.
 *   - Per-request device arrays are strided by the batch's strides (qcf_batch_get_info):
 *       t_stride = max_b (N_b + Lq_b) rows  — fused caches, position-indexed fresh rows, outputs
 *       n_stride = max_b N_b               — scores, selections
 *   - Errors: every call returns a qcf_status; nothing throws or aborts.  Arguments are validated on the
 *     host before any launch.  qcf_last_error(ctx) gives the message of the last failure on that ctx.
 *   - A ctx and its batches are not thread-safe; use one ctx per host thread / stream.
 *   - There is no CPU fallback: without an sm_100 device qcf_create fails with QCF_ERR_UNSUPPORTED.
 */
#ifndef QCF_H_
#define QCF_H_

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define QCF_API __attribute__((visibility("default")))

typedef struct qcf_ctx qcf_ctx;       /* opaque: device properties, workspace                           */
typedef struct qcf_batch qcf_batch;   /* opaque: device-resident description of a batch of requests     */

typedef enum {
  QCF_OK = 0,
  QCF_ERR_INVALID_ARG = 1,  /* null pointer, negative size, ratio outside [0,1], mis-ordered offsets     */
  QCF_ERR_UNSUPPORTED = 2,  /* head_dim not in {64,128}, Hq % Hkv != 0, G not in {1,2,4,8,16}, max_query*G > 8192,
                               no sm_100 device                                                          */
  QCF_ERR_WORKSPACE = 3,    /* batch exceeds the limits given to qcf_create                              */
  QCF_ERR_CUDA = 4          /* a CUDA runtime call failed; message holds cudaGetErrorString              */
} qcf_status;

/* Head layout of one attention layer (BASELINE.json: "head layout"). */
typedef struct {
  int32_t n_q_heads;     /* Hq                                                     */
  int32_t n_kv_heads;    /* Hkv, divides Hq                                        */
  int32_t head_dim;      /* d, 64 or 128                                           */
  float rope_theta;      /* RoPE base theta (1e6 in the BASELINE configs)          */
  float softmax_scale;   /* 0 -> 1/sqrt(d)                                         */
} qcf_layout;

/* One request C = [c_1..c_m] + U (Eq. 1).  All pointers are HOST pointers, read only during
 * qcf_batch_create.  Chunk i's PIC cache (Eq. 3) is `chunk_len[i]` consecutive rows of the
 * layer's PIC pool starting at row `chunk_row[i]` (the pool is a [pool_rows][Hkv][d] bf16 array whose base
 * pointers, one for K and one for V, are given per call because they change per layer while the chunk
 * geometry does not).  The chunk's request offset off_i is the exclusive prefix sum of chunk_len
 * (PAPER.md:112-117), N = sum chunk_len.  A chunk may be shared by many requests (BASELINE config 4). */
typedef struct {
  int32_t n_chunks;            /* m >= 0                                                               */
  int32_t n_query;             /* Lq = |U| >= 0                                                        */
  const int32_t* chunk_len;    /* host [m], each >= 0                                                  */
  const int64_t* chunk_row;    /* host [m], first pool row of chunk i's PIC cache, >= 0                */
  const int32_t* chunk_pos;    /* host [m] or NULL.  NULL: chunk i is rotated by off_i, the exclusive prefix sum of
                                  chunk_len (Eq. 4: contiguous stitching).  Non-NULL: chunk i is rotated by
                                  chunk_pos[i] >= 0 while its rows are still WRITTEN contiguously in chunk order —
                                  the anchor stitch of Eq. 15-16: "chunk" i = the |A_i| anchor rows
                                  of c_i kept compactly in an anchor pool, chunk_pos[i] = off_i of c_i in the full
                                  request, so every anchor keeps its original request position off_i + a
                                   while the anchor cache stays a compact subsequence.             */
} qcf_request;

typedef struct {
  int32_t batch;       /* B                                                                             */
  int32_t t_stride;    /* max_b (N_b + Lq_b)                                                            */
  int32_t n_stride;    /* max_b N_b                                                                     */
  int32_t q_stride;    /* max_b Lq_b                                                                    */
  int64_t total_ctx;   /* sum_b N_b                                                                     */
  int64_t pool_rows_touched; /* rows of the PIC pool the batch reads (union over requests: shared chunks count once) */
} qcf_batch_info;

/* ---------------------------------------------------------------------------------------------- lifetime */

/* Creates a context on the current CUDA device for one head layout.  max_batch / max_ctx / max_query bound
 * the batches that may be created on it (they size the internal workspace: score statistics, tile counters).
 * Fails with QCF_ERR_UNSUPPORTED if the device is not compute capability 10.x or the layout is unsupported. */
QCF_API qcf_status qcf_create(qcf_ctx** out, const qcf_layout* layout, int32_t max_batch, int32_t max_ctx,
                              int32_t max_query);
QCF_API void qcf_destroy(qcf_ctx* ctx);
/* Message of the last failure on ctx ("" if none).  With ctx == NULL returns the message of the last failed
 * qcf_create on this thread.  The pointer stays valid until the next call on the same ctx. */
QCF_API const char* qcf_last_error(const qcf_ctx* ctx);
/* Library version string, and the SM architecture the kernels were compiled for (100). */
QCF_API const char* qcf_version(void);

/* Validates `reqs[0..batch)`, computes chunk offsets off_i, the per-chunk rotation tables
 * (cos, sin)(off_i * theta^(-2j/d)) in double precision on the host (Eq. 4's Pi_i), and uploads them.
 * Synchronous (one blocking upload); not a hot-path call: a batch is built once per request set and reused by
 * all L layers.  batch == 0 is legal (every later call on it is a no-op). */
QCF_API qcf_status qcf_batch_create(qcf_ctx* ctx, const qcf_request* reqs, int32_t batch, qcf_batch** out);
QCF_API void qcf_batch_destroy(qcf_batch* b);
QCF_API qcf_status qcf_batch_get_info(const qcf_batch* b, qcf_batch_info* info);

/* |P| = floor(rho * N + 1e-6) evaluated in double (Eq. 8 constraint |P| = floor(rho N), PAPER.md:195;
 * DESIGN.md reading (g)).  Returns -1 if n_ctx < 0 or ratio is outside [0,1] or NaN. */
QCF_API int32_t qcf_n_select(int32_t n_ctx, double ratio);

/* ------------------------------------------------------------------------------------------------ a1 */

/* Eq. 4.  For every request b, chunk i, chunk row r, kv-head g, pair j < d/2:
 *     phi = off_i * theta^(-2j/d);  (a, b) = K_pic[r][g][j], K_pic[r][g][j+d/2]
 *     k_fused[b][off_i+r][g][j]     = bf16(a cos phi - b sin phi)
 *     k_fused[b][off_i+r][g][j+d/2] = bf16(b cos phi + a sin phi)
 *     v_fused[b][off_i+r][g][:]     = V_pic[r][g][:]                       (byte copy)
 * fp32 arithmetic, one bf16 rounding (RNE) on store.  A chunk at off_i = 0 is copied bit-exactly.
 *   k_pool, v_pool : dev, [pool_rows][Hkv][d] bf16, read-only (the layer's PIC pool)
 *   k_fused,v_fused: dev, [B][t_stride][Hkv][d] bf16; rows 0..N_b-1 of each request are written, the rest
 *                    (the Lq query rows and padding) are left untouched.
 * Either half may be omitted: v_pool == v_fused == NULL re-positions K only (the scoring prefetch of a critical layer
 * reads no V), k_pool == k_fused == NULL stitches V only (its V, loaded later).  QCF_ERR_INVALID_ARG if both are. */
QCF_API qcf_status qcf_rope_reposition(qcf_ctx* ctx, const qcf_batch* b, const void* k_pool, const void* v_pool,
                                       void* k_fused, void* v_fused, void* stream);

/* ------------------------------------------------------------------------------------------------ a2 */

/* Eq. 18 with Attn^l(.)_t as defined at PAPER.md:208.  For request b, context position
 * t < N_b:
 *     I(t) = 1/(Hq Lq) * sum_{i<Lq} sum_{h<Hq} softmax_{t' < N_b}( q_probe[i][h] . k_fused[t'][h/G] * scale )_t
 * (context keys only, no mask: DESIGN.md readings (b), (c), (d), (e)).  bf16 operands, fp32 accumulation and
 * softmax.  accumulate == 0: scores[b][t] = I(t);  accumulate != 0: scores[b][t] += I(t)  (Eq. 20, the sum
 * over critical layers).
 *   q_probe : dev, [B][q_stride][Hq][d] bf16 — the anchor-conditioned query states Q_U^l(C_A) (Eq. 17), RoPE
 *             at positions N_b..N_b+Lq_b-1; rows >= Lq_b of a request are ignored
 *   k_fused : dev, [B][t_stride][Hkv][d] bf16 — output of qcf_rope_reposition (rows 0..N_b-1 are read)
 *   scores  : dev, [B][n_stride] fp32; entries t >= N_b are left untouched
 * A request with Lq_b == 0 or N_b == 0 contributes nothing (its scores are zeroed when accumulate == 0). */
QCF_API qcf_status qcf_score(qcf_ctx* ctx, const qcf_batch* b, const void* q_probe, const void* k_fused,
                             float* scores, int32_t accumulate, void* stream);

/* KV-head-sharded step: the heads of a layer are independent for a1, a4 and a5, and a2
 * is a SUM over heads (Eq. 18), so a layer can be split over n_shards ranks, each with a ctx created for Hq/n_shards
 * query heads and Hkv/n_shards kv-heads and holding those heads' slices of every tensor.  After this call qcf_score on
 * this ctx divides by (Hq * n_shards) * Lq, i.e. it returns the rank's PARTIAL of Eq. 18 over all heads of the layer:
 * the element-wise sum of the ranks' score arrays (one all-reduce of [B][n_stride] fp32 — or, on one device,
 * qcf_score with accumulate != 0 on the same array) is I(t).  qcf_select_topk then runs replicated on the summed
 * scores, so every rank selects the same P.  n_shards in [1, 64]; 1 (the default) restores the plain behaviour. */
QCF_API qcf_status qcf_set_head_shards(qcf_ctx* ctx, int32_t n_shards);

/* The same step with the score exchange FUSED into a2 instead of a collective call between two launches (SURVEY.md
 * section 8(f).4): every rank owns an exchange buffer of qcf_score_exchange_bytes(n_shards, slot_elems) bytes, laid out
 *     [64 x uint32 flags][64 x uint32 acks][2 slot sets x n_shards slots x slot_elems fp32],
 *     slot_elems >= B * n_stride of every batch used,
 * and `peer_bufs[p]` (host array [n_shards]) is rank p's buffer AS MAPPED INTO THIS PROCESS (its own allocation for
 * p == rank; cudaIpcOpenMemHandle / peer access over NVLink for the others).  After this call, on this ctx:
 *   qcf_score        is epoch e (e counts this ctx's exchanging qcf_score calls from 1).  Besides writing `scores` as
 *                    before, the combine CTAs store this rank's (accumulated) partial I_rank(t) straight into slot `rank`
 *                    of slot set (e & 1) of EVERY rank's buffer (plain st.global on peer pointers), and a one-thread tail
 *                    kernel then publishes e in flag[rank] of every buffer with a system-scope release — no NCCL call, no
 *                    host involvement.  Before it starts, a one-warp head kernel waits until every peer has acknowledged
 *                    the newest selection epoch <= e - 2 (see below);
 *   qcf_select_topk  waits (system-scope acquire, bounded: a missing peer traps after ~2 s instead of hanging) until all
 *                    n_shards flags of ITS OWN buffer have reached the current epoch e, then ranks the element-wise sum
 *                    of the n_shards slots of slot set (e & 1), added in slot order (every rank forms bit-identical sums
 *                    and selects the same P); its `scores` argument is ignored.  A one-thread tail kernel then publishes e
 *                    in ack[rank] of every buffer: "this rank has finished reading epoch e".
 * Protocol invariant (what makes back-to-back steps safe when ranks drift apart): a rank overwrites slot set (e & 1),
 * last written at epoch e - 2, only after every peer has acknowledged the newest selection at an epoch <= e - 2 — so no
 * selection that could still be reading that set is outstanding — while the selection of epoch e - 1, if a slower peer has
 * yet to run it, reads the OTHER set.  A rank may therefore run up to one exchanging qcf_score ahead of its slowest peer's
 * selection; further ahead it waits.  Flags and acks only ever increase.
 * Rules for the caller: (1) the buffers are ZEROED before they are shared (qcf_set_score_exchange clears nothing: a faster
 * peer may already have published into this rank's buffer); no rank issues an exchanging call before every rank's buffer
 * is zeroed and mapped (sharded.share_exchange_buffers ends with a barrier).  (2) All ranks issue the same sequence of
 * exchanging qcf_score / qcf_select_topk calls (the epoch counts the former).  (3) Selecting twice at the same epoch is
 * allowed only while no rank has moved past the next epoch (only the first selection's ack is distinguishable).
 * n_shards == 1 or peer_bufs == NULL turns the exchange off.  Not CUDA-graph capturable (the epoch is a launch argument).
 * Unmeasured on > 1 GPU in this repository (one GPU per box); tested with two contexts on one GPU — including one rank
 * running a whole step ahead of the other's selection — and with two PROCESSES sharing one GPU through CUDA IPC handles,
 * their phases ordered on the host so that no kernel ever spins on a flag another process has yet to write. */
QCF_API int64_t qcf_score_exchange_bytes(int32_t n_shards, int64_t slot_elems);
QCF_API qcf_status qcf_set_score_exchange(qcf_ctx* ctx, int32_t rank, int32_t n_shards, void* const* peer_bufs,
                                          int64_t slot_elems);

/* ------------------------------------------------------------------------------------------------ a3 */

/* Eq. 11: per request, the k_b = qcf_n_select(N_b, ratio) context positions with the
 * largest scores over ALL context positions of the request (global budget, reading (i)); ties are broken
 * towards the lower position (reading (h)); positions are emitted in ascending order.
 *   scores : dev, [B][n_stride] fp32 (any finite values; -0 == +0; NaN unsupported)
 *   sel    : dev, [B][n_stride] int32; sel[b][0..k_b) written
 *   n_sel  : dev, [B] int32; n_sel[b] = k_b written
 * Exact (integer radix select on the order-preserving key of the fp32 score): bit-identical across runs. */
QCF_API qcf_status qcf_select_topk(qcf_ctx* ctx, const qcf_batch* b, const float* scores, double ratio,
                                   int32_t* sel, int32_t* n_sel, void* stream);

/* --------------------------------------------------------------------------------------------- a4 + a5 */

/* Eq. 7 + PAPER.md:134.  With R_b = sel[b][0..n_sel[b]) followed by the query positions N_b..N_b+Lq_b-1:
 *   a4: for p in R_b:  k_fused[b][p] = k_new[.], v_fused[b][p] = v_new[.]      (row copy; the query's own
 *       K/V are appended at N_b..)
 *   a5: for row index r (position p_r = R_b[r]) and head h:
 *       out[b][r][h] = sum_{j <= p_r} softmax_j( q_new[.][h] . k_fused[b][j][h/G] * scale ) v_fused[b][j][h/G]
 *       over the FUSED cache (unselected prefix = PIC, selected prefix = new; reading (k): all rows are
 *       independent given the fused cache).  bf16 operands, fp32 softmax/accumulate, bf16 output (RNE).
 *   sel, n_sel : dev, as written by qcf_select_topk (sel ascending, distinct, < N_b)
 *   q_new/k_new/v_new : dev bf16, fresh rows under the current request order and positions;
 *       rows_by_position != 0: [B][t_stride][H][d] indexed by request position p (only rows in R_b are read)
 *       rows_by_position == 0: [B][t_stride][H][d] compact, row r <-> R_b[r]
 *   k_fused, v_fused : dev, in/out
 *   out : dev, [B][t_stride][Hq][d] bf16, rows 0..|R_b|-1 written (compact, P ascending then U)
 *   lse : dev or NULL, [B][t_stride][Hq] fp32 natural-log-sum-exp of each output row's logits */
QCF_API qcf_status qcf_recompute_attn(qcf_ctx* ctx, const qcf_batch* b, const int32_t* sel, const int32_t* n_sel,
                                      const void* q_new, const void* k_new, const void* v_new,
                                      int32_t rows_by_position, void* k_fused, void* v_fused, void* out,
                                      float* lse, void* stream);

/* Eq. 2 at one layer: dense causal GQA attention of all T_b = N_b + Lq_b rows over
 * themselves — the rho = 1 endpoint and the "library's own full-prefill attention" comparator.
 *   q : dev [B][t_stride][Hq][d];  k, v : dev [B][t_stride][Hkv][d];  out : dev [B][t_stride][Hq][d] */
QCF_API qcf_status qcf_full_prefill_attn(qcf_ctx* ctx, const qcf_batch* b, const void* q, const void* k,
                                         const void* v, void* out, float* lse, void* stream);

/* ------------------------------------------------------------------------------------------------ a1' */

/* Anchor stitch (Eq. 15-16) is qcf_rope_reposition on a batch whose requests were created
 * with chunk_pos (see qcf_request): k_pool / v_pool are then the layer's compact ANCHOR pool, k_fused / v_fused
 * the probe cache KV^A(C_A) [B][t_stride][Hkv][d] (t_stride of that batch = max_b (|C_A|_b + Lq_b)).  With
 * v_pool == NULL and v_fused == NULL only K is re-positioned (scoring prefetch of the critical layers reads no V). */

/* ------------------------------------------------------------------------------------- Phase I: anchors */

/* Eq. 14: A_i = TopK(G_i, ceil(r_a |c_i|)) for every chunk of the batch, which must list ONE chunk
 * per request (n_chunks = 1, n_query = 0; chunk_row = the chunk's first row in k_pool).
 *   rule QCF_ANCHOR_SINK : G_i(r) = -r                  (the first positions of the chunk)
 *   rule QCF_ANCHOR_KNORM: G_i(r) = -||K_i[r]||_2       over all kv-heads and dims of the layer's PIC keys (the paper
 *                          does not say which end of the norm ranking is kept; low-norm keys, reading (o'))
 *   k_pool   : dev [pool_rows][Hkv][d] bf16 (ignored for SINK; may be NULL)
 *   scores   : dev [B][n_stride] fp32 workspace, receives G_i; accumulate != 0 adds to it (norms summed over layers:
 *              call once per layer with select_now = 0, then once with select_now != 0)
 *   anchor_idx : dev [B][n_stride] int32, chunk-local positions ascending; n_anchor : dev [B] int32
 * KVzip (a reconstruction probe over a trained model) is out of scope. */
typedef enum { QCF_ANCHOR_SINK = 0, QCF_ANCHOR_KNORM = 1 } qcf_anchor_rule;
QCF_API qcf_status qcf_anchor_rank(qcf_ctx* ctx, const qcf_batch* chunks, const void* k_pool, int32_t rule, double r_a,
                                   float* scores, int32_t accumulate, int32_t select_now, int32_t* anchor_idx,
                                   int32_t* n_anchor, void* stream);

/* Eq. 16: KV_i^A = KV_i^PIC[A_i] — the step between the ranking above and the anchor stitch (a1'):
 * the anchor rows of every chunk are copied out of a layer's PIC pool into that layer's COMPACT anchor pool, chunk after
 * chunk, anchors ascending inside a chunk — exactly the pool layout a chunk_pos batch reads (chunk i's "chunk" = its
 * |A_i| anchor rows starting at row sum_{j<i} |A_j|).
 *   chunks     : the one-chunk-per-request batch of qcf_anchor_rank (chunk_row = the chunk's first row in the PIC pool)
 *   k_pool, v_pool     : dev [pool_rows][Hkv][d] bf16, this layer's PIC pool; either may be NULL (with its output)
 *   anchor_idx, n_anchor : dev, as written by qcf_anchor_rank (chunk-local positions; counts)
 *   k_anchor, v_anchor : dev [>= sum_i n_anchor[i]][Hkv][d] bf16, written; the caller sizes them (n_anchor[i] =
 *                        ceil(r_a |c_i|) is known on the host).  Rows are byte copies; K keeps its chunk-local RoPE, which
 *                        qcf_rope_reposition on the chunk_pos batch then moves to off_i + a (Eq. 15). */
QCF_API qcf_status qcf_anchor_gather(qcf_ctx* ctx, const qcf_batch* chunks, const void* k_pool, const void* v_pool,
                                     const int32_t* anchor_idx, const int32_t* n_anchor, void* k_anchor, void* v_anchor,
                                     void* stream);

/* ------------------------------------------------------------------------------------------------ a6 */

/* Everything one layer needs, by name.  Pointers as documented at the stage entry points. */
typedef struct {
  const void* k_pool;      /* a1 in  */
  const void* v_pool;      /* a1 in  */
  void* k_fused;           /* a1 out, a2 in, a4/a5 in-out */
  void* v_fused;
  const void* q_probe;     /* a2 in (critical layers only; may be NULL otherwise) */
  float* scores;           /* a2 in-out, a3 in */
  int32_t* sel;            /* a3 out / a4,a5 in */
  int32_t* n_sel;
  const void* q_new;       /* a4/a5 in */
  const void* k_new;
  const void* v_new;
  void* out;               /* a5 out */
  float* lse;              /* a5 out, optional */
  double ratio;            /* rho, used when select_now != 0 */
  int32_t rows_by_position;
  int32_t is_critical_layer; /* != 0: run a2 on this layer (l in L*, Eq. 20) */
  int32_t accumulate;        /* a2: add to `scores` instead of overwriting */
  int32_t select_now;        /* != 0: run a3 after a2 (once, after the last critical layer) */
} qcf_layer_args;

/* Fig. 9 / PAPER.md:337-344, one layer: a1 -> [a2 if is_critical_layer] -> [a3 if select_now] -> a4 -> a5,
 * chained on `stream` with no host synchronisation. */
QCF_API qcf_status qcf_layer_step(qcf_ctx* ctx, const qcf_batch* b, const qcf_layer_args* args, void* stream);

/* The same step with every tensor in HOST memory (pinned memory recommended): uploads the PIC pool rows, probe and fresh
 * rows, runs qcf_layer_step on the context's internal device buffers, downloads the |R_b| written rows of `out`, `sel`,
 * `n_sel` (and the fused cache if k_fused / v_fused are non-NULL), and synchronises `stream` before returning.  Pointer
 * fields of `host` are host pointers with the same shapes.  Device staging buffers are allocated on first use and kept
 * by the ctx.
 *   pool_rows: rows of host->k_pool / v_pool; every chunk of the batch must lie inside them (QCF_ERR_INVALID_ARG otherwise).
 *   Only the pool rows some request of the batch reads are uploaded (qcf_batch_info.pool_rows_touched rows per tensor).
 *   With rows_by_position != 0 and q_new / k_new / v_new in pinned, device-mapped host memory (cudaHostAlloc,
 *   cudaHostRegister, torch.pin_memory) those three buffers are not uploaded at all: the a4 and a5 kernels read the |R_b|
 *   rows they need straight from host memory (zero-copy gather; P is only known on the device after a3).  Pageable
 *   buffers are staged through a full upload. */
QCF_API qcf_status qcf_layer_step_host(qcf_ctx* ctx, const qcf_batch* b, const qcf_layer_args* host,
                                       int64_t pool_rows, void* stream);

/* Per-stage device time.  qcf_set_profiling(ctx, 1) makes every qcf_layer_step record CUDA events between its
 * stages on `stream` (still asynchronous, no host synchronisation; up to 512 steps are kept).
 * qcf_get_stage_ms synchronises on the last recorded event and fills ms[5] = {a1, a2, a3, a4, a5} with the MEAN
 * over the profiled steps issued since the previous call (or since profiling was enabled), then forgets them. */
QCF_API qcf_status qcf_set_profiling(qcf_ctx* ctx, int32_t enable);
QCF_API qcf_status qcf_get_stage_ms(qcf_ctx* ctx, float* ms5);

/* Test-only launch knobs (the one debug entry point; nothing is read from the environment).  They change HOW the same
 * kernels are launched, never WHAT is computed — the parity tests use them to force launch shapes the host heuristics
 * would only pick at other problem sizes:
 *   QCF_DEBUG_PDL          value 0: plain stream-ordered launches; 1 (default): programmatic dependent launch between the
 *                          kernels of a step
 *   QCF_DEBUG_ATTN_CLUSTER value 1 / 2 / 4: split-KV cluster size of the a5 kernel; 0 (default): host heuristic
 *   QCF_DEBUG_GEMM_MT      value 1 / 2: GEMM tile height in units of 128 rows; 0 (default): host heuristic
 * QCF_ERR_INVALID_ARG for an unknown knob or value. */
typedef enum { QCF_DEBUG_PDL = 0, QCF_DEBUG_ATTN_CLUSTER = 1, QCF_DEBUG_GEMM_MT = 2 } qcf_debug_knob;
QCF_API qcf_status qcf_debug_set(qcf_ctx* ctx, int32_t knob, int32_t value);

/* ---------------------------------------------------------------------------------------- a7 / a8 (config 3) */

/* Row-wise dense projection of the recomputed rows (BASELINE config 3):
 *     c[M][N] = a[M][K] . w[N][K]^T          bf16 operands (nn.Linear layout [out][in]), fp32 accumulation
 *   epilogue QCF_EPI_STORE        : c = acc                                  (bf16, RNE)
 *            QCF_EPI_ADD_RESIDUAL : c = residual + acc   (residual [M][N] bf16; residual == c allowed)
 *            QCF_EPI_SWIGLU       : w holds (gate_j, up_j) rows INTERLEAVED (row 2j = W_g[j], 2j+1 = W_u[j]);
 *                                   c[M][N/2] = silu(acc[2j]) * acc[2j+1]
 * All dev pointers 16-byte aligned; K % 8 == 0, N % 8 == 0 (N % 16 == 0 for SWIGLU).  M, N, K tails are handled.
 * Not invariant to M in the last bit: M == 1 (a decoding row) runs a weight-streaming GEMV whose fp32 sums are formed in
 * another order than the tensor-core tiles used for M > 1, so one row computed alone and the same row inside a larger batch
 * can differ by one bf16 rounding (both are within the stated tolerance of the exact product).  Likewise the decode path
 * folds RMSNorm into the GEMV prologue ((x * inv_rms) * gain rounded to bf16 once, the same expression as the prefill's
 * RMSNorm kernel); decode == last row of a one-token-longer prefill holds within the free-running bound, not bit for bit. */
typedef enum { QCF_EPI_STORE = 0, QCF_EPI_ADD_RESIDUAL = 1, QCF_EPI_SWIGLU = 2 } qcf_epilogue;
QCF_API qcf_status qcf_linear(qcf_ctx* ctx, const void* a, const void* w, const void* residual, void* c, int32_t M,
                              int32_t N, int32_t K, int32_t epilogue, void* stream);

typedef struct qcf_stack qcf_stack;   /* opaque: weights table, activation workspace, loader stream, events */

typedef struct {
  int32_t n_layers;   /* L                                                   */
  int32_t hidden;     /* model width, % 8 == 0                               */
  int32_t ffn;        /* SwiGLU inner width, % 8 == 0                        */
  int32_t vocab;      /* rows of the embedding table                         */
  float rms_eps;      /* RMSNorm epsilon (1e-6)                              */
} qcf_stack_dims;

/* One decoder layer (readings (l), (q)): pre-norm block, QK-norm before RoPE, no biases, SwiGLU.
 * Device pointers to bf16 tensors owned by the caller; they must outlive the stack. */
typedef struct {
  const void* w_qkv;       /* [(Hq + 2 Hkv) d][hidden]: q heads, then k heads, then v heads            */
  const void* w_o;         /* [hidden][Hq d]                                                           */
  const void* w_gate_up;   /* [2 ffn][hidden], gate/up rows interleaved (see QCF_EPI_SWIGLU)           */
  const void* w_down;      /* [hidden][ffn]                                                            */
  const void* g_attn;      /* [hidden] RMSNorm gain before attention                                   */
  const void* g_ffn;       /* [hidden] RMSNorm gain before the MLP                                     */
  const void* g_q;         /* [d] per-head RMSNorm gain of q                                           */
  const void* g_k;         /* [d] per-head RMSNorm gain of k                                           */
} qcf_layer_weights;

/* layers: host array [n_layers]; embed: dev [vocab][hidden] bf16.  max_rows bounds the rows any call pushes through
 * the block (N + Lq for full prefill), max_pos the largest request position + 1 (RoPE table, evaluated in double),
 * max_pool_rows the PIC / anchor pool rows staged per layer by qcf_stack_fuse (0: fuse not used).  The head layout
 * is the ctx's.  Only single-request batches (B = 1) are supported by the stack calls. */
QCF_API qcf_status qcf_stack_create(qcf_ctx* ctx, const qcf_stack_dims* dims, const qcf_layer_weights* layers,
                                    const void* embed, int32_t max_rows, int32_t max_pos, int64_t max_pool_rows,
                                    qcf_stack** out);
QCF_API void qcf_stack_destroy(qcf_stack* s);

/* Eq. 2 / Eq. 3: all T = N + Lq rows of the batch's request, token ids tokens[T] (dev int32) at
 * positions 0..T-1, through every layer with dense causal attention.  k_cache / v_cache: host arrays [n_layers] of
 * dev pointers [T][Hkv][d] that receive each layer's K (post QK-norm, post RoPE) and V.  hidden_out: dev
 * [T][hidden] final hidden states, or NULL.  Used for the full-prefill comparator (Eq. 2) and, on a one-chunk batch
 * with Lq = 0, for building that chunk's PIC cache at chunk-local positions (Eq. 3). */
QCF_API qcf_status qcf_stack_prefill(qcf_stack* s, const qcf_batch* b, const int32_t* tokens, void* const* k_cache,
                                     void* const* v_cache, void* hidden_out, void* stream);

/* One layer of Fig. 9 stage 2 for the rows R = sel[0..n_sel) u U of the batch's request:
 *   RMSNorm -> QKV projection -> QK-norm + RoPE at the rows' request positions -> a4 scatter + a5 attention over
 *   k_fused / v_fused (which must already hold this layer's stitched PIC entries) -> O projection + residual ->
 *   RMSNorm -> SwiGLU MLP + residual.
 *   x: dev [n_rows][hidden] bf16, in/out (compact, P ascending then U); n_rows = n_sel + Lq must be given by the
 *   caller (host; qcf_n_select).  sel == NULL: dense mode — rows are positions 0..n_rows-1 and k_fused / v_fused
 *   receive their K/V (one layer of qcf_stack_prefill).  query_pos0 >= 0 overrides the request position of the
 *   first query row (default N_b): the probe stage runs U over the compact anchor cache at positions N..N+Lq-1
 *   (PAPER.md:293).  q_tap: dev [n_rows][Hq][d] or NULL, receives the post-RoPE query states (Eq. 17). */
QCF_API qcf_status qcf_stack_layer(qcf_stack* s, int32_t layer, const qcf_batch* b, const int32_t* sel,
                                   const int32_t* n_sel, int32_t n_rows, int32_t query_pos0, void* x, void* k_fused,
                                   void* v_fused, void* q_tap, void* stream);

/* The end of time-to-first-token: the first generated token from the final hidden state of the LAST query
 * row:   token = argmax_v ( RMSNorm(hidden[row]; g_final) . w_lm[v] ),  ties to the lower token id.
 *   hidden : dev [rows][hidden] bf16 (hidden_out of qcf_stack_fuse: row = n_R - 1; of qcf_stack_prefill: row = T - 1)
 *   g_final: dev [hidden] bf16;  w_lm: dev [vocab][hidden] bf16 (vocab = dims.vocab)
 *   logits : dev [vocab] fp32, written (needed as workspace);  token : dev [1] int32 */
QCF_API qcf_status qcf_stack_first_token(qcf_stack* s, const void* hidden, int32_t row, const void* g_final, const void* w_lm,
                                         float* logits, int32_t* token, void* stream);

/* Decoding over KV^Fuse (after fusion "the fused KV cache and the user query states" go to decoding;
 * TTFT ends at the first token and generation continues from it).
 *
 * qcf_decode_attn — single-row GQA attention of ONE new token over rows [0, n_keys) of a layer's cache (the token's own
 * K/V row, n_keys - 1, included):   out[h] = sum_{j < n_keys} softmax_j(q[h] . k_cache[j][h/G] * scale) v_cache[j][h/G]
 *   q : dev [Hq][d] bf16;  k_cache, v_cache : dev [>= n_keys][Hkv][d] bf16;  out : dev [Hq][d] bf16;
 *   lse : dev [Hq] fp32 natural-log-sum-exp, or NULL.  fp32 softmax / accumulation, split over key ranges and merged in
 *   split order (bit-reproducible).  n_keys >= 1. */
QCF_API qcf_status qcf_decode_attn(qcf_ctx* ctx, const void* q, const void* k_cache, const void* v_cache, int32_t n_keys,
                                   void* out, float* lse, void* stream);

/* qcf_decode_attn_static — qcf_decode_attn for callers that cannot allocate device memory.  Same operation, same kernel,
 * same arguments and result (bit-identical to qcf_decode_attn for the same layout on the same GPU), but no qcf_ctx:
 * qcf_create cudaMallocs the kernel's split-KV workspace, and that is exactly what some callers may not do — an op
 * plugged into a serving engine whose pool allocator already owns all of HBM, code inside a region its framework has
 * declared allocation-free, a monitoring tool that must leave the allocator untouched.  Here the workspace is a fixed
 * array inside the library image (about 2.1 MiB of device memory on every GPU that loads libqcf.so, held until the
 * process exits), and the call itself makes no cudaMalloc / cudaFree and uses no allocating library routine: it is one
 * 256-byte cudaMemsetAsync (the arrival counters) plus one kernel launch on `stream`.
 *   layout : host; Hq * head_dim <= 8192 and Hkv <= 64 (what the fixed workspace holds; beyond it the call fails with
 *            QCF_ERR_WORKSPACE and launches nothing — use qcf_create + qcf_decode_attn there), head_dim 64 or 128,
 *            Hq / Hkv in {1,2,4,8,16}; softmax_scale 0 -> 1/sqrt(d); rope_theta is not used.  n_keys >= 1, no upper limit.
 *   q, k_cache, v_cache, out, lse : as for qcf_decode_attn; the caller owns them.
 * First call on each device: with that device current, the library looks up the array's device address and the SM count
 * (a few driver queries, no allocation) and keeps them; make that first call outside any stream capture.
 * One workspace per GPU, shared by every caller and thread: two calls whose kernels can overlap on the GPU (different
 * streams, no ordering between them) race on it and both results are undefined; calls on one stream, or ordered by
 * events, are fine.  Each call clears the counters it needs; the rest of the array is overwritten before it is read.
 * Errors: returned as a status; the message is qcf_last_error(NULL) on the calling thread. */
QCF_API qcf_status qcf_decode_attn_static(const qcf_layout* layout, const void* q, const void* k_cache, const void* v_cache,
                                          int32_t n_keys, void* out, float* lse, void* stream);

/* qcf_stack_decode — n_new greedy tokens, one at a time through every layer:
 *   token i (i = 0: *token_in, the token qcf_stack_first_token produced; else tokens_out[i-1]) is embedded, sits at request
 *   position pos0 + i, and per layer: RMSNorm -> QKV projection -> QK-norm + RoPE at that position -> its K/V APPENDED as
 *   cache row pos0 + i -> qcf_decode_attn over rows 0..pos0+i -> O projection + residual -> RMSNorm -> SwiGLU MLP + residual;
 *   then tokens_out[i] = argmax_v(RMSNorm(x; g_final) . w_lm[v]) (ties to the lower id), logits[i][:] its fp32 logits.
 *   token_in : dev int32 [1];  pos0 = rows already in every cache (N + Lq after qcf_stack_fuse / qcf_stack_prefill)
 *   k_cache, v_cache : host arrays [L] of dev [>= pos0 + n_new][Hkv][d] — the caches qcf_stack_fuse filled (KV^Fuse), with
 *                      room for the appended rows;  pos0 + n_new <= max_pos of qcf_stack_create
 *   Limits: hidden, ffn and Hq * head_dim <= 115712 (the row a GEMV multiplies is staged whole in shared memory), else
 *   QCF_ERR_UNSUPPORTED; Hq / Hkv in {1,2,4,8,16} as for every ctx.
 *   logits : dev [n_new][vocab] fp32;  tokens_out : dev int32 [n_new]
 * Launch-only on `stream` (token ids never return to the host between steps). */
QCF_API qcf_status qcf_stack_decode(qcf_stack* s, const int32_t* token_in, int32_t pos0, int32_t n_new,
                                    void* const* k_cache, void* const* v_cache, const void* g_final, const void* w_lm,
                                    float* logits, int32_t* tokens_out, void* stream);

/* The whole online pipeline of Fig. 9 for one request.
 *   stage 1  for l = 0..max(L*): load anchor pool l, stitch (a1'), run U through layer l over the anchor cache
 *            (Eq. 17); for l in L*: load PIC pool l, stitch (a1), score (a2, Eq. 18/20); then top-k (a3, Eq. 11)
 *   stage 2  for every layer: load PIC pool l+1.. and stitch them on a second stream WHILE layer l recomputes the
 *            rows R on `stream` (a8: PAPER.md:23, 341-342), a4 + a5 + a7 per layer
 * Pools may live in pinned host memory (the paper's setting) or on the device (cudaMemcpyDefault).
 * The compressed view is an argument, not a mode: anchor pools = the PIC pools with a probe batch that lists whole chunks
 * and crit_layers = every layer gives full-view (ProphetKV-style) selection (Eq. 9-11); an empty anchor
 * pool with crit_layers = {L-1} gives query-only final-layer selection. */
typedef struct {
  const void* const* k_pic;      /* host array [L] of pointers to [pool_rows][Hkv][d] bf16 PIC pools              */
  const void* const* v_pic;
  int64_t pool_rows;             /* rows of each PIC pool; every chunk of main_batch must lie inside (else INVALID_ARG)  */
  const void* const* k_anchor;   /* host array [L] (entries l <= max(L*) are read) of compact anchor pools         */
  const void* const* v_anchor;
  int64_t anchor_rows;           /* rows of each anchor pool; every chunk of probe_batch must lie inside                  */
  const int32_t* crit_layers;    /* host [n_crit], ascending 0-based layer indices of L*                           */
  int32_t n_crit;
  double ratio;                  /* rho                                                                             */
  const int32_t* tokens;         /* dev int32 [N + Lq] token ids by request position                                */
  void* const* k_fused;          /* host array [L] of dev [t_stride][Hkv][d]: receives KV^Fuse of every layer       */
  void* const* v_fused;
  float* scores;                 /* dev [n_stride]   out: Eq. 20 scores                                             */
  int32_t* sel;                  /* dev [n_stride]   out: P ascending                                               */
  int32_t* n_sel;                /* dev [1]                                                                         */
  void* hidden_out;              /* dev [n_R][hidden] out: final hidden states of the rows R (P ascending, then U)  */
  int32_t overlap;               /* != 0: layer-ahead loading on a second stream (a8); 0: serial, for the ablation  */
  int32_t stages;                /* 0 or 3: both stages; 1: stage 1 only (scores, sel, n_sel are produced, no layer is
                                    recomputed); 2: stage 2 only (sel / n_sel are INPUTS, e.g. from another selector: they
                                    must hold EXACTLY qcf_n_select(N, ratio) positions — every stage-2 row count is derived
                                    on the host from `ratio`; pass ratio = |P| / N for an external selection of another size.
                                    This mode reads n_sel[0] back once (one stream synchronisation before the first launch)
                                    and returns QCF_ERR_INVALID_ARG on a mismatch)                                        */
  double load_gbps;              /* > 0: emulate a KV store of this bandwidth (GB/s): every pool load on the loader stream
                                    is held until bytes / load_gbps have elapsed since it started (the
                                    bandwidth-constrained loading experiment); 0: unthrottled                            */
} qcf_fuse_args;
QCF_API qcf_status qcf_stack_fuse(qcf_stack* s, const qcf_batch* main_batch, const qcf_batch* probe_batch,
                                  const qcf_fuse_args* args, void* stream);

#ifdef __cplusplus
}
#endif
#endif /* QCF_H_ */
