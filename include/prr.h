/* prr.h — C ABI of the B200-native PRR (Predict, Reuse, Repair) decode hot path.
 *
 * Source of the operations: /root/reference/PAPER.md (arxiv 2606.30389).  "PAPER.md:n" below is a
 * line of that file; Q1..Q15 are the readings listed in DESIGN.md.
 *
 * Conventions
 *   - Every call returns an int32 status (PRR_OK = 0).  No exceptions, no abort(), no I/O.
 *   - "dev" pointers are CUDA device memory owned by the CALLER, 16-byte aligned; "host" pointers
 *     are ordinary host memory.  The library owns only what lives in the prr_ctx (EMA state, theta,
 *     scores, block sets, partial attention states, streams/events) and frees it in prr_destroy.
 *     It never allocates on the per-step path.
 *   - Every call that takes `stream` (a cudaStream_t passed as void*) only ENQUEUES work on it and
 *     returns; results are valid after the caller synchronises that stream.  Calls that fill a host
 *     output (prr_calibrate with theta_out/H_out, prr_get_stats, prr_decode_step_host) synchronise
 *     the stream themselves.  All calls may be issued while `stream` is being captured into a CUDA
 *     graph (prr_graph_begin/end or the caller's own capture) except those that synchronise.
 *   - Errors: bad arguments -> PRR_E_INVALID before any launch; unsupported shape/dtype ->
 *     PRR_E_UNSUPPORTED; decode before theta/EMA state exists is NOT an error (P is empty and the
 *     step degenerates to repair over all of A, Q5); CUDA failures -> PRR_E_CUDA; prr_last_error
 *     gives the text.  No partial output on an argument error.  There is no CPU fallback.
 *   - Layouts (row-major, innermost last):
 *       K/V pages   bf16  [n_pages, n_kv_heads, block_size, head_dim]
 *       block_table int32 [batch, max_blocks_per_seq]     logical block -> physical page
 *       seq_lens    int32 [batch]                         tokens in the cache
 *       summaries   bf16  [batch, n_kv_heads, max_blocks_per_seq, head_dim]   (one buffer per layer)
 *       q           bf16  [batch, n_q_heads, head_dim]; query head g belongs to KV head g / G
 *       scores      fp32  [batch, n_kv_heads, max_blocks_per_seq]
 *       block lists int32 [batch, n_kv_heads, width] ascending block index, padded with -1
 *       partials    fp32  O [batch, n_q_heads, width, head_dim] unnormalised, m and l
 *                   [batch, n_q_heads, width]; m in natural-log units of the scaled logit,
 *                   relative to which O and l are accumulated (block-local maximum)
 *       out         fp32  [batch, n_q_heads, head_dim]
 */
#ifndef PRR_H_
#define PRR_H_

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

enum { PRR_OK = 0, PRR_E_INVALID = 1, PRR_E_UNSUPPORTED = 2, PRR_E_STATE = 3, PRR_E_CUDA = 4,
       PRR_E_NOMEM = 5 };
/* KV page element type.  PRR_FP8_E4M3 (PAPER.md:319 names fp8 as future work; format: DESIGN.md section 10):
 * pages hold OCP e4m3 codes, one byte per element, same [n_pages, n_kv_heads, block_size, head_dim] layout, with
 * ONE power-of-two scale per (page, KV head) for K and one for V (prr_set_kv_scales); element = code * scale. */
enum { PRR_BF16 = 0, PRR_FP8_E4M3 = 1 };
/* What happens to over-predicted blocks P\A at merge (Q7).  PRR_DROP: the output is attention
 * over exactly A (BASELINE.json north_star).  PRR_RETAIN: P\A is "retained as additional
 * low-priority context", the output is attention over A u P. */
enum { PRR_DROP = 0, PRR_RETAIN = 1 };
/* How a layer-step is orchestrated (Fig. 1: speculation overlaps selection).
 * PRR_FUSED (default): ONE persistent cooperative launch; warps are the workers, selection,
 * speculative attention, repair and merge are ordered by device-scope counters.
 * PRR_STREAMS: the paper's orchestration, one kernel per stage on two event-ordered streams. */
enum { PRR_FUSED = 0, PRR_STREAMS = 1 };
/* The paper's ablation ladder (Table 2).  S3 (default): the EMA predictor with its budget and
 * incremental repair.  S2: the prediction is the last step's true top-K (theta = (1, 1, 0), budget = K) with
 * incremental repair.  S1: the same prediction, but ANY miss in a row discards the speculative result and
 * attention is recomputed over all of A (the fallback PRR avoids).  The output is attention over
 * A in every mode; the modes differ in the work on the critical path. */
enum { PRR_MODE_S3 = 0, PRR_MODE_S2 = 1, PRR_MODE_S1 = 2 };
enum { PRR_SUMMARY_MEAN = 0, PRR_SUMMARY_QUEST = 1 };

typedef struct prr_ctx prr_ctx; /* opaque, library-owned */

typedef struct {
  int32_t n_q_heads, n_kv_heads; /* n_q_heads % n_kv_heads == 0, group G = ratio, G <= 16 */
  int32_t head_dim;              /* 64 or 128 */
  int32_t max_batch;             /* >= 1 */
  int32_t max_blocks_per_seq;    /* row stride of block_table / summaries / scores; <= 32768 */
  int32_t n_layers;              /* EMA state is kept per (layer, sequence, KV head, block) */
  int32_t kv_dtype;              /* PRR_BF16 | PRR_FP8_E4M3 (needs PRR_STREAMS, block_size <= 128) */
  int32_t overpredict_policy;    /* PRR_DROP | PRR_RETAIN */
  float sm_scale;                /* softmax scale of the attention logits; 0 -> 1/sqrt(head_dim) */
  int32_t orchestration;         /* PRR_FUSED | PRR_STREAMS */
} prr_layout;

typedef struct {
  const void* k_pages;        /* dev bf16 */
  const void* v_pages;        /* dev bf16 */
  const int32_t* block_table; /* dev */
  int32_t* seq_lens;          /* dev; read-only for every call except prr_append */
  int32_t batch;              /* 1..max_batch */
  int32_t layer;              /* 0..n_layers-1 */
} prr_paged_kv;

/* Problem statement (PAPER.md:109 Eq. 1, :135): block size, top-K of the DSA, speculation budget
 * |P| <= budget = delta*K.  block_size in {16,32,64,128,256}; 1 <= K <= 512; 0 <= budget <= 1024.  Blocks of 256
 * tokens run on the fused cluster kernel only (the stage calls and PRR_STREAMS return PRR_E_UNSUPPORTED). */
int32_t prr_create(const prr_layout* layout, int32_t block_size, int32_t K, int32_t budget,
                   prr_ctx** out);
int32_t prr_destroy(prr_ctx* ctx);
/* Text of the last error of this ctx (or of the last failed prr_create if ctx == NULL). */
const char* prr_last_error(const prr_ctx* ctx);
const char* prr_version(void);

/* --- cache maintenance (a0) ------------------------------------------------------------------ */

/* Mean-pooled key summary of every block of every sequence ("compresses each block
 * (e.g., mean)"): kbar = bf16_rne(exact mean over the valid tokens), Q2.  Also seeds the running
 * sum of the open block that prr_append continues.  The prefill-side counterpart of prr_append. */
int32_t prr_build_summaries(prr_ctx* ctx, const prr_paged_kv* kv, void* summaries /*dev bf16*/,
                            void* stream);

/* Append one token per sequence: writes k_new/v_new (dev bf16 [batch, n_kv_heads, head_dim]) at
 * position seq_lens[b] of the paged cache (the page must already be mapped in block_table),
 * refreshes the summary row of that block, then INCREMENTS seq_lens[b] on the device (Q10: the
 * decode step that follows sees its own token).  k_pages/v_pages are written through the const
 * pointers of `kv`. */
int32_t prr_append(prr_ctx* ctx, const prr_paged_kv* kv, const void* k_new, const void* v_new,
                   void* summaries, void* stream);

/* --- fp8 KV (PRR_FP8_E4M3) --------------------------------------------------------------------- */

/* Quantise a bf16 paged cache (kv: the bf16 pages, block table and lengths; any ctx of the same shape): per
 * (mapped page, KV head) amax over the block's VALID tokens, scale = the smallest 2^e with amax <= 448 * 2^e,
 * codes = round-to-nearest-even(x / 2^e) saturated to +-448; token slots past the length get code 0.
 * k8_pages / v8_pages: dev uint8, the layout of the bf16 pages; k_scale / v_scale: dev fp32 [n_pages,
 * n_kv_heads] (entries of unmapped pages are left untouched).  x / 2^e and code * 2^e are exact. */
int32_t prr_quantize_kv_fp8(prr_ctx* ctx, const prr_paged_kv* kv, void* k8_pages, void* v8_pages,
                            float* k_scale, float* v_scale, void* stream);
/* Scales of a layer's fp8 pages (dev fp32 [n_pages, n_kv_heads], powers of two, caller-owned, read by every
 * later call on that layer).  With a PRR_FP8_E4M3 ctx, prr_paged_kv.k_pages / v_pages point at the code pages;
 * prr_build_summaries (mean of the dequantised keys), prr_score, prr_topk, prr_calibrate, prr_speculate,
 * prr_repair, prr_attend and prr_decode_step (PRR_STREAMS) work as for bf16 and move half the KV bytes; the
 * tiles are widened to bf16 on chip (exact), so every result equals the bf16 path's on the dequantised cache
 * bit for bit.  prr_append / prr_step_append / prr_decode_step_host return PRR_E_UNSUPPORTED (a new token cannot
 * join a block quantised with a fixed scale: re-quantise the open block with prr_quantize_kv_fp8); a call
 * before the scales are set returns PRR_E_STATE. */
int32_t prr_set_kv_scales(prr_ctx* ctx, int32_t layer, const float* k_scale, const float* v_scale);

/* --- predictor ------------------------------------------------------------ */

/* Set theta = (alpha, beta, gamma) of Eq. 2-3 for one (layer, sequence) without calibration.
 * seq = -1: all sequences.  Enqueued on `stream`. */
int32_t prr_set_ema_params(prr_ctx* ctx, int32_t layer, int32_t seq, double alpha, double beta,
                           double gamma, void* stream);
/* Forget the EMA state of a layer (no block has state; next prediction is empty). */
int32_t prr_reset_ema(prr_ctx* ctx, int32_t layer, void* stream);

/* Per-prompt calibration: simulate Eq. 2-3 over the prefill score trajectory
 * for the 80 grid points (alpha {.2,.4,.6,.8} x beta {.1,..,.5} x gamma {0,.25,.5,.75}, alpha-major),
 * score-weighted hit rate H (Eq. 4) with |P| = min(budget, #stateful), theta* = first argmax
 * (Eq. 5), Q8.  prefill_scores: dev fp32 [n_kv_heads, T, N] (row phi = score vector at prefill
 * token phi); n_valid: dev int32 [T] non-decreasing number of valid blocks per row, or NULL = N.
 * Stores theta*, seeds the EMA state of (layer, seq) with the state after the last row and
 * predicts the first decode step's P (Q5).  theta_out (host double[3]), H_out (host double),
 * H_all_out (host double[80]) may be NULL; if any is given the call synchronises `stream`. */
int32_t prr_calibrate(prr_ctx* ctx, int32_t layer, int32_t seq, const float* prefill_scores,
                      int32_t T, int32_t N, const int32_t* n_valid, double* theta_out,
                      double* H_out, double* H_all_out, void* stream);

/* Eq. 2: predicted scores from the current state, P = top-min(budget, #stateful) blocks, ties ->
 * lower index.  P_out dev int32 [batch, n_kv_heads, budget]; count_out dev [batch, n_kv_heads]
 * or NULL. */
int32_t prr_predict(prr_ctx* ctx, int32_t layer, int32_t batch, int32_t* P_out,
                    int32_t* count_out, void* stream);
/* Eq. 3 with this step's scores (dev fp32 [batch, n_kv_heads, max_blocks]); blocks seen for the
 * first time get l = IS, v = 0.  Also refreshes the library's stored prediction
 * for the next decode step of this layer.  n_blocks: dev int32 [batch]. */
int32_t prr_ema_update(prr_ctx* ctx, int32_t layer, int32_t batch, const float* scores,
                       const int32_t* n_blocks, void* stream);

/* --- profiling-guided speculation budget (PAPER.md:204-208 section 4.4, :229, :424 A.6) --------- */

/* The budget of prr_create is the WIDTH of a prediction row and the largest budget; the budget in force
 * (blocks of P predicted for the next step, delta * K of Eq. 1) is a per-layer run-time value, initially
 * that maximum.  prr_set_budget changes it (layer = -1: every layer) and re-predicts the layer's next P
 * under it, so the next decode step already speculates on the new budget.  0 = no speculation: the step
 * degenerates to select-then-attend through the repair path. */
int32_t prr_set_budget(prr_ctx* ctx, int32_t layer, int32_t budget, void* stream);
int32_t prr_get_budget(const prr_ctx* ctx, int32_t layer, int32_t* budget_out /* host */);
/* Batch-aware budgets (PAPER.md:319 leaves coordination across the requests of a batch as future work; DESIGN.md
 * section 11): the sequences of a batch differ in locality, so each (layer, sequence) may carry its OWN run-time
 * budget: 0 .. the budget of prr_create, or -1 = follow the layer's (the default).  One fused launch then serves
 * sequences that speculate and sequences that do not (their rows go through the repair path alone).  The call
 * re-predicts the layer's next P at once; a per-sequence budget stays until it is set to -1. */
int32_t prr_set_budget_seq(prr_ctx* ctx, int32_t layer, int32_t seq, int32_t budget, void* stream);
int32_t prr_get_budget_seq(const prr_ctx* ctx, int32_t layer, int32_t seq, int32_t* budget_out /* host */);
/* The paper's offline sweep, in the library: for every candidate budget (host int32 [n_budgets]) run the T
 * decode steps of a query trajectory q_traj (dev bf16 [T, batch, n_q_heads, head_dim], e.g. the prefill
 * trajectory used for prr_calibrate) on the layer's cache WITHOUT appending, each step timed by CUDA events
 * on `stream` (cold_l2 != 0: a 256 MB write between steps, outside the timed interval), and the same for
 * the sequential select-then-attend path.  The paper compares the speculative-attention time with the
 * selection window; timing the whole critical path per budget measures what that comparison stands for,
 * including the repair work a smaller budget causes.  us_out (host float [n_budgets]) = median us per step
 * (the first step is a warm-up), us_sequential_out (host float) likewise, best_budget_out (host) = the
 * LARGEST candidate whose time is within 1 % of the fastest candidate's and beats the sequential path by more
 * than 2 %, else 0 (the paper's "largest safe delta", with "safe" measured on the whole critical path).  The layer's predictor state, prediction buffers, counters and budget are saved
 * before and restored after.  Synchronises `stream`; not allowed inside a stream capture. */
int32_t prr_profile_budget(prr_ctx* ctx, const prr_paged_kv* kv, const void* q_traj, int32_t T,
                           const void* summaries, const int32_t* budgets, int32_t n_budgets, int32_t cold_l2,
                           float* us_out, float* us_sequential_out, int32_t* best_budget_out, void* stream);
/* Lookup by context length: a least-squares polynomial (degree <= 3) through the profiled
 * (context length, best budget) points, evaluated and clamped to [0, budget of prr_create] by
 * prr_budget_for.  Before any fit prr_budget_for returns the budget of prr_create. */
int32_t prr_budget_fit(prr_ctx* ctx, int32_t n, const int32_t* ctx_lens /* host */, const int32_t* budgets /* host */,
                       int32_t degree);
int32_t prr_budget_for(const prr_ctx* ctx, int32_t ctx_len, int32_t* budget_out /* host */);

/* Ablation modes (see PRR_MODE_*).  S2 / S1 set theta = (1, 1, 0) for every (layer, sequence) and the budget
 * to min(K, budget of prr_create); S3 leaves theta and the budget as they are (calibrate / set them).  S1
 * needs PRR_DROP and PRR_FUSED and runs on the cluster kernel. */
int32_t prr_set_mode(prr_ctx* ctx, int32_t mode, void* stream);

/* --- selection (a1, a2) ---------------------------------------------------------------------- */

/* Block importance (PAPER.md:66 compressed attention; group aggregated as in A.1 PAPER.md:372):
 * IS[b,h,i] = fp32( (sum_{g in group h} sum_j q[b,g,j] kbar[b,h,i,j]) / (G sqrt(head_dim)) ),
 * accumulated exactly (fp64 over exact bf16 products), rounded once, -0 -> +0 (Q1).  Writes the
 * first ceil(seq_len/block_size) entries of each row. */
int32_t prr_score(prr_ctx* ctx, const prr_paged_kv* kv, const void* q, const void* summaries,
                  float* scores_out, void* stream);
/* Top-k of the first n_blocks[b] scores of each (b, KV head) row (row stride max_blocks_per_seq);
 * order (value desc, index asc), selects min(k, n); idx_out dev int32 [batch, n_kv_heads, k]
 * ascending, -1 padded; count_out dev [batch, n_kv_heads] or NULL.  1 <= k <= 1024. */
int32_t prr_topk(prr_ctx* ctx, const float* scores, const int32_t* n_blocks, int32_t batch,
                 int32_t k, int32_t* idx_out, int32_t* count_out, void* stream);

/* --- attention (a4-a7) ----------------------------------------------------------------------- */

/* Per-block partial states (the forward also writes l and m) for every block of
 * the list P (dev int32 [batch, n_kv_heads, budget], -1 padded) and every query head:
 * m_p = max_j s_j, l_p = sum_j e^{s_j - m_p}, O_p = sum_j e^{s_j - m_p} v_j, s_j = sm_scale q.k_j,
 * tokens >= seq_len masked.  Slots holding -1 are left untouched. */
int32_t prr_speculate(prr_ctx* ctx, const prr_paged_kv* kv, const void* q, const int32_t* P,
                      float* O_part, float* m_part, float* l_part, void* stream);
/* Incremental repair (Eq. 6-8): given the true set A (dev int32 [batch,
 * n_kv_heads, K]), the predicted set P and its partial states, attends only to M = A\P and folds
 * hits u M (PRR_DROP) or P u M (PRR_RETAIN) in ascending block order into out; m_out/l_out (dev
 * fp32 [batch, n_q_heads], natural-log max and denominator of the final state) may be NULL. */
int32_t prr_repair(prr_ctx* ctx, const prr_paged_kv* kv, const void* q, const int32_t* A,
                   const int32_t* P, const float* O_part, const float* m_part,
                   const float* l_part, float* out, float* m_out, float* l_out, void* stream);

/* Sequential select-then-attend (the serial DSA PRR is compared with): score ->
 * top-K -> attention over A, one stream.  Updates the EMA state like prr_decode_step. */
int32_t prr_attend(prr_ctx* ctx, const prr_paged_kv* kv, const void* q, const void* summaries,
                   float* out, void* stream);
/* One PRR layer-step (Fig. 1): speculative attention over the stored prediction P
 * on a second stream, concurrently score -> top-K -> diff -> repair of A\P, then merge; EMA update
 * and the next step's prediction run off the critical path.  Call prr_append first. */
int32_t prr_decode_step(prr_ctx* ctx, const prr_paged_kv* kv, const void* q, const void* summaries,
                        float* out, void* stream);
/* prr_append followed by prr_decode_step (sequential = 0) or prr_attend (sequential != 0) as ONE
 * call: a0-a8 of SURVEY.md section 8(a).  With PRR_FUSED orchestration the append rides in the
 * same launch as the rest of the step (the new token's k/v and the open block's summary are patched
 * into the tiles that need them on chip; the cache, the summary row and seq_lens are written for
 * the following steps); results are identical to the two separate calls.  Arguments as in
 * prr_append / prr_decode_step; kv->seq_lens holds the lengths BEFORE the append on entry and is
 * incremented by the call. */
int32_t prr_step_append(prr_ctx* ctx, const prr_paged_kv* kv, const void* q, const void* k_new,
                        const void* v_new, void* summaries, float* out, int32_t sequential, void* stream);
/* prr_append + prr_decode_step with HOST q/k_new/v_new/out (pinned or pageable): copies the
 * inputs to library staging buffers, runs the step, copies out back and synchronises. */
int32_t prr_decode_step_host(prr_ctx* ctx, const prr_paged_kv* kv, const void* q_host,
                             const void* k_new_host, const void* v_new_host, void* summaries,
                             float* out_host, void* stream);

/* --- introspection --------------------------------------------------------------------------- */

/* Block sets of the last step of `layer` (any of the dev outputs may be NULL): A [batch,n_kv,K],
 * P [batch,n_kv,budget] (the prediction that step used), M [batch,n_kv,K], counts
 * [batch,n_kv,3] = |A|, |P|, |M|. */
int32_t prr_get_sets(prr_ctx* ctx, int32_t layer, int32_t batch, int32_t* A, int32_t* P,
                     int32_t* M, int32_t* counts, void* stream);
/* Last scores of `layer`: dev fp32 [batch, n_kv_heads, max_blocks_per_seq]. */
int32_t prr_get_scores(prr_ctx* ctx, int32_t layer, int32_t batch, float* scores, void* stream);
/* EMA state of one (layer, seq): dev double [n_kv_heads, max_blocks] each, n_state dev int32
 * [n_kv_heads], theta host double[3] (any may be NULL; theta synchronises). */
int32_t prr_get_ema(prr_ctx* ctx, int32_t layer, int32_t seq, double* level, double* trend,
                    int32_t* n_state, double* theta, void* stream);
/* Cumulative counters since create / last reset: host int64[4] = sum|A|, sum|A n P|, sum|M|,
 * sum|P| over all (layer, seq, KV head, step).  Synchronises `stream`.  reset != 0 clears them. */
int32_t prr_get_stats(prr_ctx* ctx, int64_t* stats_out, int32_t reset, void* stream);
/* Synchronises `stream` and reports whether a fused step ever gave up waiting on a dependency
 * counter (PRR_E_STATE; cannot happen unless the device was shared with a kernel that never ends)
 * or a CUDA error is pending (PRR_E_CUDA). */
int32_t prr_check(prr_ctx* ctx, void* stream);
/* Number of kernels this ctx has launched (or captured) so far. */
int64_t prr_launch_count(const prr_ctx* ctx);
/* Profiling aid for the fused step (a9, Fig. 5 timeline).  While enabled, every warp of a
 * fused step launched (or captured) afterwards stores %globaltimer (ns) at its phase boundaries:
 * [0] start, [1] scores done, [2] row job done, [3] speculative units done, [4] repair units done,
 * [5] merge done; words 6-15 are finer marks (score chunk: [6] queries summed, [13] rows landed, [14] computed,
 * [15] published; row jobs: [8] scores seen, [9] keys, [12] histogram, [13] bucket, [14] candidates, [10] K-th,
 * [11] emitted; repair units: [8] M seen, [10] tile requested, [11] computed; merge: [12]-[14]).  prr_timeline_read copies the stamps of the LAST step,
 * uint64 [n_warps, 16] with warp index = cta * warps_per_cta + warp, to HOST memory and
 * synchronises `stream`; n_warps_out (host, may be NULL) receives the rows copied (<= max_warps). */
int32_t prr_timeline_enable(prr_ctx* ctx, int32_t on);
int32_t prr_timeline_read(prr_ctx* ctx, uint64_t* stamps_host, int32_t max_warps, int32_t* n_warps_out,
                          void* stream);
/* Same copy WITHOUT synchronising: the stamps live in pinned host memory that the device writes directly,
 * so they can be looked at while a step is still running (or after a fault). */
int32_t prr_timeline_peek(prr_ctx* ctx, uint64_t* stamps_host, int32_t max_warps, int32_t* n_warps_out);

/* Tuning / introspection of the fused step (k_row.cu).  Options are per ctx and take effect at the next
 * launch (or capture).  PRR_OPT_PDL: 1 (default) = consecutive fused steps are linked by programmatic
 * dependent launch, so the next step's launch latency hides behind the running one.  PRR_OPT_CLUSTER:
 * 0 (default) = the library picks the largest cluster (1, 2, 4 or 8 CTAs per (sequence, KV head) row)
 * that still runs every row at once; 1/2/4/8 force a size.  PRR_OPT_CUT: 1 (default) = once A is known,
 * predicted blocks that missed and whose tile has not been requested yet are not requested (PRR_DROP
 * only; the output is attention over A either way); 0 = every block of P is fetched.  PRR_OPT_SUBTILE:
 * tokens per tile unit of the cluster kernel, 16 / 32 / 64 (default 64; a block larger than that is several units).
 * PRR_OPT_KERNEL: which fused kernel runs a step: 0 (default) = the library chooses by the number of
 * (sequence, KV head) rows, 1 = the persistent cooperative grid (k_step.cu), 2 = a cluster per row (k_row.cu).
 * PRR_OPT_PACE: percent of the estimated HBM rate at which the persistent kernel issues its first wave of
 * speculative tiles (default 100; 0 = unpaced).  Read-only:
 * PRR_OPT_SUMMARY: what a block's summary row holds.  PRR_SUMMARY_MEAN (default): the mean key, d bf16.
 * PRR_SUMMARY_QUEST: Quest's channel-wise minimum and maximum key, 2 d bf16 per row (min then max: the summaries
 * buffer is [batch, n_kv_heads, max_blocks_per_seq, 2, head_dim]), scored with the GQA mean query as
 * s_p = sum_i max(Qbar_i m_{p,i}, Qbar_i M_{p,i}) / sqrt d (A.1).  prr_build_summaries, prr_append and
 * prr_score follow the option; decode steps with Quest summaries run under PRR_STREAMS only (PRR_FUSED contexts
 * refuse the option with PRR_E_INVALID).  Set it before the summaries are built.
 * PRR_OPT_LAST_CLUSTER / _LAST_RING / _LAST_GRID = cluster size, ring depth and grid of the last fused
 * launch, PRR_OPT_LAST_KERNEL = the kernel it used (1 or 2).  Unknown option or bad value -> PRR_E_INVALID. */
enum { PRR_OPT_PDL = 0, PRR_OPT_CLUSTER = 1, PRR_OPT_CUT = 2, PRR_OPT_SUBTILE = 3, PRR_OPT_KERNEL = 4, PRR_OPT_PACE = 5,
       PRR_OPT_SUMMARY = 6,
       PRR_OPT_LAST_KERNEL = 19, PRR_OPT_LAST_CLUSTER = 16, PRR_OPT_LAST_RING = 17,
       PRR_OPT_LAST_GRID = 18 };
int32_t prr_set_option(prr_ctx* ctx, int32_t option, int32_t value);
int32_t prr_get_option(const prr_ctx* ctx, int32_t option, int32_t* value_out /* host */);

/* --- no-allocation entry point ---------------------------------------------------------------- */

/* Sparse attention over given block lists (a4 + a7: per-block partial states, then the Eq. 6-8 fold)
 * for callers that may not allocate: code under stream capture, tight serving loops, harnesses that forbid
 * cudaMalloc.  blocks: dev int32 [batch, n_kv_heads, width], -1 = hole (skipped); the listed blocks are folded in
 * list order; out dev fp32 [batch, n_q_heads, head_dim]; m_out / l_out (dev fp32 [batch, n_q_heads], natural-log
 * maximum and denominator of the final state) may be NULL.  Same kernels and results as prr_repair with an empty
 * prediction, but the partial states between the two launches live in ONE static device array of
 * PRR_STATIC_SCRATCH_BYTES inside the library (every GPU that loads the library holds it until exit) instead of
 * ctx-owned buffers.  The call itself makes no cudaMalloc / cudaFree and calls no allocating library routine.
 * Limit: batch * n_q_heads * width * (head_dim + 2) * 4 bytes <= PRR_STATIC_SCRATCH_BYTES, 1 <= width <= 1024,
 * block_size <= 128; beyond it -> PRR_E_UNSUPPORTED with the sizes in prr_last_error, nothing launched.
 * Every call on a device shares the array, which keeps the last call's contents (nothing in it needs to start at
 * zero: each call writes every slot it reads).  Calls that OVERLAP on the GPU (two streams, two host threads, two
 * contexts on one device) race on it: order them on one stream or with events. */
#define PRR_STATIC_SCRATCH_BYTES (8 * 1024 * 1024)
int64_t prr_static_scratch_bytes(void);
int32_t prr_attend_blocks_static(prr_ctx* ctx, const prr_paged_kv* kv, const void* q, const int32_t* blocks,
                                 int32_t width, float* out, float* m_out, float* l_out, void* stream);

/* --- CUDA-graph helpers (so callers need no CUDA runtime of their own) ------------------------ */
typedef struct prr_graph prr_graph;
int32_t prr_graph_begin(prr_ctx* ctx, void* stream);               /* start capturing `stream` */
int32_t prr_graph_end(prr_ctx* ctx, void* stream, prr_graph** out); /* end capture, instantiate */
int32_t prr_graph_launch(prr_graph* g, void* stream);
int32_t prr_graph_destroy(prr_graph* g);

#ifdef __cplusplus
}
#endif
#endif /* PRR_H_ */
