/*
 * darts.h — C-ABI of the B200-native DARTS group-rollout decoder (arxiv/paper_2605_30859).
 *
 * What the library computes (citations: PAPER.md:<line>, section):
 *   For each prompt q_i of a rollout batch, M'_i = Kp[i] redundant trajectories are decoded
 *   autoregressively ("intra-prompt redundant rollout", §4.1.1) over ONE shared,
 *   paged prompt KV cache; after every lock-step decode step the distribution-aware rule of
 *   Alg. 2 (PAPER.md:465-477, prose :426-432, :479) is applied per prompt on the device:
 *     - M'_i <  M_up : dual-end length sampling — wait for the whole pool, keep the S = K - L_long
 *       shortest and the L_long longest trajectories, the longest drawn only from trajectories that
 *       did not hit the length limit (§4.1.2);
 *     - M'_i >= M_up : shortest-only sampling with proactive early stop — as soon as K valid
 *       trajectories exist the other M'_i - K are halted (§4.3.1).
 *   Finished / pruned rows are compacted out of the batch on the device.
 *   Notation: the paper's M is `K` here, M'_i is `Kp[i]`, the paper's K (short count) is K - L_long.
 *
 * Conventions
 *   - Every function returns a darts_status (0 = DARTS_OK).  No exceptions, no exit(), no stdout.
 *     darts_last_error(ctx) returns a ctx-owned, NUL-terminated description of the last failure.
 *   - "device" pointers are CUDA device pointers allocated by the caller (e.g. with torch); "host"
 *     pointers are ordinary host memory.  The library never frees caller memory.  Weights are
 *     BORROWED: the pointers in darts_weights must stay valid until darts_destroy.
 *   - The library allocates no device memory of its own: everything it needs (KV page pool, page
 *     tables, row state, activations) is carved out of the caller's workspace, whose size
 *     darts_workspace_bytes reports.  It owns a few bytes of pinned host memory for counters.
 *   - All work is enqueued on runtime_desc.stream (a cudaStream_t passed as void*).  Only
 *     darts_rollout, darts_get_results, darts_get_counters and darts_debug_* synchronise.
 *   - One ctx = one GPU = one stream; a ctx is not thread-safe.
 *   - There is no CPU fallback and no other backend: on a device that is not sm_100 every entry
 *     point that needs the GPU returns DARTS_ERR_UNSUPPORTED.
 *
 * Environment: the library as built by build.py reads none.  A -DDARTS_PROFILING build (DARTS_NVCC_FLAGS=-DDARTS_PROFILING) reads, at
 * darts_create, DARTS_NO_PDL=1 (ordinary stream launches instead of programmatic dependent launch) and DARTS_SKIP=<bitmask> (drop one
 * kernel class of every layer: results are garbage, only the step time means anything; profiles/r1_live_cost_by_kernel.md).
 *
 * Layouts
 *   - Projections are [out_features, in_features] row-major in the model dtype (F32 or BF16).
 *     wqkv rows: n_q_heads q-heads, then n_kv_heads k-heads, then n_kv_heads v-heads (head_dim rows each).
 *     wgu rows:  ffn gate rows, then ffn up rows.  MoE: wgu_e [E][2*expert_ffn][d], wd_e [E][d][expert_ffn],
 *     router wr [E][d] always F32.
 *   - Rows (trajectories) are numbered group-major: row = sum_{i'<i} Kp[i'] + j.
 *   - KV cache (library-owned, inside the workspace): pages of page_size tokens,
 *     [layer][page][kv_head][K|V][token][head_dim] (the K and V tiles of one (page, head) are adjacent; for bf16 /
 *     head_dim 128 the 16-byte chunks of a token row are XOR-permuted by token & 7); a row's page table is
 *     [its prompt's shared prefix pages || its own suffix pages]; the suffix starts on a fresh page,
 *     so the K' samples of a prompt share the prefix pages without any copy.
 */
#ifndef DARTS_H_
#define DARTS_H_

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef int32_t darts_status;
enum {
  DARTS_OK = 0,
  DARTS_ERR_INVALID_ARG = 1,       /* NULLs, K > Kp[i], Kp[i] > 32, L_long >= K, G > max_prompts, ... */
  DARTS_ERR_UNSUPPORTED = 2,       /* head_dim / page_size / dtype combination, non-sm_100 device */
  DARTS_ERR_KV_POOL_EXHAUSTED = 3, /* page pool ran dry; the rollout is stopped, nothing is corrupted */
  DARTS_ERR_WORKSPACE_TOO_SMALL = 4,
  DARTS_ERR_CUDA = 5,              /* sticky; darts_last_error carries cudaGetErrorString */
  DARTS_ERR_BAD_STATE = 6          /* e.g. darts_decode_step before darts_prefill */
};

enum { DARTS_F32 = 0, DARTS_BF16 = 1 };

/* Row status (rows "reaching the system length limit" are incomplete/invalid = TRUNC;
 * rows halted by the early-stop signal = PRUNED). */
enum { DARTS_ROW_ACTIVE = 0, DARTS_ROW_VALID = 1, DARTS_ROW_TRUNC = 2, DARTS_ROW_PRUNED = 3 };

/* Selection mode.  AUTO is the paper's rule: shortest-only + early stop iff Kp[i] >= M_up. */
enum { DARTS_MODE_AUTO = 0, DARTS_MODE_DUAL_END = 1, DARTS_MODE_SHORTEST_EARLY_STOP = 2 };

enum {
  DARTS_FLAG_DUMP_LOGITS = 1,       /* keep fp32 logits of every row of the last step for darts_debug_logits */
  DARTS_FLAG_NO_PREFIX_SHARING = 2, /* A/B switch: attention re-reads the prefix once per row, not per group */
  DARTS_FLAG_PROFILE_ATTENTION = 4, /* bracket layer 0's attention of every decode step with CUDA events (bench roofline) */
  DARTS_FLAG_LM_HEAD_TILES = 16,    /* A/B switch: decode LM head on the 128 x 128 tile kernel instead of the persistent swap-AB kernel (both
                                     * sample the same distribution from the same Philox stream) */
  DARTS_FLAG_CTA_PAIRS = 32,        /* dense projections on the CTA-pair (tcgen05 cta_group::2) stream-K kernel: two SMs share the activation block
                                     * of one MMA of 256 weight rows (a third less L2 -> SM operand traffic from ~256 live rows on) */
  DARTS_FLAG_DUMP_HIDDEN = 8        /* keep the fp32 residual stream of every layer boundary of the last pass for darts_debug_hidden
                                     * ((n_layers + 1) x rows x d_model floats of workspace; parity only) */
};

typedef struct {
  int32_t n_layers, d_model, n_q_heads, n_kv_heads, head_dim;
  int32_t ffn;                         /* dense SwiGLU width (0 for MoE / attention-only) */
  int32_t vocab;                       /* 0: attention-only context (config 2), no model weights needed */
  int32_t n_experts, top_k, expert_ffn;/* 0 => dense */
  int32_t dtype;                       /* DARTS_F32 | DARTS_BF16: weights, activations fed to GEMMs, KV cache */
  int32_t qk_norm;                     /* 1: per-head RMSNorm of q and k before RoPE */
  float rope_theta, rms_eps;
  int32_t eos_id;                      /* -1 disables natural EOS */
} darts_model_desc;

/* Device pointers; per-layer members are HOST arrays of n_layers device pointers. */
typedef struct {
  const void *embed, *final_norm, *lm_head;
  const void *const *attn_norm, *const *wqkv, *const *q_norm, *const *k_norm, *const *wo;
  const void *const *mlp_norm, *const *wgu, *const *wd;
  const void *const *wr, *const *wgu_e, *const *wd_e;
} darts_weights;

typedef struct {
  int32_t page_size;                   /* tokens per KV page (64 for the tuned bf16 path) */
  int32_t n_pages;                     /* pages in the pool (shared by all layers' slabs) */
  int32_t max_rows;                    /* >= sum Kp[i] */
  int32_t max_prompts, max_prompt_len, max_new;
  int32_t prefill_chunk;               /* max prompt tokens per prefill pass (>= max_prompt_len); 0 = default */
  uint32_t flags;
  void *workspace;                     /* device; >= darts_workspace_bytes() */
  size_t workspace_bytes;
  void *stream;                        /* cudaStream_t */
} darts_runtime_desc;

/* Per-prompt rule parameters (Alg. 2 inputs "Target Size M, Dual-End Short Size K"). */
typedef struct {
  int32_t K;                           /* keep count (paper's M) */
  int32_t L_long;                      /* dual-end long count (paper's L; 1 in all main experiments) */
  int32_t M_up;                        /* saturation threshold (paper: 2M); 0 => 2*K */
  int32_t mode;                        /* DARTS_MODE_* */
} darts_policy;

/* Caller buffers (HOST unless a member says device) filled by darts_get_results; any may be NULL. */
typedef struct {
  int32_t *tokens;                     /* [n_rows][max_new], -1 beyond len */
  int32_t *len;                        /* [n_rows] generated tokens incl. the terminal EOS */
  uint8_t *status;                     /* [n_rows] DARTS_ROW_* */
  float *margin;                       /* [n_rows][max_new] Gumbel-max top1-top2 margin per sampled token */
  int32_t *sel;                        /* [G][K] selected sample indices j, rule order */
  uint32_t *sel_mask;                  /* [G] bitset of sel */
  int32_t *close_step;                 /* [G] step index at which the group closed */
  float *len_mean, *len_var;           /* [G] mean / population variance of the pool's lengths (sigma_L^2), over ALL Kp[i]
                                        * rows at the moment the group closed: a PRUNED row enters with the length at which the early stop
                                        * cut it (R25), so the value of an early-stopped group is a censored, i.e. deflated, sigma_L^2 —
                                        * n_pruned tells the caller which groups those are (skip or correct their EMA update) */
  float *logprob;                      /* [n_rows][max_new] log softmax(z / T) of the token the sampler DREW at each step (T == 0: of
                                        * softmax(z)); where a forced stop replaced the draw by EOS the value is still the draw's.
                                        * 0 beyond len.  fp32, accumulated per 128-id vocab tile then merged. */
  int32_t *n_pruned;                   /* [G] rows of the group halted by the early-stop signal (0 for a dual-end group) */
} darts_results;

typedef struct {
  int64_t n_steps;                     /* lock-step decode iterations incl. step 0 (first token from prefill) */
  int64_t n_generated_tokens;          /* all sampled tokens, incl. rows later pruned */
  int64_t n_kept_tokens;               /* tokens of the K selected trajectories of every prompt */
  int64_t n_near_ties;                 /* sampled tokens whose margin < 1e-3 */
  int64_t n_row_steps;                 /* sum over steps of active rows (= n_generated_tokens) */
  int64_t peak_pages;                  /* high-water mark of pages in use */
  int64_t kernel_launches;             /* kernels this ctx launched since darts_create */
  int64_t pages_allocated;             /* pages popped from the free stack since darts_prefill, prefix pages included
                                        * (> n_pages: freed pages were handed out again) */
} darts_counters;

typedef struct darts_ctx darts_ctx;

/* Host-only sizing of the workspace for (model, runtime). */
darts_status darts_workspace_bytes(const darts_model_desc *m, const darts_runtime_desc *rt, size_t *out);

/* Carve the workspace, record borrowed weight pointers.  `w` may be NULL only if m->vocab == 0. */
darts_status darts_create(const darts_model_desc *m, const darts_weights *w, const darts_runtime_desc *rt,
                          darts_ctx **out);
darts_status darts_destroy(darts_ctx *ctx);
const char *darts_last_error(const darts_ctx *ctx);

/* SURVEY §8(a) rows 1-2 + the first token (step 0):  one causal forward per PROMPT (not per sample)
 * writes the shared prefix pages; the last-position logits are sampled Kp[i] times with Philox keys
 * (seed, i, j, 0).  prompt_tokens / prompt_offsets (G+1) / Kp (G) / forced_len ([G][Kp_max] row-major,
 * Kp_max = max Kp, or NULL) are DEVICE pointers; Kp_host mirrors Kp on the host (needed for sizing).
 * forced_len[i][j] == len forces token len of trajectory (i,j) to eos_id (BASELINE.json workloads). */
darts_status darts_prefill(darts_ctx *ctx, const int32_t *prompt_tokens, const int32_t *prompt_offsets_host,
                           int32_t G, const int32_t *Kp_host, const int32_t *forced_len,
                           const darts_policy *policy, float temperature, uint64_t seed);

/* SURVEY §8(a) rows 3-8 for all active rows: embed, L x [RMSNorm, QKV, RoPE + KV append,
 * prefix-shared split-KV attention, O-proj, RMSNorm, SwiGLU MLP or MoE], final norm, LM head fused
 * with temperature + Philox Gumbel-max, EOS / forced-stop / length update.  No-op when nothing is active. */
darts_status darts_decode_step(darts_ctx *ctx);

/* per-prompt rule (Alg. 2), pruning, page release, stable compaction of the
 * active row list.  n_active_out: device or pinned host int32, may be NULL. */
darts_status darts_select_and_compact(darts_ctx *ctx, int32_t *n_active_out);

/* north_star signature: prefill + loop until every prompt has closed; synchronises before returning.
 * prompts: DEVICE [G][prompt_len] int32 (equal-length prompts); Kp_scalar = K' for every prompt.
 * L_long = 1, M_up = 2K, mode AUTO (use darts_prefill + the step calls for anything else). */
darts_status darts_rollout(darts_ctx *ctx, const int32_t *prompts, int32_t prompt_len, int32_t G,
                           int32_t Kp_scalar, int32_t K, int32_t max_len, float temperature, uint64_t seed,
                           const int32_t *forced_len, darts_results *out);

/* Same loop after a caller-issued darts_prefill (ragged prompts, per-prompt Kp, explicit policy). */
darts_status darts_run_to_completion(darts_ctx *ctx, darts_results *out);

/* Token-level streaming hook (§4.3.2 "ship token chunks to the trainer once a threshold accumulates"; rollout side
 * only — the consumer is the caller's).  Same loop as darts_run_to_completion; every chunk_steps lock-step iterations the tokens
 * of steps [step_begin, step_end) are copied to pinned host memory on a second stream (overlapping the following decode steps) and
 * fn(user, step_begin, step_end, n_rows, tokens, logprob) is called on the calling thread, in step order, with tokens = HOST
 * [n_rows][step_end - step_begin] row-major (-1 where a row had already stopped; a trailing chunk may hold only -1) and logprob the
 * same shape in fp32 (darts_results.logprob's values: the sampling policy's log-probability of each drawn token, 0 where tokens is
 * -1) — what the trainer's old-policy pass would otherwise recompute with a teacher-forced forward over the chunk.  The buffers are
 * valid during the call only.  The chunks together cover steps [0, n_steps).  The library owns the two pinned staging buffers. */
typedef void (*darts_chunk_fn)(void *user, int32_t step_begin, int32_t step_end, int32_t n_rows, const int32_t *tokens_host,
                               const float *logprob_host);
darts_status darts_run_to_completion_streaming(darts_ctx *ctx, int32_t chunk_steps, darts_chunk_fn fn, void *user, darts_results *out);

/* Token-level streaming, CONSUMER side (§4.3.2: chunks "are dispatched to the training engine ... it launches the
 * forward computation"; App. E :481-489: an incremental forward over a per-trajectory KV cache).  A context of its own — the consumer's
 * copy of the model, its own KV pool — scores streamed chunks with a teacher-forced forward: the tokens of a chunk are run through ONE
 * causal pass over [shared prompt pages || the row's own pages] (chunked prefill on the decode path's kernels: weights are streamed once
 * per chunk, not once per token), their K/V are appended, and each given token gets its log-probability under softmax(z / T) of the
 * logits at the position before it (T == 0: softmax(z)).  With the rollout's weights and temperature the values reproduce
 * darts_results.logprob wherever the rollout kept the token it drew (a forced EOS is scored as the EOS it is).
 *   darts_score_begin: prompts as in darts_prefill (DEVICE tokens, HOST offsets and Kp); one causal pass per prompt, no sampling.
 *   darts_score_chunk: tokens_host HOST [n_rows][step_end - step_begin] exactly as darts_chunk_fn delivers them (-1 from a row's end on);
 *     chunks must arrive in step order; logprob_out_host HOST, same shape, 0 where tokens is -1.  Synchronises.
 * Errors: DARTS_ERR_BAD_STATE (no darts_score_begin, chunk out of order), DARTS_ERR_KV_POOL_EXHAUSTED, DARTS_ERR_WORKSPACE_TOO_SMALL
 * (a chunk longer than max_rows - 1 steps).  The step / rollout calls return DARTS_ERR_BAD_STATE on a scoring context until the next
 * darts_prefill. */
darts_status darts_score_begin(darts_ctx *ctx, const int32_t *prompt_tokens, const int32_t *prompt_offsets_host, int32_t G,
                               const int32_t *Kp_host, float temperature);
darts_status darts_score_chunk(darts_ctx *ctx, int32_t step_begin, int32_t step_end, const int32_t *tokens_host, float *logprob_out_host);

/* End-to-end convenience with HOST inputs (bench `e2e`): copies prompts / forced_len host->device,
 * runs the rollout, copies results device->host. */
darts_status darts_rollout_host(darts_ctx *ctx, const int32_t *prompts_host, int32_t prompt_len, int32_t G,
                                const int32_t *Kp_host, const int32_t *forced_len_host, const darts_policy *policy,
                                int32_t max_len, float temperature, uint64_t seed, darts_results *out);

darts_status darts_get_results(darts_ctx *ctx, darts_results *out);
darts_status darts_get_counters(darts_ctx *ctx, darts_counters *out);
darts_status darts_n_active(darts_ctx *ctx, int32_t *out_host);      /* synchronises */

/* With DARTS_FLAG_PROFILE_ATTENTION: device time (ms, CUDA events on the ctx stream) of layer 0's attention launches
 * (split-KV main kernel + merge) for every decode step since the last darts_prefill, in step order.
 * ms_host: HOST [cap]; *n_out = number of steps recorded (may exceed cap; only cap are written).  Synchronises. */
darts_status darts_get_attention_times(darts_ctx *ctx, float *ms_host, int32_t cap, int32_t *n_out);

/* Parity hooks (valid with DARTS_FLAG_DUMP_LOGITS): fp32 logits of global row `row` from the most
 * recent step that row took part in (step 0: the prompt's prefill logits).  out: HOST [vocab]. */
darts_status darts_debug_logits(darts_ctx *ctx, int32_t row, float *out_host);

/* Parity hooks for the MoE router's discrete choice (R13; MoE context with DARTS_FLAG_DUMP_LOGITS):
 * darts_debug_routing: expert ids, in selection order, that every layer's router chose for slots [slot_begin, slot_begin + n_slots)
 *   of the MOST RECENT forward pass (a decode step: slot = position in the active row list; a prefill pass: slot = index of the
 *   prompt token within the pass).  out: HOST [n_layers][n_slots][top_k].  Synchronises.
 * darts_debug_row_slots: for every global row, the slot it occupied in the last decode step it took part in and that step's index
 *   (-1: none yet).  HOST [n_rows] each.  Synchronises. */
darts_status darts_debug_routing(darts_ctx *ctx, int32_t slot_begin, int32_t n_slots, int32_t *out_host);
darts_status darts_debug_row_slots(darts_ctx *ctx, int32_t *slot_host, int32_t *step_host, int32_t n_rows);

/* Parity hook for layer-by-layer comparison at full depth (DARTS_FLAG_DUMP_HIDDEN): the fp32 residual stream ENTERING layer
 * `layer` (layer == n_layers: leaving the last layer, i.e. the input of the final norm) for slots [slot_begin, slot_begin + n_slots)
 * of the most recent forward pass (slot numbering as in darts_debug_routing).  out: HOST [n_slots][d_model].  Synchronises. */
darts_status darts_debug_hidden(darts_ctx *ctx, int32_t layer, int32_t slot_begin, int32_t n_slots, float *out_host);

/* Profiling hook for PTL(b, ctx) sweeps (SURVEY.md 8(f) row f3; PAPER.md:163-169 Eq. 4, :372-382 App. A): give every ACTIVE row a
 * generated length of new_len (1 <= new_len < max_len) without decoding the steps in between.  Page tables are extended from the free
 * stack; the K/V of the skipped positions is whatever the pool holds (zeros after darts_create), so the tokens decoded afterwards are
 * meaningless — the step TIME at that context is what the hook is for.  Asynchronous on the ctx stream. */
darts_status darts_debug_fast_forward(darts_ctx *ctx, int32_t new_len);

/* Teacher forcing for parity at bf16 (R12): overwrite the token the next decode step feeds
 * for global row `row`.  tokens: HOST [n_rows] (-1 = leave). */
darts_status darts_debug_set_last_tokens(darts_ctx *ctx, const int32_t *tokens_host, int32_t n_rows);

/* Parity hook for the tcgen05 GEMM that carries every projection of the bf16 path:
 * C[rows][N] (fp32) = X[rows][K] . W[N][K]^T with bf16 X, W.  All pointers DEVICE.  split_k >= 1 K-splits are
 * computed as separate partials in `scratch` (>= split_k * rows * N floats) and added in split order into C
 * (C == NULL: leave the partials in `scratch`, no reduction).
 * Needs K % 64 == 0 and N % 4 == 0 (DARTS_ERR_UNSUPPORTED otherwise).  Asynchronous on the ctx stream. */
/* split_k == 0 selects the stream-K weight-streaming kernel (the one the decode projections use); its pieces need
 * darts_debug_gemm_scratch_floats(...) floats of scratch. */
darts_status darts_debug_gemm_scratch_floats(darts_ctx *ctx, int32_t rows, int32_t N, int32_t K, int32_t split_k, size_t *out);
darts_status darts_debug_gemm_bf16(darts_ctx *ctx, const void *X, const void *W, float *C, float *scratch, int32_t rows,
                                   int32_t N, int32_t K, int32_t split_k);

/* ---- The same stream-K GEMM for callers that cannot allocate (CUDA-graph capture, serving loops, harnesses that forbid cudaMalloc) ------
 * darts_gemm_bf16_static: C[rows][N] (fp32, DEVICE) = X[rows][K] . W[N][K]^T (bf16, DEVICE) on the stream-K weight-streaming kernel of the
 * decode projections (always the single-CTA kernel), i.e. what darts_debug_gemm_bf16 computes with split_k == 0 —
 * bit-identical to it on a context without DARTS_FLAG_CTA_PAIRS — but WITHOUT a scratch argument: the fp32 pieces and the piece-count table
 * live in a file-scope device array of DARTS_STATIC_SCRATCH_BYTES inside the library, which every GPU that loads the library holds until
 * the process exits.  The call allocates nothing (no cudaMalloc / cudaFree / allocating library routine): tensor-map encoding on the host,
 * one 8 KB cudaMemsetAsync and two kernel launches, all asynchronous on the ctx stream.  The first call on a device also looks the array's
 * device address up (cudaGetSymbolAddress): make one call outside any stream capture.
 * Limit: 8192 + slots * rows * N * 4 bytes <= DARTS_STATIC_SCRATCH_BYTES, slots = the stream-K plan's pieces per tile (what
 * darts_debug_gemm_scratch_floats reports / (rows N)); beyond it DARTS_ERR_WORKSPACE_TOO_SMALL and darts_last_error says how much was needed.
 * Needs K % 64 == 0 and N % 4 == 0 (DARTS_ERR_UNSUPPORTED otherwise); NULL / non-positive arguments: DARTS_ERR_INVALID_ARG.
 * The array is SHARED by every call in the process on that GPU and keeps the previous call's contents (the piece-count table is cleared per
 * call; every piece a call reads it has written first): calls on one context are ordered by its stream, calls that OVERLAP on the GPU
 * (other contexts, other streams) race on it and must be serialised by the caller.
 * darts_static_scratch_bytes: *out = DARTS_STATIC_SCRATCH_BYTES as compiled into the library (host-only). */
#define DARTS_STATIC_SCRATCH_BYTES (32u << 20)
darts_status darts_static_scratch_bytes(size_t *out);
darts_status darts_gemm_bf16_static(darts_ctx *ctx, const void *X, const void *W, float *C, int32_t rows, int32_t N, int32_t K);

/* ---- Adaptive redundancy allocation (§4.2.2; App. B Eq. 6-9 :384-411; App. C Alg. 1 :413-462) --------
 * Host-only helpers for the step upstream of the rollout: per-prompt length variances (darts_results.len_var) -> EMA ->
 * total budget -> greedy plan Kp[G] for the next darts_prefill.  All pointers HOST.  No context, no GPU work.
 * darts_update_variance_ema: var_ema[i] <- (1-beta) var_ema[i] + beta len_var[i]; var_ema[i] < 0 means "no history".
 * darts_redundancy_budget:   M* = rho/(lambda k) (Eq. 8), *M_total_out = clip(floor(M*), K G, 2 K G) (Eq. 9).
 * darts_allocate_redundancy: Alg. 1 with w_i = min-max normalised sqrt(var_ema[i]) (all equal: 1), marginal gain
 *   w_i (1/M'_i - 1/(M'_i+1)) (R18), ties -> smallest i; needs G M_low <= M_total; the plan sums to
 *   min(M_total, G M_up).  DARTS_ERR_INVALID_ARG on NULLs, non-positive sizes or negative / NaN variances. */
darts_status darts_update_variance_ema(float *var_ema_host, const float *len_var_host, int32_t G, float beta);
darts_status darts_redundancy_budget(double rho, double lambda, double k, int32_t G, int32_t K, int64_t *M_total_out);
darts_status darts_allocate_redundancy(const float *var_ema_host, int32_t G, int64_t M_total, int32_t M_low, int32_t M_up,
                                       int32_t *Kp_out_host);

/* ---- Attention-only entry points (BASELINE.json config 2) -------------------
 * Build G groups of Kp rows whose KV is given explicitly, then time darts_attention alone.
 * k_prefix/v_prefix: DEVICE [G][P][n_kv_heads][head_dim]; suffix_len: HOST [R]; k_suffix/v_suffix:
 * DEVICE packed [sum suffix_len][n_kv_heads][head_dim] in row order.  Loads layer 0 of the cache. */
darts_status darts_attn_load(darts_ctx *ctx, int32_t G, int32_t P, int32_t Kp, const void *k_prefix,
                             const void *v_prefix, const int32_t *suffix_len_host, const void *k_suffix,
                             const void *v_suffix);
/* q: DEVICE [R][n_q_heads][head_dim] (model dtype); out: DEVICE same shape.  One decode-step attention
 * over all R rows on layer `layer`; asynchronous on the ctx stream. */
darts_status darts_attention(darts_ctx *ctx, int32_t layer, const void *q, void *out);

#ifdef __cplusplus
}
#endif
#endif /* DARTS_H_ */
