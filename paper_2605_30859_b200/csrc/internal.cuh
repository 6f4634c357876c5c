// Internal declarations shared by the translation units of libdarts.so (not part of the C-ABI).
#pragma once
#include <cuda.h>
#include <cuda_bf16.h>
#include <cuda_runtime.h>
#include <stdint.h>
#include <stdio.h>
#include <string.h>

#include <vector>

#include "darts.h"

#ifndef ATTN_CHUNK_PAGES
#define ATTN_CHUNK_PAGES 8        // pages (of 64 tokens) per split-KV work item of the tuned attention kernel
#endif
#define ATTN_CHUNK_TOKENS (ATTN_CHUNK_PAGES * 64)
#define DARTS_MAX_KP 32          // a group's pool is ranked by one warp (include/darts.h: Kp[i] <= 32)
#define NEAR_TIE_MARGIN 1e-3f    // north_star: "bit-exact wherever the Gumbel-max margin exceeds 1e-3"

// Device-resident scalar state of a rollout (one instance per ctx).
struct DevState {
  int32_t n_active;              // rows still decoding (== length of row_list)
  int32_t n_rows;                // sum Kp
  int32_t n_groups;
  int32_t free_top;              // number of pages on the free stack
  int32_t err;                   // sticky device-side error (DARTS_ERR_KV_POOL_EXHAUSTED)
  int32_t step;                  // index of the NEXT lock-step iteration (0 = first token)
  int32_t peak_used;
  int32_t n_open_groups;
  unsigned long long n_generated, n_near_ties, n_kept, n_row_steps;
  unsigned long long n_pops;     // pages handed out since the prefill (prefix pages + every pop of the free stack)
};

// KV cache geometry.  One layer slab = [page][kv_head][K|V][token][head_dim]; the (K,V) tiles of one
// (page, head) are adjacent so the tuned attention kernel fetches both with ONE bulk copy.  With swz set
// (bf16, head_dim 128) the 16-byte chunks of a token row are XOR-permuted by (token & 7): the layout in HBM is
// already the bank-conflict-free layout ldmatrix wants in shared memory, so a plain linear copy stages it.
struct KvGeom {
  size_t page_elems, tile_elems;
  int hd, swz;
};
__device__ __forceinline__ size_t kv_elem(const KvGeom &g, int page, int head, int kv, int tok, int d) {
  int dd = g.swz ? ((((d >> 3) ^ (tok & 7)) << 3) | (d & 7)) : d;
  return (size_t)page * g.page_elems + ((size_t)head * 2 + kv) * g.tile_elems + (size_t)tok * g.hd + dd;
}

struct XMaps { CUtensorMap m[5]; };   // one activation matrix [rows][K] with boxes of 16, 32, 64, 128, 256 rows

struct darts_ctx {
  darts_model_desc m;
  darts_runtime_desc rt;
  cudaStream_t stream;
  bool has_weights;
  // borrowed weights (host-side copies of the per-layer pointer arrays)
  const void *embed, *final_norm, *lm_head;
  const void **attn_norm, **wqkv, **q_norm, **k_norm, **wo, **mlp_norm, **wgu, **wd, **wr, **wgu_e, **wd_e;

  // geometry
  int elt;                       // sizeof model dtype
  int n_qkv;                     // (Hq + 2 Hkv) * hd
  int max_suffix_pages, max_prefix_pages;
  int act_rows;                  // rows the activation buffers hold: max(max_rows, prefill_chunk)
  size_t kv_tile_elems;          // page_size * head_dim                      (one (page, K|V, head) tile)
  size_t kv_page_elems;          // 2 * Hkv * kv_tile_elems                   (one page of one layer)
  size_t kv_layer_elems;         // n_pages * kv_page_elems
  int kv_swz;                    // 1: swizzled token rows (bf16, head_dim 128)
  KvGeom geom() const { return KvGeom{kv_page_elems, kv_tile_elems, m.head_dim, kv_swz}; }

  // carve-outs (device)
  void *kv_pool;
  DevState *st;
  int32_t *free_pages;
  int32_t *row_list, *row_list_tmp;
  int32_t *row_prompt, *row_sample, *row_len, *row_forced, *row_last_tok, *row_pages, *row_slot, *row_slot_step;
  uint8_t *row_status;
  int32_t *tokens_out;
  float *margin_out;
  float *logprob_out;            // [max_rows][max_new] log softmax(z/T) of the drawn token
  int32_t *g_off, *g_Kp, *g_plen, *g_closed, *g_sel, *g_close_step, *g_prefix_pages, *g_tok_off, *g_n_pruned;
  uint32_t *g_mask;
  float *g_len_mean, *g_len_var;
  int32_t *prompt_tokens;        // private copy of the prompt tokens [sum P]
  // per-slot plan of the current pass
  int32_t *slot_row, *slot_tok, *slot_pos, *slot_dst_page, *slot_dst_off, *slot_prompt, *slot_npre, *slot_nsuf;
  float2 *slot_cs;               // [act_rows][hd/2] (cos, sin)
  // activations
  float *h, *qkv32, *gu32, *logits, *z0, *hlast, *attn_part;
  float *hid_dump;               // [n_layers + 1][act_rows][d] residual stream at the layer boundaries (DARTS_FLAG_DUMP_HIDDEN; parity hook)
  void *xn, *q, *ao, *act;
  // attention-only mode (config 2)
  int32_t attn_rows;
  // tensor-core path (bf16, kernels_gemm_tc.cu): split-K partial buffer, LM-head top-2 partials, tensor maps
  bool tc_path;                  // every GEMM of this model runs on tcgen05
  unsigned skip_mask;            // -DDARTS_PROFILING builds only (env DARTS_SKIP, bit per kernel class of a layer): skipped launches leave stale data — timing only
  bool use_pairs;                // dense projections on the CTA-pair (cta_group::2) stream-K kernel (DARTS_FLAG_CTA_PAIRS)
  bool use_pdl;                  // launch the kernels of a step as programmatic dependents (-DDARTS_PROFILING builds: DARTS_NO_PDL=1 disables)
  float *part;                   // [S][rows][N] fp32 partials of the GEMM in flight
  size_t part_bytes;
  int32_t *sk_np;                // [SK_NP_TABLE] pieces per tile of the stream-K GEMM in flight (read by its consumer kernel)
  float *top2;                   // float4 [vocab tiles][max_rows]
  float *lse;                    // float2 [vocab tiles][max_rows]
  CUtensorMap *tm_wqkv, *tm_wo, *tm_wgu, *tm_wd, *tm_wgu_e, *tm_wd_e;   // host arrays [n_layers]
  CUtensorMap tm_lm, tm_xn, tm_ao, tm_act, tm_xs, tm_hl;                      // activations: 16-row boxes
  XMaps xm_xn, xm_ao, xm_act, xm_xs;                                            // the same matrices for the stream-K kernel
  // MoE (kernels_moe.cu)
  int32_t *moe_eid, *moe_pos, *moe_off, *moe_cnt, *moe_tok, *moe_rb, *moe_nrb, *moe_arrive;
  size_t moe_arrive_n;   // moe_rb: row blocks {row0, nrows, expert, -}   // moe_cnt: [n_layers][E], zeroed once per forward pass
  int32_t *moe_eid_dump;         // [n_layers][act_rows][top_k] expert ids of the last pass (DARTS_FLAG_DUMP_LOGITS only; parity hook)
  float *moe_w, *moe_logits, *moe_y;   // gates [rows*top_k]; router logits [rows][E]; generic path expert outputs [rows*top_k][d]
  void *xs;                      // expert-sorted copy of xn [max_rows * top_k][d]
  // tuned attention (kernels_attn_sm100.cu): per-step work list and split-KV partials
  int32_t *attn_items_pre, *attn_items_suf, *attn_nitems, *part_base, *part_cnt;
  float *part_ml, *part_acc;
  int attn_max_items;
  bool attn_plan_valid, attn_causal;   // attn_causal: the current plan is a prefill pass (row-wise causal masks)
  int n_sms;

  // policy / sampling
  darts_policy pol;
  float temperature;
  uint64_t seed;
  int32_t G, R, Kp_max, max_len;
  int32_t *forced_stage;       // device staging for host-provided forced_len
  uint32_t gen;                  // rollout generation (tags the pinned mirror)
  cudaEvent_t ev[2];
  bool prefilled;
  int32_t host_active_ub;        // stale-but-safe upper bound of n_active known to the host
  int32_t steps_issued;

  // pinned host mirror written by the compaction kernel
  volatile int32_t *pinned;      // host view: [0] n_active + [1] generation (one 64-bit store), [2] err
  int32_t *pinned_dev;           // device view of the same mapped allocation
  int64_t launches;
  // DARTS_FLAG_PROFILE_ATTENTION: event pairs around layer 0's attention of each decode step
  std::vector<cudaEvent_t> prof_ev;
  int prof_n;
  bool in_decode;
  // token-level streaming (darts_run_to_completion_streaming): copy stream, pinned double buffer, events
  cudaStream_t copy_stream;
  int32_t *chunk_stage[2];
  size_t chunk_stage_bytes;
  cudaEvent_t ev_copy_ready[2], ev_copy_done[2];
  // chunk scoring (darts_score_begin / darts_score_chunk): a context used as the CONSUMER of streamed token chunks.  Pages are handed
  // out by the host (the call takes host tokens and returns host log-probabilities anyway); device side: targets, results, pending rows.
  bool score_mode;
  std::vector<int32_t> sc_len, sc_free, sc_pages;   // tokens forwarded per row; free page ids (stack); host mirror of row_pages
  int32_t *score_tgt, *score_idx;                   // [max_rows] target id per LM-head row; [2 * max_rows] gather / scatter indices
  float *score_lp;                                  // [max_rows] log-probability per LM-head row
  void *score_pend, *pend0;                         // [max_rows][d] / [max_prompts][d] final-normed hidden awaiting its next token (model dtype)
  char err[512];
  darts_status sticky;
};

// Profiling aid, compiled out of the default build: the product never reads the environment.
#ifdef DARTS_PROFILING
#define DARTS_SKIPPED(c, bit) (((c)->skip_mask & (bit)) != 0)
#else
#define DARTS_SKIPPED(c, bit) false
#endif

#define CUDA_TRY(ctx, expr)                                                                   \
  do {                                                                                        \
    cudaError_t e__ = (expr);                                                                 \
    if (e__ != cudaSuccess) {                                                                 \
      snprintf((ctx)->err, sizeof((ctx)->err), "%s:%d: %s: %s", __FILE__, __LINE__, #expr,    \
               cudaGetErrorString(e__));                                                      \
      (ctx)->sticky = DARTS_ERR_CUDA;                                                         \
      return DARTS_ERR_CUDA;                                                                  \
    }                                                                                         \
  } while (0)

#define FAIL(ctx, code, ...)                                  \
  do {                                                        \
    snprintf((ctx)->err, sizeof((ctx)->err), __VA_ARGS__);    \
    return (code);                                            \
  } while (0)

template <typename T> __device__ __forceinline__ float to_f(T x);
template <> __device__ __forceinline__ float to_f<float>(float x) { return x; }
template <> __device__ __forceinline__ float to_f<__nv_bfloat16>(__nv_bfloat16 x) { return __bfloat162float(x); }
template <typename T> __device__ __forceinline__ T from_f(float x);
template <> __device__ __forceinline__ float from_f<float>(float x) { return x; }
template <> __device__ __forceinline__ __nv_bfloat16 from_f<__nv_bfloat16>(float x) { return __float2bfloat16_rn(x); }

// Programmatic dependent launch (PDL): a kernel that calls pdl_trigger() lets the NEXT kernel of the stream start its
// prologue (and, for the GEMMs, its weight prefetch) while this one is still running; a kernel launched with the PDL
// attribute must call pdl_wait() before it touches anything an earlier kernel wrote.  Both are no-ops otherwise.
__device__ __forceinline__ void pdl_trigger() { asm volatile("griddepcontrol.launch_dependents;" ::: "memory"); }
__device__ __forceinline__ void pdl_wait() { asm volatile("griddepcontrol.wait;" ::: "memory"); }

// Host side: launch `kernel` as a programmatic dependent of the previous kernel in the stream (plain launch if PDL is off).
template <typename... KArgs, typename... Args>
inline void launch_pdl(darts_ctx *c, void (*kernel)(KArgs...), dim3 grid, dim3 block, size_t smem, Args &&...args) {
  cudaLaunchConfig_t cfg{};
  cfg.gridDim = grid; cfg.blockDim = block; cfg.dynamicSmemBytes = smem; cfg.stream = c->stream;
  cudaLaunchAttribute at[1];
  at[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
  at[0].val.programmaticStreamSerializationAllowed = 1;
  cfg.attrs = at; cfg.numAttrs = c->use_pdl ? 1 : 0;
  cudaLaunchKernelEx(&cfg, kernel, static_cast<KArgs>(args)...);
}

__device__ __forceinline__ float warp_sum(float v) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
  return v;
}
__device__ __forceinline__ float warp_max(float v) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v = fmaxf(v, __shfl_xor_sync(0xffffffffu, v, o));
  return v;
}

// ---- launchers implemented across the .cu files (all asynchronous on ctx->stream) ----------------
// n_rows_dev: device pointer to the live row count (kernels ignore slots >= *n_rows_dev); rows_ub: host upper bound.
darts_status launch_embed(darts_ctx *c, const int32_t *tok_of_slot_src, int mode, int rows_ub, const int32_t *n_rows_dev);
darts_status launch_embed_norm_rope(darts_ctx *c, const int32_t *slot_tok, const void *w, int rows_ub, const int32_t *n_rows_dev);
darts_status launch_rmsnorm(darts_ctx *c, const float *h, const void *w, void *out, int rows_ub, const int32_t *n_rows_dev);
darts_status launch_gemm(darts_ctx *c, const void *X, const void *W, float *C, int N, int K, int rows_ub,
                         const int32_t *n_rows_dev, bool accumulate, bool w_is_f32 = false);
darts_status launch_rope_table(darts_ctx *c, int rows_ub, const int32_t *n_rows_dev);
darts_status launch_rope_append(darts_ctx *c, int layer, int rows_ub, const int32_t *n_rows_dev);
darts_status launch_attention(darts_ctx *c, int layer, const void *q, void *out, int rows_ub, const int32_t *n_rows_dev);
darts_status launch_silu_mul(darts_ctx *c, int rows_ub, const int32_t *n_rows_dev);
darts_status launch_moe(darts_ctx *c, int layer, int rows_ub, const int32_t *n_rows_dev);
darts_status launch_moe_tc(darts_ctx *c, int layer, const void *next_norm, int rows_ub, const int32_t *n_rows_dev);
darts_status launch_moe_begin_pass(darts_ctx *c);
darts_status launch_sample(darts_ctx *c, const float *logits, int step0, int rows_ub);
darts_status launch_plan_decode(darts_ctx *c, int rows_ub);
darts_status launch_fast_forward(darts_ctx *c, int new_len);
darts_status launch_plan_prefill(darts_ctx *c, int tok_begin, int n_tok, int g_begin, int g_end);
darts_status launch_gather_last(darts_ctx *c, int tok_begin, int n_tok, int g_begin, int g_end);
darts_status launch_select(darts_ctx *c);
darts_status launch_compact(darts_ctx *c, int32_t *n_active_out);
darts_status launch_init_rows(darts_ctx *c, const int32_t *forced_len, int n_prefix_pages_total);
darts_status launch_attn_load(darts_ctx *c, int G, int P, int Kp, const void *kp, const void *vp, const int32_t *suffix_len_dev,
                              const int64_t *suffix_offs_dev, const void *ks, const void *vs, long long n_suffix_tok);
darts_status launch_gemm_simt(darts_ctx *c, const void *X, const void *W, float *C, int N, int K, int rows_ub,
                              const int32_t *n_rows_dev, bool accumulate, bool w_is_f32);
// tcgen05 GEMM (kernels_gemm_tc.cu)
struct TcGemm {
  const CUtensorMap *a_map, *b_map;   // activations [rows][K] (16-row boxes), weights [N (x groups)][K] (128-row boxes)
  float *C;                           // partials [S][rows][N] (ignored when sample)
  size_t split_stride;
  int N, K, S, rows_ub;
  const int32_t *n_rows_dev;
  bool sample;                        // LM head: fused temperature + Gumbel-max epilogue -> ctx->top2
};
darts_status launch_gemm_tc(darts_ctx *c, const TcGemm &g);
darts_status tc_make_map(darts_ctx *c, CUtensorMap *out, const void *base, long long rows, int K, int box_rows);
darts_status tc_make_xmaps(darts_ctx *c, XMaps *out, const void *base, long long rows, int K);
bool tc_shape_ok(int N, int K);
// stream-K weight-streaming GEMM (kernels_gemm_sk.cu)
#define SK_ROWBLOCK 256            // activation rows per MMA N block
#ifndef SK_RB512_MAX
#define SK_RB512_MAX 384           // largest live row count served as ONE 512-row block (two MMA N blocks sharing the weight tile)
#endif
#define SK_NP_TABLE 2048           // >= tiles of a split (non whole-tile) dense launch: n_wtiles * row blocks < 8 * SMs
struct SkPlan { int nkb, n_wtiles, P, unit_tile, slots, stage_bytes, n_stages, tm_cols, n_acc; };   // stage / TMEM fields: grouped mode only
struct SkGemm {
  const CUtensorMap *w_map;           // weights [N (x groups)][K], 128-row boxes
  const XMaps *x_maps;
  float *C;                           // pieces [slot][rows][N]
  size_t slot_stride;
  int N, rows_ub;
  const int32_t *n_rows_dev;
  int32_t *np_table;                  // dense stream-K: pieces per tile, written by each tile's head piece for the consumers (NULL: not kept)
  bool pairs;                         // run on the CTA-pair kernel (plan from sk2_plan)
  const int32_t *rb_list, *n_rb_dev;  // grouped: {row0, nrows, group id, -} per row block, count on the device
  int w_rows_per_group;               // grouped: weight row base of a block = group id * w_rows_per_group
  SkPlan plan;
};
// What a consumer needs to add the pieces of element (row, col) in slot order.
struct SkView {
  const float *part;
  size_t slot_stride;
  int N, nkb, n_wtiles, P, unit_tile;
  const int32_t *np_table;            // pieces per tile, written by the GEMM that produced `part` (NULL: closed form)
  int rb512;                          // 1: the producer used sk_rb_rows (one 512-row block for 257..384 live rows); 0: 256-row blocks always (CTA-pair kernel)
};
// Activation rows per row block of a DENSE launch, decided from the LIVE row count on the device (never from the host's stale upper
// bound: the block size fixes where a tile's pieces are cut, i.e. the fp32 summation order, and that must not depend on timing).
// 257..384 live rows: one 512-row block = two MMA N blocks per stage sharing the weight tile; otherwise 256-row blocks.
__host__ __device__ __forceinline__ int sk_rb_rows(int live) { return (live > SK_ROWBLOCK && live <= SK_RB512_MAX) ? 2 * SK_ROWBLOCK : SK_ROWBLOCK; }
// CTA that owns unit u when T units are cut into P ranges [c*T/P, (c+1)*T/P)
__host__ __device__ __forceinline__ int sk_owner(int u, int P, int T) { return ((u + 1) * P - 1) / T; }
__host__ __device__ __forceinline__ int sk_view_rb_rows(const SkView &v, int live) { return v.rb512 ? sk_rb_rows(live) : SK_ROWBLOCK; }
__host__ __device__ __forceinline__ int sk_npieces(const SkView &v, int n_rb, int rb_rows, int col, int row) {
  if (v.unit_tile) return 1;
  int t = (col >> 7) * n_rb + (rb_rows == 2 * SK_ROWBLOCK ? row / (2 * SK_ROWBLOCK) : row / SK_ROWBLOCK);
#ifdef __CUDA_ARCH__
  // the producing GEMM left the count of every tile it touched (its head piece writes it): one L2 hit instead of four integer divisions
  // per warp, which were ~45 % of the instructions of the piece-summing consumers
  if (v.np_table) return __ldg(v.np_table + t);
#endif
  int T = v.n_wtiles * n_rb * v.nkb;
  return sk_owner(t * v.nkb + v.nkb - 1, v.P, T) - sk_owner(t * v.nkb, v.P, T) + 1;
}
SkPlan sk_plan(int n_sms, int N, int K, int rows_ub, int n_rb_ub_grouped, bool rows_exact);
darts_status launch_gemm_sk(darts_ctx *c, const SkGemm &g);
darts_status launch_sk_reduce(darts_ctx *c, const SkView &v, float *out, int rows);
bool sk_sample_supported(const darts_ctx *c, int rows_ub);
darts_status launch_gemm_sk_sample(darts_ctx *c, const CUtensorMap *w_map, const XMaps *x_maps, int N, int K, int rows_ub, const int32_t *n_rows_dev,
                                   const int32_t *target = nullptr);
// chunk scoring (kernels_score.cu)
darts_status launch_score_init_pend(darts_ctx *c, int R);
darts_status launch_score_gather(darts_ctx *c, int S, int n_pend);
darts_status launch_score_scatter(darts_ctx *c, int n_pend);
darts_status launch_score_finalize(darts_ctx *c, int n_tiles, int rows);
darts_status launch_score_logits(darts_ctx *c, int rows);
inline SkView sk_view(const SkGemm &g) { return SkView{g.C, g.slot_stride, g.N, g.plan.nkb, g.plan.n_wtiles, g.plan.P, g.plan.unit_tile, g.np_table, g.pairs ? 0 : 1}; }
// CTA-pair (cta_group::2) variant (kernels_gemm_sk2.cu)
SkPlan sk2_plan(int n_sms, int N, int K, int rows_ub, bool rows_exact);
darts_status launch_gemm_sk2(darts_ctx *c, const SkGemm &g);
darts_status gemm_sk2_configure(darts_ctx *c);
darts_status launch_add_rmsnorm_sk(darts_ctx *c, const SkView &v, const void *w, int rows_ub, const int32_t *n_rows_dev);
darts_status launch_silu_mul_sk(darts_ctx *c, const SkView &v, int rows_ub, const int32_t *n_rows_dev);
darts_status launch_rope_append_sk(darts_ctx *c, int layer, const SkView &v, int rows_ub, const int32_t *n_rows_dev);
// consumers of the split-K partials (kernels_fused.cu)
darts_status launch_sample_finalize(darts_ctx *c, int n_tiles, int rows_ub);
darts_status launch_sum_partials(darts_ctx *c, const float *part, float *out, int S, size_t n);
darts_status launch_gather_rows_bf16(darts_ctx *c, const void *src, void *dst, int tok_begin, int g_begin, int g_end);
darts_status launch_attention_plan_sm100(darts_ctx *c, int rows_ub, const int32_t *n_rows_dev, bool prefill = false);
bool attention_sm100_supported(const darts_ctx *c);
// per-context kernel set-up (function attributes), called by darts_create
darts_status gemm_sk_configure(darts_ctx *c);
darts_status gemm_tc_configure(darts_ctx *c);
darts_status attn_sm100_configure(darts_ctx *c);
darts_status moe_configure(darts_ctx *c);
darts_status launch_attention_ref(darts_ctx *c, int layer, const void *q, void *out, int rows_ub, const int32_t *n_rows_dev);
