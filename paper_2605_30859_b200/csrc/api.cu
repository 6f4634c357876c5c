// C-ABI entry points (include/darts.h): workspace carving, prefill, decode step, selection/compaction,
// the rollout loop and result read-back.  Host logic only; every step of the path runs in the kernels.
#include <stdlib.h>

#include <algorithm>
#include <new>
#include <vector>

#include "internal.cuh"

namespace {

struct Carver {
  char *base;
  size_t off = 0;
  explicit Carver(void *b) : base((char *)b) {}
  template <typename T> T *take(size_t n) {
    off = (off + 255) & ~(size_t)255;
    T *p = base ? (T *)(base + off) : nullptr;
    off += n * sizeof(T);
    return p;
  }
};

int ceil_div(int a, int b) { return (a + b - 1) / b; }

int default_chunk(const darts_runtime_desc *rt) {
  int c = rt->prefill_chunk > 0 ? rt->prefill_chunk : 4096;
  return std::max(c, rt->max_prompt_len);
}

// One routine lays the workspace out for both sizing (c->... pointers NULL) and creation.
size_t carve(darts_ctx *c, void *base) {
  const darts_model_desc &m = c->m;
  const darts_runtime_desc &rt = c->rt;
  Carver k(base);
  bool model = m.vocab > 0;
  c->elt = m.dtype == DARTS_F32 ? 4 : 2;
  c->n_qkv = (m.n_q_heads + 2 * m.n_kv_heads) * m.head_dim;
  c->max_suffix_pages = ceil_div(rt.max_new, rt.page_size) + 1;
  c->max_prefix_pages = std::max(1, ceil_div(rt.max_prompt_len, rt.page_size));
  c->act_rows = model ? std::max(rt.max_rows, default_chunk(&rt)) : rt.max_rows;
  c->kv_tile_elems = (size_t)rt.page_size * m.head_dim;
  c->kv_page_elems = 2 * (size_t)m.n_kv_heads * c->kv_tile_elems;
  c->kv_layer_elems = (size_t)rt.n_pages * c->kv_page_elems;
  c->kv_swz = (c->elt == 2 && m.head_dim == 128) ? 1 : 0;
  size_t R = rt.max_rows, G = rt.max_prompts, A = c->act_rows;
  c->kv_pool = k.take<char>((size_t)m.n_layers * c->kv_layer_elems * c->elt);
  c->st = k.take<DevState>(1);
  c->free_pages = k.take<int32_t>(rt.n_pages);
  c->row_list = k.take<int32_t>(R);
  c->row_list_tmp = k.take<int32_t>(R);
  c->row_prompt = k.take<int32_t>(R);
  c->row_sample = k.take<int32_t>(R);
  c->row_len = k.take<int32_t>(R);
  c->row_forced = k.take<int32_t>(R);
  c->row_last_tok = k.take<int32_t>(R);
  c->row_slot = k.take<int32_t>(R);
  c->row_slot_step = k.take<int32_t>(R);
  c->row_pages = k.take<int32_t>(R * c->max_suffix_pages);
  c->row_status = k.take<uint8_t>(R);
  c->g_off = k.take<int32_t>(G + 1);
  c->g_Kp = k.take<int32_t>(G);
  c->g_plen = k.take<int32_t>(G);
  c->g_closed = k.take<int32_t>(G);
  c->g_sel = k.take<int32_t>(G * DARTS_MAX_KP);
  c->g_close_step = k.take<int32_t>(G);
  c->g_n_pruned = k.take<int32_t>(G);
  c->g_prefix_pages = k.take<int32_t>(G * c->max_prefix_pages);
  c->g_tok_off = k.take<int32_t>(G + 1);
  c->g_mask = k.take<uint32_t>(G);
  c->g_len_mean = k.take<float>(G);
  c->g_len_var = k.take<float>(G);
  c->slot_row = k.take<int32_t>(A);
  c->slot_tok = k.take<int32_t>(A);
  c->slot_pos = k.take<int32_t>(A);
  c->slot_dst_page = k.take<int32_t>(A);
  c->slot_dst_off = k.take<int32_t>(A);
  c->slot_prompt = k.take<int32_t>(A);
  c->slot_npre = k.take<int32_t>(A);
  c->slot_nsuf = k.take<int32_t>(A);
  c->forced_stage = k.take<int32_t>(G * DARTS_MAX_KP);
  c->sk_np = k.take<int32_t>(SK_NP_TABLE);
  if (attention_sm100_supported(c)) {
    size_t npc_max = (size_t)ceil_div(rt.max_prompt_len, ATTN_CHUNK_TOKENS);
    size_t max_parts = R * (npc_max + 2) + (size_t)rt.n_pages / ATTN_CHUNK_PAGES + 16;
    if (model) max_parts = std::max(max_parts, A * npc_max + 16);            // a prefill pass: one partial per (prompt token, chunk)
    c->attn_max_items = (int)max_parts;
    c->attn_items_pre = k.take<int32_t>(max_parts * 6);
    c->attn_items_suf = k.take<int32_t>(max_parts * 6);
    c->attn_nitems = k.take<int32_t>(4);
    c->part_base = k.take<int32_t>(A);
    c->part_cnt = k.take<int32_t>(A);
    c->part_ml = k.take<float>(max_parts * m.n_q_heads * 2);
    c->part_acc = k.take<float>(max_parts * m.n_q_heads * m.head_dim);
  }
  size_t Fm = m.n_experts ? (size_t)m.top_k * m.expert_ffn : (size_t)m.ffn;
  int qd_ = m.n_q_heads * m.head_dim;
  c->tc_path = model && m.dtype == DARTS_BF16 && tc_shape_ok(c->n_qkv, m.d_model) && tc_shape_ok(m.d_model, qd_) &&
               tc_shape_ok(m.vocab, m.d_model) &&
               (m.n_experts ? (tc_shape_ok(2 * m.expert_ffn, m.d_model) && tc_shape_ok(m.d_model, m.expert_ffn))
                            : (tc_shape_ok(2 * m.ffn, m.d_model) && tc_shape_ok(m.d_model, m.ffn)));
  if (model) {
    size_t F = Fm;
    c->tokens_out = k.take<int32_t>(R * rt.max_new);
    c->margin_out = k.take<float>(R * rt.max_new);
    c->logprob_out = k.take<float>(R * rt.max_new);
    c->prompt_tokens = k.take<int32_t>(G * rt.max_prompt_len);
    c->slot_cs = k.take<float2>(A * (m.head_dim / 2));
    c->h = k.take<float>(A * m.d_model);
    if (rt.flags & DARTS_FLAG_DUMP_HIDDEN) c->hid_dump = k.take<float>((size_t)(m.n_layers + 1) * A * m.d_model);
    if (m.n_experts) {
      size_t RK = A * m.top_k;
      c->moe_logits = k.take<float>(A * m.n_experts);
      c->moe_eid = k.take<int32_t>(RK);
      c->moe_pos = k.take<int32_t>(RK);
      c->moe_w = k.take<float>(RK);
      c->moe_arrive_n = A / 4 + 1;
      c->moe_arrive = k.take<int32_t>(c->moe_arrive_n);         // router arrival counters, one per block of 4 slots; zero between launches
      if (rt.flags & DARTS_FLAG_DUMP_LOGITS) c->moe_eid_dump = k.take<int32_t>((size_t)m.n_layers * RK);
    }
    if (c->tc_path) {
      // stream-K pieces [slots][rows][N]: whole-tile mode (1 slot) for the prefill-sized passes, up to 16 slots for decode rows
      size_t maxN = std::max<size_t>(std::max<size_t>(c->n_qkv, 2 * F), m.n_experts ? (size_t)m.top_k * m.d_model : (size_t)m.d_model);
      size_t dec = 0;
      const int sms = c->n_sms > 0 ? c->n_sms : 148;       // host-only sizing assumes a full B200; darts_create re-checks
      int shapes[4][2] = {{c->n_qkv, m.d_model}, {m.d_model, qd_}, {m.n_experts ? 0 : 2 * m.ffn, m.d_model}, {m.n_experts ? 0 : m.d_model, m.ffn}};
      for (auto &sh : shapes)
        if (sh[0] > 0) {
          // a decode step re-plans with the host's current row bound: the slot count grows as the row blocks get fewer, so take
          // the largest footprint over every row-block count the context can see (launch_gemm_sk re-checks at launch)
          for (int rows = SK_ROWBLOCK; rows < rt.max_rows + SK_ROWBLOCK; rows += SK_ROWBLOCK) {
            const size_t r = (size_t)std::min(rows, rt.max_rows);
            dec = std::max(dec, (size_t)sk_plan(sms, sh[0], sh[1], (int)r, 0, false).slots * r * sh[0] * 4);
          }
          dec = std::max(dec, (size_t)sk_plan(sms, sh[0], sh[1], (int)A, 0, true).slots * A * sh[0] * 4);
        }
      c->part_bytes = std::max<size_t>(std::max<size_t>(A * maxN * 4, dec), (size_t)64 << 20);
      c->part = k.take<float>(c->part_bytes / 4);
      c->top2 = k.take<float>((size_t)4 * ceil_div(m.vocab, 128) * R * 4);    // one entry per (vocab tile, warp quadrant, row)
      c->lse = k.take<float>((size_t)4 * ceil_div(m.vocab, 128) * R * 2);
      if (rt.flags & DARTS_FLAG_DUMP_LOGITS) c->logits = k.take<float>(R * m.vocab);
      if (m.n_experts) {
        size_t RK = A * m.top_k;
        c->moe_tok = k.take<int32_t>(RK);
        c->moe_off = k.take<int32_t>(m.n_experts + 1);
        c->moe_rb = k.take<int32_t>(4 * ((size_t)m.n_experts + RK / SK_ROWBLOCK + 1));
        c->moe_nrb = k.take<int32_t>(1);
        c->moe_cnt = k.take<int32_t>((size_t)m.n_layers * m.n_experts);
        c->xs = k.take<char>(RK * m.d_model * 2);
      }
    } else {
      c->qkv32 = k.take<float>(A * c->n_qkv);
      if (m.n_experts) c->moe_y = k.take<float>(A * m.top_k * m.d_model);
      else c->gu32 = k.take<float>(A * 2 * F);
      c->logits = k.take<float>(R * m.vocab);
    }
    c->score_tgt = k.take<int32_t>(R);
    c->score_idx = k.take<int32_t>(2 * R);
    c->score_lp = k.take<float>(R);
    c->score_pend = k.take<char>(R * m.d_model * c->elt);
    c->pend0 = k.take<char>(G * m.d_model * c->elt);
    c->z0 = k.take<float>(G * m.vocab);
    c->hlast = k.take<float>(G * m.d_model);
    c->xn = k.take<char>(A * m.d_model * c->elt);
    c->q = k.take<char>(A * m.n_q_heads * m.head_dim * c->elt);
    c->ao = k.take<char>(A * m.n_q_heads * m.head_dim * c->elt);
    c->act = k.take<char>(A * F * c->elt);
  }
  return (k.off + 255) & ~(size_t)255;
}

darts_status validate(const darts_model_desc *m, const darts_runtime_desc *rt, char *err, size_t n) {
  if (!m || !rt) { snprintf(err, n, "NULL descriptor"); return DARTS_ERR_INVALID_ARG; }
  if (m->n_layers <= 0 || m->n_q_heads <= 0 || m->n_kv_heads <= 0 || m->head_dim <= 0 || m->n_q_heads % m->n_kv_heads) {
    snprintf(err, n, "bad head geometry"); return DARTS_ERR_INVALID_ARG;
  }
  if (m->dtype != DARTS_F32 && m->dtype != DARTS_BF16) { snprintf(err, n, "dtype must be F32 or BF16"); return DARTS_ERR_UNSUPPORTED; }
  if (m->head_dim % 32 || m->head_dim > 256 || (m->head_dim / 32 != 1 && m->head_dim / 32 != 2 && m->head_dim / 32 != 4 && m->head_dim / 32 != 8)) {
    snprintf(err, n, "head_dim %d not in {32,64,128,256}", m->head_dim); return DARTS_ERR_UNSUPPORTED;
  }
  if (m->n_q_heads / m->n_kv_heads > 32) { snprintf(err, n, "GQA ratio > 32"); return DARTS_ERR_UNSUPPORTED; }
  if (rt->page_size <= 0 || rt->n_pages <= 0 || rt->max_rows <= 0 || rt->max_prompts <= 0 || rt->max_new <= 0 || rt->max_prompt_len <= 0) {
    snprintf(err, n, "runtime sizes must be positive"); return DARTS_ERR_INVALID_ARG;
  }
  if (m->vocab > 0 && m->n_experts == 0 && m->ffn <= 0) { snprintf(err, n, "dense model needs ffn > 0"); return DARTS_ERR_INVALID_ARG; }
  if (m->n_experts < 0 || (m->n_experts > 0 && (m->top_k <= 0 || m->top_k > m->n_experts || m->top_k > 32 || m->expert_ffn <= 0))) {
    snprintf(err, n, "MoE needs 0 < top_k <= min(n_experts, 32) and expert_ffn > 0"); return DARTS_ERR_INVALID_ARG;
  }
  if (m->n_experts > 256) { snprintf(err, n, "n_experts > 256"); return DARTS_ERR_UNSUPPORTED; }
  if (m->vocab > 0 && m->d_model % 4) { snprintf(err, n, "d_model must be a multiple of 4"); return DARTS_ERR_UNSUPPORTED; }
  return DARTS_OK;
}

darts_status check_device(darts_ctx *c) {
  int dev = 0;
  cudaDeviceProp p;
  CUDA_TRY(c, cudaGetDevice(&dev));
  CUDA_TRY(c, cudaGetDeviceProperties(&p, dev));
  if (p.major != 10) FAIL(c, DARTS_ERR_UNSUPPORTED, "device is sm_%d%d; this library is sm_100a only (no fallback)", p.major, p.minor);
  c->n_sms = p.multiProcessorCount;
  return DARTS_OK;
}

const void **dup_ptrs(const void *const *src, int n) {
  if (!src) return nullptr;
  const void **d = new const void *[n];
  for (int i = 0; i < n; ++i) d[i] = src[i];
  return d;
}

#define TRY(x) do { darts_status s__ = (x); if (s__ != DARTS_OK) return s__; } while (0)

// Parity hook: keep the residual stream at a layer boundary (boundary b = input of layer b; b = n_layers: output of the last layer).
darts_status dump_hidden(darts_ctx *c, int boundary, int rows_ub) {
  if (!c->hid_dump) return DARTS_OK;
  CUDA_TRY(c, cudaMemcpyAsync(c->hid_dump + (size_t)boundary * c->act_rows * c->m.d_model, c->h, (size_t)rows_ub * c->m.d_model * sizeof(float),
                              cudaMemcpyDeviceToDevice, c->stream));
  return DARTS_OK;
}

// One transformer pass over `rows` slots whose plan (slot_*) is already on the device.
darts_status forward_layers(darts_ctx *c, int rows_ub, const int32_t *n_rows_dev) {
  const darts_model_desc &m = c->m;
  TRY(launch_embed(c, c->slot_tok, 0, rows_ub, n_rows_dev));
  TRY(dump_hidden(c, 0, rows_ub));
  TRY(launch_rope_table(c, rows_ub, n_rows_dev));
  int qd = m.n_q_heads * m.head_dim;
  for (int l = 0; l < m.n_layers; ++l) {
    TRY(launch_rmsnorm(c, c->h, c->attn_norm[l], c->xn, rows_ub, n_rows_dev));
    TRY(launch_gemm(c, c->xn, c->wqkv[l], c->qkv32, c->n_qkv, m.d_model, rows_ub, n_rows_dev, false));
    TRY(launch_rope_append(c, l, rows_ub, n_rows_dev));
    TRY(launch_attention(c, l, c->q, c->ao, rows_ub, n_rows_dev));
    TRY(launch_gemm(c, c->ao, c->wo[l], c->h, m.d_model, qd, rows_ub, n_rows_dev, true));
    TRY(launch_rmsnorm(c, c->h, c->mlp_norm[l], c->xn, rows_ub, n_rows_dev));
    if (m.n_experts == 0) {
      TRY(launch_gemm(c, c->xn, c->wgu[l], c->gu32, 2 * m.ffn, m.d_model, rows_ub, n_rows_dev, false));
      TRY(launch_silu_mul(c, rows_ub, n_rows_dev));
      TRY(launch_gemm(c, c->act, c->wd[l], c->h, m.d_model, m.ffn, rows_ub, n_rows_dev, true));
    } else {
      TRY(launch_moe(c, l, rows_ub, n_rows_dev));
    }
    TRY(dump_hidden(c, l + 1, rows_ub));
  }
  return DARTS_OK;
}

// Tensor-core path (bf16): every projection on the stream-K tcgen05 kernel, its pieces reduced inside the consumer
// kernels, the residual add fused with the next RMSNorm.  Leaves xn = rmsnorm(h_L) * final_norm for the LM head.
SkGemm sk_gemm(darts_ctx *c, const XMaps *x, const CUtensorMap *w, int N, int K, int rows_ub, const int32_t *n_rows_dev) {
  SkGemm g{};
  g.w_map = w; g.x_maps = x; g.C = c->part; g.N = N; g.rows_ub = rows_ub; g.n_rows_dev = n_rows_dev; g.np_table = c->sk_np;
  g.pairs = c->use_pairs;
  g.plan = g.pairs ? sk2_plan(c->n_sms, N, K, rows_ub, n_rows_dev == nullptr) : sk_plan(c->n_sms, N, K, rows_ub, 0, n_rows_dev == nullptr);
  g.slot_stride = (size_t)rows_ub * N;
  return g;
}

darts_status run_gemm_sk(darts_ctx *c, const SkGemm &g) { return g.pairs ? launch_gemm_sk2(c, g) : launch_gemm_sk(c, g); }

darts_status forward_layers_tc(darts_ctx *c, int rows_ub, const int32_t *n_rows_dev) {
  const darts_model_desc &m = c->m;
  const int d = m.d_model, qd = m.n_q_heads * m.head_dim, F = m.ffn, L = m.n_layers;
  TRY(launch_moe_begin_pass(c));
  TRY(launch_embed_norm_rope(c, c->slot_tok, c->attn_norm[0], rows_ub, n_rows_dev));     // embedding, first RMSNorm, RoPE table: one launch
  TRY(dump_hidden(c, 0, rows_ub));
  // -DDARTS_PROFILING builds: DARTS_SKIP bit k drops the k-th kernel class of every layer so that the change of the step time gives that
  // class's LIVE cost (launch-list times are serialised and cold); results are garbage in that mode.  Default build: nothing is skipped.
  for (int l = 0; l < L; ++l) {
    SkGemm g = sk_gemm(c, &c->xm_xn, &c->tm_wqkv[l], c->n_qkv, d, rows_ub, n_rows_dev);
    if (!DARTS_SKIPPED(c, 1)) TRY(run_gemm_sk(c, g));
    if (!DARTS_SKIPPED(c, 2)) TRY(launch_rope_append_sk(c, l, sk_view(g), rows_ub, n_rows_dev));
    if (!(DARTS_SKIPPED(c, 4) && DARTS_SKIPPED(c, 8))) TRY(launch_attention(c, l, c->q, c->ao, rows_ub, n_rows_dev));
    g = sk_gemm(c, &c->xm_ao, &c->tm_wo[l], d, qd, rows_ub, n_rows_dev);
    if (!DARTS_SKIPPED(c, 16)) TRY(run_gemm_sk(c, g));
    if (!DARTS_SKIPPED(c, 32)) TRY(launch_add_rmsnorm_sk(c, sk_view(g), c->mlp_norm[l], rows_ub, n_rows_dev));
    const void *next_norm = l + 1 < L ? c->attn_norm[l + 1] : c->final_norm;
    if (m.n_experts == 0) {
      g = sk_gemm(c, &c->xm_xn, &c->tm_wgu[l], 2 * F, d, rows_ub, n_rows_dev);
      if (!DARTS_SKIPPED(c, 64)) TRY(run_gemm_sk(c, g));
      if (!DARTS_SKIPPED(c, 128)) TRY(launch_silu_mul_sk(c, sk_view(g), rows_ub, n_rows_dev));
      g = sk_gemm(c, &c->xm_act, &c->tm_wd[l], d, F, rows_ub, n_rows_dev);
      if (!DARTS_SKIPPED(c, 256)) TRY(run_gemm_sk(c, g));
      if (!DARTS_SKIPPED(c, 512)) TRY(launch_add_rmsnorm_sk(c, sk_view(g), next_norm, rows_ub, n_rows_dev));
    } else {
      TRY(launch_moe_tc(c, l, next_norm, rows_ub, n_rows_dev));
    }
    TRY(dump_hidden(c, l + 1, rows_ub));
  }
  return DARTS_OK;
}

// LM head over xn (or any bf16 [rows][d] matrix behind `a`): plain logits store (prefill) or fused sampling (decode).
darts_status lm_head_tc(darts_ctx *c, const CUtensorMap *a, float *logits_out, int rows_ub, const int32_t *n_rows_dev, bool sample) {
  TcGemm g{};
  g.a_map = a; g.b_map = &c->tm_lm; g.C = logits_out; g.N = c->m.vocab; g.K = c->m.d_model; g.rows_ub = rows_ub; g.n_rows_dev = n_rows_dev;
  g.S = 1; g.split_stride = 0; g.sample = sample;
  return launch_gemm_tc(c, g);
}

darts_status make_maps(darts_ctx *c) {
  const darts_model_desc &m = c->m;
  const int d = m.d_model, qd = m.n_q_heads * m.head_dim, L = m.n_layers;
  c->tm_wqkv = new CUtensorMap[L]; c->tm_wo = new CUtensorMap[L];
  if (m.n_experts == 0) { c->tm_wgu = new CUtensorMap[L]; c->tm_wd = new CUtensorMap[L]; }
  else { c->tm_wgu_e = new CUtensorMap[L]; c->tm_wd_e = new CUtensorMap[L]; }
  for (int l = 0; l < L; ++l) {
    TRY(tc_make_map(c, &c->tm_wqkv[l], c->wqkv[l], c->n_qkv, d, 128));
    TRY(tc_make_map(c, &c->tm_wo[l], c->wo[l], d, qd, 128));
    if (m.n_experts == 0) {
      TRY(tc_make_map(c, &c->tm_wgu[l], c->wgu[l], 2 * m.ffn, d, 128));
      TRY(tc_make_map(c, &c->tm_wd[l], c->wd[l], d, m.ffn, 128));
    } else {
      TRY(tc_make_map(c, &c->tm_wgu_e[l], c->wgu_e[l], (long long)m.n_experts * 2 * m.expert_ffn, d, 128));
      TRY(tc_make_map(c, &c->tm_wd_e[l], c->wd_e[l], (long long)m.n_experts * d, m.expert_ffn, 128));
    }
  }
  TRY(tc_make_map(c, &c->tm_lm, c->lm_head, m.vocab, d, 128));
  TRY(tc_make_map(c, &c->tm_xn, c->xn, c->act_rows, d, 16));
  TRY(tc_make_map(c, &c->tm_ao, c->ao, c->act_rows, qd, 16));
  TRY(tc_make_xmaps(c, &c->xm_xn, c->xn, c->act_rows, d));
  TRY(tc_make_xmaps(c, &c->xm_ao, c->ao, c->act_rows, qd));
  TRY(tc_make_map(c, &c->tm_hl, c->hlast, c->rt.max_prompts, d, 16));
  if (m.n_experts == 0) {
    TRY(tc_make_map(c, &c->tm_act, c->act, c->act_rows, m.ffn, 16));
    TRY(tc_make_xmaps(c, &c->xm_act, c->act, c->act_rows, m.ffn));
  } else {
    TRY(tc_make_xmaps(c, &c->xm_act, c->act, (long long)c->act_rows * m.top_k, m.expert_ffn));
    TRY(tc_make_xmaps(c, &c->xm_xs, c->xs, (long long)c->act_rows * m.top_k, d));
    TRY(tc_make_map(c, &c->tm_act, c->act, (long long)c->act_rows * m.top_k, m.expert_ffn, 16));
    TRY(tc_make_map(c, &c->tm_xs, c->xs, (long long)c->act_rows * m.top_k, d, 16));
  }
  return DARTS_OK;
}

void refresh_ub(darts_ctx *c) {
  long long v = *(volatile long long *)c->pinned;          // {n_active, generation} written in one store
  if ((uint32_t)(v >> 32) == c->gen) c->host_active_ub = std::min(c->host_active_ub, (int32_t)(v & 0xffffffff));
}

darts_status prefill_impl(darts_ctx *c, const int32_t *prompt_tokens_dev, bool tokens_in_place, const int32_t *offs, int32_t G,
                          const int32_t *Kp, const int32_t *forced_len_dev, const darts_policy *pol, float temperature, uint64_t seed,
                          bool sample_step0 = true) {
  if (c->sticky) return c->sticky;
  if (!c->has_weights) FAIL(c, DARTS_ERR_BAD_STATE, "context was created without weights (attention-only)");
  if (!offs || !Kp || !pol || G <= 0 || (!tokens_in_place && !prompt_tokens_dev)) FAIL(c, DARTS_ERR_INVALID_ARG, "NULL argument or G <= 0");
  if (G > c->rt.max_prompts) FAIL(c, DARTS_ERR_INVALID_ARG, "G=%d > max_prompts=%d", G, c->rt.max_prompts);
  darts_policy p = *pol;
  if (p.M_up <= 0) p.M_up = 2 * p.K;                                            // PAPER.md:204 (M_up = 2M)
  if (p.K <= 0 || p.K > DARTS_MAX_KP || p.L_long < 0 || p.L_long >= p.K)
    FAIL(c, DARTS_ERR_INVALID_ARG, "need 0 < K <= 32 and 0 <= L_long < K (K=%d, L_long=%d)", p.K, p.L_long);
  if (p.mode < DARTS_MODE_AUTO || p.mode > DARTS_MODE_SHORTEST_EARLY_STOP) FAIL(c, DARTS_ERR_INVALID_ARG, "bad mode %d", p.mode);
  std::vector<int32_t> g_off(G + 1), plen(G), tok_off(G + 1), pre_pages((size_t)G * c->max_prefix_pages, -1);
  int R = 0, Kp_max = 0, n_prefix_pages = 0;
  for (int i = 0; i < G; ++i) {
    if (Kp[i] < p.K || Kp[i] > DARTS_MAX_KP) FAIL(c, DARTS_ERR_INVALID_ARG, "need K <= Kp[i] <= 32 (Kp[%d]=%d, K=%d)", i, Kp[i], p.K);
    int P = offs[i + 1] - offs[i];
    if (P <= 0 || P > c->rt.max_prompt_len) FAIL(c, DARTS_ERR_INVALID_ARG, "prompt %d has length %d (max %d)", i, P, c->rt.max_prompt_len);
    g_off[i] = R; plen[i] = P; tok_off[i] = offs[i] - offs[0];
    R += Kp[i]; Kp_max = std::max(Kp_max, Kp[i]);
    for (int q = 0; q < ceil_div(P, c->rt.page_size); ++q) pre_pages[(size_t)i * c->max_prefix_pages + q] = n_prefix_pages++;
  }
  g_off[G] = R; tok_off[G] = offs[G] - offs[0];
  if (R > c->rt.max_rows) FAIL(c, DARTS_ERR_INVALID_ARG, "sum Kp = %d > max_rows = %d", R, c->rt.max_rows);
  if (n_prefix_pages > c->rt.n_pages) FAIL(c, DARTS_ERR_KV_POOL_EXHAUSTED, "prefix needs %d pages, pool has %d", n_prefix_pages, c->rt.n_pages);
  c->pol = p; c->temperature = temperature; c->seed = seed; c->G = G; c->R = R; c->Kp_max = Kp_max;
  if (c->max_len <= 0 || c->max_len > c->rt.max_new) c->max_len = c->rt.max_new;
  c->gen += 1; c->host_active_ub = R; c->steps_issued = 0; c->prefilled = false; c->prof_n = 0;
  cudaStream_t s = c->stream;
  int total_tok = tok_off[G];
  if (!tokens_in_place)
    CUDA_TRY(c, cudaMemcpyAsync(c->prompt_tokens, prompt_tokens_dev + offs[0], (size_t)total_tok * 4, cudaMemcpyDeviceToDevice, s));
  CUDA_TRY(c, cudaMemcpyAsync(c->g_off, g_off.data(), (G + 1) * 4, cudaMemcpyHostToDevice, s));
  CUDA_TRY(c, cudaMemcpyAsync(c->g_Kp, Kp, G * 4, cudaMemcpyHostToDevice, s));
  CUDA_TRY(c, cudaMemcpyAsync(c->g_plen, plen.data(), G * 4, cudaMemcpyHostToDevice, s));
  CUDA_TRY(c, cudaMemcpyAsync(c->g_tok_off, tok_off.data(), (G + 1) * 4, cudaMemcpyHostToDevice, s));
  CUDA_TRY(c, cudaMemcpyAsync(c->g_prefix_pages, pre_pages.data(), pre_pages.size() * 4, cudaMemcpyHostToDevice, s));
  CUDA_TRY(c, cudaMemsetAsync(c->tokens_out, 0xFF, (size_t)R * c->rt.max_new * 4, s));
  CUDA_TRY(c, cudaMemsetAsync(c->margin_out, 0, (size_t)R * c->rt.max_new * 4, s));
  CUDA_TRY(c, cudaMemsetAsync(c->logprob_out, 0, (size_t)R * c->rt.max_new * 4, s));
  CUDA_TRY(c, cudaMemsetAsync(c->g_sel, 0xFF, (size_t)G * DARTS_MAX_KP * 4, s));
  TRY(launch_init_rows(c, forced_len_dev, n_prefix_pages));
  // one causal pass per PROMPT, in chunks of whole prompts
  int chunk = default_chunk(&c->rt);
  for (int g0 = 0; g0 < G;) {
    int g1 = g0, ntok = 0;
    while (g1 < G && ntok + plen[g1] <= chunk) ntok += plen[g1++];
    int tb = tok_off[g0];
    TRY(launch_plan_prefill(c, tb, ntok, g0, g1));
    c->attn_plan_valid = attention_sm100_supported(c);                            // causal plan: blocks of query positions x 512-token chunks
    if (c->attn_plan_valid) TRY(launch_attention_plan_sm100(c, ntok, nullptr, true));
    if (c->tc_path) {
      TRY(forward_layers_tc(c, ntok, nullptr));
      TRY(launch_gather_rows_bf16(c, c->xn, c->hlast, tb, g0, g1));             // final-normed hidden of each prompt's last token
      TRY(lm_head_tc(c, &c->tm_hl, c->z0 + (size_t)g0 * c->m.vocab, g1 - g0, nullptr, false));
    } else {
      TRY(forward_layers(c, ntok, nullptr));
      TRY(launch_gather_last(c, tb, ntok, g0, g1));
      TRY(launch_rmsnorm(c, c->hlast, c->final_norm, c->xn, g1 - g0, nullptr));
      CUDA_TRY(c, cudaMemcpyAsync((char *)c->pend0 + (size_t)g0 * c->m.d_model * c->elt, c->xn, (size_t)(g1 - g0) * c->m.d_model * c->elt,
                                  cudaMemcpyDeviceToDevice, s));                   // kept for darts_score_begin (scores every row's token 0)
      TRY(launch_gemm(c, c->xn, c->lm_head, c->z0 + (size_t)g0 * c->m.vocab, c->m.vocab, c->m.d_model, g1 - g0, nullptr, false));
    }
    g0 = g1;
  }
  if (sample_step0) TRY(launch_sample(c, c->z0, 1, R));                          // step 0: Kp[i] draws from the shared z0[i]
  c->prefilled = true;
  c->score_mode = false;
  return DARTS_OK;
}

}  // namespace

// dispatchers: the tuned sm_100a kernels take the shapes they support, the generic kernels the rest
darts_status launch_attention_sm100(darts_ctx *c, int layer, const void *q, void *out, int rows_ub, const int32_t *n_rows_dev, bool *taken);

darts_status launch_gemm(darts_ctx *c, const void *X, const void *W, float *C, int N, int K, int rows_ub, const int32_t *n_rows_dev,
                         bool accumulate, bool w_is_f32) {
  if (rows_ub <= 0) return DARTS_OK;
  return launch_gemm_simt(c, X, W, C, N, K, rows_ub, n_rows_dev, accumulate, w_is_f32);
}

darts_status launch_attention(darts_ctx *c, int layer, const void *q, void *out, int rows_ub, const int32_t *n_rows_dev) {
  if (rows_ub <= 0) return DARTS_OK;
  bool prof = (c->rt.flags & DARTS_FLAG_PROFILE_ATTENTION) && layer == 0 && c->in_decode;
  if (prof) {
    while ((int)c->prof_ev.size() < 2 * (c->prof_n + 1)) {
      cudaEvent_t e;
      CUDA_TRY(c, cudaEventCreate(&e));
      c->prof_ev.push_back(e);
    }
    CUDA_TRY(c, cudaEventRecord(c->prof_ev[2 * c->prof_n], c->stream));
  }
  bool taken = false;
  darts_status s = launch_attention_sm100(c, layer, q, out, rows_ub, n_rows_dev, &taken);
  if (s == DARTS_OK && !taken) s = launch_attention_ref(c, layer, q, out, rows_ub, n_rows_dev);
  if (prof && s == DARTS_OK) {
    CUDA_TRY(c, cudaEventRecord(c->prof_ev[2 * c->prof_n + 1], c->stream));
    c->prof_n++;
  }
  return s;
}

extern "C" {

darts_status darts_workspace_bytes(const darts_model_desc *m, const darts_runtime_desc *rt, size_t *out) {
  char err[128];
  if (!out) return DARTS_ERR_INVALID_ARG;
  darts_status s = validate(m, rt, err, sizeof(err));
  if (s != DARTS_OK) return s;
  darts_ctx tmp{};
  tmp.m = *m; tmp.rt = *rt;
  *out = carve(&tmp, nullptr);
  return DARTS_OK;
}

darts_status darts_create(const darts_model_desc *m, const darts_weights *w, const darts_runtime_desc *rt, darts_ctx **out) {
  if (!out) return DARTS_ERR_INVALID_ARG;
  *out = nullptr;
  char err[128];
  darts_status s = validate(m, rt, err, sizeof(err));
  if (s != DARTS_OK) return s;
  if (m->vocab > 0 && !w) return DARTS_ERR_INVALID_ARG;
  if (!rt->workspace) return DARTS_ERR_INVALID_ARG;
  darts_ctx *c = new (std::nothrow) darts_ctx{};
  if (!c) return DARTS_ERR_INVALID_ARG;
  c->m = *m; c->rt = *rt; c->stream = (cudaStream_t)rt->stream;
  *out = c;                                    // returned even on failure so darts_last_error can be read
  if ((s = check_device(c)) != DARTS_OK) return s;
  size_t need = carve(c, rt->workspace);
  if (need > rt->workspace_bytes) FAIL(c, DARTS_ERR_WORKSPACE_TOO_SMALL, "workspace %zu < %zu bytes", rt->workspace_bytes, need);
  if (((uintptr_t)rt->workspace & 255) != 0) FAIL(c, DARTS_ERR_INVALID_ARG, "workspace must be 256-byte aligned");
  c->has_weights = m->vocab > 0;
  c->use_pdl = true;
#ifdef DARTS_PROFILING
  c->use_pdl = getenv("DARTS_NO_PDL") == nullptr;
  c->skip_mask = getenv("DARTS_SKIP") ? (unsigned)strtoul(getenv("DARTS_SKIP"), nullptr, 0) : 0u;
#endif
  c->use_pairs = (rt->flags & DARTS_FLAG_CTA_PAIRS) != 0;
  if ((s = gemm_sk_configure(c)) != DARTS_OK || (s = gemm_sk2_configure(c)) != DARTS_OK || (s = gemm_tc_configure(c)) != DARTS_OK || (s = attn_sm100_configure(c)) != DARTS_OK ||
      (s = moe_configure(c)) != DARTS_OK)
    return s;
  if (c->has_weights) {
    int L = m->n_layers;
    c->embed = w->embed; c->final_norm = w->final_norm; c->lm_head = w->lm_head;
    c->attn_norm = dup_ptrs(w->attn_norm, L); c->wqkv = dup_ptrs(w->wqkv, L); c->wo = dup_ptrs(w->wo, L);
    c->q_norm = dup_ptrs(w->q_norm, L); c->k_norm = dup_ptrs(w->k_norm, L);
    c->mlp_norm = dup_ptrs(w->mlp_norm, L); c->wgu = dup_ptrs(w->wgu, L); c->wd = dup_ptrs(w->wd, L);
    c->wr = dup_ptrs(w->wr, L); c->wgu_e = dup_ptrs(w->wgu_e, L); c->wd_e = dup_ptrs(w->wd_e, L);
    bool ok = c->embed && c->final_norm && c->lm_head && c->attn_norm && c->wqkv && c->wo && c->mlp_norm &&
              (m->n_experts ? (c->wr && c->wgu_e && c->wd_e) : (c->wgu && c->wd)) && (!m->qk_norm || (c->q_norm && c->k_norm));
    if (!ok) FAIL(c, DARTS_ERR_INVALID_ARG, "missing weight pointers");
    if (c->tc_path && (s = make_maps(c)) != DARTS_OK) return s;
  }
  void *pin = nullptr;
  CUDA_TRY(c, cudaHostAlloc(&pin, 64, cudaHostAllocMapped));
  memset(pin, 0, 64);
  c->pinned = (volatile int32_t *)pin;
  void *pd = nullptr;
  CUDA_TRY(c, cudaHostGetDevicePointer(&pd, pin, 0));
  c->pinned_dev = (int32_t *)pd;
  CUDA_TRY(c, cudaEventCreateWithFlags(&c->ev[0], cudaEventDisableTiming));
  CUDA_TRY(c, cudaEventCreateWithFlags(&c->ev[1], cudaEventDisableTiming));
  CUDA_TRY(c, cudaMemsetAsync(c->st, 0, sizeof(DevState), c->stream));
  if (c->moe_arrive) CUDA_TRY(c, cudaMemsetAsync(c->moe_arrive, 0, c->moe_arrive_n * sizeof(int32_t), c->stream));
  // The pool must hold finite values everywhere: a partially filled page is multiplied by zero probabilities.
  CUDA_TRY(c, cudaMemsetAsync(c->kv_pool, 0, (size_t)m->n_layers * c->kv_layer_elems * c->elt, c->stream));
  return DARTS_OK;
}

darts_status darts_destroy(darts_ctx *c) {
  if (!c) return DARTS_OK;
  if (c->stream || c->pinned) cudaStreamSynchronize(c->stream);
  if (c->pinned) cudaFreeHost((void *)c->pinned);
  if (c->ev[0]) cudaEventDestroy(c->ev[0]);
  if (c->ev[1]) cudaEventDestroy(c->ev[1]);
  for (cudaEvent_t e : c->prof_ev) cudaEventDestroy(e);
  if (c->copy_stream) {
    cudaStreamSynchronize(c->copy_stream);
    cudaStreamDestroy(c->copy_stream);
    for (int b = 0; b < 2; ++b) { cudaEventDestroy(c->ev_copy_ready[b]); cudaEventDestroy(c->ev_copy_done[b]); if (c->chunk_stage[b]) cudaFreeHost(c->chunk_stage[b]); }
  }
  const void **arrs[] = {c->attn_norm, c->wqkv, c->q_norm, c->k_norm, c->wo, c->mlp_norm, c->wgu, c->wd, c->wr, c->wgu_e, c->wd_e};
  for (auto a : arrs) delete[] a;
  CUtensorMap *maps[] = {c->tm_wqkv, c->tm_wo, c->tm_wgu, c->tm_wd, c->tm_wgu_e, c->tm_wd_e};
  for (auto a : maps) delete[] a;
  delete c;
  return DARTS_OK;
}

const char *darts_last_error(const darts_ctx *c) { return c ? c->err : "NULL context"; }

darts_status darts_prefill(darts_ctx *c, const int32_t *prompt_tokens, const int32_t *prompt_offsets_host, int32_t G,
                           const int32_t *Kp_host, const int32_t *forced_len, const darts_policy *policy, float temperature, uint64_t seed) {
  if (!c) return DARTS_ERR_INVALID_ARG;
  c->max_len = c->rt.max_new;                      // the step-wise API always runs to the context's limit (darts_rollout* pass their own)
  return prefill_impl(c, prompt_tokens, false, prompt_offsets_host, G, Kp_host, forced_len, policy, temperature, seed);
}

darts_status darts_decode_step(darts_ctx *c) {
  if (!c) return DARTS_ERR_INVALID_ARG;
  if (c->sticky) return c->sticky;
  if (!c->prefilled || c->score_mode) FAIL(c, DARTS_ERR_BAD_STATE, "darts_decode_step before darts_prefill (or on a scoring context)");
  refresh_ub(c);
  int ub = c->host_active_ub;
  if (ub <= 0) return DARTS_OK;
  const int32_t *n = &c->st->n_active;
  TRY(launch_plan_decode(c, ub));
  c->attn_plan_valid = attention_sm100_supported(c);
  if (c->attn_plan_valid) TRY(launch_attention_plan_sm100(c, ub, n));
  c->in_decode = true;
  struct Leave { darts_ctx *c; ~Leave() { c->in_decode = false; } } leave{c};
  if (c->tc_path) {
    TRY(forward_layers_tc(c, ub, n));
    // logits never reach HBM (unless DUMP_LOGITS): swap-AB persistent kernel with the sampling epilogue, 4 entries per vocab tile
    if (!(c->rt.flags & DARTS_FLAG_LM_HEAD_TILES) && sk_sample_supported(c, ub)) {
      TRY(launch_gemm_sk_sample(c, &c->tm_lm, &c->xm_xn, c->m.vocab, c->m.d_model, ub, n));
      TRY(launch_sample_finalize(c, 4 * ceil_div(c->m.vocab, 128), ub));
    } else {
      TRY(lm_head_tc(c, &c->tm_xn, nullptr, ub, n, true));
      TRY(launch_sample_finalize(c, ceil_div(c->m.vocab, 128), ub));
    }
  } else {
    TRY(forward_layers(c, ub, n));
    TRY(launch_rmsnorm(c, c->h, c->final_norm, c->xn, ub, n));
    TRY(launch_gemm(c, c->xn, c->lm_head, c->logits, c->m.vocab, c->m.d_model, ub, n, false));
    TRY(launch_sample(c, c->logits, 0, ub));
  }
  c->steps_issued++;
  return DARTS_OK;
}

darts_status darts_select_and_compact(darts_ctx *c, int32_t *n_active_out) {
  if (!c) return DARTS_ERR_INVALID_ARG;
  if (c->sticky) return c->sticky;
  if (!c->prefilled || c->score_mode) FAIL(c, DARTS_ERR_BAD_STATE, "darts_select_and_compact before darts_prefill (or on a scoring context)");
  TRY(launch_select(c));
  return launch_compact(c, n_active_out);
}

darts_status darts_n_active(darts_ctx *c, int32_t *out_host) {
  if (!c || !out_host) return DARTS_ERR_INVALID_ARG;
  DevState st;
  CUDA_TRY(c, cudaMemcpyAsync(&st, c->st, sizeof(st), cudaMemcpyDeviceToHost, c->stream));
  CUDA_TRY(c, cudaStreamSynchronize(c->stream));
  *out_host = st.n_active;
  c->host_active_ub = std::min(c->host_active_ub, st.n_active);
  if (st.err) { c->sticky = st.err; FAIL(c, st.err, "KV page pool exhausted"); }
  return DARTS_OK;
}

darts_status darts_get_attention_times(darts_ctx *c, float *ms_host, int32_t cap, int32_t *n_out) {
  if (!c || !n_out || (cap > 0 && !ms_host)) return DARTS_ERR_INVALID_ARG;
  CUDA_TRY(c, cudaStreamSynchronize(c->stream));
  *n_out = c->prof_n;
  for (int k = 0; k < c->prof_n && k < cap; ++k) CUDA_TRY(c, cudaEventElapsedTime(&ms_host[k], c->prof_ev[2 * k], c->prof_ev[2 * k + 1]));
  return DARTS_OK;
}

darts_status darts_get_results(darts_ctx *c, darts_results *o) {
  if (!c || !o) return DARTS_ERR_INVALID_ARG;
  if (!c->prefilled) FAIL(c, DARTS_ERR_BAD_STATE, "no rollout to read");
  CUDA_TRY(c, cudaStreamSynchronize(c->stream));
  size_t R = c->R, G = c->G, mn = c->rt.max_new;
  if (o->tokens) CUDA_TRY(c, cudaMemcpy(o->tokens, c->tokens_out, R * mn * 4, cudaMemcpyDeviceToHost));
  if (o->margin) CUDA_TRY(c, cudaMemcpy(o->margin, c->margin_out, R * mn * 4, cudaMemcpyDeviceToHost));
  if (o->logprob) CUDA_TRY(c, cudaMemcpy(o->logprob, c->logprob_out, R * mn * 4, cudaMemcpyDeviceToHost));
  if (o->len) CUDA_TRY(c, cudaMemcpy(o->len, c->row_len, R * 4, cudaMemcpyDeviceToHost));
  if (o->status) CUDA_TRY(c, cudaMemcpy(o->status, c->row_status, R, cudaMemcpyDeviceToHost));
  if (o->sel) CUDA_TRY(c, cudaMemcpy(o->sel, c->g_sel, G * c->pol.K * 4, cudaMemcpyDeviceToHost));
  if (o->sel_mask) CUDA_TRY(c, cudaMemcpy(o->sel_mask, c->g_mask, G * 4, cudaMemcpyDeviceToHost));
  if (o->close_step) CUDA_TRY(c, cudaMemcpy(o->close_step, c->g_close_step, G * 4, cudaMemcpyDeviceToHost));
  if (o->len_mean) CUDA_TRY(c, cudaMemcpy(o->len_mean, c->g_len_mean, G * 4, cudaMemcpyDeviceToHost));
  if (o->len_var) CUDA_TRY(c, cudaMemcpy(o->len_var, c->g_len_var, G * 4, cudaMemcpyDeviceToHost));
  if (o->n_pruned) CUDA_TRY(c, cudaMemcpy(o->n_pruned, c->g_n_pruned, G * 4, cudaMemcpyDeviceToHost));
  return DARTS_OK;
}

darts_status darts_get_counters(darts_ctx *c, darts_counters *o) {
  if (!c || !o) return DARTS_ERR_INVALID_ARG;
  DevState st;
  CUDA_TRY(c, cudaMemcpyAsync(&st, c->st, sizeof(st), cudaMemcpyDeviceToHost, c->stream));
  CUDA_TRY(c, cudaStreamSynchronize(c->stream));
  o->n_steps = st.step; o->n_generated_tokens = (int64_t)st.n_generated; o->n_kept_tokens = (int64_t)st.n_kept;
  o->n_near_ties = (int64_t)st.n_near_ties; o->n_row_steps = (int64_t)st.n_row_steps; o->peak_pages = st.peak_used;
  o->kernel_launches = c->launches; o->pages_allocated = (int64_t)st.n_pops;
  return DARTS_OK;
}

// Token-level streaming (§4.3.2, App. E :481-489, rollout side only): every
// `chunk_steps` lock-step iterations the token columns produced since the last chunk are copied device->host on a second
// stream (ordered after the step that produced them by an event, overlapping the following steps) and handed to `fn`.
struct ChunkStream {
  darts_ctx *c;
  int chunk;
  darts_chunk_fn fn;
  void *user;
  int flushed = 0;
  int pend_s0[2] = {0, 0}, pend_s1[2] = {0, 0};
  bool pending[2] = {false, false};
  int next_slot = 0;

  darts_status drain(int b) {
    if (!pending[b]) return DARTS_OK;
    CUDA_TRY(c, cudaEventSynchronize(c->ev_copy_done[b]));
    fn(user, pend_s0[b], pend_s1[b], c->R, c->chunk_stage[b], (const float *)(c->chunk_stage[b] + (size_t)c->R * (pend_s1[b] - pend_s0[b])));
    pending[b] = false;
    return DARTS_OK;
  }
  darts_status issue(int s0, int s1) {
    int b = next_slot;
    next_slot ^= 1;
    darts_status st = drain(b);                               // slots alternate, so chunks are delivered in step order
    if (st != DARTS_OK) return st;
    CUDA_TRY(c, cudaEventRecord(c->ev_copy_ready[b], c->stream));
    CUDA_TRY(c, cudaStreamWaitEvent(c->copy_stream, c->ev_copy_ready[b], 0));
    CUDA_TRY(c, cudaMemcpy2DAsync(c->chunk_stage[b], (size_t)(s1 - s0) * 4, c->tokens_out + s0, (size_t)c->rt.max_new * 4, (size_t)(s1 - s0) * 4,
                                  (size_t)c->R, cudaMemcpyDeviceToHost, c->copy_stream));
    CUDA_TRY(c, cudaMemcpy2DAsync(c->chunk_stage[b] + (size_t)c->R * (s1 - s0), (size_t)(s1 - s0) * 4, c->logprob_out + s0, (size_t)c->rt.max_new * 4,
                                  (size_t)(s1 - s0) * 4, (size_t)c->R, cudaMemcpyDeviceToHost, c->copy_stream));   // log-probs behind the tokens
    CUDA_TRY(c, cudaEventRecord(c->ev_copy_done[b], c->copy_stream));
    pend_s0[b] = s0; pend_s1[b] = s1; pending[b] = true;
    flushed = s1;
    return DARTS_OK;
  }
};

static darts_status run_loop(darts_ctx *c, darts_results *out, ChunkStream *cs) {
  if (c->sticky) return c->sticky;
  if (!c->prefilled) FAIL(c, DARTS_ERR_BAD_STATE, "darts_run_to_completion before darts_prefill");
  TRY(darts_select_and_compact(c, nullptr));
  // The host never waits for a step's result: it sizes grids from a stale (monotone, hence safe) upper
  // bound of n_active mirrored in pinned memory and stays at most two iterations ahead of the device.
  for (int it = 0; it <= c->max_len + 4; ++it) {
    refresh_ub(c);
    if (c->host_active_ub <= 0) break;
    TRY(darts_decode_step(c));
    TRY(darts_select_and_compact(c, nullptr));
    CUDA_TRY(c, cudaEventRecord(c->ev[it & 1], c->stream));
    if (it >= 1) CUDA_TRY(c, cudaEventSynchronize(c->ev[(it + 1) & 1]));
    if (cs && it + 2 - cs->flushed >= cs->chunk && cs->flushed + cs->chunk <= c->max_len)   // token columns [0, it + 2) are enqueued
      TRY(cs->issue(cs->flushed, cs->flushed + cs->chunk));
  }
  CUDA_TRY(c, cudaStreamSynchronize(c->stream));
  int32_t na = 0;
  TRY(darts_n_active(c, &na));
  if (na != 0) FAIL(c, DARTS_ERR_BAD_STATE, "rollout loop ended with %d active rows", na);
  if (cs) {
    DevState st;
    CUDA_TRY(c, cudaMemcpy(&st, c->st, sizeof(st), cudaMemcpyDeviceToHost));
    while (cs->flushed < st.step) TRY(cs->issue(cs->flushed, std::min(st.step, cs->flushed + cs->chunk)));
    TRY(cs->drain(cs->next_slot));
    TRY(cs->drain(cs->next_slot ^ 1));
  }
  return out ? darts_get_results(c, out) : DARTS_OK;
}

darts_status darts_run_to_completion(darts_ctx *c, darts_results *out) {
  if (!c) return DARTS_ERR_INVALID_ARG;
  return run_loop(c, out, nullptr);
}

darts_status darts_run_to_completion_streaming(darts_ctx *c, int32_t chunk_steps, darts_chunk_fn fn, void *user, darts_results *out) {
  if (!c) return DARTS_ERR_INVALID_ARG;
  if (!fn || chunk_steps <= 0) FAIL(c, DARTS_ERR_INVALID_ARG, "chunk_steps must be positive and fn non-NULL");
  if (!c->prefilled) FAIL(c, DARTS_ERR_BAD_STATE, "darts_run_to_completion_streaming before darts_prefill");
  size_t need = (size_t)c->R * chunk_steps * 8;              // tokens + their log-probabilities
  if (!c->copy_stream) {
    CUDA_TRY(c, cudaStreamCreateWithFlags(&c->copy_stream, cudaStreamNonBlocking));
    for (int b = 0; b < 2; ++b) {
      CUDA_TRY(c, cudaEventCreateWithFlags(&c->ev_copy_ready[b], cudaEventDisableTiming));
      CUDA_TRY(c, cudaEventCreateWithFlags(&c->ev_copy_done[b], cudaEventDisableTiming));
    }
  }
  if (need > c->chunk_stage_bytes) {
    for (int b = 0; b < 2; ++b) {
      if (c->chunk_stage[b]) cudaFreeHost(c->chunk_stage[b]);
      c->chunk_stage[b] = nullptr;
      CUDA_TRY(c, cudaHostAlloc((void **)&c->chunk_stage[b], need, cudaHostAllocDefault));
    }
    c->chunk_stage_bytes = need;
  }
  ChunkStream cs{c, chunk_steps, fn, user};
  return run_loop(c, out, &cs);
}

static darts_status rollout_common(darts_ctx *c, const int32_t *prompts_dev, bool in_place, int32_t prompt_len, int32_t G,
                                   const int32_t *Kp, const int32_t *forced_dev, const darts_policy *pol, int32_t max_len,
                                   float temperature, uint64_t seed, darts_results *out) {
  if (prompt_len <= 0 || G <= 0) FAIL(c, DARTS_ERR_INVALID_ARG, "prompt_len and G must be positive");
  if (max_len <= 0 || max_len > c->rt.max_new) FAIL(c, DARTS_ERR_INVALID_ARG, "max_len %d outside (0, max_new=%d]", max_len, c->rt.max_new);
  std::vector<int32_t> offs(G + 1);
  for (int i = 0; i <= G; ++i) offs[i] = i * prompt_len;
  c->max_len = max_len;
  TRY(prefill_impl(c, prompts_dev, in_place, offs.data(), G, Kp, forced_dev, pol, temperature, seed));
  return darts_run_to_completion(c, out);
}

darts_status darts_rollout(darts_ctx *c, const int32_t *prompts, int32_t prompt_len, int32_t G, int32_t Kp_scalar, int32_t K,
                           int32_t max_len, float temperature, uint64_t seed, const int32_t *forced_len, darts_results *out) {
  if (!c) return DARTS_ERR_INVALID_ARG;
  if (!prompts) FAIL(c, DARTS_ERR_INVALID_ARG, "prompts is NULL");
  std::vector<int32_t> Kp(std::max(G, 1), Kp_scalar);
  darts_policy pol{K, K > 1 ? 1 : 0, 2 * K, DARTS_MODE_AUTO};                    // L=1, M_up=2M (:204)
  return rollout_common(c, prompts, false, prompt_len, G, Kp.data(), forced_len, &pol, max_len, temperature, seed, out);
}

darts_status darts_rollout_host(darts_ctx *c, const int32_t *prompts_host, int32_t prompt_len, int32_t G, const int32_t *Kp_host,
                                const int32_t *forced_len_host, const darts_policy *policy, int32_t max_len, float temperature,
                                uint64_t seed, darts_results *out) {
  if (!c) return DARTS_ERR_INVALID_ARG;
  if (!prompts_host || !Kp_host || !policy) FAIL(c, DARTS_ERR_INVALID_ARG, "NULL argument");
  if (G <= 0 || G > c->rt.max_prompts || prompt_len <= 0 || prompt_len > c->rt.max_prompt_len) FAIL(c, DARTS_ERR_INVALID_ARG, "bad G / prompt_len");
  if (!c->has_weights) FAIL(c, DARTS_ERR_BAD_STATE, "attention-only context");
  CUDA_TRY(c, cudaMemcpyAsync(c->prompt_tokens, prompts_host, (size_t)G * prompt_len * 4, cudaMemcpyHostToDevice, c->stream));
  const int32_t *forced_dev = nullptr;
  if (forced_len_host) {
    int Kp_max = 0;
    for (int i = 0; i < G; ++i) Kp_max = std::max(Kp_max, Kp_host[i]);
    if (Kp_max > DARTS_MAX_KP) FAIL(c, DARTS_ERR_INVALID_ARG, "Kp > 32");
    CUDA_TRY(c, cudaMemcpyAsync(c->forced_stage, forced_len_host, (size_t)G * Kp_max * 4, cudaMemcpyHostToDevice, c->stream));
    forced_dev = c->forced_stage;
  }
  return rollout_common(c, nullptr, true, prompt_len, G, Kp_host, forced_dev, policy, max_len, temperature, seed, out);
}

// ---- consumer half of token-level streaming (§4.3.2; App. E :481-489) --------------------------
darts_status darts_score_begin(darts_ctx *c, const int32_t *prompt_tokens, const int32_t *prompt_offsets_host, int32_t G, const int32_t *Kp_host,
                               float temperature) {
  if (!c) return DARTS_ERR_INVALID_ARG;
  if ((c->m.d_model * c->elt) % 16) FAIL(c, DARTS_ERR_UNSUPPORTED, "scoring needs 16-byte hidden rows");
  c->max_len = c->rt.max_new;
  darts_policy pol{1, 0, 0, DARTS_MODE_DUAL_END};              // no rule runs on a scoring context; the fields only have to be valid
  TRY(prefill_impl(c, prompt_tokens, false, prompt_offsets_host, G, Kp_host, nullptr, &pol, temperature, 0, false));
  const int R = c->R, page = c->rt.page_size;
  std::vector<int32_t> prompt_of(R);
  int n_prefix = 0, r = 0;
  for (int i = 0; i < G; ++i) {
    n_prefix += ceil_div(prompt_offsets_host[i + 1] - prompt_offsets_host[i], page);
    for (int j = 0; j < Kp_host[i]; ++j) prompt_of[r++] = i;
  }
  c->sc_len.assign(R, 0);
  c->sc_pages.assign((size_t)R * c->max_suffix_pages, -1);
  c->sc_free.clear();
  for (int p = c->rt.n_pages - 1; p >= n_prefix; --p) c->sc_free.push_back(p);      // back of the vector = lowest id = next page handed out
  CUDA_TRY(c, cudaMemcpyAsync(c->score_idx, prompt_of.data(), (size_t)R * 4, cudaMemcpyHostToDevice, c->stream));
  TRY(launch_score_init_pend(c, R));
  CUDA_TRY(c, cudaStreamSynchronize(c->stream));                                   // prompt_of is a local
  c->score_mode = true;
  return DARTS_OK;
}

// One pass: rows [r0, r1), each forwarding its m[r] leading valid tokens of the chunk.  Slots are row-major, step-minor.
static darts_status score_pass(darts_ctx *c, int r0, int r1, int s0, int n, const int32_t *tokens, const std::vector<int> &m, float *lp_out) {
  const int page = c->rt.page_size, msp = c->max_suffix_pages;
  std::vector<int32_t> g_plen(c->G), g_off(c->G + 1);
  CUDA_TRY(c, cudaMemcpy(g_plen.data(), c->g_plen, (size_t)c->G * 4, cudaMemcpyDeviceToHost));
  CUDA_TRY(c, cudaMemcpy(g_off.data(), c->g_off, (size_t)(c->G + 1) * 4, cudaMemcpyDeviceToHost));
  std::vector<int32_t> s_row, s_tok, s_pos, s_pg, s_off, s_pr, s_npre, s_nsuf, tgt, idx_rows, idx_last;
  int i = 0;
  for (int r = r0; r < r1; ++r) {
    if (m[r] == 0) continue;
    while (g_off[i + 1] <= r) ++i;
    for (int k = 0; k < m[r]; ++k) {
      const int s = s0 + k;                                   // suffix index of this token = its step
      if (s % page == 0) {
        if (c->sc_free.empty()) { c->sticky = DARTS_ERR_KV_POOL_EXHAUSTED; FAIL(c, DARTS_ERR_KV_POOL_EXHAUSTED, "scoring context ran out of KV pages"); }
        c->sc_pages[(size_t)r * msp + s / page] = c->sc_free.back();
        c->sc_free.pop_back();
      }
      s_row.push_back(r); s_tok.push_back(tokens[(size_t)r * n + k]); s_pos.push_back(g_plen[i] + s);
      s_pg.push_back(c->sc_pages[(size_t)r * msp + s / page]); s_off.push_back(s % page);
      s_pr.push_back(i); s_npre.push_back(g_plen[i]); s_nsuf.push_back(s + 1);
      tgt.push_back(k + 1 < m[r] ? tokens[(size_t)r * n + k + 1] : -1);              // this slot's logits score the row's NEXT token of the chunk
    }
    idx_rows.push_back(r);
    idx_last.push_back((int32_t)s_row.size() - 1);
    CUDA_TRY(c, cudaMemcpyAsync(c->row_pages + (size_t)r * msp, &c->sc_pages[(size_t)r * msp], (size_t)msp * 4, cudaMemcpyHostToDevice, c->stream));
  }
  const int S = (int)s_row.size(), n_pend = (int)idx_rows.size();
  if (S == 0) return DARTS_OK;
  for (int r : idx_rows) tgt.push_back(tokens[(size_t)r * n]);                       // the pending hidden scores the chunk's first token
  cudaStream_t st = c->stream;
  auto up = [&](int32_t *dst, const std::vector<int32_t> &v) { return cudaMemcpyAsync(dst, v.data(), v.size() * 4, cudaMemcpyHostToDevice, st); };
  CUDA_TRY(c, up(c->slot_row, s_row)); CUDA_TRY(c, up(c->slot_tok, s_tok)); CUDA_TRY(c, up(c->slot_pos, s_pos));
  CUDA_TRY(c, up(c->slot_dst_page, s_pg)); CUDA_TRY(c, up(c->slot_dst_off, s_off)); CUDA_TRY(c, up(c->slot_prompt, s_pr));
  CUDA_TRY(c, up(c->slot_npre, s_npre)); CUDA_TRY(c, up(c->slot_nsuf, s_nsuf)); CUDA_TRY(c, up(c->score_tgt, tgt));
  CUDA_TRY(c, up(c->score_idx, idx_rows)); CUDA_TRY(c, up(c->score_idx + c->rt.max_rows, idx_last));
  c->attn_plan_valid = attention_sm100_supported(c);
  if (c->attn_plan_valid) TRY(launch_attention_plan_sm100(c, S, nullptr));
  const int rows_lm = S + n_pend;
  if (c->tc_path) {
    TRY(forward_layers_tc(c, S, nullptr));                                          // leaves xn = rmsnorm(h_L) * final_norm for the S slots
    TRY(launch_score_gather(c, S, n_pend));
    if (!sk_sample_supported(c, rows_lm)) FAIL(c, DARTS_ERR_UNSUPPORTED, "scoring needs d_model %% 64 == 0 and vocab %% 4 == 0 on the tensor-core path");
    TRY(launch_gemm_sk_sample(c, &c->tm_lm, &c->xm_xn, c->m.vocab, c->m.d_model, rows_lm, nullptr, c->score_tgt));
    TRY(launch_score_finalize(c, 4 * ceil_div(c->m.vocab, 128), rows_lm));
  } else {
    TRY(forward_layers(c, S, nullptr));
    TRY(launch_rmsnorm(c, c->h, c->final_norm, c->xn, S, nullptr));
    TRY(launch_score_gather(c, S, n_pend));
    TRY(launch_gemm(c, c->xn, c->lm_head, c->logits, c->m.vocab, c->m.d_model, rows_lm, nullptr, false));
    TRY(launch_score_logits(c, rows_lm));
  }
  TRY(launch_score_scatter(c, n_pend));
  std::vector<float> lp(rows_lm);
  CUDA_TRY(c, cudaMemcpyAsync(lp.data(), c->score_lp, (size_t)rows_lm * 4, cudaMemcpyDeviceToHost, st));
  CUDA_TRY(c, cudaStreamSynchronize(st));                                            // the host vectors above stay alive until here
  int slot = 0;
  for (int q = 0; q < n_pend; ++q) {
    const int r = idx_rows[q];
    lp_out[(size_t)r * n] = lp[S + q];
    for (int k = 1; k < m[r]; ++k) lp_out[(size_t)r * n + k] = lp[slot + k - 1];
    slot += m[r];
    c->sc_len[r] += m[r];
  }
  return DARTS_OK;
}

darts_status darts_score_chunk(darts_ctx *c, int32_t step_begin, int32_t step_end, const int32_t *tokens_host, float *logprob_out_host) {
  if (!c) return DARTS_ERR_INVALID_ARG;
  if (c->sticky) return c->sticky;
  if (!c->score_mode) FAIL(c, DARTS_ERR_BAD_STATE, "darts_score_chunk before darts_score_begin");
  if (!tokens_host || !logprob_out_host || step_begin < 0 || step_end <= step_begin || step_end > c->rt.max_new)
    FAIL(c, DARTS_ERR_INVALID_ARG, "bad chunk [%d, %d) (max_new %d) or NULL buffers", step_begin, step_end, c->rt.max_new);
  const int R = c->R, n = step_end - step_begin, V = c->m.vocab;
  std::vector<int> m(R, 0);
  for (int r = 0; r < R; ++r) {
    int k = 0;
    while (k < n && tokens_host[(size_t)r * n + k] >= 0) {
      if (tokens_host[(size_t)r * n + k] >= V) FAIL(c, DARTS_ERR_INVALID_ARG, "token %d of row %d outside the vocabulary", tokens_host[(size_t)r * n + k], r);
      ++k;
    }
    m[r] = k;
    if (k > 0 && c->sc_len[r] != step_begin) FAIL(c, DARTS_ERR_BAD_STATE, "row %d has %d tokens scored, chunk starts at step %d (chunks must arrive in order)", r, c->sc_len[r], step_begin);
    for (int q = 0; q < n; ++q) logprob_out_host[(size_t)r * n + q] = 0.f;
  }
  // passes: slots + pending rows share the LM-head matrix (<= max_rows rows); the split-KV work list is bounded as well
  const int npc_max = ceil_div(c->rt.max_prompt_len, ATTN_CHUNK_TOKENS);
  int r0 = 0;
  while (r0 < R) {
    int r1 = r0, rows_lm = 0;
    long long parts = 0;
    while (r1 < R) {
      long long p = 0;
      for (int k = 0; k < m[r1]; ++k) p += npc_max + ceil_div(step_begin + k + 1, ATTN_CHUNK_TOKENS);
      const int add = m[r1] ? m[r1] + 1 : 0;
      if (rows_lm + add > c->rt.max_rows || (c->attn_max_items > 0 && parts + p > c->attn_max_items)) break;
      rows_lm += add; parts += p; ++r1;
    }
    if (r1 == r0) FAIL(c, DARTS_ERR_WORKSPACE_TOO_SMALL, "a chunk of %d steps does not fit a pass (max_rows %d): use shorter chunks", n, c->rt.max_rows);
    TRY(score_pass(c, r0, r1, step_begin, n, tokens_host, m, logprob_out_host));
    r0 = r1;
  }
  return DARTS_OK;
}

darts_status darts_debug_logits(darts_ctx *c, int32_t row, float *out_host) {
  if (!c || !out_host) return DARTS_ERR_INVALID_ARG;
  if (!c->prefilled || row < 0 || row >= c->R) FAIL(c, DARTS_ERR_INVALID_ARG, "bad row %d", row);
  CUDA_TRY(c, cudaStreamSynchronize(c->stream));
  int32_t slot, sstep, prompt;
  DevState st;
  CUDA_TRY(c, cudaMemcpy(&slot, c->row_slot + row, 4, cudaMemcpyDeviceToHost));
  CUDA_TRY(c, cudaMemcpy(&sstep, c->row_slot_step + row, 4, cudaMemcpyDeviceToHost));
  CUDA_TRY(c, cudaMemcpy(&prompt, c->row_prompt + row, 4, cudaMemcpyDeviceToHost));
  CUDA_TRY(c, cudaMemcpy(&st, c->st, sizeof(st), cudaMemcpyDeviceToHost));
  const float *src;
  if (sstep == 0) src = c->z0 + (size_t)prompt * c->m.vocab;
  else {
    // valid only for the most recent decode step (the logits buffer is overwritten every step)
    if (!c->logits) FAIL(c, DARTS_ERR_BAD_STATE, "decode logits are not kept: create the context with DARTS_FLAG_DUMP_LOGITS");
    if (sstep != c->steps_issued) FAIL(c, DARTS_ERR_BAD_STATE, "row %d last decoded at step %d, buffer holds step %d", row, sstep, c->steps_issued);
    src = c->logits + (size_t)slot * c->m.vocab;
  }
  CUDA_TRY(c, cudaMemcpy(out_host, src, (size_t)c->m.vocab * 4, cudaMemcpyDeviceToHost));
  return DARTS_OK;
}

darts_status darts_debug_routing(darts_ctx *c, int32_t slot_begin, int32_t n_slots, int32_t *out_host) {
  if (!c || !out_host) return DARTS_ERR_INVALID_ARG;
  if (!c->moe_eid_dump) FAIL(c, DARTS_ERR_BAD_STATE, "routing is kept only by a MoE context created with DARTS_FLAG_DUMP_LOGITS");
  if (slot_begin < 0 || n_slots <= 0 || slot_begin + n_slots > c->act_rows) FAIL(c, DARTS_ERR_INVALID_ARG, "bad slot range");
  CUDA_TRY(c, cudaStreamSynchronize(c->stream));
  const size_t k = c->m.top_k;
  CUDA_TRY(c, cudaMemcpy2D(out_host, (size_t)n_slots * k * 4, c->moe_eid_dump + (size_t)slot_begin * k, (size_t)c->act_rows * k * 4, (size_t)n_slots * k * 4,
                           (size_t)c->m.n_layers, cudaMemcpyDeviceToHost));
  return DARTS_OK;
}

darts_status darts_debug_hidden(darts_ctx *c, int32_t layer, int32_t slot_begin, int32_t n_slots, float *out_host) {
  if (!c || !out_host) return DARTS_ERR_INVALID_ARG;
  if (!c->hid_dump) FAIL(c, DARTS_ERR_BAD_STATE, "the residual stream is kept only by a context created with DARTS_FLAG_DUMP_HIDDEN");
  if (layer < 0 || layer > c->m.n_layers || slot_begin < 0 || n_slots <= 0 || slot_begin + n_slots > c->act_rows) FAIL(c, DARTS_ERR_INVALID_ARG, "bad layer / slot range");
  CUDA_TRY(c, cudaStreamSynchronize(c->stream));
  CUDA_TRY(c, cudaMemcpy(out_host, c->hid_dump + ((size_t)layer * c->act_rows + slot_begin) * c->m.d_model, (size_t)n_slots * c->m.d_model * sizeof(float),
                         cudaMemcpyDeviceToHost));
  return DARTS_OK;
}

darts_status darts_debug_row_slots(darts_ctx *c, int32_t *slot_host, int32_t *step_host, int32_t n_rows) {
  if (!c || !slot_host || !step_host) return DARTS_ERR_INVALID_ARG;
  if (!c->prefilled || n_rows != c->R) FAIL(c, DARTS_ERR_INVALID_ARG, "n_rows must equal the rollout's row count");
  CUDA_TRY(c, cudaStreamSynchronize(c->stream));
  CUDA_TRY(c, cudaMemcpy(slot_host, c->row_slot, (size_t)n_rows * 4, cudaMemcpyDeviceToHost));
  CUDA_TRY(c, cudaMemcpy(step_host, c->row_slot_step, (size_t)n_rows * 4, cudaMemcpyDeviceToHost));
  return DARTS_OK;
}

darts_status darts_debug_fast_forward(darts_ctx *c, int32_t new_len) {
  if (!c) return DARTS_ERR_INVALID_ARG;
  if (c->sticky) return c->sticky;
  if (!c->prefilled || c->score_mode) FAIL(c, DARTS_ERR_BAD_STATE, "darts_debug_fast_forward needs a prefilled rollout context");
  if (new_len < 1 || new_len >= c->max_len) FAIL(c, DARTS_ERR_INVALID_ARG, "new_len %d outside [1, max_len = %d)", new_len, c->max_len);
  return launch_fast_forward(c, new_len);
}

darts_status darts_debug_set_last_tokens(darts_ctx *c, const int32_t *tokens_host, int32_t n_rows) {
  if (!c || !tokens_host) return DARTS_ERR_INVALID_ARG;
  if (!c->prefilled || n_rows != c->R) FAIL(c, DARTS_ERR_INVALID_ARG, "n_rows must equal the rollout's row count");
  CUDA_TRY(c, cudaStreamSynchronize(c->stream));
  std::vector<int32_t> cur(n_rows);
  CUDA_TRY(c, cudaMemcpy(cur.data(), c->row_last_tok, (size_t)n_rows * 4, cudaMemcpyDeviceToHost));
  for (int r = 0; r < n_rows; ++r) if (tokens_host[r] >= 0) cur[r] = tokens_host[r];
  CUDA_TRY(c, cudaMemcpy(c->row_last_tok, cur.data(), (size_t)n_rows * 4, cudaMemcpyHostToDevice));
  return DARTS_OK;
}

darts_status darts_debug_gemm_scratch_floats(darts_ctx *c, int32_t rows, int32_t N, int32_t K, int32_t split_k, size_t *out) {
  if (!c || !out || rows <= 0 || N <= 0 || K <= 0 || split_k < 0) return DARTS_ERR_INVALID_ARG;
  if (!tc_shape_ok(N, K)) FAIL(c, DARTS_ERR_UNSUPPORTED, "tcgen05 GEMM needs K %% 64 == 0, N %% 4 == 0");
  int slots = split_k > 0 ? split_k : (c->use_pairs ? sk2_plan(c->n_sms, N, K, rows, true) : sk_plan(c->n_sms, N, K, rows, 0, true)).slots;
  *out = (size_t)slots * rows * N;
  return DARTS_OK;
}

darts_status darts_debug_gemm_bf16(darts_ctx *c, const void *X, const void *W, float *C, float *scratch, int32_t rows, int32_t N, int32_t K,
                                   int32_t split_k) {
  if (!c) return DARTS_ERR_INVALID_ARG;
  if (c->sticky) return c->sticky;
  if (!X || !W || !scratch || rows <= 0 || N <= 0 || K <= 0 || split_k < 0) FAIL(c, DARTS_ERR_INVALID_ARG, "NULL / non-positive argument");
  if (!tc_shape_ok(N, K) || split_k > K / 64) FAIL(c, DARTS_ERR_UNSUPPORTED, "tcgen05 GEMM needs K %% 64 == 0, N %% 4 == 0, split_k <= K/64");
  CUtensorMap ta, tb;
  if (split_k == 0) {                                        // the stream-K weight-streaming kernel; scratch >= slots * rows * N floats
    XMaps xm;
    TRY(tc_make_xmaps(c, &xm, X, rows, K));
    TRY(tc_make_map(c, &tb, W, N, K, 128));
    SkGemm g{};
    g.w_map = &tb; g.x_maps = &xm; g.C = scratch; g.N = N; g.rows_ub = rows; g.slot_stride = (size_t)rows * N; g.np_table = c->sk_np;
    g.pairs = c->use_pairs;
    g.plan = g.pairs ? sk2_plan(c->n_sms, N, K, rows, true) : sk_plan(c->n_sms, N, K, rows, 0, true);
    TRY(run_gemm_sk(c, g));
    if (!C) return DARTS_OK;
    return launch_sk_reduce(c, sk_view(g), C, rows);
  }
  TRY(tc_make_map(c, &ta, X, rows, K, 16));
  TRY(tc_make_map(c, &tb, W, N, K, 128));
  TcGemm g{};
  g.a_map = &ta; g.b_map = &tb; g.C = scratch; g.N = N; g.K = K; g.S = split_k; g.rows_ub = rows; g.split_stride = (size_t)rows * N;
  TRY(launch_gemm_tc(c, g));
  if (!C) return DARTS_OK;                                   // partials only (timing the GEMM kernel alone)
  return launch_sum_partials(c, scratch, C, split_k, (size_t)rows * N);
}

darts_status darts_attn_load(darts_ctx *c, int32_t G, int32_t P, int32_t Kp, const void *k_prefix, const void *v_prefix,
                             const int32_t *suffix_len_host, const void *k_suffix, const void *v_suffix) {
  if (!c) return DARTS_ERR_INVALID_ARG;
  if (c->sticky) return c->sticky;
  if (!k_prefix || !v_prefix || !suffix_len_host || !k_suffix || !v_suffix || G <= 0 || P <= 0 || Kp <= 0) FAIL(c, DARTS_ERR_INVALID_ARG, "NULL / non-positive argument");
  int R = G * Kp, page = c->rt.page_size;
  if (G > c->rt.max_prompts || R > c->rt.max_rows || P > c->rt.max_prompt_len) FAIL(c, DARTS_ERR_INVALID_ARG, "G, G*Kp or P exceed the runtime sizes");
  int npp = ceil_div(P, page);
  std::vector<int32_t> pre((size_t)G * c->max_prefix_pages, -1), rowp((size_t)R * c->max_suffix_pages, -1);
  std::vector<int32_t> sprompt(R), snpre(R, P), snsuf(R), srow(R), rlist(R);
  std::vector<int64_t> soffs(R + 1, 0);
  int next = 0;
  for (int g = 0; g < G; ++g) for (int q = 0; q < npp; ++q) pre[(size_t)g * c->max_prefix_pages + q] = next++;
  for (int r = 0; r < R; ++r) {
    int t = suffix_len_host[r];
    if (t < 0 || ceil_div(t, page) > c->max_suffix_pages) FAIL(c, DARTS_ERR_INVALID_ARG, "suffix_len[%d]=%d exceeds max_new", r, t);
    for (int q = 0; q < ceil_div(t, page); ++q) rowp[(size_t)r * c->max_suffix_pages + q] = next++;
    sprompt[r] = r / Kp; snsuf[r] = t; srow[r] = r; rlist[r] = r; soffs[r + 1] = soffs[r] + t;
  }
  if (next > c->rt.n_pages) FAIL(c, DARTS_ERR_KV_POOL_EXHAUSTED, "need %d pages, pool has %d", next, c->rt.n_pages);
  cudaStream_t s = c->stream;
  // suffix offsets (int64) and lengths are staged in the (otherwise unused here) free_pages / row_len arrays
  if ((size_t)c->rt.n_pages * 4 < (size_t)(R + 1) * 8) FAIL(c, DARTS_ERR_WORKSPACE_TOO_SMALL, "n_pages too small to stage offsets");
  int64_t *soffs_dev = (int64_t *)c->free_pages;
  CUDA_TRY(c, cudaMemcpyAsync(soffs_dev, soffs.data(), (size_t)(R + 1) * 8, cudaMemcpyHostToDevice, s));
  CUDA_TRY(c, cudaMemcpyAsync(c->row_len, suffix_len_host, (size_t)R * 4, cudaMemcpyHostToDevice, s));
  CUDA_TRY(c, cudaMemcpyAsync(c->g_prefix_pages, pre.data(), pre.size() * 4, cudaMemcpyHostToDevice, s));
  CUDA_TRY(c, cudaMemcpyAsync(c->row_pages, rowp.data(), rowp.size() * 4, cudaMemcpyHostToDevice, s));
  CUDA_TRY(c, cudaMemcpyAsync(c->slot_prompt, sprompt.data(), (size_t)R * 4, cudaMemcpyHostToDevice, s));
  CUDA_TRY(c, cudaMemcpyAsync(c->slot_npre, snpre.data(), (size_t)R * 4, cudaMemcpyHostToDevice, s));
  CUDA_TRY(c, cudaMemcpyAsync(c->slot_nsuf, snsuf.data(), (size_t)R * 4, cudaMemcpyHostToDevice, s));
  CUDA_TRY(c, cudaMemcpyAsync(c->slot_row, srow.data(), (size_t)R * 4, cudaMemcpyHostToDevice, s));
  CUDA_TRY(c, cudaMemcpyAsync(c->row_list, rlist.data(), (size_t)R * 4, cudaMemcpyHostToDevice, s));
  DevState st{};
  st.n_active = R; st.n_rows = R; st.n_groups = G; st.free_top = 0;
  CUDA_TRY(c, cudaMemcpyAsync(c->st, &st, sizeof(st), cudaMemcpyHostToDevice, s));
  darts_status rs = launch_attn_load(c, G, P, Kp, k_prefix, v_prefix, c->row_len, soffs_dev, k_suffix, v_suffix, soffs[R]);
  if (rs != DARTS_OK) return rs;
  c->attn_rows = R; c->G = G; c->R = R; c->Kp_max = Kp;
  c->attn_plan_valid = attention_sm100_supported(c);
  if (c->attn_plan_valid) TRY(launch_attention_plan_sm100(c, R, &c->st->n_active));
  return DARTS_OK;
}

darts_status darts_attention(darts_ctx *c, int32_t layer, const void *q, void *out) {
  if (!c) return DARTS_ERR_INVALID_ARG;
  if (c->sticky) return c->sticky;
  if (!q || !out || layer < 0 || layer >= c->m.n_layers) FAIL(c, DARTS_ERR_INVALID_ARG, "bad q / out / layer");
  if (c->attn_rows <= 0) FAIL(c, DARTS_ERR_BAD_STATE, "darts_attention before darts_attn_load");
  return launch_attention(c, layer, q, out, c->attn_rows, &c->st->n_active);
}

}  // extern "C"
