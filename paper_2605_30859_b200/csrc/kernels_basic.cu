// Element-wise / bookkeeping kernels of the decode step: embedding gather, RMSNorm, RoPE + KV append,
// SiLU*mul, step planning with the device page allocator.  (SURVEY.md §8(a) rows 2-4, 6.)
#include "internal.cuh"

#define DISPATCH_T(c, ...)                                        \
  if ((c)->m.dtype == DARTS_F32) { using T = float; __VA_ARGS__; } \
  else { using T = __nv_bfloat16; __VA_ARGS__; }

static inline darts_status post_launch(darts_ctx *c, const char *what) {
  c->launches++;
  cudaError_t e = cudaGetLastError();
  if (e != cudaSuccess) {
    snprintf(c->err, sizeof(c->err), "launch %s: %s", what, cudaGetErrorString(e));
    c->sticky = DARTS_ERR_CUDA;
    return DARTS_ERR_CUDA;
  }
  return DARTS_OK;
}

__device__ __forceinline__ int live_rows(const int32_t *n_rows_dev, int rows_ub) {
  return n_rows_dev ? min(*n_rows_dev, rows_ub) : rows_ub;
}

// ---------------------------------------------------------------- embedding: h[slot] = E[tok]
template <typename T>
__global__ void embed_k(const T *__restrict__ E, const int32_t *__restrict__ slot_tok, float *__restrict__ h, int d,
                        const int32_t *n_rows_dev, int rows_ub) {
  int slot = blockIdx.x;
  if (slot >= live_rows(n_rows_dev, rows_ub)) return;
  const T *src = E + (size_t)slot_tok[slot] * d;
  for (int k = threadIdx.x; k < d; k += blockDim.x) h[(size_t)slot * d + k] = to_f<T>(src[k]);
}

darts_status launch_embed(darts_ctx *c, const int32_t *slot_tok, int, int rows_ub, const int32_t *n_rows_dev) {
  if (rows_ub <= 0) return DARTS_OK;
  DISPATCH_T(c, embed_k<T><<<rows_ub, 256, 0, c->stream>>>((const T *)c->embed, slot_tok, c->h, c->m.d_model, n_rows_dev, rows_ub));
  return post_launch(c, "embed");
}

// ---------------------------------------------------------------- RMSNorm: out = x * w / sqrt(mean(x^2) + eps)
template <typename T>
__global__ void rmsnorm_k(const float *__restrict__ h, const T *__restrict__ w, T *__restrict__ out, int d, float eps,
                          const int32_t *n_rows_dev, int rows_ub) {
  pdl_trigger();
  int slot = blockIdx.x;
  if (slot >= live_rows(n_rows_dev, rows_ub)) return;
  const float *x = h + (size_t)slot * d;
  float ss = 0.f;
  for (int k = threadIdx.x; k < d; k += blockDim.x) ss += x[k] * x[k];
  __shared__ float red[32];
  ss = warp_sum(ss);
  if ((threadIdx.x & 31) == 0) red[threadIdx.x >> 5] = ss;
  __syncthreads();
  if (threadIdx.x < 32) {
    float v = threadIdx.x < (blockDim.x >> 5) ? red[threadIdx.x] : 0.f;
    v = warp_sum(v);
    if (threadIdx.x == 0) red[0] = v;
  }
  __syncthreads();
  float r = 1.0f / sqrtf(red[0] / d + eps);
  for (int k = threadIdx.x; k < d; k += blockDim.x) out[(size_t)slot * d + k] = from_f<T>(x[k] * r * to_f<T>(w[k]));
}

darts_status launch_rmsnorm(darts_ctx *c, const float *h, const void *w, void *out, int rows_ub, const int32_t *n_rows_dev) {
  if (rows_ub <= 0) return DARTS_OK;
  DISPATCH_T(c, rmsnorm_k<T><<<rows_ub, 256, 0, c->stream>>>(h, (const T *)w, (T *)out, c->m.d_model, c->m.rms_eps, n_rows_dev, rows_ub));
  return post_launch(c, "rmsnorm");
}

// ---------------------------------------------------------------- embed + first RMSNorm + RoPE table in one launch (tensor-core path)
// Same arithmetic as embed_k, rmsnorm_k and rope_table_k one after the other (same thread -> element mapping, same reduction
// order); three step-boundary launches become one.
template <typename T>
__global__ void __launch_bounds__(256) embed_norm_rope_k(const T *__restrict__ E, const int32_t *__restrict__ slot_tok, float *__restrict__ h,
                                                         const T *__restrict__ w, T *__restrict__ out, int d, float eps,
                                                         const int32_t *__restrict__ slot_pos, float2 *__restrict__ cs, int half, double theta,
                                                         const int32_t *n_rows_dev, int rows_ub) {
  pdl_trigger();
  int slot = blockIdx.x;
  if (slot >= live_rows(n_rows_dev, rows_ub)) return;
  const T *src = E + (size_t)slot_tok[slot] * d;
  float *x = h + (size_t)slot * d;
  float ss = 0.f;
  for (int k = threadIdx.x; k < d; k += blockDim.x) { float v = to_f<T>(src[k]); x[k] = v; ss += v * v; }
  __shared__ float red[32];
  ss = warp_sum(ss);
  if ((threadIdx.x & 31) == 0) red[threadIdx.x >> 5] = ss;
  __syncthreads();
  if (threadIdx.x < 32) {
    float v = threadIdx.x < (blockDim.x >> 5) ? red[threadIdx.x] : 0.f;
    v = warp_sum(v);
    if (threadIdx.x == 0) red[0] = v;
  }
  __syncthreads();
  float r = 1.0f / sqrtf(red[0] / d + eps);
  for (int k = threadIdx.x; k < d; k += blockDim.x) out[(size_t)slot * d + k] = from_f<T>(to_f<T>(src[k]) * r * to_f<T>(w[k]));
  for (int p = threadIdx.x; p < half; p += blockDim.x) {
    double inv_freq = pow(theta, -(double)p / (double)half);
    double s, co;
    sincos((double)slot_pos[slot] * inv_freq, &s, &co);
    cs[(size_t)slot * half + p] = make_float2((float)co, (float)s);
  }
}

darts_status launch_embed_norm_rope(darts_ctx *c, const int32_t *slot_tok, const void *w, int rows_ub, const int32_t *n_rows_dev) {
  if (rows_ub <= 0) return DARTS_OK;
  DISPATCH_T(c, embed_norm_rope_k<T><<<rows_ub, 256, 0, c->stream>>>((const T *)c->embed, slot_tok, c->h, (const T *)w, (T *)c->xn, c->m.d_model,
                                                                     c->m.rms_eps, c->slot_pos, c->slot_cs, c->m.head_dim / 2,
                                                                     (double)c->m.rope_theta, n_rows_dev, rows_ub));
  return post_launch(c, "embed_norm_rope");
}

// ---------------------------------------------------------------- SiLU(gate) * up
template <typename T>
__global__ void silu_mul_k(const float *__restrict__ gu, T *__restrict__ act, int F, const int32_t *n_rows_dev, int rows_ub) {
  int slot = blockIdx.y;
  if (slot >= live_rows(n_rows_dev, rows_ub)) return;
  int k = blockIdx.x * blockDim.x + threadIdx.x;
  if (k >= F) return;
  float g = gu[(size_t)slot * 2 * F + k], u = gu[(size_t)slot * 2 * F + F + k];
  act[(size_t)slot * F + k] = from_f<T>(g / (1.0f + expf(-g)) * u);
}

darts_status launch_silu_mul(darts_ctx *c, int rows_ub, const int32_t *n_rows_dev) {
  if (rows_ub <= 0) return DARTS_OK;
  int F = c->m.ffn;
  dim3 grid((F + 255) / 256, rows_ub);
  DISPATCH_T(c, silu_mul_k<T><<<grid, 256, 0, c->stream>>>(c->gu32, (T *)c->act, F, n_rows_dev, rows_ub));
  return post_launch(c, "silu_mul");
}

// ---------------------------------------------------------------- RoPE angle table (double precision angles)
// cs[slot][p] = (cos, sin)(pos * theta^(-2p/hd)); shared by all layers and heads of the step.
__global__ void rope_table_k(const int32_t *__restrict__ slot_pos, float2 *__restrict__ cs, int half, double theta,
                             const int32_t *n_rows_dev, int rows_ub) {
  int slot = blockIdx.x;
  if (slot >= live_rows(n_rows_dev, rows_ub)) return;
  for (int p = threadIdx.x; p < half; p += blockDim.x) {
    double inv_freq = pow(theta, -(double)p / (double)half);
    double s, co;
    sincos((double)slot_pos[slot] * inv_freq, &s, &co);
    cs[(size_t)slot * half + p] = make_float2((float)co, (float)s);
  }
}

darts_status launch_rope_table(darts_ctx *c, int rows_ub, const int32_t *n_rows_dev) {
  if (rows_ub <= 0) return DARTS_OK;
  rope_table_k<<<rows_ub, 64, 0, c->stream>>>(c->slot_pos, c->slot_cs, c->m.head_dim / 2, (double)c->m.rope_theta, n_rows_dev, rows_ub);
  return post_launch(c, "rope_table");
}

// ---------------------------------------------------------------- (QK-norm) + RoPE + KV append
// One warp per head of one slot.  q -> q buffer (model dtype); k, v -> the slot's destination page.
template <typename T>
__global__ void rope_append_k(const float *__restrict__ qkv, T *__restrict__ q_out, T *__restrict__ kv_layer,
                              const int32_t *__restrict__ slot_dst_page, const int32_t *__restrict__ slot_dst_off,
                              const float2 *__restrict__ cs, const T *__restrict__ q_norm, const T *__restrict__ k_norm,
                              int Hq, int Hkv, int hd, float eps, KvGeom geo, int S, size_t split_stride,
                              const int32_t *n_rows_dev, int rows_ub) {
  int slot = blockIdx.y;
  if (slot >= live_rows(n_rows_dev, rows_ub)) return;
  int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  int head = blockIdx.x * 4 + warp;
  if (head >= Hq + 2 * Hkv) return;
  const float *src = qkv + (size_t)slot * (Hq + 2 * Hkv) * hd + (size_t)head * hd;
  // split-K partials (tensor-core path): element = sum over splits in split order; S == 1 for the SIMT path
  auto ld = [&](int k) { float v = src[k]; for (int s = 1; s < S; ++s) v += src[(size_t)s * split_stride + k]; return v; };
  int half = hd >> 1;
  int page = slot_dst_page[slot], off = slot_dst_off[slot];
  if (head >= Hq + Hkv) {  // v: plain copy
    if (page < 0) return;
    for (int k = lane; k < hd; k += 32) kv_layer[kv_elem(geo, page, head - Hq - Hkv, 1, off, k)] = from_f<T>(ld(k));
    return;
  }
  bool is_q = head < Hq;
  const T *nw = is_q ? q_norm : k_norm;
  float r = 1.f;
  if (nw) {
    float ss = 0.f;
    for (int k = lane; k < hd; k += 32) { float v = ld(k); ss += v * v; }
    ss = warp_sum(ss);
    r = 1.0f / sqrtf(ss / hd + eps);
  }
  if (!is_q && page < 0) return;
  T *qdst = q_out + (size_t)slot * Hq * hd + (size_t)head * hd;
  for (int p = lane; p < half; p += 32) {
    float x1 = ld(p), x2 = ld(p + half);
    if (nw) { x1 = x1 * r * to_f<T>(nw[p]); x2 = x2 * r * to_f<T>(nw[p + half]); }
    float2 t = cs[(size_t)slot * half + p];
    T y1 = from_f<T>(x1 * t.x - x2 * t.y), y2 = from_f<T>(x2 * t.x + x1 * t.y);
    if (is_q) { qdst[p] = y1; qdst[p + half] = y2; }
    else {
      kv_layer[kv_elem(geo, page, head - Hq, 0, off, p)] = y1;
      kv_layer[kv_elem(geo, page, head - Hq, 0, off, p + half)] = y2;
    }
  }
}

darts_status launch_rope_append(darts_ctx *c, int layer, int rows_ub, const int32_t *n_rows_dev) {
  if (rows_ub <= 0) return DARTS_OK;
  int nh = c->m.n_q_heads + 2 * c->m.n_kv_heads;
  dim3 grid((nh + 3) / 4, rows_ub);
  DISPATCH_T(c, rope_append_k<T><<<grid, 128, 0, c->stream>>>(
                    c->qkv32, (T *)c->q, (T *)c->kv_pool + (size_t)layer * c->kv_layer_elems, c->slot_dst_page, c->slot_dst_off,
                    c->slot_cs, c->m.qk_norm ? (const T *)c->q_norm[layer] : nullptr,
                    c->m.qk_norm ? (const T *)c->k_norm[layer] : nullptr, c->m.n_q_heads, c->m.n_kv_heads, c->m.head_dim,
                    c->m.rms_eps, c->geom(), 1, 0, n_rows_dev, rows_ub));
  return post_launch(c, "rope_append");
}

// ---------------------------------------------------------------- block-wide exclusive scan helper (<= 1024 threads)
__device__ __forceinline__ int block_excl_scan(int v, int *total, int *smem /*[33]*/) {
  int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  int incl = v;
#pragma unroll
  for (int o = 1; o < 32; o <<= 1) {
    int t = __shfl_up_sync(0xffffffffu, incl, o);
    if (lane >= o) incl += t;
  }
  if (lane == 31) smem[warp] = incl;
  __syncthreads();
  if (warp == 0) {
    int w = lane < (int)(blockDim.x >> 5) ? smem[lane] : 0;
    int wi = w;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
      int t = __shfl_up_sync(0xffffffffu, wi, o);
      if (lane >= o) wi += t;
    }
    smem[lane] = wi - w;                       // exclusive warp offsets
    if (lane == 31) smem[32] = wi;             // block total
  }
  __syncthreads();
  int res = smem[warp] + incl - v;
  *total = smem[32];
  __syncthreads();
  return res;
}

// ---------------------------------------------------------------- decode-step plan + page allocation (one CTA)
// For every active slot: the token to feed, its position, and where its K/V go.  Rows whose suffix
// index t = len-1 starts a page pop one page from the free stack in slot order (deterministic).
__global__ void plan_decode_k(DevState *st, const int32_t *__restrict__ row_list, const int32_t *__restrict__ row_len,
                              const int32_t *__restrict__ row_prompt, const int32_t *__restrict__ row_last_tok,
                              int32_t *__restrict__ row_pages, const int32_t *__restrict__ g_plen,
                              int32_t *__restrict__ free_pages, int32_t *slot_row, int32_t *slot_tok, int32_t *slot_pos,
                              int32_t *slot_dst_page, int32_t *slot_dst_off, int32_t *slot_prompt, int32_t *slot_npre,
                              int32_t *slot_nsuf, int page, int msp, int32_t *pinned) {
  __shared__ int sm[33];
  __shared__ int s_base;
  int n = st->n_active;
  int free_top = st->free_top;
  if (threadIdx.x == 0) s_base = 0;
  __syncthreads();
  for (int base = 0; base < n; base += blockDim.x) {
    int slot = base + threadIdx.x;
    int row = -1, t = 0, need = 0;
    if (slot < n) {
      row = row_list[slot];
      t = row_len[row] - 1;
      need = (t % page) == 0;
    }
    int total;
    int excl = block_excl_scan(need, &total, sm);
    int b = s_base;
    if (slot < n) {
      int i = row_prompt[row];
      if (need) {
        int idx = free_top - 1 - (b + excl);
        row_pages[(size_t)row * msp + t / page] = idx >= 0 ? free_pages[idx] : -1;
      }
      slot_row[slot] = row;
      slot_tok[slot] = row_last_tok[row];
      slot_pos[slot] = g_plen[i] + t;
      slot_dst_page[slot] = row_pages[(size_t)row * msp + t / page];
      slot_dst_off[slot] = t % page;
      slot_prompt[slot] = i;
      slot_npre[slot] = g_plen[i];
      slot_nsuf[slot] = t + 1;
    }
    __syncthreads();
    if (threadIdx.x == 0) s_base = b + total;
    __syncthreads();
  }
  if (threadIdx.x == 0) {
    if (s_base > free_top) {               // pool ran dry: stop the rollout, never write through a bad page
      st->err = DARTS_ERR_KV_POOL_EXHAUSTED;
      st->n_active = 0;
      pinned[2] = DARTS_ERR_KV_POOL_EXHAUSTED;
    } else {
      st->free_top = free_top - s_base;
      st->n_pops += (unsigned long long)s_base;
    }
  }
}

// Profiling hook (PTL(b, ctx) sweeps): give every active row a generated length of new_len without decoding the
// steps in between — page tables are extended from the free stack, the cache content of the skipped positions is whatever the pool holds
// (finite: the pool is zeroed at darts_create), which changes no timing.  One thread: a tool's hook, not a step of the path.
__global__ void fast_forward_k(DevState *st, const int32_t *__restrict__ row_list, int32_t *row_len, int32_t *row_pages,
                               const int32_t *__restrict__ free_pages, int page, int msp, int new_len, int32_t *pinned) {
  if (threadIdx.x || blockIdx.x) return;
  int top = st->free_top;
  for (int s = 0; s < st->n_active; ++s) {
    const int row = row_list[s];
    const int t_old = row_len[row] - 1, t_new = new_len - 1;
    if (t_new <= t_old) continue;
    for (int p = (t_old + page - 1) / page; p < (t_new + page - 1) / page; ++p) {
      if (top <= 0) { st->err = DARTS_ERR_KV_POOL_EXHAUSTED; st->n_active = 0; pinned[2] = DARTS_ERR_KV_POOL_EXHAUSTED; return; }
      row_pages[(size_t)row * msp + p] = free_pages[--top];
    }
    row_len[row] = new_len;
  }
  st->n_pops += (unsigned long long)(st->free_top - top);
  st->free_top = top;
}

darts_status launch_fast_forward(darts_ctx *c, int new_len) {
  fast_forward_k<<<1, 32, 0, c->stream>>>(c->st, c->row_list, c->row_len, c->row_pages, c->free_pages, c->rt.page_size, c->max_suffix_pages, new_len,
                                          c->pinned_dev);
  return post_launch(c, "fast_forward");
}

darts_status launch_plan_decode(darts_ctx *c, int) {
  plan_decode_k<<<1, 1024, 0, c->stream>>>(c->st, c->row_list, c->row_len, c->row_prompt, c->row_last_tok, c->row_pages, c->g_plen,
                                           c->free_pages, c->slot_row, c->slot_tok, c->slot_pos, c->slot_dst_page, c->slot_dst_off,
                                           c->slot_prompt, c->slot_npre, c->slot_nsuf, c->rt.page_size, c->max_suffix_pages, c->pinned_dev);
  return post_launch(c, "plan_decode");
}

// ---------------------------------------------------------------- prefill plan: slot = prompt token
__global__ void plan_prefill_k(const int32_t *__restrict__ prompt_tokens, const int32_t *__restrict__ g_tok_off,
                               const int32_t *__restrict__ g_prefix_pages, int32_t *slot_tok, int32_t *slot_pos,
                               int32_t *slot_dst_page, int32_t *slot_dst_off, int32_t *slot_prompt, int32_t *slot_npre,
                               int32_t *slot_nsuf, int32_t *slot_row, int tok_begin, int n_tok, int g_begin, int g_end,
                               int page, int mpp) {
  int slot = blockIdx.x * blockDim.x + threadIdx.x;
  if (slot >= n_tok) return;
  int idx = tok_begin + slot;
  int lo = g_begin, hi = g_end;            // find prompt i with g_tok_off[i] <= idx < g_tok_off[i+1]
  while (hi - lo > 1) {
    int mid = (lo + hi) >> 1;
    if (g_tok_off[mid] <= idx) lo = mid; else hi = mid;
  }
  int i = lo, p = idx - g_tok_off[i];
  slot_tok[slot] = prompt_tokens[idx];
  slot_pos[slot] = p;
  slot_dst_page[slot] = g_prefix_pages[(size_t)i * mpp + p / page];
  slot_dst_off[slot] = p % page;
  slot_prompt[slot] = i;
  slot_npre[slot] = p + 1;                 // causal: sees prompt positions 0..p
  slot_nsuf[slot] = 0;
  slot_row[slot] = 0;
}

darts_status launch_plan_prefill(darts_ctx *c, int tok_begin, int n_tok, int g_begin, int g_end) {
  plan_prefill_k<<<(n_tok + 255) / 256, 256, 0, c->stream>>>(c->prompt_tokens, c->g_tok_off, c->g_prefix_pages, c->slot_tok, c->slot_pos,
                                                             c->slot_dst_page, c->slot_dst_off, c->slot_prompt, c->slot_npre, c->slot_nsuf,
                                                             c->slot_row, tok_begin, n_tok, g_begin, g_end, c->rt.page_size, c->max_prefix_pages);
  return post_launch(c, "plan_prefill");
}

// hlast[i] = h[slot of the last token of prompt i]
__global__ void gather_last_k(const float *__restrict__ h, float *__restrict__ hlast, const int32_t *__restrict__ g_tok_off,
                              int tok_begin, int g_begin, int d) {
  int i = g_begin + blockIdx.x;
  int slot = g_tok_off[i + 1] - 1 - tok_begin;
  for (int k = threadIdx.x; k < d; k += blockDim.x) hlast[(size_t)blockIdx.x * d + k] = h[(size_t)slot * d + k];
}

darts_status launch_gather_last(darts_ctx *c, int tok_begin, int, int g_begin, int g_end) {
  gather_last_k<<<g_end - g_begin, 256, 0, c->stream>>>(c->h, c->hlast, c->g_tok_off, tok_begin, g_begin, c->m.d_model);
  return post_launch(c, "gather_last");
}
