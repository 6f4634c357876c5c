// Group selection (Alg. 2, :465-477; §4.1.2 :140; §4.3.1 :222-224) and active-set compaction with
// page release, plus row/group initialisation.  Integer work, bit-exact by design.
#include <limits.h>

#include "internal.cuh"

namespace {

// count, over lanes flagged `in_set`, of lanes whose key (len, lane) orders before mine.
// desc == true orders by (larger len first, then smaller lane).
__device__ __forceinline__ int rank_among(bool in_set, int len, bool desc) {
  int lane = threadIdx.x & 31, r = 0;
  unsigned set = __ballot_sync(0xffffffffu, in_set);
#pragma unroll 4
  for (int o = 0; o < 32; ++o) {
    int lo = __shfl_sync(0xffffffffu, len, o);
    if ((set >> o) & 1u) {
      bool before = desc ? (lo > len || (lo == len && o < lane)) : (lo < len || (lo == len && o < lane));
      r += before ? 1 : 0;
    }
  }
  return r;
}

// One warp per prompt; lane j = sample j (Kp <= 32).
__global__ void select_k(DevState *st, const int32_t *__restrict__ g_off, const int32_t *__restrict__ g_Kp, int32_t *g_closed,
                         int32_t *g_sel, uint32_t *g_mask, int32_t *g_close_step, float *g_len_mean, float *g_len_var, int32_t *g_n_pruned,
                         const int32_t *__restrict__ row_len, uint8_t *row_status, int G, int K, int L_long, int M_up, int mode) {
  int g = blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5);
  int lane = threadIdx.x & 31;
  if (g >= G || g_closed[g]) return;
  int Kp = g_Kp[g], off = g_off[g];
  bool has = lane < Kp;
  int len = has ? row_len[off + lane] : INT_MAX;
  int stt = has ? (int)row_status[off + lane] : 255;
  unsigned active = __ballot_sync(0xffffffffu, has && stt == DARTS_ROW_ACTIVE);
  unsigned valid = __ballot_sync(0xffffffffu, has && stt == DARTS_ROW_VALID);
  bool early = mode == DARTS_MODE_SHORTEST_EARLY_STOP || (mode == DARTS_MODE_AUTO && Kp >= M_up);
  if (early && __popc(valid) >= K && active) {   // proactive early stop
    if (has && stt == DARTS_ROW_ACTIVE) { stt = DARTS_ROW_PRUNED; row_status[off + lane] = DARTS_ROW_PRUNED; }
    active = 0;
  }
  if (active) return;
  // ---- the group closes at this step: emit exactly K sample indices
  bool chosen;
  if (early) {
    // order by (class, len, j), class VALID < TRUNC < PRUNED: fold the class into the key's high bits
    int cls = stt == DARTS_ROW_VALID ? 0 : (stt == DARTS_ROW_TRUNC ? 1 : 2);
    int key = has ? (cls << 28) | len : INT_MAX;
    int r = rank_among(has, key, false);
    chosen = has && r < K;
    if (chosen) g_sel[(size_t)g * K + r] = lane;
  } else {
    int S = K - L_long;
    int ra = rank_among(has, len, false);
    bool in_short = has && ra < S;
    bool cand = has && !in_short && stt == DARTS_ROW_VALID;        // longest excludes limit-hitting rows
    int nc = __popc(__ballot_sync(0xffffffffu, cand));
    int rd = rank_among(cand, len, true);
    bool in_long = cand && rd < L_long;
    int nfill = L_long - min(L_long, nc);
    bool rest = has && !in_short && !in_long;
    int rf = rank_among(rest, len, false);
    bool in_fill = rest && rf < nfill;
    bool longsel = in_long || in_fill;
    int rl = rank_among(longsel, len, false);
    if (in_short) g_sel[(size_t)g * K + ra] = lane;
    if (longsel) g_sel[(size_t)g * K + S + rl] = lane;
    chosen = in_short || longsel;
  }
  unsigned mask = __ballot_sync(0xffffffffu, chosen);
  unsigned pruned_mask = __ballot_sync(0xffffffffu, has && stt == DARTS_ROW_PRUNED);
  float fl = has ? (float)len : 0.f;
  float mean = warp_sum(fl) / Kp;
  float dv = has ? (fl - mean) * (fl - mean) : 0.f;
  float var = warp_sum(dv) / Kp;
  int kept = chosen ? len : 0;
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) kept += __shfl_xor_sync(0xffffffffu, kept, o);
  if (lane == 0) {
    g_mask[g] = mask;
    g_closed[g] = 1;                      // 1 = closed this step (prefix pages still to be released)
    g_close_step[g] = st->step;
    g_len_mean[g] = mean;
    g_len_var[g] = var;
    g_n_pruned[g] = __popc(pruned_mask);
    atomicAdd(&st->n_kept, (unsigned long long)kept);
  }
}

__device__ __forceinline__ int block_excl_scan2(int v, int *total, int *smem /*[33]*/) {
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
    smem[lane] = wi - w;
    if (lane == 31) smem[32] = wi;
  }
  __syncthreads();
  int res = smem[warp] + incl - v;
  *total = smem[32];
  __syncthreads();
  return res;
}

// One CTA: stable partition of row_list keeping ACTIVE rows; pages of rows that left are pushed back on
// the free stack in slot order, then the prefix pages of groups that closed this step.
__global__ void compact_k(DevState *st, int32_t *row_list, int32_t *row_list_tmp, const uint8_t *__restrict__ row_status,
                          const int32_t *__restrict__ row_len, const int32_t *__restrict__ row_pages, int32_t *free_pages,
                          int32_t *g_closed, const int32_t *__restrict__ g_plen, const int32_t *__restrict__ g_prefix_pages, int G,
                          int page, int msp, int mpp, int n_pages, int32_t *pinned, int32_t *n_active_out, int gen) {
  __shared__ int sm[33];
  __shared__ int s_keep, s_free;
  int n = st->n_active;
  if (threadIdx.x == 0) { s_keep = 0; s_free = st->free_top; }
  __syncthreads();
  for (int base = 0; base < n; base += blockDim.x) {
    int slot = base + threadIdx.x;
    int row = -1, keep = 0, npg = 0;
    if (slot < n) {
      row = row_list[slot];
      keep = row_status[row] == DARTS_ROW_ACTIVE;
      if (!keep) npg = (row_len[row] - 1 + page - 1) / page;     // tokens fed = len-1 (the last one never is)
    }
    int tk, tf;
    int ek = block_excl_scan2(keep, &tk, sm);
    int ef = block_excl_scan2(npg, &tf, sm);
    int bk = s_keep, bf = s_free;
    if (slot < n) {
      if (keep) row_list_tmp[bk + ek] = row;
      else
        for (int p = 0; p < npg; ++p) free_pages[bf + ef + p] = row_pages[(size_t)row * msp + p];
    }
    __syncthreads();
    if (threadIdx.x == 0) { s_keep = bk + tk; s_free = bf + tf; }
    __syncthreads();
  }
  int n_new = s_keep;
  for (int s = threadIdx.x; s < n_new; s += blockDim.x) row_list[s] = row_list_tmp[s];
  if (threadIdx.x == 0) {
    int ft = s_free;
    for (int g = 0; g < G; ++g) {
      if (g_closed[g] == 1) {
        int np = (g_plen[g] + page - 1) / page;
        for (int p = 0; p < np; ++p) free_pages[ft++] = g_prefix_pages[(size_t)g * mpp + p];
        g_closed[g] = 2;
      }
    }
    int used_before = n_pages - st->free_top;
    if (used_before > st->peak_used) st->peak_used = used_before;
    st->free_top = ft;
    if (n > 0) { st->n_row_steps += (unsigned long long)n; st->step += 1; }
    st->n_active = n_new;
    pinned[2] = st->err;
    *(volatile long long *)pinned = ((long long)gen << 32) | (unsigned)n_new;   // {n_active, generation} in one store
    if (n_active_out) *n_active_out = n_new;
  }
}

__global__ void init_rows_k(DevState *st, const int32_t *__restrict__ g_off, const int32_t *__restrict__ forced_len, int G, int R,
                            int Kp_max, int32_t *row_list, int32_t *row_prompt, int32_t *row_sample, int32_t *row_len,
                            int32_t *row_forced, int32_t *row_last_tok, int32_t *row_slot_step, uint8_t *row_status,
                            int32_t *g_closed, int32_t *free_pages, int n_pages, int n_prefix_pages, int32_t *pinned) {
  int t = blockIdx.x * blockDim.x + threadIdx.x;
  if (t < R) {
    int lo = 0, hi = G;
    while (hi - lo > 1) {
      int mid = (lo + hi) >> 1;
      if (g_off[mid] <= t) lo = mid; else hi = mid;
    }
    int i = lo, j = t - g_off[i];
    row_list[t] = t;
    row_prompt[t] = i;
    row_sample[t] = j;
    row_len[t] = 0;
    row_forced[t] = forced_len ? forced_len[(size_t)i * Kp_max + j] : 0;
    row_last_tok[t] = 0;
    row_slot_step[t] = -1;
    row_status[t] = DARTS_ROW_ACTIVE;
  }
  if (t < G) g_closed[t] = 0;
  int nfree = n_pages - n_prefix_pages;
  for (int k = t; k < nfree; k += gridDim.x * blockDim.x) free_pages[k] = n_pages - 1 - k;   // top of stack = lowest id
  if (t == 0) {
    st->n_active = R; st->n_rows = R; st->n_groups = G; st->free_top = nfree; st->err = 0; st->step = 0;
    st->peak_used = n_prefix_pages; st->n_open_groups = G;
    st->n_generated = 0; st->n_near_ties = 0; st->n_kept = 0; st->n_row_steps = 0; st->n_pops = (unsigned long long)n_prefix_pages;
    pinned[2] = 0;
  }
}

// Config-2 loader: scatter explicit K/V into the paged cache (layer 0) and fill the static plan.
template <typename T>
__global__ void attn_load_k(T *kv_layer, const T *__restrict__ kp, const T *__restrict__ vp, const T *__restrict__ ks,
                            const T *__restrict__ vs, const int32_t *__restrict__ suffix_len, const int64_t *__restrict__ suffix_offs,
                            const int32_t *__restrict__ g_prefix_pages, const int32_t *__restrict__ row_pages, int G, int P, int Kp,
                            int Hkv, int hd, int page, int mpp, int msp, KvGeom geo, long long n_prefix_tok, long long n_tok) {
  long long tok = blockIdx.x;
  if (tok >= n_tok) return;
  const T *srck, *srcv;
  int pg, off;
  if (tok < n_prefix_tok) {
    int g = (int)(tok / P), p = (int)(tok % P);
    srck = kp + (size_t)tok * Hkv * hd; srcv = vp + (size_t)tok * Hkv * hd;
    pg = g_prefix_pages[(size_t)g * mpp + p / page]; off = p % page;
  } else {
    long long st = tok - n_prefix_tok;
    int lo = 0, hi = G * Kp;
    while (hi - lo > 1) {
      int mid = (lo + hi) >> 1;
      if (suffix_offs[mid] <= st) lo = mid; else hi = mid;
    }
    int row = lo, t = (int)(st - suffix_offs[row]);
    srck = ks + (size_t)st * Hkv * hd; srcv = vs + (size_t)st * Hkv * hd;
    pg = row_pages[(size_t)row * msp + t / page]; off = t % page;
  }
  for (int e = threadIdx.x; e < Hkv * hd; e += blockDim.x) {
    int h = e / hd, d = e % hd;
    kv_layer[kv_elem(geo, pg, h, 0, off, d)] = srck[e];
    kv_layer[kv_elem(geo, pg, h, 1, off, d)] = srcv[e];
  }
}

}  // namespace

darts_status launch_select(darts_ctx *c) {
  int G = c->G;
  select_k<<<(G + 3) / 4, 128, 0, c->stream>>>(c->st, c->g_off, c->g_Kp, c->g_closed, c->g_sel, c->g_mask, c->g_close_step, c->g_len_mean,
                                               c->g_len_var, c->g_n_pruned, c->row_len, c->row_status, G, c->pol.K, c->pol.L_long, c->pol.M_up, c->pol.mode);
  c->launches++;
  if (cudaGetLastError() != cudaSuccess) FAIL(c, DARTS_ERR_CUDA, "launch select failed");
  return DARTS_OK;
}

darts_status launch_compact(darts_ctx *c, int32_t *n_active_out) {
  compact_k<<<1, 1024, 0, c->stream>>>(c->st, c->row_list, c->row_list_tmp, c->row_status, c->row_len, c->row_pages, c->free_pages,
                                       c->g_closed, c->g_plen, c->g_prefix_pages, c->G, c->rt.page_size, c->max_suffix_pages,
                                       c->max_prefix_pages, c->rt.n_pages, c->pinned_dev, n_active_out, (int)c->gen);
  c->launches++;
  if (cudaGetLastError() != cudaSuccess) FAIL(c, DARTS_ERR_CUDA, "launch compact failed");
  return DARTS_OK;
}

darts_status launch_init_rows(darts_ctx *c, const int32_t *forced_len, int n_prefix_pages_total) {
  int n = max(max(c->R, c->G), 1024);
  init_rows_k<<<(n + 255) / 256, 256, 0, c->stream>>>(c->st, c->g_off, forced_len, c->G, c->R, c->Kp_max, c->row_list, c->row_prompt,
                                                      c->row_sample, c->row_len, c->row_forced, c->row_last_tok, c->row_slot_step,
                                                      c->row_status, c->g_closed, c->free_pages, c->rt.n_pages, n_prefix_pages_total,
                                                      c->pinned_dev);
  c->launches++;
  if (cudaGetLastError() != cudaSuccess) FAIL(c, DARTS_ERR_CUDA, "launch init_rows failed");
  return DARTS_OK;
}

darts_status launch_attn_load(darts_ctx *c, int G, int P, int Kp, const void *kp, const void *vp, const int32_t *suffix_len_dev,
                              const int64_t *suffix_offs_dev, const void *ks, const void *vs, long long n_suffix_tok) {
  long long n_pre = (long long)G * P, n_tok = n_pre + n_suffix_tok;
  if (c->m.dtype == DARTS_F32)
    attn_load_k<float><<<(unsigned)n_tok, 128, 0, c->stream>>>((float *)c->kv_pool, (const float *)kp, (const float *)vp, (const float *)ks,
                                                               (const float *)vs, suffix_len_dev, suffix_offs_dev, c->g_prefix_pages,
                                                               c->row_pages, G, P, Kp, c->m.n_kv_heads, c->m.head_dim, c->rt.page_size,
                                                               c->max_prefix_pages, c->max_suffix_pages, c->geom(), n_pre, n_tok);
  else
    attn_load_k<__nv_bfloat16><<<(unsigned)n_tok, 128, 0, c->stream>>>(
        (__nv_bfloat16 *)c->kv_pool, (const __nv_bfloat16 *)kp, (const __nv_bfloat16 *)vp, (const __nv_bfloat16 *)ks,
        (const __nv_bfloat16 *)vs, suffix_len_dev, suffix_offs_dev, c->g_prefix_pages, c->row_pages, G, P, Kp, c->m.n_kv_heads,
        c->m.head_dim, c->rt.page_size, c->max_prefix_pages, c->max_suffix_pages, c->geom(), n_pre, n_tok);
  c->launches++;
  if (cudaGetLastError() != cudaSuccess) FAIL(c, DARTS_ERR_CUDA, "launch attn_load failed");
  return DARTS_OK;
}
