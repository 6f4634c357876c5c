// Consumer half of token-level streaming (§4.3.2 "dispatched to the training engine ... it launches the forward
// computation"; App. E :481-489, incremental forward over a per-trajectory KV cache): small kernels around the
// chunked teacher-forced forward of darts_score_chunk (api.cu).  The forward itself runs on the kernels of the decode step; here:
//   score_init_pend   pend[row] = final-normed hidden of the row's prompt's last token (its logits score the row's token 0)
//   score_gather      xn[S + k] = pend[row_k]: the pending rows join the pass's LM-head matrix behind the S forwarded slots
//   score_scatter     pend[row_k] = xn[last slot of row_k]: the hidden whose logits score the first token of the NEXT chunk
//   score_finalize    merge the LM-head epilogue's per-tile (target z / T, log-sum-exp) entries: lp = z_tgt / T - logsumexp(z / T)
//   score_logits      the same from materialised fp32 logits (generic / fp32 path)
#include "internal.cuh"

namespace {

darts_status post(darts_ctx *c, const char *what) {
  c->launches++;
  cudaError_t e = cudaGetLastError();
  if (e != cudaSuccess) {
    snprintf(c->err, sizeof(c->err), "launch %s: %s", what, cudaGetErrorString(e));
    c->sticky = DARTS_ERR_CUDA;
    return DARTS_ERR_CUDA;
  }
  return DARTS_OK;
}

// dst[dst_idx[k]] = src[src_idx[k]] over rows of `bytes` bytes (16-byte multiples); idx == NULL: identity
__global__ void copy_rows_k(const uint4 *__restrict__ src, uint4 *__restrict__ dst, const int32_t *__restrict__ src_idx, int src_off,
                            const int32_t *__restrict__ dst_idx, int dst_off, int vec) {
  const int k = blockIdx.x;
  const uint4 *s = src + (size_t)(src_idx ? src_idx[k] : src_off + k) * vec;
  uint4 *d = dst + (size_t)(dst_idx ? dst_idx[k] : dst_off + k) * vec;
  for (int i = threadIdx.x; i < vec; i += blockDim.x) d[i] = s[i];
}

struct Lse { float m, s; };
__device__ __forceinline__ Lse lse_merge(const Lse &a, const Lse &b) {
  if (b.m == -INFINITY) return a;
  if (a.m == -INFINITY) return b;
  float mn = fmaxf(a.m, b.m);
  return Lse{mn, a.s * __expf(a.m - mn) + b.s * __expf(b.m - mn)};
}

// One CTA per LM-head row.  top2[k][row] = (z_tgt / T or -inf, -, id, z_tgt / T) from the tile that holds the target; lse[k][row] = (max, sum).
__global__ void __launch_bounds__(512) score_finalize_k(const float4 *__restrict__ top2, const float2 *__restrict__ lse, int n_tiles, int rows,
                                                        const int32_t *__restrict__ tgt, float *__restrict__ lp) {
  const int row = blockIdx.x;
  float zt = -INFINITY;
  Lse l{-INFINITY, 0.f};
  for (int k = threadIdx.x; k < n_tiles; k += blockDim.x) {
    const float4 v = __ldcs(&top2[(size_t)k * rows + row]);
    const float2 w = __ldcs(&lse[(size_t)k * rows + row]);
    zt = fmaxf(zt, v.x);                                  // exactly one entry is finite
    l = lse_merge(l, Lse{w.x, w.y});
  }
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) {
    zt = fmaxf(zt, __shfl_xor_sync(0xffffffffu, zt, o));
    l = lse_merge(l, Lse{__shfl_xor_sync(0xffffffffu, l.m, o), __shfl_xor_sync(0xffffffffu, l.s, o)});
  }
  __shared__ float rz[16];
  __shared__ Lse rl[16];
  if ((threadIdx.x & 31) == 0) { rz[threadIdx.x >> 5] = zt; rl[threadIdx.x >> 5] = l; }
  __syncthreads();
  if (threadIdx.x == 0) {
    for (int w = 1; w < (int)(blockDim.x >> 5); ++w) { zt = fmaxf(zt, rz[w]); l = lse_merge(l, rl[w]); }
    lp[row] = tgt[row] >= 0 ? zt - (l.m + logf(l.s)) : 0.f;
  }
}

// Generic path: lp[row] = z[tgt] / T - logsumexp(z / T) over one row of fp32 logits (T == 0: of softmax(z), R23).
__global__ void __launch_bounds__(256) score_logits_k(const float *__restrict__ logits, int V, const int32_t *__restrict__ tgt, float T,
                                                      float *__restrict__ lp) {
  const int row = blockIdx.x;
  const float *z = logits + (size_t)row * V;
  float m = -INFINITY;
  for (int v = threadIdx.x; v < V; v += blockDim.x) m = fmaxf(m, T != 0.f ? z[v] / T : z[v]);
  m = warp_max(m);
  __shared__ float red[8];
  if ((threadIdx.x & 31) == 0) red[threadIdx.x >> 5] = m;
  __syncthreads();
  m = red[0];
  for (int w = 1; w < 8; ++w) m = fmaxf(m, red[w]);
  __syncthreads();
  float s = 0.f;
  for (int v = threadIdx.x; v < V; v += blockDim.x) s += expf((T != 0.f ? z[v] / T : z[v]) - m);
  s = warp_sum(s);
  if ((threadIdx.x & 31) == 0) red[threadIdx.x >> 5] = s;
  __syncthreads();
  if (threadIdx.x == 0) {
    float t = 0.f;
    for (int w = 0; w < 8; ++w) t += red[w];
    const int g = tgt[row];
    lp[row] = g >= 0 ? (T != 0.f ? z[g] / T : z[g]) - (m + logf(t)) : 0.f;
  }
}

}  // namespace

// pend[row] = (tensor-core path: hlast, generic path: pend0)[row_prompt[row]]; the gather indices were uploaded to score_idx[0..R)
darts_status launch_score_init_pend(darts_ctx *c, int R) {
  const int vec = c->m.d_model * c->elt / 16;
  const void *src = c->tc_path ? (const void *)c->hlast : c->pend0;
  copy_rows_k<<<R, 128, 0, c->stream>>>((const uint4 *)src, (uint4 *)c->score_pend, c->score_idx, 0, nullptr, 0, vec);
  return post(c, "score_init_pend");
}

// xn[S + k] = pend[score_idx[k]]
darts_status launch_score_gather(darts_ctx *c, int S, int n_pend) {
  if (n_pend <= 0) return DARTS_OK;
  const int vec = c->m.d_model * c->elt / 16;
  copy_rows_k<<<n_pend, 128, 0, c->stream>>>((const uint4 *)c->score_pend, (uint4 *)c->xn, c->score_idx, 0, nullptr, S, vec);
  return post(c, "score_gather");
}

// pend[score_idx[k]] = xn[score_idx[max_rows + k]]
darts_status launch_score_scatter(darts_ctx *c, int n_pend) {
  if (n_pend <= 0) return DARTS_OK;
  const int vec = c->m.d_model * c->elt / 16;
  copy_rows_k<<<n_pend, 128, 0, c->stream>>>((const uint4 *)c->xn, (uint4 *)c->score_pend, c->score_idx + c->rt.max_rows, 0, c->score_idx, 0, vec);
  return post(c, "score_scatter");
}

darts_status launch_score_finalize(darts_ctx *c, int n_tiles, int rows) {
  score_finalize_k<<<rows, 512, 0, c->stream>>>((const float4 *)c->top2, (const float2 *)c->lse, n_tiles, rows, c->score_tgt, c->score_lp);
  return post(c, "score_finalize");
}

darts_status launch_score_logits(darts_ctx *c, int rows) {
  score_logits_k<<<rows, 256, 0, c->stream>>>(c->logits, c->m.vocab, c->score_tgt, c->temperature, c->score_lp);
  return post(c, "score_logits");
}
