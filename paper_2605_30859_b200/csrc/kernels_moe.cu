// Mixture-of-experts MLP (BASELINE.json configs[4]; R5, R13, R19):
//   p = softmax(b Wr^T) over E experts in fp32, b = rmsnorm(h) un-rounded;  top-k by p (ties -> lower expert id);
//   w = p_top / sum(p_top);  m = sum_e w_e expert_e(b);  h += m.
// Kernels (all sized from a host upper bound of the row count, live count read on the device):
//   moe_router_k     router logits [slot][E] straight from the fp32 residual stream (the bf16 xn is NOT used: the
//                    discrete top-k decision is taken in fp32 on both sides, R13); the last CTA to finish a block of
//                    slots then takes their top-k, one warp per slot: softmax, k rounds of warp arg-max, renormalised
//                    gates, per-expert counts
//   moe_place_k      (tensor-core path) one CTA per expert: exclusive scan of the counts, stable ballot ranking of the
//                    expert's assignments, gather of their bf16 activation rows into the expert-sorted matrix xs
//   [grouped stream-K tcgen05 GEMMs of kernels_gemm_sk.cu: gate/up then down, one row block per (expert, <= 256 rows)]
//   moe_expert_simt_k (fp32 / generic path) one CTA per (slot, k): the expert's SwiGLU MLP as warp dot products
//   moe_combine_k    h += sum_k w_k y_k in selection order (+ the next RMSNorm on the tensor-core path)
// Weight bytes streamed per step scale with the DISTINCT experts hit: groups with no rows exit before any load.
#include <algorithm>

#include "internal.cuh"

namespace {

constexpr int RROWS = 4;       // slots per router CTA (Wr tile reuse)
constexpr int REXP = 8;        // experts per router CTA (one per warp: the grid, not a loop, covers the experts)
constexpr int MAX_E_PER_LANE = 8;   // E <= 256

__device__ __forceinline__ int live_rows(const int32_t *n_rows_dev, int rows_ub) { return n_rows_dev ? min(*n_rows_dev, rows_ub) : rows_ub; }

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

// grid (ceil(rows_ub / RROWS), ceil(E / REXP)), 256 threads, dynamic smem RROWS * d floats.  d % 4 == 0.
// One warp per slot.  Ordering is taken on the logits (monotone in p, so identical to ordering by p in exact arithmetic).
__device__ __forceinline__ void topk_row(const float *logits, int E, int top_k, int32_t *__restrict__ eid, float *__restrict__ gate,
                                         int32_t *__restrict__ pos, int32_t *__restrict__ cnt, int32_t *__restrict__ eid_dump, int slot, int lane) {
  float z[MAX_E_PER_LANE];
  float mx = -INFINITY;
#pragma unroll
  for (int q = 0; q < MAX_E_PER_LANE; ++q) {
    int e = q * 32 + lane;
    z[q] = e < E ? __ldcg(&logits[(size_t)slot * E + e]) : -INFINITY;
    mx = fmaxf(mx, z[q]);
  }
  mx = warp_max(mx);
  float sum = 0.f;
#pragma unroll
  for (int q = 0; q < MAX_E_PER_LANE; ++q) sum += (q * 32 + lane) < E ? expf(z[q] - mx) : 0.f;
  sum = warp_sum(sum);
  unsigned taken = 0;
  float my_p = 0.f, psum = 0.f;
  int my_e = -1;
  for (int k = 0; k < top_k; ++k) {
    float bz = -INFINITY;
    int be = 0x7fffffff;
#pragma unroll
    for (int q = 0; q < MAX_E_PER_LANE; ++q) {
      int e = q * 32 + lane;
      if (e < E && !((taken >> q) & 1u) && (z[q] > bz)) { bz = z[q]; be = e; }     // ascending e: strict > keeps the lower id
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
      float oz = __shfl_xor_sync(0xffffffffu, bz, o);
      int oe = __shfl_xor_sync(0xffffffffu, be, o);
      if (oz > bz || (oz == bz && oe < be)) { bz = oz; be = oe; }
    }
    if ((be & 31) == lane) taken |= 1u << (be >> 5);
    float p = expf(bz - mx) / sum;
    psum += p;
    if (lane == k) { my_p = p; my_e = be; }
  }
  if (lane < top_k) {
    int a = slot * top_k + lane;
    eid[a] = my_e;
    if (eid_dump) eid_dump[a] = my_e;                    // parity hook (darts_debug_routing): this layer's choices survive the pass
    gate[a] = my_p / psum;
    pos[a] = a;                                        // identity; moe_place_k overwrites it on the tensor-core path
    if (cnt) atomicAdd(&cnt[my_e], 1);
  }
}


template <typename T>
__global__ void __launch_bounds__(256) moe_router_k(const float *__restrict__ h, const T *__restrict__ wnorm, const float *__restrict__ wr,
                                                    float *logits, int d, int E, float eps, int top_k, int32_t *__restrict__ eid,
                                                    float *__restrict__ gate, int32_t *__restrict__ pos, int32_t *__restrict__ cnt,
                                                    int32_t *arrive, int32_t *eid_dump, const int32_t *n_rows_dev, int rows_ub) {
  pdl_trigger();
  pdl_wait();
  extern __shared__ float xs[];                       // [RROWS][d] normalised rows
  __shared__ float red[RROWS][8];
  __shared__ int s_last;
  const int n = live_rows(n_rows_dev, rows_ub);
  const int s0 = blockIdx.x * RROWS;
  if (s0 >= n) return;
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  float ss[RROWS];
#pragma unroll
  for (int r = 0; r < RROWS; ++r) {
    ss[r] = 0.f;
    if (s0 + r < n)
      for (int k = threadIdx.x; k < d; k += blockDim.x) { float v = h[(size_t)(s0 + r) * d + k]; xs[r * d + k] = v; ss[r] += v * v; }
    else
      for (int k = threadIdx.x; k < d; k += blockDim.x) xs[r * d + k] = 0.f;
    ss[r] = warp_sum(ss[r]);
    if (lane == 0) red[r][warp] = ss[r];
  }
  __syncthreads();
#pragma unroll
  for (int r = 0; r < RROWS; ++r) {
    float tot = 0.f;
    for (int w = 0; w < 8; ++w) tot += red[r][w];
    float rinv = 1.0f / sqrtf(tot / d + eps);
    for (int k = threadIdx.x; k < d; k += blockDim.x) xs[r * d + k] = xs[r * d + k] * rinv * to_f<T>(wnorm[k]);
  }
  __syncthreads();
  for (int e = blockIdx.y * REXP + warp; e < min(E, (int)(blockIdx.y + 1) * REXP); e += 8) {
    float acc[RROWS] = {};
    const float4 *wrow = reinterpret_cast<const float4 *>(wr + (size_t)e * d);
#pragma unroll 4
    for (int k4 = lane; k4 < d / 4; k4 += 32) {
      float4 w = __ldg(wrow + k4);
#pragma unroll
      for (int r = 0; r < RROWS; ++r) {
        float4 x = *reinterpret_cast<const float4 *>(&xs[r * d + 4 * k4]);
        acc[r] = fmaf(w.x, x.x, fmaf(w.y, x.y, fmaf(w.z, x.z, fmaf(w.w, x.w, acc[r]))));
      }
    }
#pragma unroll
    for (int r = 0; r < RROWS; ++r) {
      float v = warp_sum(acc[r]);
      if (lane == 0 && s0 + r < n) logits[(size_t)(s0 + r) * E + e] = v;
    }
  }
  // the CTA that completes a slot block's logits (last of gridDim.y to arrive) takes its top-k: one warp per slot
  __threadfence();
  __syncthreads();
  if (threadIdx.x == 0) s_last = atomicAdd(&arrive[blockIdx.x], 1) == (int)gridDim.y - 1;
  __syncthreads();
  if (!s_last) return;
  __threadfence();
  if (threadIdx.x == 0) arrive[blockIdx.x] = 0;       // ready for the next layer's launch
  if (warp < RROWS && s0 + warp < n) topk_row(logits, E, top_k, eid, gate, pos, cnt, eid_dump, s0 + warp, lane);
}

// One CTA per expert (tensor-core path).  off[e] = sum_{e'<e} cnt[e'];  the expert's assignments keep their slot
// order (stable), so the layout of xs is a pure function of the routing.  xs[off[e] + rank] = xn[slot of assignment].
__global__ void __launch_bounds__(256) moe_place_k(const int32_t *__restrict__ cnt, const int32_t *__restrict__ eid, int32_t *__restrict__ pos,
                                                   int32_t *__restrict__ tok, int32_t *__restrict__ off_out, int32_t *__restrict__ rb_list,
                                                   int32_t *__restrict__ n_rb_out, const __nv_bfloat16 *__restrict__ xn,
                                                   __nv_bfloat16 *__restrict__ xs, int E, int top_k, int d, const int32_t *n_rows_dev,
                                                   int rows_ub) {
  pdl_trigger();
  pdl_wait();
  __shared__ int s_red[8], s_redb[8];
  __shared__ int s_off, s_blk;
  const int e = blockIdx.x, warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int n_assign = live_rows(n_rows_dev, rows_ub) * top_k;
  int part = 0, partb = 0;                               // rows / 256-row blocks of the experts before this one
  for (int q = threadIdx.x; q < e; q += blockDim.x) { int cq = cnt[q]; part += cq; partb += (cq + SK_ROWBLOCK - 1) / SK_ROWBLOCK; }
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) { part += __shfl_xor_sync(0xffffffffu, part, o); partb += __shfl_xor_sync(0xffffffffu, partb, o); }
  if (lane == 0) { s_red[warp] = part; s_redb[warp] = partb; }
  __syncthreads();
  if (threadIdx.x == 0) {
    int t = 0, tb = 0;
    for (int w = 0; w < 8; ++w) { t += s_red[w]; tb += s_redb[w]; }
    s_off = t; s_blk = tb;
    off_out[e] = t;
    if (e == E - 1) { off_out[E] = t + cnt[e]; *n_rb_out = tb + (cnt[e] + SK_ROWBLOCK - 1) / SK_ROWBLOCK; }
  }
  __syncthreads();
  const int off = s_off, mine = cnt[e];
  if (mine == 0) return;
  for (int i = threadIdx.x; i < (mine + SK_ROWBLOCK - 1) / SK_ROWBLOCK; i += blockDim.x) {   // this expert's row blocks for the grouped GEMM
    int32_t *rb = rb_list + 4 * (s_blk + i);
    rb[0] = off + i * SK_ROWBLOCK; rb[1] = min(SK_ROWBLOCK, mine - i * SK_ROWBLOCK); rb[2] = e; rb[3] = 0;
  }
  if (warp == 0) {
    int base = off;
    for (int a0 = 0; a0 < n_assign; a0 += 32) {
      int a = a0 + lane;
      bool m = a < n_assign && eid[a] == e;
      unsigned mask = __ballot_sync(0xffffffffu, m);
      if (m) {
        int p = base + __popc(mask & ((1u << lane) - 1u));
        pos[a] = p;
        tok[p] = a;
      }
      base += __popc(mask);
    }
  }
  __syncthreads();
  const int vec = d / 8;                                  // uint4 = 8 bf16
  for (int i = warp; i < mine; i += 8) {
    int slot = tok[off + i] / top_k;
    const uint4 *src = reinterpret_cast<const uint4 *>(xn + (size_t)slot * d);
    uint4 *dst = reinterpret_cast<uint4 *>(xs + (size_t)(off + i) * d);
    for (int k = lane; k < vec; k += 32) dst[k] = src[k];
  }
}

// act[p][f] = silu(g) * u over the expert-sorted rows p < live * top_k;  g = sum_s P_s[p][f], u = sum_s P_s[p][F + f].
__global__ void __launch_bounds__(256) moe_silu_mul_k(const float *__restrict__ part, int S, size_t split_stride, __nv_bfloat16 *__restrict__ act,
                                                      int F, int top_k, const int32_t *n_rows_dev, int rows_ub) {
  pdl_trigger();
  pdl_wait();
  int p = blockIdx.y;
  if (p >= live_rows(n_rows_dev, rows_ub) * top_k) return;
  int k = (blockIdx.x * blockDim.x + threadIdx.x) * 4;
  if (k >= F) return;
  const float *row = part + (size_t)p * 2 * F;
  float4 g = *reinterpret_cast<const float4 *>(row + k), u = *reinterpret_cast<const float4 *>(row + F + k);
  for (int s = 1; s < S; ++s) {
    float4 a = *reinterpret_cast<const float4 *>(row + s * split_stride + k), b = *reinterpret_cast<const float4 *>(row + s * split_stride + F + k);
    g.x += a.x; g.y += a.y; g.z += a.z; g.w += a.w;
    u.x += b.x; u.y += b.y; u.z += b.z; u.w += b.w;
  }
  auto f = [](float gg, float uu) { return gg / (1.0f + expf(-gg)) * uu; };
  __nv_bfloat162 o0 = __floats2bfloat162_rn(f(g.x, u.x), f(g.y, u.y)), o1 = __floats2bfloat162_rn(f(g.z, u.z), f(g.w, u.w));
  uint2 o;
  o.x = *reinterpret_cast<uint32_t *>(&o0);
  o.y = *reinterpret_cast<uint32_t *>(&o1);
  *reinterpret_cast<uint2 *>(act + (size_t)p * F + k) = o;
}

// Generic path: one CTA per assignment a = slot * top_k + k.  y[a] = Wd_e (silu(Wg_e x) * (Wu_e x)), fp32 throughout.
template <typename T>
__global__ void __launch_bounds__(256) moe_expert_simt_k(const T *__restrict__ xn, const T *__restrict__ wgu_e, const T *__restrict__ wd_e,
                                                         const int32_t *__restrict__ eid, float *__restrict__ y, int d, int F, int top_k,
                                                         const int32_t *n_rows_dev, int rows_ub) {
  pdl_trigger();
  pdl_wait();
  extern __shared__ float sm_f[];                      // x [d], act [F]
  float *x = sm_f, *act = sm_f + d;
  const int a = blockIdx.x, slot = a / top_k;
  if (slot >= live_rows(n_rows_dev, rows_ub)) return;
  const int e = eid[a], warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  for (int k = threadIdx.x; k < d; k += blockDim.x) x[k] = to_f<T>(xn[(size_t)slot * d + k]);
  __syncthreads();
  const T *wg = wgu_e + (size_t)e * 2 * F * d;
  for (int f = warp; f < F; f += 8) {
    float g = 0.f, u = 0.f;
    for (int k = lane; k < d; k += 32) { g = fmaf(to_f<T>(wg[(size_t)f * d + k]), x[k], g); u = fmaf(to_f<T>(wg[(size_t)(F + f) * d + k]), x[k], u); }
    g = warp_sum(g); u = warp_sum(u);
    if (lane == 0) act[f] = g / (1.0f + expf(-g)) * u;
  }
  __syncthreads();
  const T *wd = wd_e + (size_t)e * d * F;
  for (int nn = warp; nn < d; nn += 8) {
    float v = 0.f;
    for (int k = lane; k < F; k += 32) v = fmaf(to_f<T>(wd[(size_t)nn * F + k]), act[k], v);
    v = warp_sum(v);
    if (lane == 0) y[(size_t)a * d + nn] = v;
  }
}

// h[slot] += sum_k gate_k * (sum_s Y_s[pos_k]) in selection order;  if wnorm: out = rmsnorm(h[slot]) * wnorm (next GEMM input).
template <typename T>
__global__ void __launch_bounds__(256) moe_combine_k(float *__restrict__ h, const float *__restrict__ y, int S, size_t split_stride,
                                                     const int32_t *__restrict__ pos, const float *__restrict__ gate, int top_k,
                                                     const T *__restrict__ wnorm, T *__restrict__ out, int d, float eps,
                                                     const int32_t *n_rows_dev, int rows_ub) {
  pdl_trigger();
  pdl_wait();
  int slot = blockIdx.x;
  if (slot >= live_rows(n_rows_dev, rows_ub)) return;
  float4 *hr = reinterpret_cast<float4 *>(h + (size_t)slot * d);
  float ss = 0.f;
  for (int k = threadIdx.x; k < d / 4; k += blockDim.x) {
    float4 v = hr[k];
    for (int kk = 0; kk < top_k; ++kk) {
      int p = pos[slot * top_k + kk];
      float g = gate[slot * top_k + kk];
      const float4 *yr = reinterpret_cast<const float4 *>(y + (size_t)p * d) + k;
      float4 a = yr[0];
      for (int s = 1; s < S; ++s) { float4 b = yr[s * (split_stride / 4)]; a.x += b.x; a.y += b.y; a.z += b.z; a.w += b.w; }
      v.x = fmaf(g, a.x, v.x); v.y = fmaf(g, a.y, v.y); v.z = fmaf(g, a.z, v.z); v.w = fmaf(g, a.w, v.w);
    }
    hr[k] = v;
    ss += v.x * v.x + v.y * v.y + v.z * v.z + v.w * v.w;
  }
  if (!wnorm) return;
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
  for (int k = threadIdx.x; k < d / 4; k += blockDim.x) {
    float4 v = hr[k];
    T *o = out + (size_t)slot * d + 4 * k;
    o[0] = from_f<T>(v.x * r * to_f<T>(wnorm[4 * k])); o[1] = from_f<T>(v.y * r * to_f<T>(wnorm[4 * k + 1]));
    o[2] = from_f<T>(v.z * r * to_f<T>(wnorm[4 * k + 2])); o[3] = from_f<T>(v.w * r * to_f<T>(wnorm[4 * k + 3]));
  }
}

template <typename T>
darts_status route(darts_ctx *c, int layer, int rows_ub, const int32_t *n_rows_dev, int32_t *cnt) {
  const darts_model_desc &m = c->m;
  dim3 grid((rows_ub + RROWS - 1) / RROWS, (m.n_experts + REXP - 1) / REXP);
  size_t smem = (size_t)RROWS * m.d_model * sizeof(float);
  launch_pdl(c, moe_router_k<T>, grid, dim3(256), smem, c->h, (const T *)c->mlp_norm[layer], (const float *)c->wr[layer], c->moe_logits, m.d_model,
             m.n_experts, m.rms_eps, m.top_k, c->moe_eid, c->moe_w, c->moe_pos, cnt, c->moe_arrive,
             c->moe_eid_dump ? c->moe_eid_dump + (size_t)layer * c->act_rows * m.top_k : nullptr, n_rows_dev, rows_ub);
  return post(c, "moe_router");
}

}  // namespace

darts_status moe_configure(darts_ctx *c) {
  if (!c->m.n_experts) return DARTS_OK;
  const size_t smem = (size_t)RROWS * c->m.d_model * sizeof(float);
  if (smem > 48 * 1024) {
    CUDA_TRY(c, cudaFuncSetAttribute(moe_router_k<float>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    CUDA_TRY(c, cudaFuncSetAttribute(moe_router_k<__nv_bfloat16>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
  }
  return DARTS_OK;
}

// Zero the per-layer expert counters of one forward pass (tensor-core path; one memset per pass).
darts_status launch_moe_begin_pass(darts_ctx *c) {
  if (!c->m.n_experts || !c->tc_path) return DARTS_OK;
  CUDA_TRY(c, cudaMemsetAsync(c->moe_cnt, 0, (size_t)c->m.n_layers * c->m.n_experts * sizeof(int32_t), c->stream));
  return DARTS_OK;
}

// Generic path (fp32 models, shapes the tcgen05 GEMM does not take): xn = rmsnorm(h) * mlp_norm is already in c->xn.
darts_status launch_moe(darts_ctx *c, int layer, int rows_ub, const int32_t *n_rows_dev) {
  if (rows_ub <= 0) return DARTS_OK;
  const darts_model_desc &m = c->m;
  darts_status s;
  size_t smem = (size_t)(m.d_model + m.expert_ffn) * sizeof(float);
  if (smem > 48 * 1024) FAIL(c, DARTS_ERR_UNSUPPORTED, "generic MoE path needs d_model + expert_ffn <= 12288");
  if (m.dtype == DARTS_F32) {
    if ((s = route<float>(c, layer, rows_ub, n_rows_dev, nullptr)) != DARTS_OK) return s;
    moe_expert_simt_k<float><<<rows_ub * m.top_k, 256, smem, c->stream>>>((const float *)c->xn, (const float *)c->wgu_e[layer], (const float *)c->wd_e[layer],
                                                                           c->moe_eid, c->moe_y, m.d_model, m.expert_ffn, m.top_k, n_rows_dev, rows_ub);
    if ((s = post(c, "moe_expert_simt")) != DARTS_OK) return s;
    moe_combine_k<float><<<rows_ub, 256, 0, c->stream>>>(c->h, c->moe_y, 1, 0, c->moe_pos, c->moe_w, m.top_k, nullptr, nullptr, m.d_model, m.rms_eps,
                                                         n_rows_dev, rows_ub);
  } else {
    using T = __nv_bfloat16;
    if ((s = route<T>(c, layer, rows_ub, n_rows_dev, nullptr)) != DARTS_OK) return s;
    moe_expert_simt_k<T><<<rows_ub * m.top_k, 256, smem, c->stream>>>((const T *)c->xn, (const T *)c->wgu_e[layer], (const T *)c->wd_e[layer], c->moe_eid,
                                                                       c->moe_y, m.d_model, m.expert_ffn, m.top_k, n_rows_dev, rows_ub);
    if ((s = post(c, "moe_expert_simt")) != DARTS_OK) return s;
    moe_combine_k<T><<<rows_ub, 256, 0, c->stream>>>(c->h, c->moe_y, 1, 0, c->moe_pos, c->moe_w, m.top_k, nullptr, nullptr, m.d_model, m.rms_eps,
                                                     n_rows_dev, rows_ub);
  }
  return post(c, "moe_combine");
}

// Tensor-core path: router -> top-k -> expert-sorted gather -> grouped gate/up GEMM -> SiLU*mul -> grouped down GEMM ->
// gated combine + residual + next RMSNorm (leaves xn ready for the next layer's QKV GEMM / the LM head).
darts_status launch_moe_tc(darts_ctx *c, int layer, const void *next_norm, int rows_ub, const int32_t *n_rows_dev) {
  if (rows_ub <= 0) return DARTS_OK;
  using T = __nv_bfloat16;
  const darts_model_desc &m = c->m;
  const int E = m.n_experts, F = m.expert_ffn, d = m.d_model, RK = rows_ub * m.top_k;
  int32_t *cnt = c->moe_cnt + (size_t)layer * E;
  darts_status s;
  if ((s = route<T>(c, layer, rows_ub, n_rows_dev, cnt)) != DARTS_OK) return s;
  launch_pdl(c, moe_place_k, dim3(E), dim3(256), 0, cnt, c->moe_eid, c->moe_pos, c->moe_tok, c->moe_off, c->moe_rb, c->moe_nrb, (const T *)c->xn, (T *)c->xs, E,
                                        m.top_k, d, n_rows_dev, rows_ub);
  if ((s = post(c, "moe_place")) != DARTS_OK) return s;
  // grouped stream-K GEMMs: one row block per (expert, <= 256 of its rows); experts nobody chose cost nothing
  const int n_rb_ub = std::min(E, RK) + RK / SK_ROWBLOCK;
  SkGemm g{};
  g.w_map = &c->tm_wgu_e[layer]; g.x_maps = &c->xm_xs; g.C = c->part; g.N = 2 * F; g.rows_ub = rows_ub;      // <= rows_ub rows per expert
  g.rb_list = c->moe_rb; g.n_rb_dev = c->moe_nrb; g.w_rows_per_group = 2 * F;
  g.plan = sk_plan(c->n_sms, g.N, d, rows_ub, n_rb_ub, false);
  g.slot_stride = 0;
  if ((s = launch_gemm_sk(c, g)) != DARTS_OK) return s;
  dim3 grid((F / 4 + 255) / 256, RK);
  launch_pdl(c, moe_silu_mul_k, grid, dim3(256), 0, c->part, 1, (size_t)0, (T *)c->act, F, m.top_k, n_rows_dev, rows_ub);
  if ((s = post(c, "moe_silu_mul")) != DARTS_OK) return s;
  g.w_map = &c->tm_wd_e[layer]; g.x_maps = &c->xm_act; g.N = d; g.w_rows_per_group = d;
  g.plan = sk_plan(c->n_sms, g.N, F, rows_ub, n_rb_ub, false);
  if ((s = launch_gemm_sk(c, g)) != DARTS_OK) return s;
  launch_pdl(c, moe_combine_k<T>, dim3(rows_ub), dim3(256), 0, c->h, c->part, 1, (size_t)0, c->moe_pos, c->moe_w, m.top_k, (const T *)next_norm, (T *)c->xn, d,
                                                   m.rms_eps, n_rows_dev, rows_ub);
  return post(c, "moe_combine");
}
