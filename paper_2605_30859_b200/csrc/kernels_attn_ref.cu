// Generic paged GQA attention (any head_dim multiple of 32, any page size, fp32 or bf16 cache):
// one warp per (slot, q-head), online softmax over [visible prefix tokens || own suffix tokens].
// Used for the fp32 path (config 1), for prefill (causal: slot = prompt token) and as the
// in-library cross-check of the tuned bf16 kernel (kernels_attn_sm100.cu).
#include "internal.cuh"

namespace {

template <typename T, int DPL>
__global__ void attn_ref_k(const T *__restrict__ q, T *__restrict__ out, const T *__restrict__ kv_layer,
                           const int32_t *__restrict__ slot_prompt, const int32_t *__restrict__ slot_npre,
                           const int32_t *__restrict__ slot_nsuf, const int32_t *__restrict__ slot_row,
                           const int32_t *__restrict__ g_prefix_pages, const int32_t *__restrict__ row_pages, int mpp, int msp,
                           int Hq, int Hkv, int page, KvGeom geo, float scale,
                           const int32_t *n_rows_dev, int rows_ub) {
  constexpr int hd = DPL * 32;
  int slot = blockIdx.y;
  int R = n_rows_dev ? min(*n_rows_dev, rows_ub) : rows_ub;
  if (slot >= R) return;
  int rep = Hq / Hkv;
  int kvh = blockIdx.x, warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  int h = kvh * rep + warp;
  float qr[DPL], acc[DPL];
#pragma unroll
  for (int k = 0; k < DPL; ++k) {
    qr[k] = to_f<T>(q[((size_t)slot * Hq + h) * hd + lane * DPL + k]) * scale;
    acc[k] = 0.f;
  }
  float m = -INFINITY, l = 0.f;
  for (int seg = 0; seg < 2; ++seg) {
    int count = seg == 0 ? slot_npre[slot] : slot_nsuf[slot];
    const int32_t *pages = seg == 0 ? g_prefix_pages + (size_t)slot_prompt[slot] * mpp : row_pages + (size_t)slot_row[slot] * msp;
    for (int n = 0; n < count; ++n) {
      int pg = pages[n / page], off = n % page;
      const T *kp = kv_layer + kv_elem(geo, pg, kvh, 0, off, lane * DPL);   // DPL <= 8 dims stay inside one 16-byte chunk
      const T *vp = kv_layer + kv_elem(geo, pg, kvh, 1, off, lane * DPL);
      float s = 0.f;
#pragma unroll
      for (int k = 0; k < DPL; ++k) s = fmaf(qr[k], to_f<T>(kp[k]), s);
      s = warp_sum(s);
      float mn = fmaxf(m, s);
      float corr = expf(m - mn), p = expf(s - mn);
      l = l * corr + p;
#pragma unroll
      for (int k = 0; k < DPL; ++k) acc[k] = acc[k] * corr + p * to_f<T>(vp[k]);
      m = mn;
    }
  }
  float inv = 1.0f / l;
#pragma unroll
  for (int k = 0; k < DPL; ++k) out[((size_t)slot * Hq + h) * hd + lane * DPL + k] = from_f<T>(acc[k] * inv);
}

template <typename T>
darts_status run(darts_ctx *c, int layer, const void *q, void *out, int rows_ub, const int32_t *n_rows_dev) {
  const auto &m = c->m;
  int rep = m.n_q_heads / m.n_kv_heads;
  dim3 grid(m.n_kv_heads, rows_ub), block(rep * 32);
  const T *kv = (const T *)c->kv_pool + (size_t)layer * c->kv_layer_elems;
  float scale = 1.0f / sqrtf((float)m.head_dim);
#define ARGS (const T *)q, (T *)out, kv, c->slot_prompt, c->slot_npre, c->slot_nsuf, c->slot_row, c->g_prefix_pages, c->row_pages, \
             c->max_prefix_pages, c->max_suffix_pages, m.n_q_heads, m.n_kv_heads, c->rt.page_size, c->geom(),                     \
             scale, n_rows_dev, rows_ub
  switch (m.head_dim / 32) {
    case 1: attn_ref_k<T, 1><<<grid, block, 0, c->stream>>>(ARGS); break;
    case 2: attn_ref_k<T, 2><<<grid, block, 0, c->stream>>>(ARGS); break;
    case 4: attn_ref_k<T, 4><<<grid, block, 0, c->stream>>>(ARGS); break;
    case 8: attn_ref_k<T, 8><<<grid, block, 0, c->stream>>>(ARGS); break;
    default: FAIL(c, DARTS_ERR_UNSUPPORTED, "head_dim %d not in {32,64,128,256}", m.head_dim);
  }
#undef ARGS
  c->launches++;
  cudaError_t e = cudaGetLastError();
  if (e != cudaSuccess) {
    snprintf(c->err, sizeof(c->err), "launch attn_ref: %s", cudaGetErrorString(e));
    c->sticky = DARTS_ERR_CUDA;
    return DARTS_ERR_CUDA;
  }
  return DARTS_OK;
}

}  // namespace

darts_status launch_attention_ref(darts_ctx *c, int layer, const void *q, void *out, int rows_ub, const int32_t *n_rows_dev) {
  if (rows_ub <= 0) return DARTS_OK;
  if (c->m.dtype == DARTS_F32) return run<float>(c, layer, q, out, rows_ub, n_rows_dev);
  return run<__nv_bfloat16>(c, layer, q, out, rows_ub, n_rows_dev);
}
