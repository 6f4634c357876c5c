// Consumers of the tensor-core GEMM's split-K partials (bf16 path).  Every kernel adds the S partials of an element
// in split order (deterministic), so no GEMM output makes a second trip through HBM as a reduced matrix:
//   add_rmsnorm    h += sum_s P_s (O-proj / down-proj residual), then xn = rmsnorm(h) * w for the next GEMM
//   silu_mul_part  act = silu(sum_s gate_s) * (sum_s up_s)
//   (rope_append_k in kernels_basic.cu does the same for the QKV partials)
#include "internal.cuh"

namespace {

__device__ __forceinline__ int live_rows(const int32_t *n_rows_dev, int rows_ub) { return n_rows_dev ? min(*n_rows_dev, rows_ub) : rows_ub; }

// one CTA per slot; d % 4 == 0
__global__ void __launch_bounds__(256) add_rmsnorm_k(float *__restrict__ h, const float *__restrict__ part, int S, size_t split_stride,
                                                     const __nv_bfloat16 *__restrict__ w, __nv_bfloat16 *__restrict__ out, int d, float eps,
                                                     const int32_t *n_rows_dev, int rows_ub) {
  int slot = blockIdx.x;
  if (slot >= live_rows(n_rows_dev, rows_ub)) return;
  float4 *hr = reinterpret_cast<float4 *>(h + (size_t)slot * d);
  const float4 *pr = reinterpret_cast<const float4 *>(part + (size_t)slot * d);
  float ss = 0.f;
  for (int k = threadIdx.x; k < d / 4; k += blockDim.x) {
    float4 v = hr[k];
    for (int s = 0; s < S; ++s) {
      float4 a = pr[s * (split_stride / 4) + k];
      v.x += a.x; v.y += a.y; v.z += a.z; v.w += a.w;
    }
    hr[k] = v;
    ss += v.x * v.x + v.y * v.y + v.z * v.z + v.w * v.w;
  }
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
    float4 v = hr[k];                                       // written by this thread above
    const __nv_bfloat162 *wp = reinterpret_cast<const __nv_bfloat162 *>(w + 4 * k);
    float2 w0 = __bfloat1622float2(wp[0]), w1 = __bfloat1622float2(wp[1]);
    __nv_bfloat162 o0 = __floats2bfloat162_rn(v.x * r * w0.x, v.y * r * w0.y), o1 = __floats2bfloat162_rn(v.z * r * w1.x, v.w * r * w1.y);
    uint2 o;
    o.x = *reinterpret_cast<uint32_t *>(&o0);
    o.y = *reinterpret_cast<uint32_t *>(&o1);
    *reinterpret_cast<uint2 *>(out + (size_t)slot * d + 4 * k) = o;
  }
}

// act[slot][k] = silu(g) * u,  g = sum_s P_s[slot][k], u = sum_s P_s[slot][F + k];  F % 4 == 0
__global__ void __launch_bounds__(256) silu_mul_part_k(const float *__restrict__ part, int S, size_t split_stride, __nv_bfloat16 *__restrict__ act,
                                                       int F, const int32_t *n_rows_dev, int rows_ub) {
  int slot = blockIdx.y;
  if (slot >= live_rows(n_rows_dev, rows_ub)) return;
  int k = (blockIdx.x * blockDim.x + threadIdx.x) * 4;
  if (k >= F) return;
  const float *row = part + (size_t)slot * 2 * F;
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
  *reinterpret_cast<uint2 *>(act + (size_t)slot * F + k) = o;
}

// dst[i - g_begin] = src[slot of the last token of prompt i]   (bf16 rows of d elements)
__global__ void gather_rows_bf16_k(const __nv_bfloat16 *__restrict__ src, __nv_bfloat16 *__restrict__ dst, const int32_t *__restrict__ g_tok_off,
                                   int tok_begin, int g_begin, int d) {
  int i = g_begin + blockIdx.x;
  int slot = g_tok_off[i + 1] - 1 - tok_begin;
  for (int k = threadIdx.x; k < d; k += blockDim.x) dst[(size_t)blockIdx.x * d + k] = src[(size_t)slot * d + k];
}

__global__ void sum_partials_k(const float *__restrict__ part, float *__restrict__ out, int S, size_t n) {
  size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n) return;
  float v = part[i];
  for (int s = 1; s < S; ++s) v += part[(size_t)s * n + i];
  out[i] = v;
}

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

}  // namespace

darts_status launch_add_rmsnorm(darts_ctx *c, const float *part, int S, size_t split_stride, const void *w, int rows_ub, const int32_t *n_rows_dev) {
  if (rows_ub <= 0) return DARTS_OK;
  add_rmsnorm_k<<<rows_ub, 256, 0, c->stream>>>(c->h, part, S, split_stride, (const __nv_bfloat16 *)w, (__nv_bfloat16 *)c->xn, c->m.d_model,
                                                c->m.rms_eps, n_rows_dev, rows_ub);
  return post(c, "add_rmsnorm");
}

darts_status launch_silu_mul_part(darts_ctx *c, int S, int rows_ub, const int32_t *n_rows_dev) {
  if (rows_ub <= 0) return DARTS_OK;
  int F = c->m.ffn;
  dim3 grid((F / 4 + 255) / 256, rows_ub);
  silu_mul_part_k<<<grid, 256, 0, c->stream>>>(c->part, S, (size_t)rows_ub * 2 * F, (__nv_bfloat16 *)c->act, F, n_rows_dev, rows_ub);
  return post(c, "silu_mul_part");
}

darts_status launch_gather_rows_bf16(darts_ctx *c, const void *src, void *dst, int tok_begin, int g_begin, int g_end) {
  gather_rows_bf16_k<<<g_end - g_begin, 256, 0, c->stream>>>((const __nv_bfloat16 *)src, (__nv_bfloat16 *)dst, c->g_tok_off, tok_begin, g_begin,
                                                             c->m.d_model);
  return post(c, "gather_rows_bf16");
}

darts_status launch_sum_partials(darts_ctx *c, const float *part, float *out, int S, size_t n) {
  sum_partials_k<<<(unsigned)((n + 255) / 256), 256, 0, c->stream>>>(part, out, S, n);
  return post(c, "sum_partials");
}
