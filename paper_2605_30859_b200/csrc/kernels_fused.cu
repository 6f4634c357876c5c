// Consumers of the stream-K GEMM's pieces (bf16 path).  Every kernel adds the pieces of an element in slot order
// (deterministic), so no GEMM output makes a second trip through HBM as a reduced matrix:
//   add_rmsnorm_sk    h += sum of pieces (O-proj / down-proj residual), then xn = rmsnorm(h) * w for the next GEMM
//   silu_mul_sk       act = silu(sum gate pieces) * (sum up pieces)
//   rope_append_sk    (QK-norm) + RoPE + KV append from the QKV pieces
#include <stdlib.h>

#include <algorithm>

#include "internal.cuh"

namespace {

__device__ __forceinline__ int live_rows(const int32_t *n_rows_dev, int rows_ub) { return n_rows_dev ? min(*n_rows_dev, rows_ub) : rows_ub; }

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

// ---- consumers of the stream-K pieces (kernels_gemm_sk.cu): element (row, col) = sum of its tile's pieces in slot order.

// Piece loads are issued four at a time before their adds (memory-level parallelism at a low register cost, so that
// occupancy hides the rest of the latency); the adds run in slot order.
__device__ __forceinline__ float4 sk_sum4(const SkView &v, int np, size_t idx) {
  const float4 *p = reinterpret_cast<const float4 *>(v.part + idx);
  const size_t st = v.slot_stride / 4;
  float4 a = make_float4(0.f, 0.f, 0.f, 0.f);              // 0 + x == x: the sum is still piece 0 + piece 1 + ... in slot order
  for (int s0 = 0; s0 < np; s0 += 4) {
    float4 x[4];
#pragma unroll
    for (int s = 0; s < 4; ++s)
      if (s0 + s < np) x[s] = __ldg(p + (size_t)(s0 + s) * st);
#pragma unroll
    for (int s = 0; s < 4; ++s)
      if (s0 + s < np) { a.x += x[s].x; a.y += x[s].y; a.z += x[s].z; a.w += x[s].w; }
  }
  return a;
}

// Two elements at once (gate / up, the two halves of a rotary pair): both first pieces, then both tails, so the loads of the two
// sums overlap instead of forming two dependent round trips to L2.
__device__ __forceinline__ void sk_sum4x2(const SkView &v, int npa, size_t ia, int npb, size_t ib, float4 &a, float4 &b) {
  const float4 *pa = reinterpret_cast<const float4 *>(v.part + ia), *pb = reinterpret_cast<const float4 *>(v.part + ib);
  const size_t st = v.slot_stride / 4;
  a = __ldg(pa);
  b = __ldg(pb);
  const int np = max(npa, npb);
  for (int s0 = 1; s0 < np; s0 += 2) {
    float4 xa[2], xb[2];
#pragma unroll
    for (int s = 0; s < 2; ++s) {
      if (s0 + s < npa) xa[s] = __ldg(pa + (size_t)(s0 + s) * st);
      if (s0 + s < npb) xb[s] = __ldg(pb + (size_t)(s0 + s) * st);
    }
#pragma unroll
    for (int s = 0; s < 2; ++s) {
      if (s0 + s < npa) { a.x += xa[s].x; a.y += xa[s].y; a.z += xa[s].z; a.w += xa[s].w; }
      if (s0 + s < npb) { b.x += xb[s].x; b.y += xb[s].y; b.z += xb[s].z; b.w += xb[s].w; }
    }
  }
}

__device__ __forceinline__ uint2 pack4_bf16(float a, float b, float c, float d) {
  __nv_bfloat162 o0 = __floats2bfloat162_rn(a, b), o1 = __floats2bfloat162_rn(c, d);
  uint2 o;
  o.x = *reinterpret_cast<uint32_t *>(&o0);
  o.y = *reinterpret_cast<uint32_t *>(&o1);
  return o;
}

// h[slot] += pieces;  out = rmsnorm(h[slot]) * w.   One CTA per slot, one float4 per thread per pass (d % 4 == 0).
__global__ void __launch_bounds__(256) add_rmsnorm_sk_k(float *__restrict__ h, SkView v, const __nv_bfloat16 *__restrict__ w,
                                                        __nv_bfloat16 *__restrict__ out, int d, float eps, const int32_t *n_rows_dev, int rows_ub) {
  pdl_trigger();
  pdl_wait();
  const int slot = blockIdx.x, live = live_rows(n_rows_dev, rows_ub);
  if (slot >= live) return;
  const int rbr = sk_view_rb_rows(v, live), n_rb = (live + rbr - 1) / rbr;
  float4 *hr = reinterpret_cast<float4 *>(h + (size_t)slot * d);
  float ss = 0.f;
  for (int k = threadIdx.x; k < d / 4; k += blockDim.x) {
    float4 x = hr[k];                                       // in flight together with the piece loads
    float4 a = sk_sum4(v, sk_npieces(v, n_rb, rbr, 4 * k, slot), (size_t)slot * d + 4 * k);
    x.x += a.x; x.y += a.y; x.z += a.z; x.w += a.w;
    hr[k] = x;
    ss += x.x * x.x + x.y * x.y + x.z * x.z + x.w * x.w;
  }
  __shared__ float red[32];
  ss = warp_sum(ss);
  if ((threadIdx.x & 31) == 0) red[threadIdx.x >> 5] = ss;
  __syncthreads();
  if (threadIdx.x < 32) {
    float t = threadIdx.x < (blockDim.x >> 5) ? red[threadIdx.x] : 0.f;
    t = warp_sum(t);
    if (threadIdx.x == 0) red[0] = t;
  }
  __syncthreads();
  const float r = 1.0f / sqrtf(red[0] / d + eps);
  for (int k = threadIdx.x; k < d / 4; k += blockDim.x) {
    float4 x = hr[k];                                       // written by this thread above
    const __nv_bfloat162 *wp = reinterpret_cast<const __nv_bfloat162 *>(w + 4 * k);
    float2 w0 = __bfloat1622float2(wp[0]), w1 = __bfloat1622float2(wp[1]);
    *reinterpret_cast<uint2 *>(out + (size_t)slot * d + 4 * k) = pack4_bf16(x.x * r * w0.x, x.y * r * w0.y, x.z * r * w1.x, x.w * r * w1.y);
  }
}

// act[slot][k] = silu(g) * u with g = pieces(slot, k), u = pieces(slot, F + k)
__global__ void __launch_bounds__(256) silu_mul_sk_k(SkView v, __nv_bfloat16 *__restrict__ act, int F, const int32_t *n_rows_dev, int rows_ub) {
  pdl_trigger();
  pdl_wait();
  const int slot = blockIdx.y, live = live_rows(n_rows_dev, rows_ub);
  if (slot >= live) return;
  const int k = (blockIdx.x * blockDim.x + threadIdx.x) * 4;
  if (k >= F) return;
  const int rbr = sk_view_rb_rows(v, live), n_rb = (live + rbr - 1) / rbr;
  const size_t row = (size_t)slot * 2 * F;
  float4 g, u;
  sk_sum4x2(v, sk_npieces(v, n_rb, rbr, k, slot), row + k, sk_npieces(v, n_rb, rbr, F + k, slot), row + F + k, g, u);
  // fast exp / division (a few ulp, against 2^-9 of the bf16 store that follows): the IEEE forms were ~160 of this kernel's ~210
  // instructions per warp and the kernel is issue-bound (ncu: issue slots 53 % busy, L2 15 % — profiles/r2_consumers.md)
  auto f = [](float gg, float uu) { return __fdividef(gg, 1.0f + __expf(-gg)) * uu; };
  *reinterpret_cast<uint2 *>(act + (size_t)slot * F + k) = pack4_bf16(f(g.x, u.x), f(g.y, u.y), f(g.z, u.z), f(g.w, u.w));
}

// (QK-norm) + RoPE + KV append from the QKV pieces.  One warp per (slot, head); lane l owns elements 4l..4l+3 of the
// head's rotate-half pairs: x1 = head[4j..], x2 = head[hd/2 + 4j..] for j < hd/8 (hd in {64, 128, 256}; hd % 8 == 0).
__global__ void __launch_bounds__(128) rope_append_sk_k(SkView v, __nv_bfloat16 *__restrict__ q_out, __nv_bfloat16 *__restrict__ kv_layer,
                                                       const int32_t *__restrict__ slot_dst_page, const int32_t *__restrict__ slot_dst_off,
                                                       const float2 *__restrict__ cs, const __nv_bfloat16 *__restrict__ q_norm,
                                                       const __nv_bfloat16 *__restrict__ k_norm, int Hq, int Hkv, int hd, float eps, KvGeom geo,
                                                       const int32_t *n_rows_dev, int rows_ub) {
  pdl_trigger();
  pdl_wait();
  const int slot = blockIdx.y, live = live_rows(n_rows_dev, rows_ub);
  if (slot >= live) return;
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int head = blockIdx.x * 4 + warp;
  if (head >= Hq + 2 * Hkv) return;
  const int rbr = sk_view_rb_rows(v, live), n_rb = (live + rbr - 1) / rbr;
  const int half = hd >> 1, col0 = head * hd;
  const size_t row = (size_t)slot * (Hq + 2 * Hkv) * hd + col0;
  const int page = slot_dst_page[slot], off = slot_dst_off[slot];
  const bool is_q = head < Hq, is_v = head >= Hq + Hkv;
  if (!is_q && page < 0) return;
  const bool act = lane < half / 4;                        // hd <= 256: one pass, the head lives in <= 32 lanes
  const int p = 4 * lane;
  float a1[4] = {0.f, 0.f, 0.f, 0.f}, a2[4] = {0.f, 0.f, 0.f, 0.f};
  if (act) {
    float4 x1, x2;
    sk_sum4x2(v, sk_npieces(v, n_rb, rbr, col0 + p, slot), row + p, sk_npieces(v, n_rb, rbr, col0 + half + p, slot), row + half + p, x1, x2);
    a1[0] = x1.x; a1[1] = x1.y; a1[2] = x1.z; a1[3] = x1.w;
    a2[0] = x2.x; a2[1] = x2.y; a2[2] = x2.z; a2[3] = x2.w;
  }
  // p is a multiple of 4: the four elements of each half stay adjacent under the 16-byte-chunk swizzle of kv_elem -> one 8-byte store
  if (is_v) {
    if (act) {
      *reinterpret_cast<uint2 *>(&kv_layer[kv_elem(geo, page, head - Hq - Hkv, 1, off, p)]) = pack4_bf16(a1[0], a1[1], a1[2], a1[3]);
      *reinterpret_cast<uint2 *>(&kv_layer[kv_elem(geo, page, head - Hq - Hkv, 1, off, half + p)]) = pack4_bf16(a2[0], a2[1], a2[2], a2[3]);
    }
    return;
  }
  const __nv_bfloat16 *nw = is_q ? q_norm : k_norm;
  if (nw) {                                                // per-head RMSNorm (warp-uniform branch)
    float ss = 0.f;
#pragma unroll
    for (int e = 0; e < 4; ++e) ss += a1[e] * a1[e] + a2[e] * a2[e];
    ss = warp_sum(ss);
    const float r = 1.0f / sqrtf(ss / hd + eps);
    if (act) {
#pragma unroll
      for (int e = 0; e < 4; ++e) { a1[e] *= r * __bfloat162float(nw[p + e]); a2[e] *= r * __bfloat162float(nw[half + p + e]); }
    }
  }
  if (!act) return;
  const float4 *tp = reinterpret_cast<const float4 *>(cs + (size_t)slot * half + p);   // (cos, sin) of pairs p .. p+3: two 16-byte loads
  const float4 t01 = tp[0], t23 = tp[1];
  const float co[4] = {t01.x, t01.z, t23.x, t23.z}, si[4] = {t01.y, t01.w, t23.y, t23.w};
  float y1[4], y2[4];
#pragma unroll
  for (int e = 0; e < 4; ++e) { y1[e] = a1[e] * co[e] - a2[e] * si[e]; y2[e] = a2[e] * co[e] + a1[e] * si[e]; }
  const uint2 o1 = pack4_bf16(y1[0], y1[1], y1[2], y1[3]), o2 = pack4_bf16(y2[0], y2[1], y2[2], y2[3]);
  if (is_q) {
    __nv_bfloat16 *qdst = q_out + (size_t)slot * Hq * hd + (size_t)head * hd;
    *reinterpret_cast<uint2 *>(qdst + p) = o1;
    *reinterpret_cast<uint2 *>(qdst + half + p) = o2;
  } else {
    *reinterpret_cast<uint2 *>(&kv_layer[kv_elem(geo, page, head - Hq, 0, off, p)]) = o1;
    *reinterpret_cast<uint2 *>(&kv_layer[kv_elem(geo, page, head - Hq, 0, off, half + p)]) = o2;
  }
}

// ---- one-CTA-per-row forms (round 2, profiles/r2_consumers.md): every thread issues ALL the loads of its element — up to eight pieces —
// before the first add.  The sums are still piece 0 + piece 1 + ... in slot order.

// Up to NP pieces of one float4, all in flight together (np > NP: further rounds of NP)
template <int NP>
__device__ __forceinline__ float4 sk_sum4_wide(const float4 *p, size_t st, int np) {
  float4 a = make_float4(0.f, 0.f, 0.f, 0.f);
  for (int s0 = 0; s0 < np; s0 += NP) {
    float4 y[NP];
#pragma unroll
    for (int s = 0; s < NP; ++s)
      if (s0 + s < np) y[s] = __ldg(p + (size_t)(s0 + s) * st);
#pragma unroll
    for (int s = 0; s < NP; ++s)
      if (s0 + s < np) { a.x += y[s].x; a.y += y[s].y; a.z += y[s].z; a.w += y[s].w; }
  }
  return a;
}

// h[slot] += pieces;  out = rmsnorm(h[slot]) * w.   One CTA per slot, ONE float4 per thread (blockDim >= d / 4, d <= 4096).
__global__ void __launch_bounds__(1024) add_rmsnorm_sk_wide_k(float *__restrict__ h, SkView v, const __nv_bfloat16 *__restrict__ w,
                                                             __nv_bfloat16 *__restrict__ out, int d, float eps, const int32_t *n_rows_dev,
                                                             int rows_ub) {
  pdl_trigger();
  const int slot = blockIdx.x, k = threadIdx.x, live = live_rows(n_rows_dev, rows_ub);   // the row count is fixed for the step
  const bool ok = k < d / 4;
  float2 w0 = make_float2(0.f, 0.f), w1 = w0;
  if (ok) {                                                  // weights do not depend on the previous kernel
    const __nv_bfloat162 *wp = reinterpret_cast<const __nv_bfloat162 *>(w + 4 * k);
    w0 = __bfloat1622float2(wp[0]);
    w1 = __bfloat1622float2(wp[1]);
  }
  pdl_wait();
  if (slot >= live) return;
  const int rbr = sk_view_rb_rows(v, live), n_rb = (live + rbr - 1) / rbr;
  float4 x = make_float4(0.f, 0.f, 0.f, 0.f);
  float4 *hr = reinterpret_cast<float4 *>(h + (size_t)slot * d);
  if (ok) {
    x = hr[k];
    const float4 a = sk_sum4_wide<8>(reinterpret_cast<const float4 *>(v.part + (size_t)slot * d) + k, v.slot_stride / 4,
                                     sk_npieces(v, n_rb, rbr, 4 * k, slot));
    x.x += a.x; x.y += a.y; x.z += a.z; x.w += a.w;
    hr[k] = x;
  }
  // sum of squares in the ORDER of add_rmsnorm_sk_k (256 partial sums over k = t, t + 256, ..., then the warp tree, then the eight warps):
  // the two kernels are chosen on the host's row bound, which may lag the live count, so they must agree to the bit
  __shared__ float e[1024], red[32];
  e[k] = x.x * x.x + x.y * x.y + x.z * x.z + x.w * x.w;
  __syncthreads();
  if (threadIdx.x < 256) {
    float ss = 0.f;
    for (int q = threadIdx.x; q < d / 4; q += 256) ss += e[q];
    ss = warp_sum(ss);
    if ((threadIdx.x & 31) == 0) red[threadIdx.x >> 5] = ss;
  }
  __syncthreads();
  if (threadIdx.x < 32) {
    float t = threadIdx.x < 8 ? red[threadIdx.x] : 0.f;
    t = warp_sum(t);
    if (threadIdx.x == 0) red[0] = t;
  }
  __syncthreads();
  const float r = 1.0f / sqrtf(red[0] / d + eps);
  if (ok) *reinterpret_cast<uint2 *>(out + (size_t)slot * d + 4 * k) = pack4_bf16(x.x * r * w0.x, x.y * r * w0.y, x.z * r * w1.x, x.w * r * w1.y);
}

// (QK-norm) + RoPE + KV append, one CTA per slot: thread = (head, j) with j < hd / 8 owning elements 4j..4j+3 of both rotate-half halves
// (hd in {64, 128, 256}: 8, 16 or 32 threads per head, a head never straddles a warp).
__global__ void __launch_bounds__(768) rope_append_sk_row_k(SkView v, __nv_bfloat16 *__restrict__ q_out, __nv_bfloat16 *__restrict__ kv_layer,
                                                            const int32_t *__restrict__ slot_dst_page, const int32_t *__restrict__ slot_dst_off,
                                                            const float2 *__restrict__ cs, const __nv_bfloat16 *__restrict__ q_norm,
                                                            const __nv_bfloat16 *__restrict__ k_norm, int Hq, int Hkv, int hd, int lph_shift, float eps,
                                                            KvGeom geo, const int32_t *n_rows_dev, int rows_ub) {
  pdl_trigger();
  const int slot = blockIdx.x, live = live_rows(n_rows_dev, rows_ub);
  const int head = threadIdx.x >> lph_shift, j = threadIdx.x & ((1 << lph_shift) - 1);
  const int half = hd >> 1, col0 = head * hd, p = 4 * j;
  const bool is_q = head < Hq, is_v = head >= Hq + Hkv;
  if (slot >= live) return;                                // the row count and the append targets were fixed at the step boundary
  const int page = slot_dst_page[slot], off = slot_dst_off[slot];
  const bool act = head < Hq + 2 * Hkv && (is_q || page >= 0);
  pdl_wait();
  const int rbr = sk_view_rb_rows(v, live), n_rb = (live + rbr - 1) / rbr;
  float4 x1 = make_float4(0.f, 0.f, 0.f, 0.f), x2 = x1, t01 = x1, t23 = x1;
  if (act) {
    const float4 *pp = reinterpret_cast<const float4 *>(v.part + (size_t)slot * (Hq + 2 * Hkv) * hd + col0 + p);
    const int np1 = sk_npieces(v, n_rb, rbr, col0 + p, slot), np2 = sk_npieces(v, n_rb, rbr, col0 + half + p, slot);
    if (!is_v) {
      const float4 *tp = reinterpret_cast<const float4 *>(cs + (size_t)slot * half + p);   // (cos, sin) of pairs p .. p+3
      t01 = tp[0];
      t23 = tp[1];
    }
    const size_t st = v.slot_stride / 4;
    float4 y1[4], y2[4];                                    // a QKV tile has 2-3 pieces (48 weight tiles on 148 CTAs): one round
#pragma unroll
    for (int s = 0; s < 4; ++s) {
      if (s < np1) y1[s] = __ldg(pp + s * st);
      if (s < np2) y2[s] = __ldg(pp + half / 4 + s * st);
    }
#pragma unroll
    for (int s = 0; s < 4; ++s) {
      if (s < np1) { x1.x += y1[s].x; x1.y += y1[s].y; x1.z += y1[s].z; x1.w += y1[s].w; }
      if (s < np2) { x2.x += y2[s].x; x2.y += y2[s].y; x2.z += y2[s].z; x2.w += y2[s].w; }
    }
    if (np1 > 4) { const float4 a = sk_sum4_wide<4>(pp + 4 * st, st, np1 - 4); x1.x += a.x; x1.y += a.y; x1.z += a.z; x1.w += a.w; }
    if (np2 > 4) { const float4 a = sk_sum4_wide<4>(pp + half / 4 + 4 * st, st, np2 - 4); x2.x += a.x; x2.y += a.y; x2.z += a.z; x2.w += a.w; }
  }
  float a1[4] = {x1.x, x1.y, x1.z, x1.w}, a2[4] = {x2.x, x2.y, x2.z, x2.w};
  if (is_v) {
    if (act) {
      *reinterpret_cast<uint2 *>(&kv_layer[kv_elem(geo, page, head - Hq - Hkv, 1, off, p)]) = pack4_bf16(a1[0], a1[1], a1[2], a1[3]);
      *reinterpret_cast<uint2 *>(&kv_layer[kv_elem(geo, page, head - Hq - Hkv, 1, off, half + p)]) = pack4_bf16(a2[0], a2[1], a2[2], a2[3]);
    }
  }
  const bool rot = act && !is_v;
  if (q_norm) {                                            // per-head RMSNorm over the head's 1 << lph_shift lanes (every lane of the warp takes the shuffles)
    const __nv_bfloat16 *nw = is_q ? q_norm : k_norm;
    float ss = 0.f;
#pragma unroll
    for (int e = 0; e < 4; ++e) ss += a1[e] * a1[e] + a2[e] * a2[e];
    for (int o = (1 << lph_shift) >> 1; o > 0; o >>= 1) ss += __shfl_xor_sync(0xffffffffu, ss, o);
    const float r = 1.0f / sqrtf(ss / hd + eps);
    if (rot) {
#pragma unroll
      for (int e = 0; e < 4; ++e) { a1[e] *= r * __bfloat162float(nw[p + e]); a2[e] *= r * __bfloat162float(nw[half + p + e]); }
    }
  }
  if (!rot) return;
  const float co[4] = {t01.x, t01.z, t23.x, t23.z}, si[4] = {t01.y, t01.w, t23.y, t23.w};
  float y1[4], y2[4];
#pragma unroll
  for (int e = 0; e < 4; ++e) { y1[e] = a1[e] * co[e] - a2[e] * si[e]; y2[e] = a2[e] * co[e] + a1[e] * si[e]; }
  const uint2 o1 = pack4_bf16(y1[0], y1[1], y1[2], y1[3]), o2 = pack4_bf16(y2[0], y2[1], y2[2], y2[3]);
  if (is_q) {
    __nv_bfloat16 *qdst = q_out + (size_t)slot * Hq * hd + (size_t)head * hd;
    *reinterpret_cast<uint2 *>(qdst + p) = o1;
    *reinterpret_cast<uint2 *>(qdst + half + p) = o2;
  } else {
    *reinterpret_cast<uint2 *>(&kv_layer[kv_elem(geo, page, head - Hq, 0, off, p)]) = o1;
    *reinterpret_cast<uint2 *>(&kv_layer[kv_elem(geo, page, head - Hq, 0, off, half + p)]) = o2;
  }
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

darts_status launch_gather_rows_bf16(darts_ctx *c, const void *src, void *dst, int tok_begin, int g_begin, int g_end) {
  gather_rows_bf16_k<<<g_end - g_begin, 256, 0, c->stream>>>((const __nv_bfloat16 *)src, (__nv_bfloat16 *)dst, c->g_tok_off, tok_begin, g_begin,
                                                             c->m.d_model);
  return post(c, "gather_rows_bf16");
}

darts_status launch_sum_partials(darts_ctx *c, const float *part, float *out, int S, size_t n) {
  sum_partials_k<<<(unsigned)((n + 255) / 256), 256, 0, c->stream>>>(part, out, S, n);
  return post(c, "sum_partials");
}

darts_status launch_add_rmsnorm_sk(darts_ctx *c, const SkView &v, const void *w, int rows_ub, const int32_t *n_rows_dev) {
  if (rows_ub <= 0) return DARTS_OK;
  const int d = c->m.d_model;
  const __nv_bfloat16 *wn = (const __nv_bfloat16 *)w;
  __nv_bfloat16 *xn = (__nv_bfloat16 *)c->xn;
  // Up to 128 rows (measured cross-over: profiles/r2_consumers.md) one float4 per thread with every load of the row in flight at once; above,
  // 256 threads walk the row (more rows resident per SM).  Same bits either way.
  if (rows_ub <= 128 && d / 4 <= 1024 && d / 4 >= 256) launch_pdl(c, add_rmsnorm_sk_wide_k, dim3(rows_ub), dim3((d / 4 + 31) & ~31), 0, c->h, v, wn, xn, d, c->m.rms_eps, n_rows_dev, rows_ub);
  else launch_pdl(c, add_rmsnorm_sk_k, dim3(rows_ub), dim3(256), 0, c->h, v, wn, xn, d, c->m.rms_eps, n_rows_dev, rows_ub);
  return post(c, "add_rmsnorm_sk");
}

darts_status launch_silu_mul_sk(darts_ctx *c, const SkView &v, int rows_ub, const int32_t *n_rows_dev) {
  if (rows_ub <= 0) return DARTS_OK;
  int F = c->m.ffn;
  launch_pdl(c, silu_mul_sk_k, dim3((F / 4 + 255) / 256, rows_ub), dim3(256), 0, v, (__nv_bfloat16 *)c->act, F, n_rows_dev, rows_ub);
  return post(c, "silu_mul_sk");
}

darts_status launch_rope_append_sk(darts_ctx *c, int layer, const SkView &v, int rows_ub, const int32_t *n_rows_dev) {
  if (rows_ub <= 0) return DARTS_OK;
  using T = __nv_bfloat16;
  const int nh = c->m.n_q_heads + 2 * c->m.n_kv_heads, hd = c->m.head_dim;
  T *kv = (T *)c->kv_pool + (size_t)layer * c->kv_layer_elems;
  const T *qn = c->m.qk_norm ? (const T *)c->q_norm[layer] : nullptr, *kn = c->m.qk_norm ? (const T *)c->k_norm[layer] : nullptr;
  const int lph = hd / 8;                                  // threads per head
  if ((hd == 64 || hd == 128 || hd == 256) && nh * lph <= 768) {
    const int lph_shift = hd == 64 ? 3 : hd == 128 ? 4 : 5;
    launch_pdl(c, rope_append_sk_row_k, dim3(rows_ub), dim3((nh * lph + 31) & ~31), 0, v, (T *)c->q, kv, c->slot_dst_page, c->slot_dst_off, c->slot_cs, qn, kn,
               c->m.n_q_heads, c->m.n_kv_heads, hd, lph_shift, c->m.rms_eps, c->geom(), n_rows_dev, rows_ub);
  } else {
    launch_pdl(c, rope_append_sk_k, dim3((nh + 3) / 4, rows_ub), dim3(128), 0, v, (T *)c->q, kv, c->slot_dst_page, c->slot_dst_off, c->slot_cs, qn, kn,
               c->m.n_q_heads, c->m.n_kv_heads, hd, c->m.rms_eps, c->geom(), n_rows_dev, rows_ub);
  }
  return post(c, "rope_append_sk");
}
