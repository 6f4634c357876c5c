// Temperature + Philox Gumbel-max sampling over a row of fp32 logits, fused with EOS / forced-stop /
// length update.  DESIGN.md R4: counter = (v>>2, step, sample, prompt),
// key = (seed_lo, seed_hi), lane v&3, u = ((x>>9)+0.5)*2^-23, g = -ln(-ln u); ties -> lowest v.
#include "internal.cuh"
#include "philox.cuh"

namespace {

struct Top2 {
  float b1, b2;
  int i1;
  float z1;                     // z / T of the best entry (its log-probability = z1 - logsumexp)
};
// running log-sum-exp of z / T: sum = s * e^m
struct Lse {
  float m, s;
};
__device__ __forceinline__ void lse_push4(Lse &a, float z0, float z1, float z2, float z3) {
  float mn = fmaxf(fmaxf(a.m, fmaxf(z0, z1)), fmaxf(z2, z3));
  a.s = a.s * __expf(a.m - mn) + ((__expf(z0 - mn) + __expf(z1 - mn)) + (__expf(z2 - mn) + __expf(z3 - mn)));
  a.m = mn;
}
__device__ __forceinline__ Lse lse_merge(const Lse &a, const Lse &b) {
  if (b.m == -INFINITY) return a;
  if (a.m == -INFINITY) return b;
  float mn = fmaxf(a.m, b.m);
  return Lse{mn, a.s * __expf(a.m - mn) + b.s * __expf(b.m - mn)};
}

__device__ __forceinline__ bool better(float y, int i, float yb, int ib) { return y > yb || (y == yb && i < ib); }

__device__ __forceinline__ void top2_push(Top2 &t, float y, int i, float z) {
  if (better(y, i, t.b1, t.i1)) { t.b2 = t.b1; t.b1 = y; t.i1 = i; t.z1 = z; }
  else if (y > t.b2) t.b2 = y;
}

__device__ __forceinline__ Top2 top2_merge(const Top2 &a, const Top2 &b) {
  Top2 r;
  if (better(a.b1, a.i1, b.b1, b.i1)) { r.b1 = a.b1; r.i1 = a.i1; r.z1 = a.z1; r.b2 = fmaxf(a.b2, b.b1); }
  else { r.b1 = b.b1; r.i1 = b.i1; r.z1 = b.z1; r.b2 = fmaxf(b.b2, a.b1); }
  return r;
}

// Stop rules in the order of SURVEY.md §8(c) step 5, bookkeeping of the sampled token (one thread per row).
__device__ __forceinline__ void finish_row(DevState *st, int row, int slot, int s, const Top2 &t, const Lse &l, int32_t *row_len,
                                           uint8_t *row_status, const int32_t *row_forced, int32_t *row_last_tok, int32_t *row_slot,
                                           int32_t *row_slot_step, int32_t *tokens_out, float *margin_out, float *logprob_out,
                                           int max_new_stride, int max_len, int eos_id) {
  int tok = t.i1 == 0x7fffffff ? 0 : t.i1;              // every y was NaN (cannot happen with finite weights): stay inside the vocabulary
  float margin = t.b1 - t.b2;
  int len = s + 1;
  uint8_t status = DARTS_ROW_ACTIVE;
  if (row_forced[row] == len) { tok = eos_id; status = DARTS_ROW_VALID; }   // forced EOS (BASELINE.json workloads)
  else if (eos_id >= 0 && tok == eos_id) status = DARTS_ROW_VALID;          // natural EOS
  else if (len == max_len) status = DARTS_ROW_TRUNC;                        // length limit
  tokens_out[(size_t)row * max_new_stride + s] = tok;
  margin_out[(size_t)row * max_new_stride + s] = margin;
  logprob_out[(size_t)row * max_new_stride + s] = t.z1 - (l.m + logf(l.s));   // of the DRAWN token (a forced EOS replaces it afterwards)
  row_last_tok[row] = tok;
  row_len[row] = len;
  row_status[row] = status;
  row_slot[row] = slot;
  row_slot_step[row] = st->step;
  atomicAdd(&st->n_generated, 1ULL);
  if (margin < NEAR_TIE_MARGIN) atomicAdd(&st->n_near_ties, 1ULL);
}

__global__ void __launch_bounds__(256) sample_k(DevState *st, const float *__restrict__ logits, int V, int step0,
                                                const int32_t *__restrict__ row_list, const int32_t *__restrict__ row_prompt,
                                                const int32_t *__restrict__ row_sample, int32_t *row_len, uint8_t *row_status,
                                                const int32_t *__restrict__ row_forced, int32_t *row_last_tok, int32_t *row_slot,
                                                int32_t *row_slot_step, int32_t *tokens_out, float *margin_out, float *logprob_out,
                                                int max_new_stride, int max_len, int eos_id, float temperature, uint32_t k0, uint32_t k1) {
  int slot = blockIdx.x;
  if (slot >= st->n_active) return;
  int row = row_list[slot];
  int i = row_prompt[row], j = row_sample[row], s = row_len[row];
  const float *z = logits + (size_t)(step0 ? i : slot) * V;
  Top2 t{-INFINITY, -INFINITY, 0x7fffffff, 0.f};
  Lse l{-INFINITY, 0.f};
  int nv4 = (V + 3) >> 2;
  for (int v4 = threadIdx.x; v4 < nv4; v4 += blockDim.x) {
    uint32_t x[4];
    if (temperature != 0.f) philox4x32_10((uint32_t)v4, (uint32_t)s, (uint32_t)j, (uint32_t)i, k0, k1, x);
    float zt[4];
#pragma unroll
    for (int k = 0; k < 4; ++k) {
      int v = v4 * 4 + k;
      zt[k] = -INFINITY;
      if (v < V) {
        zt[k] = temperature != 0.f ? z[v] / temperature : z[v];
        float y = temperature != 0.f ? zt[k] + gumbel_from_bits(x[k]) : z[v];
        top2_push(t, y, v, zt[k]);
      }
    }
    lse_push4(l, zt[0], zt[1], zt[2], zt[3]);
  }
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) {
    Top2 u;
    u.b1 = __shfl_xor_sync(0xffffffffu, t.b1, o);
    u.b2 = __shfl_xor_sync(0xffffffffu, t.b2, o);
    u.i1 = __shfl_xor_sync(0xffffffffu, t.i1, o);
    u.z1 = __shfl_xor_sync(0xffffffffu, t.z1, o);
    t = top2_merge(t, u);
    Lse lu{__shfl_xor_sync(0xffffffffu, l.m, o), __shfl_xor_sync(0xffffffffu, l.s, o)};
    l = lse_merge(l, lu);
  }
  __shared__ Top2 red[8];
  __shared__ Lse redl[8];
  if ((threadIdx.x & 31) == 0) { red[threadIdx.x >> 5] = t; redl[threadIdx.x >> 5] = l; }
  __syncthreads();
  if (threadIdx.x == 0) {
    for (int w = 1; w < (int)(blockDim.x >> 5); ++w) { t = top2_merge(t, red[w]); l = lse_merge(l, redl[w]); }
    finish_row(st, row, slot, s, t, l, row_len, row_status, row_forced, row_last_tok, row_slot, row_slot_step, tokens_out, margin_out,
               logprob_out, max_new_stride, max_len, eos_id);
  }
}

// LM-head tensor-core path: the GEMM epilogue left one (best, second, argbest) per (vocab tile, slot); merge the tiles
// (max with lowest-id tie-break is order-independent) and apply the stop rules.
__global__ void __launch_bounds__(512) sample_finalize_k(DevState *st, const float4 *__restrict__ top2, const float2 *__restrict__ lse,
                                                         int n_tiles, int rows_ub,
                                                         const int32_t *__restrict__ row_list, int32_t *row_len, uint8_t *row_status,
                                                         const int32_t *__restrict__ row_forced, int32_t *row_last_tok, int32_t *row_slot,
                                                         int32_t *row_slot_step, int32_t *tokens_out, float *margin_out, float *logprob_out,
                                                         int max_new_stride, int max_len, int eos_id) {
  int slot = blockIdx.x;
  if (slot >= st->n_active) return;
  int row = row_list[slot];
  int s = row_len[row];
  Top2 t{-INFINITY, -INFINITY, 0x7fffffff, 0.f};
  Lse l{-INFINITY, 0.f};
#pragma unroll 4
  for (int k = threadIdx.x; k < n_tiles; k += blockDim.x) {      // independent loads: unrolled so several are in flight per thread
    float4 v = __ldcs(&top2[(size_t)k * rows_ub + slot]);
    float2 w = __ldcs(&lse[(size_t)k * rows_ub + slot]);
    Top2 u{v.x, v.y, __float_as_int(v.z), v.w};
    t = top2_merge(t, u);
    l = lse_merge(l, Lse{w.x, w.y});
  }
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) {
    Top2 u;
    u.b1 = __shfl_xor_sync(0xffffffffu, t.b1, o);
    u.b2 = __shfl_xor_sync(0xffffffffu, t.b2, o);
    u.i1 = __shfl_xor_sync(0xffffffffu, t.i1, o);
    u.z1 = __shfl_xor_sync(0xffffffffu, t.z1, o);
    t = top2_merge(t, u);
    Lse lu{__shfl_xor_sync(0xffffffffu, l.m, o), __shfl_xor_sync(0xffffffffu, l.s, o)};
    l = lse_merge(l, lu);
  }
  __shared__ Top2 red[16];
  __shared__ Lse redl[16];
  if ((threadIdx.x & 31) == 0) { red[threadIdx.x >> 5] = t; redl[threadIdx.x >> 5] = l; }
  __syncthreads();
  if (threadIdx.x == 0) {
    for (int w = 1; w < (int)(blockDim.x >> 5); ++w) { t = top2_merge(t, red[w]); l = lse_merge(l, redl[w]); }
    finish_row(st, row, slot, s, t, l, row_len, row_status, row_forced, row_last_tok, row_slot, row_slot_step, tokens_out, margin_out,
               logprob_out, max_new_stride, max_len, eos_id);
  }
}

}  // namespace

darts_status launch_sample(darts_ctx *c, const float *logits, int step0, int rows_ub) {
  if (rows_ub <= 0) return DARTS_OK;
  sample_k<<<rows_ub, 256, 0, c->stream>>>(c->st, logits, c->m.vocab, step0, c->row_list, c->row_prompt, c->row_sample, c->row_len,
                                           c->row_status, c->row_forced, c->row_last_tok, c->row_slot, c->row_slot_step, c->tokens_out,
                                           c->margin_out, c->logprob_out, c->rt.max_new, c->max_len, c->m.eos_id, c->temperature,
                                           (uint32_t)(c->seed & 0xffffffffu), (uint32_t)(c->seed >> 32));
  c->launches++;
  cudaError_t e = cudaGetLastError();
  if (e != cudaSuccess) {
    snprintf(c->err, sizeof(c->err), "launch sample: %s", cudaGetErrorString(e));
    c->sticky = DARTS_ERR_CUDA;
    return DARTS_ERR_CUDA;
  }
  return DARTS_OK;
}

darts_status launch_sample_finalize(darts_ctx *c, int n_tiles, int rows_ub) {
  if (rows_ub <= 0) return DARTS_OK;
  sample_finalize_k<<<rows_ub, 512, 0, c->stream>>>(c->st, (const float4 *)c->top2, (const float2 *)c->lse, n_tiles, rows_ub, c->row_list, c->row_len,
                                                    c->row_status, c->row_forced, c->row_last_tok, c->row_slot, c->row_slot_step, c->tokens_out,
                                                    c->margin_out, c->logprob_out, c->rt.max_new, c->max_len, c->m.eos_id);
  c->launches++;
  cudaError_t e = cudaGetLastError();
  if (e != cudaSuccess) {
    snprintf(c->err, sizeof(c->err), "launch sample_finalize: %s", cudaGetErrorString(e));
    c->sticky = DARTS_ERR_CUDA;
    return DARTS_ERR_CUDA;
  }
  return DARTS_OK;
}
