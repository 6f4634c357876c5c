// tcgen05 / TMEM tile GEMM (the LM head with its fused sampling epilogue; also the prefill logits and the
// split-K parity hook):   P[s][r][n] = sum_{k in split s} X[r][k] W[n][k].   The layer projections run on kernels_gemm_sk.cu.
//
// One CTA computes a 128 (activation rows) x BN (weight rows) tile of one K-split:
//   warp 0   TMA producer: per 64-wide k-block one box of W (BN x 64, 128-byte swizzle) and ceil(live rows / 16) boxes
//            of X (16 x 64) into a STAGES-deep shared-memory ring, completion on mbarriers (expect_tx);
//   warp 1   allocates TMEM, one lane issues tcgen05.mma (M=128, N=BN, K=16; A and B from shared memory through
//            UMMA descriptors, fp32 accumulator in TMEM) and commits each stage back to the producer;
//   warps 2-5 epilogue: tcgen05.ld the accumulator (lane = activation row, column = weight row) and either store the
//            fp32 partial, or (LM head) apply temperature + Philox Gumbel noise and keep a per-row running top-2, so
//            the logits never reach HBM (SURVEY.md §7 hard part 1).
// Decode GEMMs are weight-streaming (HBM-bound) below ~250 active rows: the grid is filled by splitting K
// (deterministic: every split writes its own partial, the consumer kernel adds them in split order).  Rows of the
// 128-row MMA tile beyond the live row count hold stale shared memory; they only produce their own (never stored) rows.
#include "internal.cuh"
#include "philox.cuh"
#include "sm100_ptx.cuh"

namespace {

using namespace ptx;

constexpr int BM = 128, BK = 64;
constexpr int A_BOX_ROWS = 16;
constexpr int A_STAGE_BYTES = BM * BK * 2;       // 16 KB
constexpr int GEMM_THREADS = 192;

enum { EPI_STORE = 0, EPI_SAMPLE = 1 };

struct GemmParams {
  float *C;                       // EPI_STORE: partial base [S][c_rows][N]
  size_t split_stride;            // elements between consecutive splits
  int N, K, S;
  int rows_ub;
  const int32_t *n_rows_dev;      // live row count on the device (nullable)
  // EPI_SAMPLE
  float4 *top2;                   // [n_tiles][rows] (best y, second y, bits(best index), z/T of the best)
  float2 *lse;                    // [n_tiles][rows] (max, sum e^(z/T - max)) over the tile: log-probability of the drawn token
  float *logits_dump;             // optional [rows][N]
  const int32_t *row_list, *row_prompt, *row_sample, *row_len;
  float temperature;
  uint32_t k0, k1;
};

template <int BN, int STAGES>
struct GemmSmem {
  alignas(1024) unsigned char a[STAGES][A_STAGE_BYTES];
  alignas(1024) unsigned char b[STAGES][BN * BK * 2];
  unsigned long long full[STAGES], empty[STAGES], acc_full;
  uint32_t tmem_base;
};

template <int BN, int STAGES, int EPI>
__global__ void __launch_bounds__(GEMM_THREADS) gemm_tc_k(const __grid_constant__ CUtensorMap tmA, const __grid_constant__ CUtensorMap tmB,
                                                          GemmParams p) {
  extern __shared__ unsigned char smem_raw[];
  using Smem = GemmSmem<BN, STAGES>;
  Smem &sm = *reinterpret_cast<Smem *>(((uintptr_t)smem_raw + 1023) & ~(uintptr_t)1023);
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int split = blockIdx.z;

  // ---- which rows does this tile cover? (uniform over the CTA; exit before any barrier / TMEM allocation)
  int row_begin, row_end;
  row_begin = 0;
  row_end = p.n_rows_dev ? min(*p.n_rows_dev, p.rows_ub) : p.rows_ub;
  const int m0 = row_begin + blockIdx.x * BM;             // row tiles vary fastest: the CTAs that share a weight tile run together (L2 reuse)
  if (m0 >= row_end) return;
  const int live = min(BM, row_end - m0);                // live rows of this tile
  const int n0 = blockIdx.y * BN;
  const int nkb = p.K / BK;
  const int kb0 = (int)((long long)split * nkb / p.S), kb1 = (int)((long long)(split + 1) * nkb / p.S);

  if (threadIdx.x == 0) {
    prefetch_tmap(&tmA);
    prefetch_tmap(&tmB);
    for (int s = 0; s < STAGES; ++s) { mbar_init(&sm.full[s], 1); mbar_init(&sm.empty[s], 1); }
    mbar_init(&sm.acc_full, 1);
    fence_mbar_init();
  }
  if (warp == 1) tmem_alloc(&sm.tmem_base, BN);
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  const uint32_t tmem = sm.tmem_base;

  if (warp == 0) {
    // ------------------------------------------------------------------------------------------ TMA producer
    if (lane == 0) {
      const int nbox = (live + A_BOX_ROWS - 1) / A_BOX_ROWS;
      const int tx = nbox * (A_BOX_ROWS * BK * 2) + BN * BK * 2;
      const int brow = n0;
      int stage = 0, phase = 0;
      for (int kb = kb0; kb < kb1; ++kb) {
        mbar_wait(&sm.empty[stage], phase ^ 1);
        mbar_expect_tx(&sm.full[stage], tx);
        tma_load_2d_hint(sm.b[stage], &tmB, kb * BK, brow, &sm.full[stage], HINT_EVICT_FIRST);      // weights: streamed once
        for (int bx = 0; bx < nbox; ++bx)
          tma_load_2d_hint(sm.a[stage] + bx * (A_BOX_ROWS * BK * 2), &tmA, kb * BK, m0 + bx * A_BOX_ROWS, &sm.full[stage], HINT_EVICT_LAST);
        if (++stage == STAGES) { stage = 0; phase ^= 1; }
      }
    }
  } else if (warp == 1) {
    // ------------------------------------------------------------------------------------------ MMA issuer
    if (lane == 0) {
      constexpr uint32_t idesc = umma_idesc_bf16(BM, BN);
      int stage = 0, phase = 0;
      for (int kb = kb0; kb < kb1; ++kb) {
        mbar_wait(&sm.full[stage], phase);
        tc_fence_after();
        const uint64_t da = umma_desc_sw128(smem_u32(sm.a[stage])), db = umma_desc_sw128(smem_u32(sm.b[stage]));
#pragma unroll
        for (int k = 0; k < BK / 16; ++k)       // +32 bytes (2 x 16-byte units) per K=16 step inside the 128-byte swizzle row
          mma_bf16_ss(tmem, da + 2 * k, db + 2 * k, idesc, (kb > kb0 || k > 0) ? 1u : 0u);
        mma_commit(&sm.empty[stage]);
        if (++stage == STAGES) { stage = 0; phase ^= 1; }
      }
      mma_commit(&sm.acc_full);
    }
  } else {
    // ------------------------------------------------------------------------------------------ epilogue
    const int q = warp & 3;                                // TMEM lane quadrant this warp may read
    const int r_local = q * 32 + lane;
    mbar_wait(&sm.acc_full, 0);
    tc_fence_after();
    if (q * 32 < live) {                                   // warp-uniform: skip quadrants with no live row
      const bool row_ok = r_local < live;
      const int r = m0 + r_local;
      if constexpr (EPI == EPI_STORE) {
        float *dst = p.C + (size_t)split * p.split_stride + (size_t)r * p.N + n0;
#pragma unroll 1
        for (int c = 0; c < BN; c += 32) {
          uint32_t v[32];
          tmem_ld32(tmem + ((uint32_t)(q * 32) << 16) + c, v);
          tmem_ld_wait();
          if (row_ok) {
#pragma unroll
            for (int j = 0; j < 32; j += 4)
              if (n0 + c + j < p.N)
                *reinterpret_cast<float4 *>(dst + c + j) = make_float4(__uint_as_float(v[j]), __uint_as_float(v[j + 1]), __uint_as_float(v[j + 2]), __uint_as_float(v[j + 3]));
          }
        }
      } else {
        // fused temperature + Gumbel-max: y_v = z_v / T + g_v, running (best, second, argbest) over this tile's BN vocab ids
        int pi = 0, pj = 0, ps = 0;
        if (row_ok) {
          int row = p.row_list[r];
          pi = p.row_prompt[row]; pj = p.row_sample[row]; ps = p.row_len[row];
        }
        float b1 = -INFINITY, b2 = -INFINITY, z1 = 0.f;
        int i1 = 0x7fffffff;
        float lm = -INFINITY, ls = 0.f;
#pragma unroll 1
        for (int c = 0; c < BN; c += 32) {
          uint32_t v[32];
          tmem_ld32(tmem + ((uint32_t)(q * 32) << 16) + c, v);
          tmem_ld_wait();
          if (row_ok) {
            if (p.logits_dump) {
#pragma unroll
              for (int j = 0; j < 32; j += 4)
                if (n0 + c + j < p.N)
                  *reinterpret_cast<float4 *>(p.logits_dump + (size_t)r * p.N + n0 + c + j) =
                      make_float4(__uint_as_float(v[j]), __uint_as_float(v[j + 1]), __uint_as_float(v[j + 2]), __uint_as_float(v[j + 3]));
            }
#pragma unroll
            for (int j = 0; j < 32; j += 4) {
              const int vid = n0 + c + j;                    // multiple of 4: one Philox block serves 4 vocab ids
              if (vid < p.N) {
                uint32_t x[4];
                if (p.temperature != 0.f) philox4x32_10((uint32_t)(vid >> 2), (uint32_t)ps, (uint32_t)pj, (uint32_t)pi, p.k0, p.k1, x);
                float zt[4];
#pragma unroll
                for (int e = 0; e < 4; ++e) {
                  float z = __uint_as_float(v[j + e]);
                  zt[e] = p.temperature != 0.f ? z / p.temperature : z;
                  float y = p.temperature != 0.f ? zt[e] + gumbel_from_bits(x[e]) : z;
                  if (y > b1) { b2 = b1; b1 = y; i1 = vid + e; z1 = zt[e]; }       // ids ascend: strict > keeps the lowest id on ties
                  else if (y > b2) b2 = y;
                }
                float mn = fmaxf(fmaxf(lm, fmaxf(zt[0], zt[1])), fmaxf(zt[2], zt[3]));     // running log-sum-exp of z / T, four at a time
                ls = ls * __expf(lm - mn) + ((__expf(zt[0] - mn) + __expf(zt[1] - mn)) + (__expf(zt[2] - mn) + __expf(zt[3] - mn)));
                lm = mn;
              }
            }
          }
        }
        if (row_ok) {
          p.top2[(size_t)blockIdx.y * p.rows_ub + r] = make_float4(b1, b2, __int_as_float(i1), z1);
          p.lse[(size_t)blockIdx.y * p.rows_ub + r] = make_float2(lm, ls);
        }
      }
    }
  }
  tc_fence_before();
  __syncthreads();
  if (warp == 1) tmem_dealloc(tmem, BN);
}

// ---- tensor maps ------------------------------------------------------------------------------------------------------
typedef CUresult (*EncodeTiledFn)(CUtensorMap *, CUtensorMapDataType, cuuint32_t, void *, const cuuint64_t *, const cuuint64_t *,
                                  const cuuint32_t *, const cuuint32_t *, CUtensorMapInterleave, CUtensorMapSwizzle,
                                  CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

EncodeTiledFn encode_fn() {
  static EncodeTiledFn fn = nullptr;
  if (!fn) {
    void *p = nullptr;
    cudaDriverEntryPointQueryResult q;
    if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &p, cudaEnableDefault, &q) == cudaSuccess && q == cudaDriverEntryPointSuccess)
      fn = (EncodeTiledFn)p;
  }
  return fn;
}

template <int BN, int STAGES, int EPI>
darts_status launch_cfg(darts_ctx *c, const CUtensorMap &a, const CUtensorMap &b, const GemmParams &p, dim3 grid) {
  size_t smem = sizeof(GemmSmem<BN, STAGES>) + 1024;
  gemm_tc_k<BN, STAGES, EPI><<<grid, GEMM_THREADS, smem, c->stream>>>(a, b, p);
  c->launches++;
  cudaError_t e = cudaGetLastError();
  if (e != cudaSuccess) {
    snprintf(c->err, sizeof(c->err), "launch gemm_tc: %s", cudaGetErrorString(e));
    c->sticky = DARTS_ERR_CUDA;
    return DARTS_ERR_CUDA;
  }
  return DARTS_OK;
}

}  // namespace

// bf16 [rows][K] row-major matrix -> 2-D tensor map with a (box_rows x 64) box and the 128-byte swizzle.
darts_status tc_make_map(darts_ctx *c, CUtensorMap *out, const void *base, long long rows, int K, int box_rows) {
  EncodeTiledFn fn = encode_fn();
  if (!fn) FAIL(c, DARTS_ERR_CUDA, "cuTensorMapEncodeTiled entry point not found");
  if (K % 8 || ((uintptr_t)base & 15)) FAIL(c, DARTS_ERR_INVALID_ARG, "tensor map needs 16-byte aligned rows (K=%d)", K);
  cuuint64_t dims[2] = {(cuuint64_t)K, (cuuint64_t)rows};
  cuuint64_t strides[1] = {(cuuint64_t)K * 2};
  cuuint32_t box[2] = {(cuuint32_t)BK, (cuuint32_t)box_rows};
  cuuint32_t estr[2] = {1, 1};
  CUresult r = fn(out, CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, 2, const_cast<void *>(base), dims, strides, box, estr, CU_TENSOR_MAP_INTERLEAVE_NONE,
                  CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_256B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
  if (r != CUDA_SUCCESS) FAIL(c, DARTS_ERR_CUDA, "cuTensorMapEncodeTiled failed (%d) rows=%lld K=%d", (int)r, rows, K);
  return DARTS_OK;
}

darts_status tc_make_xmaps(darts_ctx *c, XMaps *out, const void *base, long long rows, int K) {
  for (int b = 0; b < 5; ++b) {
    darts_status s = tc_make_map(c, &out->m[b], base, rows, K, 16 << b);
    if (s != DARTS_OK) return s;
  }
  return DARTS_OK;
}

darts_status gemm_tc_configure(darts_ctx *c) {
  CUDA_TRY(c, cudaFuncSetAttribute(gemm_tc_k<128, 3, EPI_STORE>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sizeof(GemmSmem<128, 3>) + 1024));
  CUDA_TRY(c, cudaFuncSetAttribute(gemm_tc_k<128, 2, EPI_SAMPLE>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sizeof(GemmSmem<128, 2>) + 1024));
  return DARTS_OK;
}

bool tc_shape_ok(int N, int K) { return K % BK == 0 && K >= BK && N % 4 == 0; }

darts_status launch_gemm_tc(darts_ctx *c, const TcGemm &g) {
  if (g.rows_ub <= 0) return DARTS_OK;
  GemmParams p{};
  p.C = g.C; p.split_stride = g.split_stride; p.N = g.N; p.K = g.K; p.S = g.S; p.rows_ub = g.rows_ub; p.n_rows_dev = g.n_rows_dev;
  dim3 grid((g.rows_ub + BM - 1) / BM, (g.N + 127) / 128, g.S);
  if (!g.sample) return launch_cfg<128, 3, EPI_STORE>(c, *g.a_map, *g.b_map, p, grid);
  p.top2 = (float4 *)c->top2; p.lse = (float2 *)c->lse; p.logits_dump = (c->rt.flags & DARTS_FLAG_DUMP_LOGITS) ? c->logits : nullptr;
  p.row_list = c->row_list; p.row_prompt = c->row_prompt; p.row_sample = c->row_sample; p.row_len = c->row_len;
  p.temperature = c->temperature; p.k0 = (uint32_t)(c->seed & 0xffffffffu); p.k1 = (uint32_t)(c->seed >> 32);
  // Sampling on this kernel is the A/B path (DARTS_FLAG_LM_HEAD_TILES); the decode LM head runs on gemm_sk_k<SK_EPI_SAMPLE>.
  // Two stages (65 KB): three CTAs per SM, so one CTA's sampling epilogue and pipeline ramp hide behind two others' loads.  Measured on the
  // non-layer part of a c3 step (LM head + boundary kernels) at 16 / 288 / 512 rows: 0.47 / 1.03 / 1.37 ms with 3 stages (2 CTAs per SM),
  // 0.43 / 0.91 / 1.17 ms with 2, 0.59 / 1.51 / 2.10 ms with 4 (1 CTA per SM); a 32-row activation slot (more stages in the same
  // shared memory) changed nothing: the tile kernel at few rows is bound by its 128-row MMA, not by bytes in flight.
  return launch_cfg<128, 2, EPI_SAMPLE>(c, *g.a_map, *g.b_map, p, grid);
}
