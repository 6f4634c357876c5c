// CTA-pair (tcgen05 cta_group::2) variant of the weight-streaming stream-K GEMM of kernels_gemm_sk.cu:
//     P[slot][r][n] = sum_{k in piece} X[r][k] W[n][k]
//
// Why: from ~256 live rows on the projections are bound by L2 -> SM operand traffic, not by the tensor pipe or HBM: one CTA per weight
// tile re-reads the whole activation block (256 rows x 64 k = 32 KB per k-block) for its 16 KB of weights (gate/up of config 3 at 512
// rows: 583 MB per launch against ~12 TB/s of L2).  Two CTAs of one cluster (an SM pair) issue ONE MMA of M = 256 weight rows:
// each CTA stages its own 128 weight rows and only HALF of the activation rows; the tensor cores read both halves.  Operand bytes per
// flop drop by a third (48 -> 32 KB per CTA and k-block), the ring gets deeper (32 KB stages), TMEM stays double-buffered.
//
// Layout of the work: a unit is (PAIR of weight tiles, 256-row block, 64-wide k-block); the units are cut into equal contiguous ranges,
// one per CTA pair (stream-K); pieces, slots and the piece-count table are exactly those of kernels_gemm_sk.cu, so the consumer kernels
// do not care which kernel produced them (SkView::rb512 = 0: this kernel never uses the 512-row bucket).
// Roles per CTA: warp 0 TMA producer (own weight tile + own half of the rows into its OWN shared memory), warp 1 MMA side, warps 2-5
// epilogue (each CTA drains the 128 accumulator lanes of its own weight tile).  Only the leader CTA (cluster rank 0) issues MMAs; the peer's
// warp 1 forwards "my stage s has landed" to the leader with a remote mbarrier arrive.  tcgen05.commit with a cluster multicast frees the
// stage in both CTAs and publishes the accumulator to both epilogues; the peer's epilogue releases the accumulator with remote arrives.
#include <algorithm>

#include "internal.cuh"
#include "sm100_ptx.cuh"

namespace {

using namespace ptx;

constexpr int BMW = 128, BK = 64;
constexpr int W_STAGE_BYTES = BMW * BK * 2;      // 16 KB: this CTA's weight tile of a k-block
constexpr int BOX_ROWS = 16, BOX_BYTES = BOX_ROWS * BK * 2;
constexpr int MAX_STAGES = 10;
constexpr int SK2_THREADS = 192;
constexpr int SMEM_BUDGET = 200 * 1024;

struct Sk2Params {
  float *C;
  size_t slot_stride;
  int N, nkb, n_wtiles, n_wpairs, rows_ub;
  const int32_t *n_rows_dev;
  int32_t *np_table;
  int unit_tile;
};

struct Sk2Bars {
  unsigned long long full[MAX_STAGES], peer_full[MAX_STAGES], empty[MAX_STAGES], acc_full[2], acc_empty[2];
  uint32_t tmem_base;
};

// ---- cluster / cta_group::2 PTX -------------------------------------------------------------------------------------------------
__device__ __forceinline__ uint32_t cluster_ctarank() {
  uint32_t r;
  asm volatile("mov.u32 %0, %%cluster_ctarank;" : "=r"(r));
  return r;
}
__device__ __forceinline__ void cluster_sync_all() {
  asm volatile("barrier.cluster.arrive.release.aligned;" ::: "memory");
  asm volatile("barrier.cluster.wait.acquire.aligned;" ::: "memory");
}
// address of the same shared-memory object in CTA `rank` of the cluster (shared::cluster window)
__device__ __forceinline__ uint32_t map_to_cta(const void *p, uint32_t rank) {
  uint32_t r;
  asm volatile("mapa.shared::cluster.u32 %0, %1, %2;" : "=r"(r) : "r"(smem_u32(p)), "r"(rank));
  return r;
}
// Plain (CTA-scope) arrive / wait semantics on purpose: what crosses the pair is written by TMA and read by the tensor cores (async proxy)
// or ordered by the tcgen05 fences; a cluster-scope acquire in the wait loop compiles to an L1 invalidate per poll (measured: the MMA
// thread then spends ~1 us per k-block in its waits and the kernel runs at half the speed of the single-CTA one).
__device__ __forceinline__ void mbar_arrive_remote(uint32_t cluster_addr) {
  asm volatile("mbarrier.arrive.shared::cluster.b64 _, [%0];" ::"r"(cluster_addr) : "memory");
}
__device__ __forceinline__ void mbar_wait_cluster(void *bar, int parity) { mbar_wait(bar, parity); }
__device__ __forceinline__ void tmem_alloc2(uint32_t *dst, int cols) {
  asm volatile("tcgen05.alloc.cta_group::2.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(smem_u32(dst)), "r"(cols) : "memory");
  asm volatile("tcgen05.relinquish_alloc_permit.cta_group::2.sync.aligned;" ::: "memory");
}
__device__ __forceinline__ void tmem_dealloc2(uint32_t taddr, int cols) {
  asm volatile("tcgen05.dealloc.cta_group::2.sync.aligned.b32 %0, %1;" ::"r"(taddr), "r"(cols) : "memory");
}
// D[tmem of both CTAs] (+)= A[256 rows: 128 per CTA, shared memory] . B[N rows: N/2 per CTA]^T; issued by ONE thread of the leader CTA
__device__ __forceinline__ void mma2_bf16_ss(uint32_t tmem_d, uint64_t desc_a, uint64_t desc_b, uint32_t idesc, uint32_t accumulate) {
  asm volatile(
      "{\n.reg .pred p;\n"
      "setp.ne.b32 p, %4, 0;\n"
      "tcgen05.mma.cta_group::2.kind::f16 [%0], %1, %2, %3, p;\n}" ::"r"(tmem_d),
      "l"(desc_a), "l"(desc_b), "r"(idesc), "r"(accumulate)
      : "memory");
}
// arrives on the barrier at this shared-memory offset in BOTH CTAs when all MMAs issued so far have completed
__device__ __forceinline__ void mma2_commit_both(void *bar) {
  asm volatile("tcgen05.commit.cta_group::2.mbarrier::arrive::one.shared::cluster.multicast::cluster.b64 [%0], %1;" ::"r"(smem_u32(bar)),
               "h"((uint16_t)3)
               : "memory");
}

struct Piece2 {
  int wpair, row0, nrows, kb0, kb1, slot, tile, npieces;
};
struct Piece2Iter {
  int u, u1, T, P, nkb, n_rb, unit_tile, pair, live;
  __device__ bool next(Piece2 &p) {
    if (u >= u1) return false;
    int tile = unit_tile ? u : u / nkb;
    p.kb0 = unit_tile ? 0 : u - tile * nkb;
    p.kb1 = unit_tile ? nkb : min(nkb, p.kb0 + (u1 - u));
    p.wpair = tile / n_rb;
    int rb = tile - p.wpair * n_rb;
    p.row0 = rb * SK_ROWBLOCK;
    p.nrows = min(SK_ROWBLOCK, live - p.row0);
    p.slot = unit_tile ? 0 : pair - sk_owner(tile * nkb, P, T);
    p.tile = tile;
    p.npieces = unit_tile ? 1 : sk_owner(tile * nkb + nkb - 1, P, T) - sk_owner(tile * nkb, P, T) + 1;
    u += unit_tile ? 1 : p.kb1 - p.kb0;
    return true;
  }
};

__global__ void __cluster_dims__(2, 1, 1) __launch_bounds__(SK2_THREADS, 1)
    gemm_sk2_k(const __grid_constant__ CUtensorMap tmW, const __grid_constant__ XMaps tmX, Sk2Params p) {
  extern __shared__ unsigned char smem_raw[];
  unsigned char *stage_base = reinterpret_cast<unsigned char *>(((uintptr_t)smem_raw + 1023) & ~(uintptr_t)1023);
  Sk2Bars &bar = *reinterpret_cast<Sk2Bars *>(stage_base + SMEM_BUDGET);
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const uint32_t rank = cluster_ctarank();
  const bool leader = rank == 0;

  pdl_trigger();
  // ---- this pair's unit range (identical in both CTAs of the cluster: every early exit below is taken by both or by neither)
  Piece2Iter it0;
  it0.nkb = p.nkb; it0.unit_tile = p.unit_tile; it0.P = gridDim.x >> 1; it0.pair = blockIdx.x >> 1;
  it0.live = p.n_rows_dev ? min(*p.n_rows_dev, p.rows_ub) : p.rows_ub;
  it0.n_rb = (it0.live + SK_ROWBLOCK - 1) / SK_ROWBLOCK;
  if (it0.n_rb <= 0) return;
  it0.T = p.n_wpairs * it0.n_rb * (p.unit_tile ? 1 : p.nkb);
  it0.u = (int)((long long)it0.pair * it0.T / it0.P);
  it0.u1 = (int)((long long)(it0.pair + 1) * it0.T / it0.P);
  if (it0.u >= it0.u1) return;
  // MMA N = the block's rows rounded up to 32 (each CTA holds N / 2 rows, a multiple of 16 for the TMA boxes)
  const int cap = (min(SK_ROWBLOCK, it0.live) + 31) & ~31;
  const int stage_bytes = W_STAGE_BYTES + (cap / 2) / BOX_ROWS * BOX_BYTES;
  const int n_stages = min(MAX_STAGES, SMEM_BUDGET / stage_bytes);
  int tm_cols = 32;
  while (tm_cols < cap) tm_cols *= 2;

  if (threadIdx.x == 0) {
    prefetch_tmap(&tmW);
    for (int b = 0; b < 4; ++b) prefetch_tmap(&tmX.m[b]);
    for (int s = 0; s < n_stages; ++s) { mbar_init(&bar.full[s], 1); mbar_init(&bar.peer_full[s], 1); mbar_init(&bar.empty[s], 1); }
    for (int b = 0; b < 2; ++b) { mbar_init(&bar.acc_full[b], 1); mbar_init(&bar.acc_empty[b], 8); }   // 4 epilogue warps of each CTA
    fence_mbar_init();
  }
  if (warp == 1) tmem_alloc2(&bar.tmem_base, 2 * tm_cols);
  tc_fence_before();
  __syncthreads();
  cluster_sync_all();                                      // the peer's barriers are initialised before anything arrives on them
  tc_fence_after();
  const uint32_t tmem = bar.tmem_base;

  if (warp == 0) {
    // ------------------------------------------------------------------------------------------ TMA producer (both CTAs, own shared memory)
    const uint64_t w_hint = it0.n_rb > 1 ? HINT_EVICT_LAST : HINT_EVICT_FIRST;
    auto wrow = [&](const Piece2 &pc) { return (2 * pc.wpair + (int)rank) * BMW; };   // rows past N are zero-filled by the tensor map
    int n_pre = 0;
    {
      Piece2Iter it = it0;
      Piece2 pc;
      while (n_pre < n_stages && it.next(pc)) {
        const int nh16 = ((pc.nrows + 31) & ~31) / 2 / BOX_ROWS;
        for (int kb = pc.kb0; kb < pc.kb1 && n_pre < n_stages; ++kb, ++n_pre)
          if (lane == 0) {
            unsigned char *st = stage_base + (size_t)n_pre * stage_bytes;
            mbar_expect_tx(&bar.full[n_pre], W_STAGE_BYTES + nh16 * BOX_BYTES);
            tma_load_2d_hint(st, &tmW, kb * BK, wrow(pc), &bar.full[n_pre], w_hint);   // weights do not depend on the producer kernel
          }
      }
    }
    pdl_wait();
    Piece2Iter it = it0;
    Piece2 pc;
    int stage = 0, phase = 0, i = 0;
    while (it.next(pc)) {
      const int nh = ((pc.nrows + 31) & ~31) / 2;            // activation rows staged by EACH CTA
      const int nh16 = nh / BOX_ROWS;
      const int tx = W_STAGE_BYTES + nh16 * BOX_BYTES;
      const int bit = lane;
      const bool mine = bit < 4 && ((nh16 >> bit) & 1);    // binary decomposition of nh into boxes of 128 / 64 / 32 / 16 rows
      const int my_row = (nh16 & ~((2 << bit) - 1)) * BOX_ROWS;
      for (int kb = pc.kb0; kb < pc.kb1; ++kb, ++i) {
        unsigned char *st = stage_base + (size_t)stage * stage_bytes;
        if (i >= n_pre) {
          mbar_wait_cluster(&bar.empty[stage], phase ^ 1);
          if (lane == 0) {
            mbar_expect_tx(&bar.full[stage], tx);
            tma_load_2d_hint(st, &tmW, kb * BK, wrow(pc), &bar.full[stage], w_hint);
          }
          __syncwarp();
        }
        if (mine)
          tma_load_2d_hint(st + W_STAGE_BYTES + my_row * (BK * 2), &tmX.m[bit], kb * BK, pc.row0 + (int)rank * nh + my_row, &bar.full[stage],
                           HINT_EVICT_LAST);
        if (++stage == n_stages) { stage = 0; phase ^= 1; }
      }
    }
  } else if (warp == 1) {
    if (lane == 0) {
      Piece2Iter it = it0;
      Piece2 pc;
      int stage = 0, phase = 0, piece = 0;
      if (!leader) {
        // ---------------------------------------------------------------------------------------- peer: forward "my stage has landed"
        while (it.next(pc))
          for (int kb = pc.kb0; kb < pc.kb1; ++kb) {
            mbar_wait(&bar.full[stage], phase);
            mbar_arrive_remote(map_to_cta(&bar.peer_full[stage], 0));
            if (++stage == n_stages) { stage = 0; phase ^= 1; }
          }
      } else {
        // ---------------------------------------------------------------------------------------- leader: the MMA issuer of the pair
        while (it.next(pc)) {
          const int buf = piece & 1, use = piece >> 1;
          const int Nmma = (pc.nrows + 31) & ~31;
          const uint32_t idesc = umma_idesc_bf16(2 * BMW, Nmma);
          mbar_wait_cluster(&bar.acc_empty[buf], (use & 1) ^ 1);
          tc_fence_after();
          const uint32_t d = tmem + (uint32_t)(buf * tm_cols);
          for (int kb = pc.kb0; kb < pc.kb1; ++kb) {
            mbar_wait(&bar.full[stage], phase);
            mbar_wait_cluster(&bar.peer_full[stage], phase);
            tc_fence_after();
            const uint32_t sa = smem_u32(stage_base + (size_t)stage * stage_bytes);
            const uint64_t dw = umma_desc_sw128(sa), dx = umma_desc_sw128(sa + W_STAGE_BYTES);
#pragma unroll
            for (int k = 0; k < BK / 16; ++k) mma2_bf16_ss(d, dw + 2 * k, dx + 2 * k, idesc, (kb > pc.kb0 || k > 0) ? 1u : 0u);
            mma2_commit_both(&bar.empty[stage]);
            if (++stage == n_stages) { stage = 0; phase ^= 1; }
          }
          mma2_commit_both(&bar.acc_full[buf]);
          ++piece;
        }
      }
    }
  } else {
    // ------------------------------------------------------------------------------------------ epilogue (both CTAs, own accumulator lanes)
    const int q = warp & 3;
    const uint32_t acc_empty_leader[2] = {map_to_cta(&bar.acc_empty[0], 0), map_to_cta(&bar.acc_empty[1], 0)};
    Piece2Iter it = it0;
    Piece2 pc;
    int piece = 0;
    while (it.next(pc)) {
      const int buf = piece & 1, use = piece >> 1;
      mbar_wait_cluster(&bar.acc_full[buf], use & 1);
      tc_fence_after();
      const int wtile = 2 * pc.wpair + (int)rank;
      const int n = wtile * BMW + q * 32 + lane;             // output column = weight row
      const bool n_ok = n < p.N;
      if (p.np_table && !p.unit_tile && pc.slot == 0 && q == 0 && lane == 0 && wtile < p.n_wtiles) {
        const int t128 = wtile * it0.n_rb + (pc.tile - pc.wpair * it0.n_rb);     // the consumers index 128-column tiles
        if (t128 < SK_NP_TABLE) p.np_table[t128] = pc.npieces;
      }
      float *dst = p.C + (size_t)pc.slot * p.slot_stride + (size_t)pc.row0 * p.N + n;
      const uint32_t src = tmem + ((uint32_t)(q * 32) << 16) + (uint32_t)(buf * tm_cols);
      const size_t ldc = (size_t)p.N;
#pragma unroll 1
      for (int c = 0; c < pc.nrows; c += 32) {
        uint32_t v[32];
        tmem_ld32(src + c, v);
        tmem_ld_wait();
        if (n_ok) {
          float *o = dst + (size_t)c * ldc;
          if (c + 32 <= pc.nrows) {
#pragma unroll
            for (int j = 0; j < 32; ++j, o += ldc) *o = __uint_as_float(v[j]);
          } else {
#pragma unroll
            for (int j = 0; j < 32; ++j, o += ldc)
              if (c + j < pc.nrows) *o = __uint_as_float(v[j]);
          }
        }
      }
      tc_fence_before();
      __syncwarp();
      if (lane == 0) mbar_arrive_remote(acc_empty_leader[buf]);   // the leader's MMA thread waits for both CTAs' drains
      ++piece;
    }
  }
  tc_fence_before();
  __syncthreads();
  cluster_sync_all();                                      // nobody frees TMEM or leaves while the peer may still touch this CTA
  if (warp == 1) tmem_dealloc2(tmem, 2 * tm_cols);
}

}  // namespace

darts_status gemm_sk2_configure(darts_ctx *c) {
  CUDA_TRY(c, cudaFuncSetAttribute(gemm_sk2_k, cudaFuncAttributeMaxDynamicSharedMemorySize, SMEM_BUDGET + (int)sizeof(Sk2Bars) + 2048));
  return DARTS_OK;
}

// Plan for the pair kernel: the same stream-K cut as sk_plan, over weight-tile PAIRS and n_sms / 2 CTA pairs.
SkPlan sk2_plan(int n_sms, int N, int K, int rows_ub, bool rows_exact) {
  SkPlan pl{};
  pl.nkb = K / BK;
  pl.n_wtiles = (N + BMW - 1) / BMW;
  const int n_wpairs = (pl.n_wtiles + 1) / 2, n_pairs = std::max(1, n_sms / 2);
  const int n_rb_ub = (rows_ub + SK_ROWBLOCK - 1) / SK_ROWBLOCK;
  const long long tiles_ub = (long long)n_wpairs * n_rb_ub;
  pl.unit_tile = tiles_ub >= 8LL * n_pairs;
  if (pl.unit_tile) {
    pl.P = (int)std::min<long long>(n_pairs, tiles_ub);
    pl.slots = 1;
  } else {
    const int T_min = n_wpairs * pl.nkb * (rows_exact ? n_rb_ub : 1);
    pl.P = std::max(1, std::min(n_pairs, T_min / 4));
    for (;;) {
      const int per = T_min / pl.P;
      pl.slots = std::min(pl.nkb, (pl.nkb + per - 1) / per + 1);
      if (pl.slots <= 16 || pl.P == 1) break;
      pl.P = std::max(1, pl.P * 3 / 4);
    }
  }
  return pl;
}

darts_status launch_gemm_sk2(darts_ctx *c, const SkGemm &g) {
  if (g.rows_ub <= 0) return DARTS_OK;
  const SkPlan &pl = g.plan;
  if (g.rb_list) FAIL(c, DARTS_ERR_UNSUPPORTED, "the CTA-pair GEMM is dense only");
  if (g.C == c->part && !pl.unit_tile && (size_t)pl.slots * g.slot_stride * sizeof(float) > c->part_bytes)
    FAIL(c, DARTS_ERR_WORKSPACE_TOO_SMALL, "stream-K piece buffer: %d slots x %zu floats > %zu bytes", pl.slots, g.slot_stride, c->part_bytes);
  Sk2Params p{};
  p.C = g.C; p.slot_stride = g.slot_stride; p.N = g.N; p.nkb = pl.nkb; p.n_wtiles = pl.n_wtiles; p.n_wpairs = (pl.n_wtiles + 1) / 2;
  p.rows_ub = g.rows_ub; p.n_rows_dev = g.n_rows_dev; p.np_table = g.np_table; p.unit_tile = pl.unit_tile;
  if (p.np_table && !pl.unit_tile && (long long)pl.n_wtiles * ((g.rows_ub + SK_ROWBLOCK - 1) / SK_ROWBLOCK) > SK_NP_TABLE)
    FAIL(c, DARTS_ERR_UNSUPPORTED, "stream-K piece-count table too small for %d weight tiles x %d rows", pl.n_wtiles, g.rows_ub);
  cudaLaunchConfig_t cfg{};
  cfg.gridDim = dim3(2 * pl.P); cfg.blockDim = dim3(SK2_THREADS);
  cfg.dynamicSmemBytes = SMEM_BUDGET + sizeof(Sk2Bars) + 1024; cfg.stream = c->stream;
  cudaLaunchAttribute at[1];
  at[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
  at[0].val.programmaticStreamSerializationAllowed = 1;
  cfg.attrs = at; cfg.numAttrs = c->use_pdl ? 1 : 0;            // the cluster shape is the kernel's __cluster_dims__
  cudaLaunchKernelEx(&cfg, gemm_sk2_k, *g.w_map, *g.x_maps, p);
  c->launches++;
  cudaError_t e = cudaGetLastError();
  if (e != cudaSuccess) {
    snprintf(c->err, sizeof(c->err), "launch gemm_sk2: %s", cudaGetErrorString(e));
    c->sticky = DARTS_ERR_CUDA;
    return DARTS_ERR_CUDA;
  }
  return DARTS_OK;
}
