// Weight-streaming tcgen05 / TMEM GEMM for the projections of the bf16 path:
//     P[slot][r][n] = sum_{k in piece} X[r][k] W[n][k]
//
// Decode projections are bound by streaming the weights from HBM once per step, so the kernel is built
// around the weight stream, not around the (small) activation matrix:
//   * "swap-AB": the 128-row MMA dimension M is a tile of WEIGHT rows, the MMA N dimension is the block of activation
//     rows (runtime N = live rows rounded up to 16, at most 256), so tensor work and activation loads scale with the
//     live row count and every weight byte is fetched once per 256-row block;
//   * persistent, one CTA per SM, stream-K: the (weight tile, row block, k-block) units of a GEMM are cut into gridDim.x
//     equal contiguous ranges, so every SM streams the same number of weight bytes whatever the tile count (152 tiles
//     on 148 SMs would otherwise cost two waves).  A tile that straddles CTAs is emitted as several partial "pieces";
//     piece s of a tile is written to slot s (slot = CTA index - first CTA of the tile), and the consumer kernels add
//     the pieces in slot order (internal.cuh: sk_npieces) — deterministic, no atomics;
//   * a deep TMA ring (stage = 16 KB of weights + 2 KB per 16 live rows; as many stages as fit in ~200 KB) keeps
//     >= 100 KB of weight loads in flight per SM, which is what it takes to cover HBM latency at 44 GB/s per SM;
//   * two TMEM accumulators: the epilogue warps drain piece i while the MMA warp accumulates piece i+1.
// Warp roles: warp 0 TMA producer, warp 1 MMA issuer (+ TMEM alloc), warps 2-5 epilogue (TMEM lane = weight row,
// column = activation row; a warp's 32 lanes store 32 consecutive output columns of one row: coalesced 128 B).
// Grouped mode (MoE): row blocks come from a device list {row0, nrows, weight row base}, units are whole tiles.
// Sampling mode (EPI_SAMPLE, the LM head of a decode step): whole (vocab tile, 256-row block) units; the
// epilogue never stores the logits: each warp transposes its 32 ids x 32 rows blocks through shared memory so that a thread owns a
// row, perturbs that row's 32 logits (z / T + Gumbel from Philox keyed by the row), keeps best / second / argbest and the
// log-sum-exp of z / T in registers, and leaves one entry per (tile, warp quadrant, row) for sample_finalize_k to merge.
#include <algorithm>

#include "internal.cuh"
#include "philox.cuh"
#include "sm100_ptx.cuh"

namespace {

using namespace ptx;

constexpr int BMW = 128, BK = 64;
constexpr int W_STAGE_BYTES = BMW * BK * 2;      // 16 KB
constexpr int BOX_ROWS = 16, BOX_BYTES = BOX_ROWS * BK * 2;
constexpr int MAX_STAGES = 10;
constexpr int SK_THREADS = 192;
constexpr int SMEM_BUDGET = 200 * 1024;

struct SkParams {
  float *C;
  size_t slot_stride;
  int N, nkb, n_wtiles, w_rows_per_group;
  int rows_ub;
  const int32_t *n_rows_dev;
  const int32_t *rb_list, *n_rb_dev;             // grouped mode
  int unit_tile;
  int stage_bytes, n_stages, tm_cols;            // tm_cols: columns of ONE accumulator (power of two >= 32)
  int n_acc;                                     // TMEM accumulators: 2 (epilogue overlaps the next piece) | 1 (one 512-column accumulator)
  int32_t *np_table;                             // dense split mode: [tile] = pieces of the tile, written by its head piece (nullable)
};

struct SkSampleArgs {
  float4 *top2;                                  // [4 * n_wtiles][rows_ub] (best y, second y, bits(argbest), z/T of the best)
  float2 *lse;                                   // [4 * n_wtiles][rows_ub] (max, sum e^(z/T - max))
  float *logits_dump;                            // [rows][N] or NULL
  const int32_t *row_list, *row_prompt, *row_sample, *row_len;
  float temperature;
  uint32_t k0, k1;
  const int32_t *target;                         // scoring (darts_score_chunk): [rows_ub] vocabulary id whose z / T is wanted per row (-1: none);
                                                 // no noise is drawn, the entry's "best" is the target's z / T, the log-sum-exp is unchanged
};
enum { SK_EPI_PIECES = 0, SK_EPI_SAMPLE = 1 };
constexpr int SK_TILE_OFF = 512;                 // behind the barriers: 32 x 33 fp32 transpose tiles, one per epilogue warp
constexpr int SK_SAMPLE_EPI_WARPS = 8;           // two per TMEM lane quadrant (alternate 32-column chunks): one warp per scheduler cannot hide its own latencies
constexpr int SK_TILE_BYTES = SK_SAMPLE_EPI_WARPS * 32 * 33 * 4;
constexpr int SK_SAMPLE_RING = 184 * 1024;       // the ring gives 16 KB to the tiles
constexpr int SK_SAMPLE_THREADS = 64 + SK_SAMPLE_EPI_WARPS * 32;

struct SkBars {
  unsigned long long full[MAX_STAGES], empty[MAX_STAGES], acc_full[2], acc_empty[2];
  uint32_t tmem_base;
};

struct Piece {
  int wtile, row0, nrows, wbase, kb0, kb1, slot, tile, npieces;
};

// Walks the pieces of CTA `cta`; the three roles call it with identical arguments and so see the same sequence.
struct PieceIter {
  int u, u1, T, P, nkb, n_rb, unit_tile, cta, w_rows_per_group, rb_rows;
  const int32_t *rb_list;
  int live;
  __device__ bool next(Piece &p) {
    if (u >= u1) return false;
    int tile = unit_tile ? u : u / nkb;
    p.kb0 = unit_tile ? 0 : u - tile * nkb;
    p.kb1 = unit_tile ? nkb : min(nkb, p.kb0 + (u1 - u));
    p.wtile = tile / n_rb;
    int rb = tile - p.wtile * n_rb;
    if (rb_list) { p.row0 = rb_list[4 * rb]; p.nrows = rb_list[4 * rb + 1]; p.wbase = rb_list[4 * rb + 2] * w_rows_per_group; }
    else { p.row0 = rb * rb_rows; p.nrows = min(rb_rows, live - p.row0); p.wbase = 0; }
    p.slot = unit_tile ? 0 : cta - sk_owner(tile * nkb, P, T);
    p.tile = tile;
    p.npieces = unit_tile ? 1 : sk_owner(tile * nkb + nkb - 1, P, T) - sk_owner(tile * nkb, P, T) + 1;
    u += unit_tile ? 1 : p.kb1 - p.kb0;
    return true;
  }
};

template <int EPI>
__global__ void __launch_bounds__(EPI == SK_EPI_SAMPLE ? SK_SAMPLE_THREADS : SK_THREADS, 1) gemm_sk_k(const __grid_constant__ CUtensorMap tmW, const __grid_constant__ XMaps tmX,
                                                           SkParams p, SkSampleArgs sa) {
  extern __shared__ unsigned char smem_raw[];
  unsigned char *stage_base = reinterpret_cast<unsigned char *>(((uintptr_t)smem_raw + 1023) & ~(uintptr_t)1023);
  constexpr int RING = EPI == SK_EPI_SAMPLE ? SK_SAMPLE_RING : SMEM_BUDGET;
  SkBars &bar = *reinterpret_cast<SkBars *>(stage_base + RING);
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;

  pdl_trigger();
  // ---- this CTA's unit range (uniform over the CTA; leave before any barrier / TMEM allocation if it is empty)
  PieceIter it0;
  it0.rb_list = p.rb_list; it0.w_rows_per_group = p.w_rows_per_group; it0.nkb = p.nkb; it0.unit_tile = p.unit_tile; it0.P = gridDim.x; it0.cta = blockIdx.x; it0.rb_rows = SK_ROWBLOCK;
  if (p.rb_list) { pdl_wait(); it0.n_rb = *p.n_rb_dev; it0.live = 0; }
  else {
    // dense: block size, ring depth and TMEM split follow the LIVE row count (device value), not the host's bound
    it0.live = p.n_rows_dev ? min(*p.n_rows_dev, p.rows_ub) : p.rows_ub;
    it0.rb_rows = EPI == SK_EPI_SAMPLE ? SK_ROWBLOCK : sk_rb_rows(it0.live);   // sampling needs both accumulators (epilogue overlap)
    it0.n_rb = (it0.live + it0.rb_rows - 1) / it0.rb_rows;
    const int cap = (min(it0.rb_rows, it0.live) + 15) & ~15;
    p.stage_bytes = W_STAGE_BYTES + cap / BOX_ROWS * BOX_BYTES;
    p.n_stages = min(MAX_STAGES, RING / p.stage_bytes);
    p.tm_cols = 32;
    while (p.tm_cols < cap) p.tm_cols *= 2;
    p.n_acc = p.tm_cols > 256 ? 1 : 2;
  }
  if (it0.n_rb <= 0) return;
  it0.T = p.n_wtiles * it0.n_rb * (p.unit_tile ? 1 : p.nkb);
  it0.u = (int)((long long)blockIdx.x * it0.T / gridDim.x);
  it0.u1 = (int)((long long)(blockIdx.x + 1) * it0.T / gridDim.x);
  if (it0.u >= it0.u1) return;

  if (threadIdx.x == 0) {
    prefetch_tmap(&tmW);
    for (int b = 0; b < 5; ++b) prefetch_tmap(&tmX.m[b]);
    for (int s = 0; s < p.n_stages; ++s) { mbar_init(&bar.full[s], 1); mbar_init(&bar.empty[s], 1); }
    for (int b = 0; b < 2; ++b) { mbar_init(&bar.acc_full[b], 1); mbar_init(&bar.acc_empty[b], EPI == SK_EPI_SAMPLE ? SK_SAMPLE_EPI_WARPS : 4); }
    fence_mbar_init();
  }
  if (warp == 1) tmem_alloc(&bar.tmem_base, p.n_acc * p.tm_cols);
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  const uint32_t tmem = bar.tmem_base;

  if (warp == 0) {
    // ------------------------------------------------------------------------------------------ TMA producer
    // The whole warp walks the ring; lane 0 arms the barrier and fetches the weight tile; the activation rows
    // (rounded up to 16) are fetched as the binary decomposition of their count into boxes of 256/128/64/32/16 rows,
    // lane b taking the box of 16 << b rows: at most five bulk-tensor copies per stage, issued by one warp instruction
    // (the copy COUNT, not the bytes, is what bounds a single-producer TMA ring).
    // Programmatic dependent launch: this kernel may start while the kernel that produces X is still running.  The weights
    // do not depend on it, so the first ring-full of weight tiles is requested BEFORE griddepcontrol.wait; only the
    // activation boxes wait.  (Grouped mode reads its row-block list first and therefore waits at the top.)
    // One row block: every weight byte is used once (evict-first).  Several row blocks re-read a weight tile a few k-blocks
    // later: keep it in L2 (evict-last), or the second pass goes back to HBM (measured: 2x DRAM reads on the gate/up GEMM).
    const uint64_t w_hint = (!p.rb_list && it0.n_rb > 1) ? HINT_EVICT_LAST : HINT_EVICT_FIRST;
    int n_pre = 0;
    if (!p.rb_list) {
      PieceIter it = it0;
      Piece pc;
      while (n_pre < p.n_stages && it.next(pc)) {
        const int n16 = (pc.nrows + BOX_ROWS - 1) / BOX_ROWS;
        for (int kb = pc.kb0; kb < pc.kb1 && n_pre < p.n_stages; ++kb, ++n_pre)
          if (lane == 0) {
            unsigned char *st = stage_base + (size_t)n_pre * p.stage_bytes;
            mbar_expect_tx(&bar.full[n_pre], W_STAGE_BYTES + n16 * BOX_BYTES);
            tma_load_2d_hint(st, &tmW, kb * BK, pc.wbase + pc.wtile * BMW, &bar.full[n_pre], w_hint);
          }
      }
    }
    pdl_wait();
    PieceIter it = it0;
    Piece pc;
    int stage = 0, phase = 0, i = 0;
    while (it.next(pc)) {
      const int n16 = (pc.nrows + BOX_ROWS - 1) / BOX_ROWS;
      const int tx = W_STAGE_BYTES + n16 * BOX_BYTES;
      const int wrow = pc.wbase + pc.wtile * BMW;
      // sub-block A = rows [0, 256) on lanes 0-4, sub-block B = rows [256, 512) on lanes 8-12 (only with rb_rows = 512)
      const int sub = lane >> 3, bit = lane & 7;
      const int n16s = sub == 0 ? min(n16, 16) : n16 - min(n16, 16);
      const bool mine = sub < 2 && bit < 5 && ((n16s >> bit) & 1);
      const int my_row = sub * 256 + (n16s & ~((2 << bit) - 1)) * BOX_ROWS;   // rows covered by the larger boxes of this sub-block
      for (int kb = pc.kb0; kb < pc.kb1; ++kb, ++i) {
        unsigned char *st = stage_base + (size_t)stage * p.stage_bytes;
        if (i >= n_pre) {
          mbar_wait(&bar.empty[stage], phase ^ 1);
          if (lane == 0) {
            mbar_expect_tx(&bar.full[stage], tx);
            tma_load_2d_hint(st, &tmW, kb * BK, wrow, &bar.full[stage], w_hint);
          }
          __syncwarp();
        }
        if (mine)
          tma_load_2d_hint(st + W_STAGE_BYTES + my_row * (BK * 2), &tmX.m[bit], kb * BK, pc.row0 + my_row, &bar.full[stage], HINT_EVICT_LAST);
        if (++stage == p.n_stages) { stage = 0; phase ^= 1; }
      }
    }
  } else if (warp == 1) {
    // ------------------------------------------------------------------------------------------ MMA issuer
    if (lane == 0) {
      PieceIter it = it0;
      Piece pc;
      int stage = 0, phase = 0, piece = 0;
      while (it.next(pc)) {
        const int buf = piece % p.n_acc, use = piece / p.n_acc;
        const int nA = min(pc.nrows, 256), nB = pc.nrows - nA;                  // two MMA N blocks share the weight tile of a stage
        const uint32_t idesc = umma_idesc_bf16(BMW, (nA + 15) & ~15), idescB = umma_idesc_bf16(BMW, (nB + 15) & ~15);
        mbar_wait(&bar.acc_empty[buf], (use & 1) ^ 1);
        tc_fence_after();
        const uint32_t d = tmem + (uint32_t)(buf * p.tm_cols);
        for (int kb = pc.kb0; kb < pc.kb1; ++kb) {
          mbar_wait(&bar.full[stage], phase);
          tc_fence_after();
          const uint32_t sa = smem_u32(stage_base + (size_t)stage * p.stage_bytes);
          const uint64_t dw = umma_desc_sw128(sa), dx = umma_desc_sw128(sa + W_STAGE_BYTES);
#pragma unroll
          for (int k = 0; k < BK / 16; ++k) mma_bf16_ss(d, dw + 2 * k, dx + 2 * k, idesc, (kb > pc.kb0 || k > 0) ? 1u : 0u);
          if (nB > 0) {
            const uint64_t dxb = umma_desc_sw128(sa + W_STAGE_BYTES + 256 * BK * 2);
#pragma unroll
            for (int k = 0; k < BK / 16; ++k) mma_bf16_ss(d + 256, dw + 2 * k, dxb + 2 * k, idescB, (kb > pc.kb0 || k > 0) ? 1u : 0u);
          }
          mma_commit(&bar.empty[stage]);
          if (++stage == p.n_stages) { stage = 0; phase ^= 1; }
        }
        mma_commit(&bar.acc_full[buf]);
        ++piece;
      }
    }
  } else {
    // ------------------------------------------------------------------------------------------ epilogue
    const int q = warp & 3;                                // TMEM lane quadrant this warp may read
    if constexpr (EPI == SK_EPI_SAMPLE) {
      // A TMEM lane is a vocabulary id and a column an activation row; sampling wants the opposite (one thread walking the ids of ONE
      // row: Philox block shared by 4 consecutive ids, running top-2 and log-sum-exp in registers, no warp-wide step).  Each 32 x 32
      // (id x row) block is therefore transposed through a padded shared-memory tile private to the warp.
      const int half = (warp - 2) >> 2;                    // the two warps of a quadrant take alternate 32-column chunks
      float *tile = reinterpret_cast<float *>(stage_base + RING + SK_TILE_OFF) + (half * 4 + q) * (32 * 33);
      pdl_wait();
      const float T = sa.temperature;
      PieceIter it = it0;
      Piece pc;
      int piece = 0;
      while (it.next(pc)) {
        const int buf = piece % p.n_acc, use = piece / p.n_acc;
        mbar_wait(&bar.acc_full[buf], use & 1);
        tc_fence_after();
        const int nb = pc.wtile * BMW + q * 32;              // first vocabulary id of this warp (multiple of 32)
        const uint32_t src = tmem + ((uint32_t)(q * 32) << 16) + (uint32_t)(buf * p.tm_cols);
        const size_t ent = (size_t)(pc.wtile * 4 + q) * p.rows_ub + pc.row0;
#pragma unroll 1
        for (int c = half * 32; c < pc.nrows; c += 32 * (SK_SAMPLE_EPI_WARPS / 4)) {
          uint32_t v[32];
          tmem_ld32(src + c, v);
          tmem_ld_wait();
          if (sa.logits_dump && nb + lane < p.N) {
#pragma unroll
            for (int j = 0; j < 32; ++j)
              if (c + j < pc.nrows) sa.logits_dump[(size_t)(pc.row0 + c + j) * p.N + nb + lane] = __uint_as_float(v[j]);
          }
#pragma unroll
          for (int j = 0; j < 32; ++j) tile[lane * 33 + j] = __uint_as_float(v[j]);       // bank (lane + j) % 32: conflict-free
          __syncwarp();
          const bool row_ok = c + lane < pc.nrows;
          int pi = 0, pj = 0, ps = 0, tgt = -1;
          if (row_ok && !sa.target) {
            const int row = sa.row_list[pc.row0 + c + lane];
            pi = sa.row_prompt[row]; pj = sa.row_sample[row]; ps = sa.row_len[row];
          }
          if (row_ok && sa.target) tgt = sa.target[pc.row0 + c + lane];
          float b1 = -INFINITY, b2 = -INFINITY, z1 = 0.f, lm = -INFINITY, ls = 0.f;
          int i1 = 0x7fffffff;
#pragma unroll
          for (int k = 0; k < 32; k += 4) {
            const int vid = nb + k;                          // multiple of 4: one Philox block serves 4 vocabulary ids
            if (vid < p.N) {                                 // warp-uniform (N % 4 == 0)
              uint32_t x[4] = {0u, 0u, 0u, 0u};
              if (T != 0.f && !sa.target) philox4x32_10((uint32_t)(vid >> 2), (uint32_t)ps, (uint32_t)pj, (uint32_t)pi, sa.k0, sa.k1, x);
              float zt[4];
#pragma unroll
              for (int e = 0; e < 4; ++e) {
                const float z = tile[(k + e) * 33 + lane];   // consecutive lanes, consecutive words
                zt[e] = T != 0.f ? z / T : z;
                if (sa.target) {                             // warp-uniform: scoring a GIVEN token
                  if (vid + e == tgt) { b1 = zt[e]; z1 = zt[e]; i1 = tgt; }
                } else {
                  const float y = T != 0.f ? zt[e] + gumbel_from_bits(x[e]) : z;
                  if (y > b1) { b2 = b1; b1 = y; i1 = vid + e; z1 = zt[e]; }        // ids ascend: strict > keeps the lowest id on ties
                  else if (y > b2) b2 = y;
                }
              }
              const float mn = fmaxf(fmaxf(lm, fmaxf(zt[0], zt[1])), fmaxf(zt[2], zt[3]));
              ls = ls * __expf(lm - mn) + ((__expf(zt[0] - mn) + __expf(zt[1] - mn)) + (__expf(zt[2] - mn) + __expf(zt[3] - mn)));
              lm = mn;
            }
          }
          __syncwarp();                                      // the tile is rewritten by the next chunk
          if (row_ok) {
            sa.top2[ent + c + lane] = make_float4(b1, b2, __int_as_float(i1), z1);
            sa.lse[ent + c + lane] = make_float2(lm, ls);
          }
        }
        tc_fence_before();
        __syncwarp();
        if (lane == 0) mbar_arrive(&bar.acc_empty[buf]);
        ++piece;
      }
    } else {
      PieceIter it = it0;
      Piece pc;
      int piece = 0;
      while (it.next(pc)) {
        const int buf = piece % p.n_acc, use = piece / p.n_acc;
        mbar_wait(&bar.acc_full[buf], use & 1);
        tc_fence_after();
        const int n = pc.wtile * BMW + q * 32 + lane;        // output column = weight row
        const bool n_ok = n < p.N;
        if (p.np_table && !p.unit_tile && pc.slot == 0 && q == 0 && lane == 0 && pc.tile < SK_NP_TABLE) p.np_table[pc.tile] = pc.npieces;
        float *dst = p.C + (size_t)pc.slot * p.slot_stride + (size_t)pc.row0 * p.N + n;
        const uint32_t src = tmem + ((uint32_t)(q * 32) << 16) + (uint32_t)(buf * p.tm_cols);
        const size_t ldc = (size_t)p.N;
#pragma unroll 1
        for (int c = 0; c < pc.nrows; c += 32) {
          uint32_t v[32];
          tmem_ld32(src + c, v);
          tmem_ld_wait();
          if (n_ok) {
            float *q = dst + (size_t)c * ldc;                // one pointer bump per store, no per-element predicate on full chunks
            if (c + 32 <= pc.nrows) {
#pragma unroll
              for (int j = 0; j < 32; ++j, q += ldc) *q = __uint_as_float(v[j]);
            } else {
#pragma unroll
              for (int j = 0; j < 32; ++j, q += ldc)
                if (c + j < pc.nrows) *q = __uint_as_float(v[j]);
            }
          }
        }
        tc_fence_before();
        __syncwarp();
        if (lane == 0) mbar_arrive(&bar.acc_empty[buf]);
        ++piece;
      }
    }
  }
  tc_fence_before();
  __syncthreads();
  if (warp == 1) tmem_dealloc(tmem, p.n_acc * p.tm_cols);
}

// out[r][n] = sum of the pieces of (r, n) in slot order (debug / test hook)
__global__ void sk_reduce_k(SkView v, float *__restrict__ out, int rows) {
  size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= (size_t)rows * v.N) return;
  int r = (int)(i / v.N), n = (int)(i % v.N);
  int rbr = sk_view_rb_rows(v, rows), n_rb = (rows + rbr - 1) / rbr;
  int np = sk_npieces(v, n_rb, rbr, n, r);
  float a = v.part[i];
  for (int s = 1; s < np; ++s) a += v.part[(size_t)s * v.slot_stride + i];
  out[i] = a;
}

}  // namespace

// Host-side plan: mode, grid, slots.  rows_ub bounds the live rows (dense; rows_exact: it IS the row count) or the rows
// of one group (grouped, at most n_rb_ub_grouped row blocks in all).
SkPlan sk_plan(int n_sms, int N, int K, int rows_ub, int n_rb_ub_grouped, bool rows_exact) {
  SkPlan pl{};
  pl.nkb = K / BK;
  pl.n_wtiles = (N + BMW - 1) / BMW;
  const bool grouped = n_rb_ub_grouped > 0;
  const int n_rb_ub = grouped ? n_rb_ub_grouped : (rows_ub + SK_ROWBLOCK - 1) / SK_ROWBLOCK;   // dense 512-row blocks only lower it
  const long long tiles_ub = (long long)pl.n_wtiles * n_rb_ub;
  pl.unit_tile = grouped || tiles_ub >= 8LL * n_sms;
  if (pl.unit_tile) {
    pl.P = (int)std::min<long long>(n_sms, tiles_ub);
    pl.slots = 1;
  } else {
    // fewest units a launch can see: one row block when the live count is only bounded; the exact count's blocks otherwise
    // (257..384 rows are ONE 512-row block, sk_rb_rows: counting two there under-sized the slot count)
    const int T_min = pl.n_wtiles * pl.nkb * (rows_exact ? (rows_ub + sk_rb_rows(rows_ub) - 1) / sk_rb_rows(rows_ub) : 1);
    pl.P = std::max(1, std::min(n_sms, T_min / 4));                        // >= 4 k-blocks (64 KB of weights) per CTA
    for (;;) {
      const int per = T_min / pl.P;                                        // every CTA range holds >= per units
      pl.slots = std::min(pl.nkb, (pl.nkb + per - 1) / per + 1);
      if (pl.slots <= 16 || pl.P == 1) break;                              // consumers hold <= 16 pieces in registers
      pl.P = std::max(1, pl.P * 3 / 4);
    }
  }
  int cap = std::min(SK_ROWBLOCK, (rows_ub + 15) & ~15);              // grouped mode; dense launches derive these on the device
  pl.stage_bytes = W_STAGE_BYTES + cap / BOX_ROWS * BOX_BYTES;
  pl.n_stages = std::min(MAX_STAGES, SMEM_BUDGET / pl.stage_bytes);
  pl.tm_cols = 32;
  while (pl.tm_cols < cap) pl.tm_cols *= 2;
  pl.n_acc = pl.tm_cols > 256 ? 1 : 2;
  return pl;
}

// Per-context set-up (darts_create): function attributes belong to the device / context the library was created on, not to the process.
darts_status gemm_sk_configure(darts_ctx *c) {
  CUDA_TRY(c, cudaFuncSetAttribute(gemm_sk_k<SK_EPI_PIECES>, cudaFuncAttributeMaxDynamicSharedMemorySize, SMEM_BUDGET + (int)sizeof(SkBars) + 2048));
  CUDA_TRY(c, cudaFuncSetAttribute(gemm_sk_k<SK_EPI_SAMPLE>, cudaFuncAttributeMaxDynamicSharedMemorySize, SK_SAMPLE_RING + SK_TILE_OFF + SK_TILE_BYTES + 1024));
  return DARTS_OK;
}

darts_status launch_gemm_sk(darts_ctx *c, const SkGemm &g) {
  if (g.rows_ub <= 0) return DARTS_OK;
  const SkPlan &pl = g.plan;
  if (g.C == c->part && !pl.unit_tile && (size_t)pl.slots * g.slot_stride * sizeof(float) > c->part_bytes)
    FAIL(c, DARTS_ERR_WORKSPACE_TOO_SMALL, "stream-K piece buffer: %d slots x %zu floats > %zu bytes", pl.slots, g.slot_stride, c->part_bytes);
  SkParams p{};
  p.C = g.C; p.slot_stride = g.slot_stride; p.N = g.N; p.nkb = pl.nkb; p.n_wtiles = pl.n_wtiles; p.rows_ub = g.rows_ub; p.n_rows_dev = g.n_rows_dev;
  p.rb_list = g.rb_list; p.n_rb_dev = g.n_rb_dev; p.w_rows_per_group = g.w_rows_per_group; p.unit_tile = pl.unit_tile; p.stage_bytes = pl.stage_bytes; p.n_stages = pl.n_stages;
  p.tm_cols = pl.tm_cols; p.n_acc = pl.n_acc;
  p.np_table = g.rb_list ? nullptr : g.np_table;
  if (p.np_table && !pl.unit_tile && (long long)pl.n_wtiles * ((g.rows_ub + SK_ROWBLOCK - 1) / SK_ROWBLOCK) > SK_NP_TABLE)
    FAIL(c, DARTS_ERR_UNSUPPORTED, "stream-K piece-count table too small for %d weight tiles x %d rows", pl.n_wtiles, g.rows_ub);
  size_t smem = SMEM_BUDGET + sizeof(SkBars) + 1024;
  launch_pdl(c, gemm_sk_k<SK_EPI_PIECES>, dim3(pl.P), dim3(SK_THREADS), smem, *g.w_map, *g.x_maps, p, SkSampleArgs{});
  c->launches++;
  cudaError_t e = cudaGetLastError();
  if (e != cudaSuccess) {
    snprintf(c->err, sizeof(c->err), "launch gemm_sk: %s", cudaGetErrorString(e));
    c->sticky = DARTS_ERR_CUDA;
    return DARTS_ERR_CUDA;
  }
  return DARTS_OK;
}

// LM head of a decode step with the sampling epilogue (whole tiles, 256-row blocks); sample_finalize_k merges 4 entries per vocab tile.
bool sk_sample_supported(const darts_ctx *c, int rows_ub) { return rows_ub > 0 && c->m.d_model % BK == 0 && c->m.vocab % 4 == 0; }

darts_status launch_gemm_sk_sample(darts_ctx *c, const CUtensorMap *w_map, const XMaps *x_maps, int N, int K, int rows_ub, const int32_t *n_rows_dev,
                                   const int32_t *target) {
  if (rows_ub <= 0) return DARTS_OK;
  static_assert(sizeof(SkBars) <= SK_TILE_OFF, "transpose tiles overlap the barriers");
  SkParams p{};
  p.N = N; p.nkb = K / BK; p.n_wtiles = (N + BMW - 1) / BMW; p.rows_ub = rows_ub; p.n_rows_dev = n_rows_dev; p.unit_tile = 1;
  SkSampleArgs sa{};
  sa.top2 = (float4 *)c->top2; sa.lse = (float2 *)c->lse; sa.logits_dump = ((c->rt.flags & DARTS_FLAG_DUMP_LOGITS) && !target) ? c->logits : nullptr;
  sa.target = target;
  sa.row_list = c->row_list; sa.row_prompt = c->row_prompt; sa.row_sample = c->row_sample; sa.row_len = c->row_len;
  sa.temperature = c->temperature; sa.k0 = (uint32_t)(c->seed & 0xffffffffu); sa.k1 = (uint32_t)(c->seed >> 32);
  const int smem = SK_SAMPLE_RING + SK_TILE_OFF + SK_TILE_BYTES + 1024;
  const int n_sms = c->n_sms > 0 ? c->n_sms : 148;
  launch_pdl(c, gemm_sk_k<SK_EPI_SAMPLE>, dim3(std::min(n_sms, p.n_wtiles)), dim3(SK_SAMPLE_THREADS), (size_t)smem, *w_map, *x_maps, p, sa);
  c->launches++;
  cudaError_t e = cudaGetLastError();
  if (e != cudaSuccess) {
    snprintf(c->err, sizeof(c->err), "launch gemm_sk (sampling): %s", cudaGetErrorString(e));
    c->sticky = DARTS_ERR_CUDA;
    return DARTS_ERR_CUDA;
  }
  return DARTS_OK;
}

darts_status launch_sk_reduce(darts_ctx *c, const SkView &v, float *out, int rows) {
  size_t n = (size_t)rows * v.N;
  sk_reduce_k<<<(unsigned)((n + 255) / 256), 256, 0, c->stream>>>(v, out, rows);
  c->launches++;
  if (cudaGetLastError() != cudaSuccess) FAIL(c, DARTS_ERR_CUDA, "launch sk_reduce failed");
  return DARTS_OK;
}
