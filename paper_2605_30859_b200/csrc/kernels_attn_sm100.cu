// Prefix-shared split-KV GQA decode attention for the bf16 path (head_dim 128, page 64).   SURVEY.md §8(a) row 5.
//
// Work is cut into ITEMS of at most CH_PAGES pages (512 tokens) of ONE page table:
//   prefix item  = (group of active rows of one prompt, chunk of the prompt's shared prefix pages):
//                  every page is fetched ONCE for all the group's rows ("reads each prompt-prefix page once per
//                  group", north_star); query rows = rows x (Hq/Hkv) heads, up to 64 per item;
//   suffix item  = (one row, chunk of its own pages).
// Items x kv-heads are strided over a persistent grid (2 CTAs per SM).  Inside a CTA one producer warp streams
// the (page, head) K+V tile pairs — 32 KB, contiguous in HBM by construction of the cache layout — into a
// 3-stage shared-memory ring with cp.async.bulk (the TMA bulk-copy engine) + mbarrier transaction counts, and
// four consumer warps run QK^T / PV on tensor cores (mma.sync m16n8k16 bf16, fp32 accumulate) with an online
// softmax in fp32.  Two inner loops: an item of more than 8 query rows (a prefix item) puts the query rows on the
// MMA's m dimension (one 16-row m-tile per warp, every warp walks the whole page); an item of <= 8 query rows (a
// row's own pages when Hq/Hkv <= 8) puts each warp's 16 tokens on m and the query rows on n = 8 (tpath_unit: half
// the MMAs and accumulators), in a software-pipelined loop over the CTA's suffix units.  The cache is stored pre-swizzled (internal.cuh: kv_elem), so the linear copy lands in the
// bank-conflict-free layout ldmatrix needs.  Every item writes one un-normalised partial (m, l, acc) per query
// row; attn_merge_k combines a row's partials by log-sum-exp in chunk order.  The split depends only on a row's
// own lengths (fixed 512-token chunks), so a row's arithmetic does not depend on which other rows are active,
// apart from which row block of its group it falls in.
#include "internal.cuh"

namespace {

constexpr int CH_PAGES = ATTN_CHUNK_PAGES;   // pages per item
constexpr int PAGE = 64, HD = 128;
constexpr int CH_TOK = CH_PAGES * PAGE;
constexpr int STAGES = 3;
constexpr int STAGE_BYTES = 2 * PAGE * HD * 2;   // K tile + V tile of one (page, head)
constexpr int N_CONS = 4;                   // consumer warps
constexpr int THREADS = (N_CONS + 1) * 32;
#ifndef ATTN_TPATH
#define ATTN_TPATH 1                        // units with <= 8 query rows: S^T = K Q^T (tokens on the MMA's m) (A/B switch: -DATTN_TPATH=0)
#endif
#ifndef ATTN_CHUNK_MAJOR
#define ATTN_CHUNK_MAJOR 1                 // plan: suffix items chunk-major when all rows have the same number of chunks (A/B switch: =0)
#endif
#ifndef ATTN_PARTIAL_LAST_PAGE
#define ATTN_PARTIAL_LAST_PAGE 1            // fetch only the valid part of a row's newest page (A/B switch: -DATTN_PARTIAL_LAST_PAGE=0)
#endif
constexpr int ITEM_INTS = 6;                // first_slot, n_slots, page_begin, n_tokens, chunk_k, is_prefix

struct Smem {
  alignas(128) unsigned char stage[STAGES][STAGE_BYTES];
  float scratch[N_CONS][4][HD];             // cross-warp merge of TOKSPLIT items, 4 query rows per round
  float ml[2][N_CONS][16][2];               // (max, sum) of the warps' partials; two buffers, alternating per unit
  unsigned long long full[STAGES], empty[STAGES];
};

// ------------------------------------------------------------------------------------------------ PTX helpers
__device__ __forceinline__ uint32_t smem_u32(const void *p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(void *bar, int count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count));
}
__device__ __forceinline__ void mbar_expect_tx(void *bar, int bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_arrive(void *bar) {
  asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(smem_u32(bar)) : "memory");
}
// Bounded wait (as in sm100_ptx.cuh): a protocol bug traps, the launch fails with an error, nothing hangs.
__device__ __forceinline__ void mbar_wait(void *bar, int parity) {
  for (uint32_t spins = 0;; ++spins) {
    uint32_t ok;
    asm volatile(
        "{\n.reg .pred p;\n"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n"
        "selp.u32 %0, 1, 0, p;\n}"
        : "=r"(ok)
        : "r"(smem_u32(bar)), "r"(parity)
        : "memory");
    if (ok) return;
    if (spins > (1u << 26)) __trap();
  }
}
__device__ __forceinline__ void bulk_g2s(void *dst, const void *src, int bytes, void *bar) {
  asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(smem_u32(dst)),
               "l"(src), "r"(bytes), "r"(smem_u32(bar))
               : "memory");
}
__device__ __forceinline__ void ldsm4(uint32_t addr, uint32_t &r0, uint32_t &r1, uint32_t &r2, uint32_t &r3) {
  asm volatile("ldmatrix.sync.aligned.m8n8.x4.shared.b16 {%0,%1,%2,%3}, [%4];" : "=r"(r0), "=r"(r1), "=r"(r2), "=r"(r3) : "r"(addr));
}
__device__ __forceinline__ void ldsm4t(uint32_t addr, uint32_t &r0, uint32_t &r1, uint32_t &r2, uint32_t &r3) {
  asm volatile("ldmatrix.sync.aligned.m8n8.x4.trans.shared.b16 {%0,%1,%2,%3}, [%4];" : "=r"(r0), "=r"(r1), "=r"(r2), "=r"(r3) : "r"(addr));
}
__device__ __forceinline__ void mma16816(float (&c)[4], uint32_t a0, uint32_t a1, uint32_t a2, uint32_t a3, uint32_t b0, uint32_t b1) {
  asm volatile("mma.sync.aligned.m16n8k16.row.col.f32.bf16.bf16.f32 {%0,%1,%2,%3}, {%4,%5,%6,%7}, {%8,%9}, {%0,%1,%2,%3};"
               : "+f"(c[0]), "+f"(c[1]), "+f"(c[2]), "+f"(c[3])
               : "r"(a0), "r"(a1), "r"(a2), "r"(a3), "r"(b0), "r"(b1));
}
__device__ __forceinline__ void movmatrix_t(uint32_t a, uint32_t &d) {
  asm volatile("movmatrix.sync.aligned.m8n8.trans.b16 %0, %1;" : "=r"(d) : "r"(a));
}
__device__ __forceinline__ uint32_t pack_bf16(float lo, float hi) {
  __nv_bfloat162 v = __floats2bfloat162_rn(lo, hi);
  return *reinterpret_cast<uint32_t *>(&v);
}
__device__ __forceinline__ void cons_bar() { asm volatile("bar.sync 1, %0;" ::"n"(N_CONS * 32) : "memory"); }

struct Params {
  const __nv_bfloat16 *q;                   // [slot][Hq][128]
  const __nv_bfloat16 *kv_layer;
  const int32_t *items_pre, *items_suf, *n_items;   // n_items[0] = prefix items, [1] = suffix items
  const int32_t *slot_prompt, *slot_row, *slot_npre, *g_prefix_pages, *row_pages, *part_base;
  int causal;                               // prefill pass: query row of slot s sees tokens < slot_npre[s] only
  float *part_ml, *part_acc;
  int mpp, msp, Hq, Hkv, rep, rep_shift;  // rep = Hq / Hkv = 1 << rep_shift (attention_sm100_supported)
  size_t page_elems, tile_elems;
  float c;                                  // softmax scale * log2(e)
};

// Online-softmax update of NT score n-tiles (two row sets: g and g+8).  Emits P (bf16x2) and rescales O.
template <int NT>
__device__ __forceinline__ void softmax_update(float (&S)[NT][4], float (&m)[2], float (&l)[2], float (&O)[16][4],
                                               uint32_t (&P)[NT][2], float c) {
#pragma unroll
  for (int rs = 0; rs < 2; ++rs) {
    float mx = -INFINITY;
#pragma unroll
    for (int nt = 0; nt < NT; ++nt) mx = fmaxf(mx, fmaxf(S[nt][2 * rs], S[nt][2 * rs + 1]));
    mx = fmaxf(mx, __shfl_xor_sync(0xffffffffu, mx, 1));
    mx = fmaxf(mx, __shfl_xor_sync(0xffffffffu, mx, 2));
    float mn = fmaxf(m[rs], mx);
    float ms = mn == -INFINITY ? 0.f : mn;
    float corr = exp2f((m[rs] - ms) * c);
    float msc = ms * c, sum = 0.f;
#pragma unroll
    for (int nt = 0; nt < NT; ++nt) {
      float p0 = exp2f(fmaf(S[nt][2 * rs], c, -msc)), p1 = exp2f(fmaf(S[nt][2 * rs + 1], c, -msc));
      sum += p0 + p1;
      P[nt][rs] = pack_bf16(p0, p1);
    }
    l[rs] = l[rs] * corr + sum;
    m[rs] = mn;
#pragma unroll
    for (int nt = 0; nt < 16; ++nt) { O[nt][2 * rs] *= corr; O[nt][2 * rs + 1] *= corr; }
  }
}

// scores of n-tile pair starting at token tok0 (16 tokens) for all 8 k-steps
__device__ __forceinline__ void qk_16tok(uint32_t sK, int tok0, const uint32_t (&Qa)[8][4], float (&S0)[4], float (&S1)[4], int lane) {
  int mat = lane >> 3, r = lane & 7;
  int token = tok0 + (mat >> 1) * 8 + r;
  uint32_t rowaddr = sK + token * (HD * 2);
#pragma unroll
  for (int ks = 0; ks < 8; ++ks) {
    int chunk = 2 * ks + (mat & 1);
    uint32_t b0, b1, b2, b3;
    ldsm4(rowaddr + ((chunk ^ r) << 4), b0, b1, b2, b3);
    mma16816(S0, Qa[ks][0], Qa[ks][1], Qa[ks][2], Qa[ks][3], b0, b1);
    mma16816(S1, Qa[ks][0], Qa[ks][1], Qa[ks][2], Qa[ks][3], b2, b3);
  }
}

// O += P(16 rows x 16 tokens starting at tokb) . V
__device__ __forceinline__ void pv_16tok(uint32_t sV, int tokb, uint32_t a0, uint32_t a1, uint32_t a2, uint32_t a3, float (&O)[16][4], int lane) {
  int mat = lane >> 3, r = lane & 7;
  int token = tokb + (mat & 1) * 8 + r;
  uint32_t rowaddr = sV + token * (HD * 2);
#pragma unroll
  for (int np = 0; np < 8; ++np) {
    int chunk = 2 * np + (mat >> 1);
    uint32_t b0, b1, b2, b3;
    ldsm4t(rowaddr + ((chunk ^ r) << 4), b0, b1, b2, b3);
    mma16816(O[2 * np], a0, a1, a2, a3, b0, b1);
    mma16816(O[2 * np + 1], a0, a1, a2, a3, b2, b3);
  }
}

// A work item of the plan (ITEM_INTS ints, 8-byte aligned): first slot, slots, first page, tokens, partial index within the row, prefix?
struct Hdr { int first, n_slots, page_begin, n_tok, chunk_k, is_pre; };
__device__ __forceinline__ Hdr load_hdr(const Params &p, int n_pre, int item) {
  const int2 *it = reinterpret_cast<const int2 *>(item < n_pre ? p.items_pre + (size_t)item * ITEM_INTS : p.items_suf + (size_t)(item - n_pre) * ITEM_INTS);
  const int2 a = it[0], b = it[1], c = it[2];
  return Hdr{a.x, a.y, b.x, b.y, c.x, c.y};
}
// B-operand fragments of Q^T for a unit of <= 8 query rows: lane (g, t) holds row g, dims 16 ks + 2 t (+1) and + 8
__device__ __forceinline__ void load_qb(const Params &p, int first, int n_rows, int kvh, int lane, uint32_t (&Qb)[8][2]) {
  const int g = lane >> 2, t = lane & 3;
  const __nv_bfloat16 *q = g < n_rows ? p.q + ((size_t)(first + (g >> p.rep_shift)) * p.Hq + kvh * p.rep + (g & (p.rep - 1))) * HD : nullptr;
#pragma unroll
  for (int ks = 0; ks < 8; ++ks) {
    const int d = 16 * ks + 2 * t;
    Qb[ks][0] = q ? *reinterpret_cast<const uint32_t *>(q + d) : 0u;
    Qb[ks][1] = q ? *reinterpret_cast<const uint32_t *>(q + d + 8) : 0u;
  }
}

// One token-split unit of <= 8 query rows (a decode row's own pages: n_rows = rep), transposed: S^T = K . Q^T puts the warp's 16 tokens
// on the MMA's m dimension and the query rows on n = 8 — one MMA per k-step instead of two, O^T (128 dims x 8 rows) in 32 accumulators
// instead of 64.  C fragment of S^T: c0/c1 = token g, rows 2t/2t+1; c2/c3 = token g+8.  The four warps' partials meet in the unit's LAST
// page stage — each warp overwrites its own 16 K rows (4 KB = 8 rows x 128 fp32), which nobody else reads — so the merge needs one CTA
// barrier and no scratch of its own; the stage goes back to the producer after the merge.  pbase = part_base[first] (used when n_slots == 1).
__device__ __forceinline__ void tpath_unit(Smem &sm, const Params &p, const Hdr &h, int kvh, int pbase, const uint32_t (&Qb)[8][2],
                                           int &stage, int &phase, int &ubuf, int warp, int lane) {
  const int g = lane >> 2, t = lane & 3;
  const int n_rows = h.n_slots << p.rep_shift, n_tok = h.n_tok;
  int limA = n_tok, limB = n_tok;                                  // token limits of rows 2t and 2t+1
  if (p.causal) {
    const int rA = 2 * t, rB = rA + 1, tok_begin = h.page_begin * PAGE;
    limA = rA < n_rows ? min(n_tok, p.slot_npre[h.first + (rA >> p.rep_shift)] - tok_begin) : 0;
    limB = rB < n_rows ? min(n_tok, p.slot_npre[h.first + (rB >> p.rep_shift)] - tok_begin) : 0;
  }
  float OT[8][4];
#pragma unroll
  for (int i = 0; i < 8; ++i) OT[i][0] = OT[i][1] = OT[i][2] = OT[i][3] = 0.f;
  float mA = -INFINITY, mB = -INFINITY, lA = 0.f, lB = 0.f;
  const int npg = (n_tok + PAGE - 1) / PAGE;
  const int mat = lane >> 3, r8 = lane & 7;
  int last_stage = stage;
  for (int pg = 0; pg < npg; ++pg) {
    mbar_wait(&sm.full[stage], phase);
    const uint32_t sK = smem_u32(sm.stage[stage]), sV = sK + PAGE * HD * 2;
    const int valid = min(PAGE, n_tok - pg * PAGE);
    const int tok0 = warp * 16;
    if (tok0 < valid) {
      float c[4] = {0.f, 0.f, 0.f, 0.f}, c2[4] = {0.f, 0.f, 0.f, 0.f};     // two accumulation chains over the k-steps
      {
        const uint32_t rowaddr = sK + (tok0 + (mat & 1) * 8 + r8) * (HD * 2);
#pragma unroll
        for (int ks = 0; ks < 8; ks += 2) {
          uint32_t a0, a1, a2, a3, e0, e1, e2, e3;
          ldsm4(rowaddr + (((2 * ks + (mat >> 1)) ^ r8) << 4), a0, a1, a2, a3);
          ldsm4(rowaddr + (((2 * ks + 2 + (mat >> 1)) ^ r8) << 4), e0, e1, e2, e3);
          mma16816(c, a0, a1, a2, a3, Qb[ks][0], Qb[ks][1]);
          mma16816(c2, e0, e1, e2, e3, Qb[ks + 1][0], Qb[ks + 1][1]);
        }
#pragma unroll
        for (int j = 0; j < 4; ++j) c[j] += c2[j];
      }
      const int vA = limA - pg * PAGE, vB = limB - pg * PAGE, tkA = tok0 + g, tkB = tkA + 8;
      if (tkA >= vA) c[0] = -INFINITY;
      if (tkA >= vB) c[1] = -INFINITY;
      if (tkB >= vA) c[2] = -INFINITY;
      if (tkB >= vB) c[3] = -INFINITY;
      float mxA = fmaxf(c[0], c[2]), mxB = fmaxf(c[1], c[3]);
#pragma unroll
      for (int o = 4; o <= 16; o <<= 1) {
        mxA = fmaxf(mxA, __shfl_xor_sync(0xffffffffu, mxA, o));
        mxB = fmaxf(mxB, __shfl_xor_sync(0xffffffffu, mxB, o));
      }
      const float mnA = fmaxf(mA, mxA), mnB = fmaxf(mB, mxB);
      const float msA = mnA == -INFINITY ? 0.f : mnA, msB = mnB == -INFINITY ? 0.f : mnB;
      const float corrA = exp2f((mA - msA) * p.c), corrB = exp2f((mB - msB) * p.c);
      const float p0 = exp2f(fmaf(c[0], p.c, -msA * p.c)), p2 = exp2f(fmaf(c[2], p.c, -msA * p.c));
      const float p1 = exp2f(fmaf(c[1], p.c, -msB * p.c)), p3 = exp2f(fmaf(c[3], p.c, -msB * p.c));
      lA = lA * corrA + p0 + p2;
      lB = lB * corrB + p1 + p3;
      mA = mnA;
      mB = mnB;
#pragma unroll
      for (int i = 0; i < 8; ++i) { OT[i][0] *= corrA; OT[i][2] *= corrA; OT[i][1] *= corrB; OT[i][3] *= corrB; }
      // P^T (tokens x rows) -> the B operand (k = tokens, n = rows): transpose the two 8x8 blocks
      uint32_t b0, b1;
      movmatrix_t(pack_bf16(p0, p1), b0);
      movmatrix_t(pack_bf16(p2, p3), b1);
      {
        const uint32_t rowaddr = sV + (tok0 + (mat >> 1) * 8 + r8) * (HD * 2);
#pragma unroll
        for (int i = 0; i < 8; ++i) {
          uint32_t a0, a1, a2, a3;
          ldsm4t(rowaddr + (((2 * i + (mat & 1)) ^ r8) << 4), a0, a1, a2, a3);
          mma16816(OT[i], a0, a1, a2, a3, b0, b1);
        }
      }
    }
    __syncwarp();
    if (pg + 1 < npg) {
      if (lane == 0) mbar_arrive(&sm.empty[stage]);
    } else {
      last_stage = stage;                                          // kept until the merge below has read it
    }
    if (++stage == STAGES) { stage = 0; phase ^= 1; }
  }
#pragma unroll
  for (int o = 4; o <= 16; o <<= 1) {
    lA += __shfl_xor_sync(0xffffffffu, lA, o);
    lB += __shfl_xor_sync(0xffffffffu, lB, o);
  }
  float (*ml)[16][2] = sm.ml[ubuf];
  ubuf ^= 1;
  if (g == 0) {
    ml[warp][2 * t][0] = mA; ml[warp][2 * t][1] = lA;
    ml[warp][2 * t + 1][0] = mB; ml[warp][2 * t + 1][1] = lB;
  }
  // partial of this warp: [row][128] fp32, the columns of rows 2t, 2t+1 rotated by 8 t (bank-conflict-free writes)
  unsigned char *part = sm.stage[last_stage];
  if (2 * t < n_rows) {
    float *mine = reinterpret_cast<float *>(part + warp * 4096) + 2 * t * HD;
#pragma unroll
    for (int i = 0; i < 8; ++i) {
      const int c0 = (16 * i + g + 8 * t) & (HD - 1), c1 = (c0 + 8) & (HD - 1);
      mine[c0] = OT[i][0]; mine[HD + c0] = OT[i][1];
      mine[c1] = OT[i][2]; mine[HD + c1] = OT[i][3];
    }
  }
  cons_bar();
  for (int r = warp; r < n_rows; r += N_CONS) {
    float M = -INFINITY;
#pragma unroll
    for (int wv = 0; wv < N_CONS; ++wv) M = fmaxf(M, ml[wv][r][0]);
    float L = 0.f, a0 = 0.f, a1 = 0.f, a2 = 0.f, a3 = 0.f;
    const int col = (lane * 4 + 8 * (r >> 1)) & (HD - 1);
#pragma unroll
    for (int wv = 0; wv < N_CONS; ++wv) {
      const float sc = exp2f((ml[wv][r][0] - M) * p.c);
      const float4 v = *reinterpret_cast<const float4 *>(reinterpret_cast<const float *>(part + wv * 4096) + r * HD + col);
      L += sc * ml[wv][r][1];
      a0 += sc * v.x; a1 += sc * v.y; a2 += sc * v.z; a3 += sc * v.w;
    }
    const int slot = h.first + (r >> p.rep_shift), head = kvh * p.rep + (r & (p.rep - 1));
    const int pb = h.n_slots == 1 ? pbase : p.part_base[slot];
    const size_t pi = (size_t)(pb + h.chunk_k) * p.Hq + head;
    if (lane == 0) { p.part_ml[pi * 2] = M; p.part_ml[pi * 2 + 1] = L; }
    *reinterpret_cast<float4 *>(p.part_acc + pi * HD + lane * 4) = make_float4(a0, a1, a2, a3);
  }
  // the stage's next user is the producer's bulk copy (async proxy): order this warp's generic accesses before it
  asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
  __syncwarp();
  if (lane == 0) mbar_arrive(&sm.empty[last_stage]);
}

// One round of the cross-warp merge of a token-split unit: rows 4 rb .. 4 rb + 3, one consumer warp per row, 4 dims per lane.
__device__ __forceinline__ void merge_round(Smem &sm, const float (*ml)[16][2], const Params &p, int rb, int n_rows, int first, int kvh, int chunk_k) {
  int rr = threadIdx.x >> 5, d4 = (threadIdx.x & 31) * 4;     // 128 consumer threads: row rr, dims d4..d4+3
  int r = rb * 4 + rr;
  if (r < n_rows) {
    float M = -INFINITY;
#pragma unroll
    for (int wv = 0; wv < N_CONS; ++wv) M = fmaxf(M, ml[wv][r][0]);
    float L = 0.f, a0 = 0.f, a1 = 0.f, a2 = 0.f, a3 = 0.f;
#pragma unroll
    for (int wv = 0; wv < N_CONS; ++wv) {
      float sc = exp2f((ml[wv][r][0] - M) * p.c);
      float4 v = *reinterpret_cast<const float4 *>(&sm.scratch[wv][rr][d4]);
      L += sc * ml[wv][r][1];
      a0 += sc * v.x; a1 += sc * v.y; a2 += sc * v.z; a3 += sc * v.w;
    }
    int slot = first + (r >> p.rep_shift), head = kvh * p.rep + (r & (p.rep - 1));
    size_t pi = (size_t)(p.part_base[slot] + chunk_k) * p.Hq + head;
    if ((threadIdx.x & 31) == 0) { p.part_ml[pi * 2] = M; p.part_ml[pi * 2 + 1] = L; }
    *reinterpret_cast<float4 *>(p.part_acc + pi * HD + d4) = make_float4(a0, a1, a2, a3);
  }
}

__global__ void __launch_bounds__(THREADS, 2) attn_main_k(Params p) {
  extern __shared__ unsigned char smem_raw[];
  Smem &sm = *reinterpret_cast<Smem *>(((uintptr_t)smem_raw + 127) & ~(uintptr_t)127);
  int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  if (threadIdx.x == 0) {
    for (int s = 0; s < STAGES; ++s) { mbar_init(&sm.full[s], 1); mbar_init(&sm.empty[s], N_CONS); }
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  pdl_trigger();
  // The plan (items, partial indices) and the page tables were written at the step boundary, by ordinary launches that everything in the
  // layer chain comes after: they are read BEFORE the wait.  q and the KV rows appended this step come from the previous kernel.
  int n_pre = p.n_items[0], n_suf = p.n_items[1];
  const int total = (n_pre + n_suf) * p.Hkv;            // work units (item, kv head); attn_max_items * Hkv < 2^31
  const int d_item = (int)gridDim.x / p.Hkv, d_kvh = (int)gridDim.x % p.Hkv;
  int stage = 0, phase = 0;
  Hdr h_first{};                                        // producer lane: its first unit's item, page table and first page id
  const int32_t *table_first = nullptr;
  int page_first = 0;
  if (threadIdx.x == N_CONS * 32 && (int)blockIdx.x < total) {
    h_first = load_hdr(p, n_pre, (int)blockIdx.x / p.Hkv);
    table_first = h_first.is_pre ? p.g_prefix_pages + (size_t)p.slot_prompt[h_first.first] * p.mpp : p.row_pages + (size_t)p.slot_row[h_first.first] * p.msp;
    page_first = table_first[h_first.page_begin];
  }
  pdl_wait();
  __syncthreads();

  if (warp == N_CONS) {
    // ------------------------------------------------------------------ producer: one lane streams the pages
    if (lane == 0) {
      int item = (int)blockIdx.x / p.Hkv, kvh = (int)blockIdx.x % p.Hkv;
      for (int w = blockIdx.x; w < total; w += gridDim.x, item += d_item, kvh += d_kvh) {
        if (kvh >= p.Hkv) { kvh -= p.Hkv; ++item; }
        const bool first_unit = w == (int)blockIdx.x;
        const Hdr h = first_unit ? h_first : load_hdr(p, n_pre, item);
        const int first = h.first, page_begin = h.page_begin, n_tok = h.n_tok;
        const int32_t *table = first_unit ? table_first
                               : h.is_pre ? p.g_prefix_pages + (size_t)p.slot_prompt[first] * p.mpp : p.row_pages + (size_t)p.slot_row[first] * p.msp;
        int npg = (n_tok + PAGE - 1) / PAGE;
        // A row's NEWEST page is on average half empty, and a whole tile pair is 32 KB: at 512 rows that is ~67 MB per layer of bytes nobody
        // reads.  For a unit whose query rows fit one m-tile (the token-split path: a warp skips a 16-token group that lies wholly beyond the
        // valid tokens, so un-copied shared memory is never touched) the last page is fetched as the valid part of K and of V, rounded up to
        // 16 tokens — two smaller copies; only when that saves at least half of the tile.
        const bool tok_split = ATTN_PARTIAL_LAST_PAGE && h.n_slots * p.rep <= 16 && !p.causal;
        for (int pg = 0; pg < npg; ++pg) {
          mbar_wait(&sm.empty[stage], phase ^ 1);
          const int page_id = first_unit && pg == 0 ? page_first : table[page_begin + pg];
          const __nv_bfloat16 *src = p.kv_layer + (size_t)page_id * p.page_elems + (size_t)kvh * 2 * p.tile_elems;
          const int v16 = (min(PAGE, n_tok - pg * PAGE) + 15) & ~15;
          if (tok_split && v16 <= PAGE / 2) {
            const int bytes = v16 * HD * 2;
            mbar_expect_tx(&sm.full[stage], 2 * bytes);
            bulk_g2s(sm.stage[stage], src, bytes, &sm.full[stage]);
            bulk_g2s(sm.stage[stage] + PAGE * HD * 2, src + PAGE * HD, bytes, &sm.full[stage]);
          } else {
            mbar_expect_tx(&sm.full[stage], STAGE_BYTES);
            bulk_g2s(sm.stage[stage], src, STAGE_BYTES, &sm.full[stage]);
          }
          if (++stage == STAGES) { stage = 0; phase ^= 1; }
        }
      }
    }
    return;
  }

  // -------------------------------------------------------------------- consumers
  int g = lane >> 2, t = lane & 3;
  int item = (int)blockIdx.x / p.Hkv, kvh = (int)blockIdx.x % p.Hkv;
  int ubuf = 0;                                                    // which sm.ml buffer the next unit uses
  // With rep <= 8 every suffix unit (one row's own pages) takes the transposed path: those run in a software-pipelined loop of their
  // own below; this loop then serves the prefix units only.
  const bool suffix_t = ATTN_TPATH && p.rep <= 8;
  const int gen_end = suffix_t ? n_pre * p.Hkv : total;
  int w = blockIdx.x;
  for (; w < gen_end; w += gridDim.x, item += d_item, kvh += d_kvh) {
    if (kvh >= p.Hkv) { kvh -= p.Hkv; ++item; }
    const Hdr hd = load_hdr(p, n_pre, item);
    int first = hd.first, n_slots = hd.n_slots, n_tok = hd.n_tok, chunk_k = hd.chunk_k;
    int n_rows = n_slots * p.rep;
    const int tok_begin = hd.page_begin * PAGE;                    // first token of this item within its page table
    if (ATTN_TPATH && n_rows <= 8) {
      uint32_t Qb[8][2];
      load_qb(p, hd.first, n_rows, kvh, lane, Qb);
      tpath_unit(sm, p, hd, kvh, p.part_base[hd.first], Qb, stage, phase, ubuf, warp, lane);
      continue;
    }
    bool rowsplit = n_rows > 16;
    int mt = rowsplit ? warp : 0;                                  // m-tile this warp works on
    bool warp_has_rows = mt * 16 < n_rows;
    // Q fragments (A operand) of this warp's m-tile: rows r = 16 mt + g (+8)
    uint32_t Qa[8][4];
    {
      int r0 = mt * 16 + g, r1 = r0 + 8;
      const __nv_bfloat16 *q0 = r0 < n_rows ? p.q + ((size_t)(first + (r0 >> p.rep_shift)) * p.Hq + kvh * p.rep + (r0 & (p.rep - 1))) * HD : nullptr;
      const __nv_bfloat16 *q1 = r1 < n_rows ? p.q + ((size_t)(first + (r1 >> p.rep_shift)) * p.Hq + kvh * p.rep + (r1 & (p.rep - 1))) * HD : nullptr;
#pragma unroll
      for (int ks = 0; ks < 8; ++ks) {
        int d = 16 * ks + 2 * t;
        Qa[ks][0] = q0 ? *reinterpret_cast<const uint32_t *>(q0 + d) : 0u;
        Qa[ks][1] = q1 ? *reinterpret_cast<const uint32_t *>(q1 + d) : 0u;
        Qa[ks][2] = q0 ? *reinterpret_cast<const uint32_t *>(q0 + d + 8) : 0u;
        Qa[ks][3] = q1 ? *reinterpret_cast<const uint32_t *>(q1 + d + 8) : 0u;
      }
    }
    // per-row token limit inside this item (rows g and g+8 of the warp's m-tile): n_tok, or the causal bound of a prefill pass
    int lim0 = n_tok, lim1 = n_tok;
    if (p.causal) {
      int r0 = mt * 16 + g, r1 = r0 + 8;
      lim0 = r0 < n_rows ? min(n_tok, p.slot_npre[first + (r0 >> p.rep_shift)] - tok_begin) : 0;
      lim1 = r1 < n_rows ? min(n_tok, p.slot_npre[first + (r1 >> p.rep_shift)] - tok_begin) : 0;
    }
    float O[16][4];
#pragma unroll
    for (int nt = 0; nt < 16; ++nt) O[nt][0] = O[nt][1] = O[nt][2] = O[nt][3] = 0.f;
    float m[2] = {-INFINITY, -INFINITY}, l[2] = {0.f, 0.f};
    int npg = (n_tok + PAGE - 1) / PAGE;
    for (int pg = 0; pg < npg; ++pg) {
      mbar_wait(&sm.full[stage], phase);
      uint32_t sK = smem_u32(sm.stage[stage]), sV = sK + PAGE * HD * 2;
      int valid = min(PAGE, n_tok - pg * PAGE);
      const int v0 = lim0 - pg * PAGE, v1 = lim1 - pg * PAGE;       // row-wise valid tokens of this page (may be <= 0 or >= PAGE)
      if (!rowsplit) {
        int tok0 = warp * 16;                                      // this warp's 16 tokens of the page
        if (tok0 < valid) {
          float S[2][4] = {};
          qk_16tok(sK, tok0, Qa, S[0], S[1], lane);
#pragma unroll
          for (int nt = 0; nt < 2; ++nt) {
            int tk = tok0 + nt * 8 + 2 * t;
            if (tk >= v0) S[nt][0] = -INFINITY;
            if (tk + 1 >= v0) S[nt][1] = -INFINITY;
            if (tk >= v1) S[nt][2] = -INFINITY;
            if (tk + 1 >= v1) S[nt][3] = -INFINITY;
          }
          uint32_t P[2][2];
          softmax_update<2>(S, m, l, O, P, p.c);
          pv_16tok(sV, tok0, P[0][0], P[0][1], P[1][0], P[1][1], O, lane);
        }
      } else if (warp_has_rows) {
        float S[8][4] = {};
        {
          // k-step outermost: the eight accumulators are independent MMA chains (one 16-token group at a time is two chains of eight
          // dependent MMAs, and two warps per scheduler cannot hide their latency)
          const int mat = lane >> 3, r = lane & 7;
          const uint32_t rowaddr = sK + ((mat >> 1) * 8 + r) * (HD * 2);
#pragma unroll
          for (int ks = 0; ks < 8; ++ks) {
            const uint32_t off = ((2 * ks + (mat & 1)) ^ r) << 4;
#pragma unroll
            for (int np = 0; np < 4; ++np) {
              uint32_t b0, b1, b2, b3;
              ldsm4(rowaddr + np * 16 * (HD * 2) + off, b0, b1, b2, b3);
              mma16816(S[2 * np], Qa[ks][0], Qa[ks][1], Qa[ks][2], Qa[ks][3], b0, b1);
              mma16816(S[2 * np + 1], Qa[ks][0], Qa[ks][1], Qa[ks][2], Qa[ks][3], b2, b3);
            }
          }
        }
        if (min(v0, v1) < PAGE) {
#pragma unroll
          for (int nt = 0; nt < 8; ++nt) {
            int tk = nt * 8 + 2 * t;
            if (tk >= v0) S[nt][0] = -INFINITY;
            if (tk + 1 >= v0) S[nt][1] = -INFINITY;
            if (tk >= v1) S[nt][2] = -INFINITY;
            if (tk + 1 >= v1) S[nt][3] = -INFINITY;
          }
        }
        uint32_t P[8][2];
        softmax_update<8>(S, m, l, O, P, p.c);
#pragma unroll
        for (int kt = 0; kt < 4; ++kt) pv_16tok(sV, kt * 16, P[2 * kt][0], P[2 * kt][1], P[2 * kt + 1][0], P[2 * kt + 1][1], O, lane);
      }
      __syncwarp();
      if (lane == 0) mbar_arrive(&sm.empty[stage]);
      if (++stage == STAGES) { stage = 0; phase ^= 1; }
    }
    // row sums live in quads: reduce
#pragma unroll
    for (int rs = 0; rs < 2; ++rs) {
      l[rs] += __shfl_xor_sync(0xffffffffu, l[rs], 1);
      l[rs] += __shfl_xor_sync(0xffffffffu, l[rs], 2);
    }
    if (rowsplit) {
      // each warp owns its rows: write the partial directly
#pragma unroll
      for (int rs = 0; rs < 2; ++rs) {
        int r = mt * 16 + g + 8 * rs;
        if (r < n_rows) {
          int slot = first + (r >> p.rep_shift), head = kvh * p.rep + (r & (p.rep - 1));
          size_t pi = (size_t)(p.part_base[slot] + chunk_k) * p.Hq + head;
          if (t == 0) { p.part_ml[pi * 2] = m[rs]; p.part_ml[pi * 2 + 1] = l[rs]; }
#pragma unroll
          for (int nt = 0; nt < 16; ++nt)
            *reinterpret_cast<float2 *>(p.part_acc + pi * HD + nt * 8 + 2 * t) = make_float2(O[nt][2 * rs], O[nt][2 * rs + 1]);
        }
      }
    } else {
      // the four warps hold partials over disjoint tokens of the same <= 16 rows: merge through shared memory
      float (*ml)[16][2] = sm.ml[ubuf];
      ubuf ^= 1;
      if (t == 0) {
        ml[warp][g][0] = m[0]; ml[warp][g][1] = l[0];
        ml[warp][g + 8][0] = m[1]; ml[warp][g + 8][1] = l[1];
      }
      int rounds = (n_rows + 3) >> 2;
      for (int rb = 0; rb < rounds; ++rb) {
        int rs = rb >> 1, glo = (rb & 1) * 4;
        if (g >= glo && g < glo + 4) {
#pragma unroll
          for (int nt = 0; nt < 16; ++nt)
            *reinterpret_cast<float2 *>(&sm.scratch[warp][g - glo][nt * 8 + 2 * t]) = rs == 0 ? make_float2(O[nt][0], O[nt][1]) : make_float2(O[nt][2], O[nt][3]);
        }
        cons_bar();
        merge_round(sm, ml, p, rb, n_rows, first, kvh, chunk_k);
        cons_bar();
      }
    }
  }
  if (!suffix_t || w >= total) return;
  // ---- suffix units, software-pipelined: a unit's header is loaded two units ahead, its Q fragments and partial index one unit ahead,
  // so that no dependent global load is left at a unit's start (at short contexts a unit is one page: the chain was most of its time)
  if (kvh >= p.Hkv) { kvh -= p.Hkv; ++item; }
  Hdr h = load_hdr(p, n_pre, item);
  int w1 = w + gridDim.x, item1 = item + d_item, kvh1 = kvh + d_kvh;
  if (kvh1 >= p.Hkv) { kvh1 -= p.Hkv; ++item1; }
  Hdr h1 = w1 < total ? load_hdr(p, n_pre, item1) : h;
  uint32_t Qb[8][2];
  load_qb(p, h.first, p.rep, kvh, lane, Qb);
  int pb = p.part_base[h.first];
  while (true) {
    const bool has1 = w1 < total;
    int w2 = w1 + gridDim.x, item2 = item1 + d_item, kvh2 = kvh1 + d_kvh;
    if (kvh2 >= p.Hkv) { kvh2 -= p.Hkv; ++item2; }
    uint32_t Qn[8][2];
    int pbn = 0;
    Hdr h2 = h1;
    if (has1) {
      load_qb(p, h1.first, p.rep, kvh1, lane, Qn);
      pbn = p.part_base[h1.first];
      if (w2 < total) h2 = load_hdr(p, n_pre, item2);
    }
    tpath_unit(sm, p, h, kvh, pb, Qb, stage, phase, ubuf, warp, lane);
    if (!has1) break;
    h = h1; kvh = kvh1; pb = pbn;
#pragma unroll
    for (int ks = 0; ks < 8; ++ks) { Qb[ks][0] = Qn[ks][0]; Qb[ks][1] = Qn[ks][1]; }
    h1 = h2; w1 = w2; item1 = item2; kvh1 = kvh2;
  }
}

// ------------------------------------------------------------------------------------------------ merge
// out[slot][h] = sum_k w_k acc_k / sum_k w_k l_k,  w_k = 2^((m_k - M) c), over the row's partials in chunk order.
__global__ void attn_merge_k(const float *__restrict__ part_ml, const float *__restrict__ part_acc, const int32_t *__restrict__ part_base,
                             const int32_t *__restrict__ part_cnt, __nv_bfloat16 *__restrict__ out, int Hq, float c,
                             const int32_t *n_rows_dev, int rows_ub) {
  pdl_trigger();
  int slot = blockIdx.x;
  int R = n_rows_dev ? min(*n_rows_dev, rows_ub) : rows_ub;   // row count and plan: fixed at the step boundary, read before the wait
  if (slot >= R) return;
  int lane = threadIdx.x & 31;
  int base = part_base[slot], cnt = part_cnt[slot];
  pdl_wait();
  for (int h = blockIdx.y * (blockDim.x >> 5) + (threadIdx.x >> 5); h < Hq; h += gridDim.y * (blockDim.x >> 5)) {   // one head per warp
    float M = -INFINITY, L = 0.f;
    float4 a = make_float4(0.f, 0.f, 0.f, 0.f);
    if (cnt <= 4) {
      // the common case (prefix chunk + up to three suffix chunks): every load of the row is issued before the first use — one L2
      // round trip instead of two dependent passes; the sums below run in chunk order as in the general loop
      float2 ml[4];
      float4 v[4];
#pragma unroll
      for (int k = 0; k < 4; ++k)
        if (k < cnt) {
          const size_t pi = (size_t)(base + k) * Hq + h;
          ml[k] = *reinterpret_cast<const float2 *>(part_ml + pi * 2);
          v[k] = *reinterpret_cast<const float4 *>(part_acc + pi * HD + lane * 4);
        }
#pragma unroll
      for (int k = 0; k < 4; ++k)
        if (k < cnt) M = fmaxf(M, ml[k].x);
#pragma unroll
      for (int k = 0; k < 4; ++k)
        if (k < cnt) {
          const float sc = exp2f((ml[k].x - M) * c);
          L += sc * ml[k].y;
          a.x += sc * v[k].x; a.y += sc * v[k].y; a.z += sc * v[k].z; a.w += sc * v[k].w;
        }
    } else {
      for (int k = 0; k < cnt; ++k) M = fmaxf(M, part_ml[((size_t)(base + k) * Hq + h) * 2]);
      for (int k = 0; k < cnt; ++k) {
        size_t pi = (size_t)(base + k) * Hq + h;
        float sc = exp2f((part_ml[pi * 2] - M) * c);
        L += sc * part_ml[pi * 2 + 1];
        float4 v = *reinterpret_cast<const float4 *>(part_acc + pi * HD + lane * 4);
        a.x += sc * v.x; a.y += sc * v.y; a.z += sc * v.z; a.w += sc * v.w;
      }
    }
    float inv = 1.0f / L;
    uint2 o;
    o.x = pack_bf16(a.x * inv, a.y * inv);
    o.y = pack_bf16(a.z * inv, a.w * inv);
    *reinterpret_cast<uint2 *>(out + ((size_t)slot * Hq + h) * HD + lane * 4) = o;
  }
}

// ------------------------------------------------------------------------------------------------ plan (one CTA)
__device__ __forceinline__ int scan1024(int v, int *total, int *smem) {
  int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  int incl = v;
#pragma unroll
  for (int o = 1; o < 32; o <<= 1) {
    int x = __shfl_up_sync(0xffffffffu, incl, o);
    if (lane >= o) incl += x;
  }
  if (lane == 31) smem[warp] = incl;
  __syncthreads();
  if (warp == 0) {
    int wv = lane < (int)(blockDim.x >> 5) ? smem[lane] : 0, wi = wv;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
      int x = __shfl_up_sync(0xffffffffu, wi, o);
      if (lane >= o) wi += x;
    }
    smem[lane] = wi - wv;
    if (lane == 31) smem[32] = wi;
  }
  __syncthreads();
  int res = smem[warp] + incl - v;
  *total = smem[32];
  __syncthreads();
  return res;
}

__global__ void attn_plan_k(const int32_t *__restrict__ slot_prompt, const int32_t *__restrict__ slot_npre,
                            const int32_t *__restrict__ slot_nsuf, int32_t *items_pre, int32_t *items_suf, int32_t *n_items,
                            int32_t *part_base, int32_t *part_cnt, int rep, int no_share, int prefill, int max_items,
                            const int32_t *n_rows_dev, int rows_ub, int cm_max_items) {
  __shared__ int sm[33];
  __shared__ int b_part, b_pre, b_suf;
  int n = n_rows_dev ? min(*n_rows_dev, rows_ub) : rows_ub;
  if (threadIdx.x == 0) { b_part = 0; b_pre = 0; b_suf = 0; }
  __syncthreads();
  int RB = 64 / rep;                                   // slots per ROWSPLIT item (64 query rows)
  // In a rollout every live row has the same generated length (lock step), hence the same number of suffix chunks.  While a launch has
  // only a few units per CTA (n x chunks <= cm_max_items: the thin tail of a rollout) the suffix items are written CHUNK-major (all rows'
  // chunk 0, then chunk 1, ...), so that the last round of the kernel's strided unit assignment is made of the rows' short newest chunks
  // instead of whole 512-token ones: -2 % per decode step at <= 64 rows.  With many units per CTA the row-major order wins by 1-2 % (a row's
  // consecutive pages) and is kept.  The order of the items changes nothing else: every unit's arithmetic and partial index are its own.
  // Rows of different lengths (chunk scoring, the attention-only entry) keep the row-major order.
  int uniform_nsc = 0;
  if (ATTN_CHUNK_MAJOR && !prefill && n > 0) {
    const int nsc0 = (slot_nsuf[0] + CH_TOK - 1) / CH_TOK;
    bool same = (long long)n * nsc0 <= cm_max_items;
    for (int slot = threadIdx.x; slot < n; slot += blockDim.x) same &= (slot_nsuf[slot] + CH_TOK - 1) / CH_TOK == nsc0;
    if (__syncthreads_and(same)) uniform_nsc = nsc0;
  }
  for (int base = 0; base < n; base += blockDim.x) {
    int slot = base + threadIdx.x;
    int npc = 0, nsc = 0, gsize = 0, nblk = 0, npre_items = 0;
    if (slot < n) {
      npc = (slot_npre[slot] + CH_TOK - 1) / CH_TOK;
      nsc = (slot_nsuf[slot] + CH_TOK - 1) / CH_TOK;
      int pr = slot_prompt[slot];
      if (prefill) {
        // causal pass over prompt tokens: slot = token at position npre-1.  A block = RB consecutive positions of one prompt
        // (RB divides the 512-token chunk, so its slots need the same chunks); its items run up to the block's LAST position
        // and the kernel masks row-wise (Params::causal).
        bool leader = (slot_npre[slot] - 1) % RB == 0;
        if (leader) {
          gsize = 1;
          while (gsize < RB && slot + gsize < n && slot_prompt[slot + gsize] == pr) ++gsize;
          nblk = 1;
          npre_items = slot_npre[slot + gsize - 1];
        }
      } else {
        bool leader = no_share || slot == 0 || slot_prompt[slot - 1] != pr;
        if (leader) {
          gsize = 1;
          if (!no_share) while (slot + gsize < n && slot_prompt[slot + gsize] == pr) ++gsize;
          nblk = gsize * rep <= 16 ? 1 : (gsize + RB - 1) / RB;
          npre_items = slot_npre[slot];
        }
      }
    }
    int tp, tq, ts;
    int ep = scan1024(npc + nsc, &tp, sm);
    int eq = scan1024(nblk * npc, &tq, sm);
    int es = scan1024(nsc, &ts, sm);
    int bp = b_part, bq = b_pre, bs = b_suf;
    if (slot < n) {
      part_base[slot] = bp + ep;
      part_cnt[slot] = npc + nsc;
      int idx = bq + eq;
      int per = nblk <= 1 ? gsize : RB;
      for (int b = 0; b < nblk; ++b)
        for (int ck = 0; ck < npc; ++ck, ++idx) {
          if (idx >= max_items) continue;
          int32_t *it = items_pre + (size_t)idx * ITEM_INTS;
          it[0] = slot + b * per;
          it[1] = min(per, gsize - b * per);
          it[2] = ck * CH_PAGES;
          it[3] = min(CH_TOK, npre_items - ck * CH_TOK);
          it[4] = ck;
          it[5] = 1;
        }
      for (int ck = 0; ck < nsc; ++ck) {
        idx = uniform_nsc ? ck * n + slot : bs + es + ck;
        if (idx >= max_items) continue;
        int32_t *it = items_suf + (size_t)idx * ITEM_INTS;
        it[0] = slot; it[1] = 1; it[2] = ck * CH_PAGES;
        it[3] = min(CH_TOK, slot_nsuf[slot] - ck * CH_TOK);
        it[4] = npc + ck; it[5] = 0;
      }
    }
    __syncthreads();
    if (threadIdx.x == 0) { b_part = bp + tp; b_pre = bq + tq; b_suf = bs + ts; }
    __syncthreads();
  }
  if (threadIdx.x == 0) { n_items[0] = min(b_pre, max_items); n_items[1] = min(b_suf, max_items); n_items[2] = b_part; }
}

}  // namespace

size_t attn_sm100_smem_bytes() { return sizeof(Smem) + 128; }

// Plan once per decode step (the lengths are the same for every layer), then per layer: main + merge.
darts_status launch_attention_plan_sm100(darts_ctx *c, int rows_ub, const int32_t *n_rows_dev, bool prefill) {
  int rep = c->m.n_q_heads / c->m.n_kv_heads;
  attn_plan_k<<<1, 1024, 0, c->stream>>>(c->slot_prompt, c->slot_npre, c->slot_nsuf, c->attn_items_pre, c->attn_items_suf, c->attn_nitems,
                                         c->part_base, c->part_cnt, rep, (c->rt.flags & DARTS_FLAG_NO_PREFIX_SHARING) ? 1 : 0, prefill ? 1 : 0,
                                         c->attn_max_items, n_rows_dev, rows_ub, 8 * (2 * c->n_sms) / c->m.n_kv_heads);   // <= 8 suffix units per CTA
  c->attn_causal = prefill;
  c->launches++;
  if (cudaGetLastError() != cudaSuccess) FAIL(c, DARTS_ERR_CUDA, "launch attn_plan failed");
  return DARTS_OK;
}

darts_status attn_sm100_configure(darts_ctx *c) {
  CUDA_TRY(c, cudaFuncSetAttribute(attn_main_k, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)attn_sm100_smem_bytes()));
  return DARTS_OK;
}

bool attention_sm100_supported(const darts_ctx *c) {
  int rep = c->m.n_q_heads / c->m.n_kv_heads;
  return c->m.dtype == DARTS_BF16 && c->m.head_dim == HD && c->rt.page_size == PAGE && (rep == 1 || rep == 2 || rep == 4 || rep == 8 || rep == 16);
}

darts_status launch_attention_sm100(darts_ctx *c, int layer, const void *q, void *out, int rows_ub, const int32_t *n_rows_dev, bool *taken) {
  *taken = false;
  if (!attention_sm100_supported(c) || !c->attn_plan_valid) return DARTS_OK;
  *taken = true;
  size_t smem = attn_sm100_smem_bytes();
  Params p;
  p.q = (const __nv_bfloat16 *)q;
  p.kv_layer = (const __nv_bfloat16 *)c->kv_pool + (size_t)layer * c->kv_layer_elems;
  p.items_pre = c->attn_items_pre; p.items_suf = c->attn_items_suf; p.n_items = c->attn_nitems;
  p.slot_prompt = c->slot_prompt; p.slot_row = c->slot_row; p.slot_npre = c->slot_npre; p.causal = c->attn_causal ? 1 : 0; p.g_prefix_pages = c->g_prefix_pages; p.row_pages = c->row_pages;
  p.part_base = c->part_base; p.part_ml = c->part_ml; p.part_acc = c->part_acc;
  p.mpp = c->max_prefix_pages; p.msp = c->max_suffix_pages; p.Hq = c->m.n_q_heads; p.Hkv = c->m.n_kv_heads; p.rep = p.Hq / p.Hkv;
  p.rep_shift = 31 - __builtin_clz((unsigned)p.rep);
  p.page_elems = c->kv_page_elems; p.tile_elems = c->kv_tile_elems;
  p.c = 1.4426950408889634f / sqrtf((float)HD);
  int grid = c->n_sms * 2;
  if (!DARTS_SKIPPED(c, 4)) launch_pdl(c, attn_main_k, dim3(grid), dim3(THREADS), smem, p);
  c->launches++;
  if (cudaGetLastError() != cudaSuccess) FAIL(c, DARTS_ERR_CUDA, "launch attn_main failed: %s", cudaGetErrorString(cudaGetLastError()));
  if (!DARTS_SKIPPED(c, 8)) launch_pdl(c, attn_merge_k, dim3(rows_ub, (p.Hq + 7) / 8), dim3(256), 0, c->part_ml, c->part_acc, c->part_base, c->part_cnt, (__nv_bfloat16 *)out, p.Hq, p.c, n_rows_dev, rows_ub);
  c->launches++;
  if (cudaGetLastError() != cudaSuccess) FAIL(c, DARTS_ERR_CUDA, "launch attn_merge failed");
  return DARTS_OK;
}
