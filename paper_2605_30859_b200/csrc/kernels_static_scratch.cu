// darts_gemm_bf16_static (include/darts.h): the stream-K tcgen05 GEMM of the decode projections for callers
// that cannot allocate — CUDA-graph capture, tight serving loops, harnesses that forbid cudaMalloc.  The kernel cuts every 128-row weight
// tile's K range into fp32 PIECES that a second kernel adds in slot order (kernels_gemm_sk.cu); on the other paths those pieces live in the
// caller's workspace (decode step) or in a caller-provided buffer (darts_debug_gemm_bf16).  Here they live in ONE file-scope device array
// of DARTS_STATIC_SCRATCH_BYTES that every GPU holds from the moment it loads the library until the process exits; the caller passes only
// the inputs and the output.
//
// The call allocates nothing: no cudaMalloc / cudaFree / cudaMallocHost, no allocating library routine — tensor-map encoding is host
// arithmetic, the rest is two kernel launches and one 8 KB cudaMemsetAsync on the context's stream.
//
// The array is SHARED by every call in the process on that GPU and keeps the last call's contents:
//   * layout: [0, 8 KB) the piece-count table of the stream-K plan (int32 per tile), [8 KB, ...) the pieces [slot][rows][N] fp32;
//   * every piece and every piece count a call reads is written by that call's own GEMM first; the piece-count table is nevertheless cleared
//     at the start of every call (an entry the GEMM failed to write would otherwise be a stale count from another shape);
//   * two calls that overlap on the GPU (different contexts / streams, or two processes' worth of threads on one context) RACE on it.
//     Calls on one context are ordered by its stream and are safe back to back.
#include <mutex>

#include "internal.cuh"

static __device__ __align__(256) unsigned char g_static_scratch[DARTS_STATIC_SCRATCH_BYTES];

namespace {

#define TRY(x) do { darts_status s__ = (x); if (s__ != DARTS_OK) return s__; } while (0)

constexpr int MAX_DEVICES = 64;
constexpr size_t NP_BYTES = (size_t)SK_NP_TABLE * sizeof(int32_t);   // 8 KB, keeps the pieces 256-byte aligned
static_assert(NP_BYTES % 256 == 0, "pieces must stay 256-byte aligned behind the table");
static_assert(DARTS_STATIC_SCRATCH_BYTES > NP_BYTES, "static scratch smaller than its own header");

std::mutex g_mu;
void *g_dev_ptr[MAX_DEVICES];                         // device address of g_static_scratch on each device, looked up once per device

// In host code `g_static_scratch` is only the symbol's host-side stand-in, NOT a device address: the address a kernel can use comes from
// cudaGetSymbolAddress, with the device in question current.
darts_status static_scratch_base(darts_ctx *c, unsigned char **out) {
  int dev = -1;
  CUDA_TRY(c, cudaGetDevice(&dev));
  if (dev < 0 || dev >= MAX_DEVICES) FAIL(c, DARTS_ERR_UNSUPPORTED, "device ordinal %d outside [0, %d)", dev, MAX_DEVICES);
  std::lock_guard<std::mutex> lock(g_mu);
  if (!g_dev_ptr[dev]) {
    void *p = nullptr;
    cudaError_t e = cudaGetSymbolAddress(&p, g_static_scratch);
    if (e != cudaSuccess || !p) {
      snprintf(c->err, sizeof(c->err), "cudaGetSymbolAddress(static scratch) on device %d: %s", dev, cudaGetErrorString(e));
      return DARTS_ERR_CUDA;
    }
    g_dev_ptr[dev] = p;
  }
  *out = (unsigned char *)g_dev_ptr[dev];
  return DARTS_OK;
}

}  // namespace

extern "C" darts_status darts_static_scratch_bytes(size_t *out) {
  if (!out) return DARTS_ERR_INVALID_ARG;
  *out = (size_t)DARTS_STATIC_SCRATCH_BYTES;
  return DARTS_OK;
}

extern "C" darts_status darts_gemm_bf16_static(darts_ctx *c, const void *X, const void *W, float *C, int32_t rows, int32_t N, int32_t K) {
  if (!c) return DARTS_ERR_INVALID_ARG;
  if (c->sticky) return c->sticky;
  if (!X || !W || !C || rows <= 0 || N <= 0 || K <= 0) FAIL(c, DARTS_ERR_INVALID_ARG, "NULL / non-positive argument");
  if (!tc_shape_ok(N, K)) FAIL(c, DARTS_ERR_UNSUPPORTED, "tcgen05 GEMM needs K %% 64 == 0, N %% 4 == 0");
  const SkPlan plan = sk_plan(c->n_sms, N, K, rows, 0, true);
  const size_t need = NP_BYTES + (size_t)plan.slots * rows * N * sizeof(float);
  if (need > (size_t)DARTS_STATIC_SCRATCH_BYTES)
    FAIL(c, DARTS_ERR_WORKSPACE_TOO_SMALL,
         "darts_gemm_bf16_static: rows=%d N=%d K=%d needs %zu bytes of pieces (%d slots), the static scratch holds %zu; use darts_debug_gemm_bf16 "
         "with a caller-provided buffer",
         rows, N, K, need, plan.slots, (size_t)DARTS_STATIC_SCRATCH_BYTES);
  unsigned char *base = nullptr;
  TRY(static_scratch_base(c, &base));
  CUDA_TRY(c, cudaMemsetAsync(base, 0, NP_BYTES, c->stream));      // the only part whose stale contents could be mistaken for this call's
  CUtensorMap tw;
  XMaps xm;
  TRY(tc_make_xmaps(c, &xm, X, rows, K));
  TRY(tc_make_map(c, &tw, W, N, K, 128));
  SkGemm g{};
  g.w_map = &tw; g.x_maps = &xm; g.C = (float *)(base + NP_BYTES); g.N = N; g.rows_ub = rows; g.slot_stride = (size_t)rows * N;
  g.np_table = (int32_t *)base;
  g.pairs = false;                                                 // always the single-CTA kernel, whatever the context's flags say
  g.plan = plan;
  TRY(launch_gemm_sk(c, g));
  return launch_sk_reduce(c, sk_view(g), C, rows);
}
