// SIMT GEMM  C[R,N] (+)= X[R,K] . W[N,K]^T  with fp32 accumulation.
// This is the fp32 path (config 1) and the fallback for shapes the tcgen05 kernel does not take.
#include "internal.cuh"

namespace {

constexpr int BM = 64, BN = 64, BK = 16;

template <typename TX, typename TW, bool ACC>
__global__ void __launch_bounds__(256) gemm_simt_k(const TX *__restrict__ X, const TW *__restrict__ W, float *__restrict__ C,
                                                   int N, int K, const int32_t *n_rows_dev, int rows_ub) {
  int R = n_rows_dev ? min(*n_rows_dev, rows_ub) : rows_ub;
  int r0 = blockIdx.y * BM, n0 = blockIdx.x * BN;
  if (r0 >= R) return;
  __shared__ float Xs[BK][BM + 4];
  __shared__ float Ws[BK][BN + 4];
  int tid = threadIdx.x, tx = tid & 15, ty = tid >> 4;
  int lrow = tid >> 2, lk = (tid & 3) * 4;     // each thread stages 4 consecutive k of one row of each operand
  float acc[4][4] = {};
  for (int k0 = 0; k0 < K; k0 += BK) {
#pragma unroll
    for (int q = 0; q < 4; ++q) {
      int k = k0 + lk + q;
      int r = r0 + lrow, n = n0 + lrow;
      Xs[lk + q][lrow] = (r < R && k < K) ? to_f<TX>(X[(size_t)r * K + k]) : 0.f;
      Ws[lk + q][lrow] = (n < N && k < K) ? to_f<TW>(W[(size_t)n * K + k]) : 0.f;
    }
    __syncthreads();
#pragma unroll
    for (int k = 0; k < BK; ++k) {
      float a[4], b[4];
#pragma unroll
      for (int i = 0; i < 4; ++i) a[i] = Xs[k][ty * 4 + i];
#pragma unroll
      for (int j = 0; j < 4; ++j) b[j] = Ws[k][tx * 4 + j];
#pragma unroll
      for (int i = 0; i < 4; ++i)
#pragma unroll
        for (int j = 0; j < 4; ++j) acc[i][j] = fmaf(a[i], b[j], acc[i][j]);
    }
    __syncthreads();
  }
#pragma unroll
  for (int i = 0; i < 4; ++i) {
    int r = r0 + ty * 4 + i;
    if (r >= R) continue;
#pragma unroll
    for (int j = 0; j < 4; ++j) {
      int n = n0 + tx * 4 + j;
      if (n >= N) continue;
      size_t o = (size_t)r * N + n;
      C[o] = ACC ? C[o] + acc[i][j] : acc[i][j];
    }
  }
}

template <typename TX, typename TW>
void launch_t(darts_ctx *c, const void *X, const void *W, float *C, int N, int K, int rows_ub, const int32_t *n_rows_dev, bool acc) {
  dim3 grid((N + BN - 1) / BN, (rows_ub + BM - 1) / BM);
  if (acc) gemm_simt_k<TX, TW, true><<<grid, 256, 0, c->stream>>>((const TX *)X, (const TW *)W, C, N, K, n_rows_dev, rows_ub);
  else gemm_simt_k<TX, TW, false><<<grid, 256, 0, c->stream>>>((const TX *)X, (const TW *)W, C, N, K, n_rows_dev, rows_ub);
}

}  // namespace

darts_status launch_gemm_simt(darts_ctx *c, const void *X, const void *W, float *C, int N, int K, int rows_ub,
                              const int32_t *n_rows_dev, bool accumulate, bool w_is_f32) {
  if (rows_ub <= 0) return DARTS_OK;
  if (c->m.dtype == DARTS_F32) launch_t<float, float>(c, X, W, C, N, K, rows_ub, n_rows_dev, accumulate);
  else if (w_is_f32) launch_t<__nv_bfloat16, float>(c, X, W, C, N, K, rows_ub, n_rows_dev, accumulate);
  else launch_t<__nv_bfloat16, __nv_bfloat16>(c, X, W, C, N, K, rows_ub, n_rows_dev, accumulate);
  c->launches++;
  cudaError_t e = cudaGetLastError();
  if (e != cudaSuccess) {
    snprintf(c->err, sizeof(c->err), "launch gemm_simt: %s", cudaGetErrorString(e));
    c->sticky = DARTS_ERR_CUDA;
    return DARTS_ERR_CUDA;
  }
  return DARTS_OK;
}
