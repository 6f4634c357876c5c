// tcgen05 / TMEM GEMM for the bf16 path (placeholder until the sm_100a kernel lands: declines every shape).
#include "internal.cuh"
darts_status launch_gemm_tc(darts_ctx *, const void *, const void *, float *, int, int, int, const int32_t *, bool, bool *taken) {
  *taken = false;
  return DARTS_OK;
}
