// Prefix-shared split-KV attention for bf16 / head_dim 128 / page 64 (placeholder: declines every shape).
#include "internal.cuh"
darts_status launch_attention_sm100(darts_ctx *, int, const void *, void *, int, const int32_t *, bool *taken) {
  *taken = false;
  return DARTS_OK;
}
