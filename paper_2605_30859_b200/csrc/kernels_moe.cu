// MoE router + expert MLPs (not built yet).
#include "internal.cuh"
darts_status launch_moe(darts_ctx *c, int, int, const int32_t *) { FAIL(c, DARTS_ERR_UNSUPPORTED, "MoE path not built yet"); }
darts_status launch_moe_tc(darts_ctx *c, int, const void *, int, const int32_t *) { FAIL(c, DARTS_ERR_UNSUPPORTED, "MoE path not built yet"); }
