// S1+S2 tensor path (TACG_PATH_MMA) -- placeholder until the tcgen05 kernel lands.
#include "tacg_common.cuh"

bool tacg_coact_mma_supported(int, int, int) { return false; }

int tacg_launch_coact_mma(tacg_ctx* ctx, const int16_t*, const int8_t*, int64_t, int, int, int, int, uint32_t*,
                          uint32_t*) {
    snprintf(ctx->detail, sizeof(ctx->detail), "coact: the tcgen05 path is not built");
    return TACG_ERR_SHAPE;
}
