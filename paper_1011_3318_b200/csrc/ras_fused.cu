// ras_fused.cu -- tier 2 of the RAS block solver (north_star (c)): placeholder until the on-chip solver lands.
#include "wcras_internal.cuh"
namespace wc {
int ras_fused_supported(const wcras_ctx*, const int*, const int*, int) { return 0; }
int ras_fused_block_solve(wcras_ctx* ctx, const float4*, float4*, bool) {
    snprintf(ctx->err, sizeof ctx->err, "fused tier not available");
    return WCRAS_UNSUPPORTED;
}
}  // namespace wc
