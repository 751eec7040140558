// temporary: bf16 tensor-core path not built yet
#include "common.cuh"
#include "edge.cuh"
int mlip_gemm_bf16(mlip_ctx* ctx, const GemmArgs&) { ctx->set_error("bf16 path not built"); return MLIP_ERR_UNSUPPORTED; }
int64_t mlip_edge_bf16_tiles(int64_t E) { return (E + 127) / 128; }
int mlip_edge_forward_bf16(mlip_ctx* ctx, int, const EdgeArgs&) { ctx->set_error("bf16 path not built"); return MLIP_ERR_UNSUPPORTED; }
int mlip_edge_backward_bf16(mlip_ctx* ctx, int, const EdgeArgs&) { ctx->set_error("bf16 path not built"); return MLIP_ERR_UNSUPPORTED; }
int mlip_gather_rev_bf16(mlip_ctx* ctx, int64_t, int, const int32_t*, const int32_t*, const __nv_bfloat16*, float*) { ctx->set_error("bf16 path not built"); return MLIP_ERR_UNSUPPORTED; }
