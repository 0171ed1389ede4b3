// contract.cu -- placeholder until the fused contraction lands
#include "kernels.h"
tm_status tm_contract_internal(tm_ctx* ctx, void*, const void*, const void*, double, double, const int*, int, tm_prec, cudaStream_t) { return tm_fail(ctx, TM_EARG, "not implemented"); }
extern "C" tm_status loop_contract_project(tm_ctx* ctx, void*, const void*, const void*, double, double, const int*, int, tm_prec, void*) { return tm_fail(ctx, TM_EARG, "not implemented"); }
extern "C" tm_status tsm_estimate(tm_ctx* ctx, void*, void*, const tsm_params*, tsm_info*, void*) { return tm_fail(ctx, TM_EARG, "not implemented"); }
extern "C" tm_status tsm_estimate_host(tm_ctx* ctx, void*, const unsigned char*, const tsm_params*, tsm_info*, void*) { return tm_fail(ctx, TM_EARG, "not implemented"); }
