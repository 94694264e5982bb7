// temporary stubs while the stages are being written
#include "hh_internal.cuh"
int hh_aca_batch(hh_ctx* ctx, int64_t first, int64_t* next) { return hh_fail(ctx, HH_ERR_UNSUPPORTED, "aca: not built yet"); }
int hh_far_apply(hh_ctx* ctx) { return hh_fail(ctx, HH_ERR_UNSUPPORTED, "far: not built yet"); }
int hh_three_apply(hh_ctx* ctx) { return hh_fail(ctx, HH_ERR_UNSUPPORTED, "three: not built yet"); }
int hh_factors_fetch(hh_ctx* ctx, int64_t block, int32_t* rank, int32_t* flag, int32_t cap_rank,
                     int32_t* piv_i, int32_t* piv_j, float* C, float* Q) { return hh_fail(ctx, HH_ERR_UNSUPPORTED, "factors: not built yet"); }
