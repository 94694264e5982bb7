// temporary stubs while the stages are being written
#include "hh_internal.cuh"
int hh_three_apply(hh_ctx* ctx) { return hh_fail(ctx, HH_ERR_UNSUPPORTED, "three: not built yet"); }
