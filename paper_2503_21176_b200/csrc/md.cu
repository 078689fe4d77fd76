// md.cu -- a-11: shadow XL-BOMD step driver.  (placeholder until implemented)
#include "common.cuh"

extern "C" int sqeq_shadow_md_init(sqeq_ctx* ctx, const sqeq_nlist*, int64_t, const float*, const double*,
                                   const sqeq_md_params*, const float*, const float*, double, int,
                                   double*, float*, double*)
{
    return sqeq_fail(ctx, SQEQ_EINVAL, "sqeq_shadow_md_init: not implemented yet");
}

extern "C" int sqeq_shadow_md_step(sqeq_ctx* ctx, const sqeq_nlist*, int64_t, float*, float*, const float*,
                                   const double*, const sqeq_md_params*, const float*, const float*,
                                   double*, float*, double*)
{
    return sqeq_fail(ctx, SQEQ_EINVAL, "sqeq_shadow_md_step: not implemented yet");
}
