// plan_rates.cu -- host code: reaction chunks, per-chunk incidence lists and re-laid-out coefficient
// tables of rates_staged.cu (see RatesPlan in crf_internal.h).
#include "host_plan.h"

RatesPlanOffsets build_rates_plan(const crf_tables *t, BlockBuilder &b)
{
    (void)t;
    (void)b;
    return RatesPlanOffsets{};
}
