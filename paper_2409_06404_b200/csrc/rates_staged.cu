#include "crf_internal.h"
#include "launch.h"
cudaError_t launch_rates_staged(const DevTables &, const double *, const double *, const double *, int64_t, double *,
                                double *, cudaStream_t)
{
    return cudaErrorNotSupported;
}
