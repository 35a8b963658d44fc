// row_io.cuh -- global-memory rows of the species-major fields as seen by the lanes-are-points kernels (rates_group.cu,
// transport_tiled.cu): a lane owns PPL adjacent points i0, i0 + 1, so that a row is one 128-bit access per lane when
// PPL = 2 and n is even (rows are then 16-byte aligned); otherwise scalar accesses, clamped / guarded at the ragged end.
#pragma once
#include <stdint.h>

namespace crf {

template <int PPL>
__device__ __forceinline__ void load_row(const double *__restrict__ row, int64_t i0, int64_t n, bool vec, double (&v)[PPL])
{
    if (PPL == 2 && vec && i0 + 1 < n) {
        const double2 t = *reinterpret_cast<const double2 *>(row + i0);
        v[0] = t.x, v[PPL - 1] = t.y;
    } else {
#pragma unroll
        for (int u = 0; u < PPL; ++u) v[u] = row[min(i0 + u, n - 1)];
    }
}
template <int PPL>
__device__ __forceinline__ void store_row(double *__restrict__ row, int64_t i0, int64_t n, bool vec, const double (&v)[PPL])
{
    if (PPL == 2 && vec && i0 + 1 < n) {
        *reinterpret_cast<double2 *>(row + i0) = make_double2(v[0], v[PPL - 1]);
    } else {
#pragma unroll
        for (int u = 0; u < PPL; ++u)
            if (i0 + u < n) row[i0 + u] = v[u];
    }
}

}  // namespace crf
