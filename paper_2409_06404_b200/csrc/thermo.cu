// thermo.cu -- crf_thermo / crf_thermo_species kernels.
//
// HBM-bound streaming kernels: one thread per grid point, Y[k*n + i] read once with
// coalesced loads (a warp reads 256 contiguous bytes per species), NASA-7 coefficients
// staged once per block into shared memory in the Horner forms of crf_internal.h.
// The per-lane range select (T <= Tmid_k) is a shared-memory address select, not a branch.
#include "crf_internal.h"
#include "launch.h"

namespace {

constexpr int TB = 256;

// smem: [2][11][Ns] = cpc(5) then hc(6) per range
__global__ void __launch_bounds__(TB) thermo_kernel(DevTables m, const double *__restrict__ T,
                                                    const double *__restrict__ Y, int64_t n,
                                                    double *__restrict__ cp, double *__restrict__ h)
{
    extern __shared__ double sm[];
    const int Ns = m.Ns;
    double *s_tmid = sm;            // [Ns]
    double *s_rW = sm + Ns;         // [Ns]
    double *s_co = sm + 2 * Ns;     // [2][11][Ns]
    for (int idx = threadIdx.x; idx < Ns; idx += TB) {
        s_tmid[idx] = m.Tmid[idx];
        s_rW[idx] = m.rW[idx];
    }
    for (int idx = threadIdx.x; idx < 2 * 5 * Ns; idx += TB) {
        int rg = idx / (5 * Ns), rem = idx % (5 * Ns);
        s_co[rg * 11 * Ns + rem] = m.cpc[idx];
    }
    for (int idx = threadIdx.x; idx < 2 * 6 * Ns; idx += TB) {
        int rg = idx / (6 * Ns), rem = idx % (6 * Ns);
        s_co[rg * 11 * Ns + 5 * Ns + rem] = m.hc[idx];
    }
    __syncthreads();
    const int64_t i = (int64_t)blockIdx.x * TB + threadIdx.x;
    if (i >= n) return;
    const double Ti = T[i];
    const double rT = 1.0 / Ti;
    double cpm = 0.0, hm = 0.0;
#pragma unroll 2
    for (int k = 0; k < Ns; ++k) {
        const double y = Y[(int64_t)k * n + i] * s_rW[k];
        const double *c = s_co + ((Ti <= s_tmid[k]) ? 0 : 11 * Ns) + k;
        double cpk = fma(Ti, c[4 * Ns], c[3 * Ns]);
        cpk = fma(Ti, cpk, c[2 * Ns]);
        cpk = fma(Ti, cpk, c[1 * Ns]);
        cpk = fma(Ti, cpk, c[0]);
        const double *d = c + 5 * Ns;
        double hk = fma(Ti, d[4 * Ns], d[3 * Ns]);
        hk = fma(Ti, hk, d[2 * Ns]);
        hk = fma(Ti, hk, d[1 * Ns]);
        hk = fma(Ti, hk, d[0]);
        hk = fma(d[5 * Ns], rT, hk);
        cpm = fma(y, cpk, cpm);
        hm = fma(y, hk, hm);
    }
    cp[i] = cpm * CRF_R_GAS;
    h[i] = hm * (CRF_R_GAS * Ti);
}

__global__ void __launch_bounds__(TB) thermo_species_kernel(DevTables m, const double *__restrict__ T, int64_t n,
                                                            double *__restrict__ cpk_o, double *__restrict__ hk_o,
                                                            double *__restrict__ sk_o)
{
    const int64_t i = (int64_t)blockIdx.x * TB + threadIdx.x;
    if (i >= n) return;
    const int Ns = m.Ns;
    const double Ti = T[i];
    const double rT = 1.0 / Ti, lnT = log(Ti);
    for (int k = 0; k < Ns; ++k) {
        const int rg = (Ti <= __ldg(m.Tmid + k)) ? 0 : 1;
        const double *c = m.cpc + rg * 5 * Ns + k;
        double v = fma(Ti, __ldg(c + 4 * Ns), __ldg(c + 3 * Ns));
        v = fma(Ti, v, __ldg(c + 2 * Ns));
        v = fma(Ti, v, __ldg(c + Ns));
        v = fma(Ti, v, __ldg(c));
        if (cpk_o) cpk_o[(int64_t)k * n + i] = v * CRF_R_GAS;
        const double *d = m.hc + rg * 6 * Ns + k;
        v = fma(Ti, __ldg(d + 4 * Ns), __ldg(d + 3 * Ns));
        v = fma(Ti, v, __ldg(d + 2 * Ns));
        v = fma(Ti, v, __ldg(d + Ns));
        v = fma(Ti, v, __ldg(d));
        v = fma(__ldg(d + 5 * Ns), rT, v);
        if (hk_o) hk_o[(int64_t)k * n + i] = v * (CRF_R_GAS * Ti);
        const double *e = m.sc + rg * 6 * Ns + k;
        v = fma(Ti, __ldg(e + 4 * Ns), __ldg(e + 3 * Ns));
        v = fma(Ti, v, __ldg(e + 2 * Ns));
        v = fma(Ti, v, __ldg(e + Ns));
        v = fma(Ti, v, __ldg(e + 5 * Ns));
        v = fma(__ldg(e), lnT, v);
        if (sk_o) sk_o[(int64_t)k * n + i] = v * CRF_R_GAS;
    }
}

}  // namespace

cudaError_t launch_thermo(const DevTables &m, const double *T, const double *Y, int64_t n, double *cp, double *h,
                          cudaStream_t st)
{
    const size_t smem = sizeof(double) * (size_t)(2 + 22) * m.Ns;
    static bool attr_done = false;
    if (!attr_done) {
        cudaFuncSetAttribute(thermo_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, 200 * 1024);
        attr_done = true;
    }
    const int64_t blocks = (n + TB - 1) / TB;
    thermo_kernel<<<(unsigned)blocks, TB, smem, st>>>(m, T, Y, n, cp, h);
    crf_count_launch();
    return cudaGetLastError();
}

cudaError_t launch_thermo_species(const DevTables &m, const double *T, int64_t n, double *cpk, double *hk, double *sk,
                                  cudaStream_t st)
{
    const int64_t blocks = (n + TB - 1) / TB;
    thermo_species_kernel<<<(unsigned)blocks, TB, 0, st>>>(m, T, n, cpk, hk, sk);
    crf_count_launch();
    return cudaGetLastError();
}
