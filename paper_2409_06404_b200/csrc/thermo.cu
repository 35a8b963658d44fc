// thermo.cu -- crf_thermo / crf_thermo_species kernels.
//
// crf_thermo is an HBM stream: Y[k*n + i] is read once, 8 (Ns + 1) + 16 bytes per point.  To stay under the stream's
// time on the FP64 pipe the mixture sums are accumulated as MOMENTS of the NASA-7 coefficients,
//     M_c = sum_k (Y_k / W_k) a_{c+1,k}(range of T),  c = 0..4,   M_5 = sum_k (Y_k / W_k) a_{6,k}
//     c_p = R (M_0 + T (M_1 + T (M_2 + T (M_3 + T M_4))))
//     h   = R T (M_0 + T (M_1/2 + T (M_2/3 + T (M_3/4 + T M_4/5))) + M_5/T)
// six FMAs per species and point instead of the thirteen of two Horner evaluations (c_p and h share their
// coefficients).  The table (a_c/W_k: the six of the low range, then the six of the high range, so that a lane's range
// select is an address offset of 48 bytes and a set is three 128-bit loads) is staged once
// per block into shared memory; a thread owns two adjacent points (128-bit loads of the Y rows), the species loop
// is unrolled by four so that four row loads are in flight per thread, and a block walks several point groups.
// The range select T <= T_mid compares the bit patterns as integers (both are positive): no FP64 pipe instruction.
// Two instances (crf_plan_options.thermo_sets).  <false>: a lane reads the coefficient set of its own range: a broadcast (one
// shared-memory wavefront per load) where the lanes of a warp agree, one wavefront per quarter warp where they do not (fields
// without spatial coherence in T: the shared-memory pipe then takes as long as the HBM stream).  <true>, the default: both
// sets at warp-uniform addresses and twelve FMAs, the mass fraction routed to the set of the point's range.
#include "crf_internal.h"
#include <algorithm>

#include "launch.h"

namespace {

constexpr int TB = 256;
constexpr int TH_MINB = 3;    // blocks per SM (80 registers: no spills; measured against 2 and 4)
constexpr int TH_UNROLL = 4;  // species rows in flight per thread
constexpr int TH_STRIDE = 14;  // doubles per species in the table: 6 low-range, 6 high-range coefficients, T_mid, pad

template <int P>
__device__ __forceinline__ void thermo_species_step(const double *__restrict__ tab, int k, const double (&y)[P],
                                                    const long long (&Tbits)[P], double (&M)[6][P])
{
    const double *row = tab + TH_STRIDE * k;
    const long long tmid = __double_as_longlong(row[12]);
#pragma unroll
    for (int u = 0; u < P; ++u) {
        const double2 *c = reinterpret_cast<const double2 *>(row + (Tbits[u] <= tmid ? 0 : 6));
        const double2 c01 = c[0], c23 = c[1], c45 = c[2];
        M[0][u] = fma(y[u], c01.x, M[0][u]), M[1][u] = fma(y[u], c01.y, M[1][u]);
        M[2][u] = fma(y[u], c23.x, M[2][u]), M[3][u] = fma(y[u], c23.y, M[3][u]);
        M[4][u] = fma(y[u], c45.x, M[4][u]), M[5][u] = fma(y[u], c45.y, M[5][u]);
    }
}

// The same sums with BOTH coefficient sets read at warp-uniform addresses (six broadcast loads: one shared-memory wavefront
// each) and the point's mass fraction routed to the set of its range: twelve FMAs per species and point instead of six,
// a quarter of the shared-memory wavefronts when the lanes of a warp sit in different ranges (crf_plan_options.thermo_sets).
template <int P>
__device__ __forceinline__ void thermo_species_step_both(const double *__restrict__ tab, int k, const double (&y)[P],
                                                         const long long (&Tbits)[P], double (&M)[6][P])
{
    const double2 *c = reinterpret_cast<const double2 *>(tab + TH_STRIDE * k);
    const long long tmid = __double_as_longlong(tab[TH_STRIDE * k + 12]);
    const double2 l01 = c[0], l23 = c[1], l45 = c[2], h01 = c[3], h23 = c[4], h45 = c[5];
#pragma unroll
    for (int u = 0; u < P; ++u) {
        const bool lo = Tbits[u] <= tmid;
        const double yl = lo ? y[u] : 0.0, yh = lo ? 0.0 : y[u];
        M[0][u] = fma(yl, l01.x, M[0][u]), M[1][u] = fma(yl, l01.y, M[1][u]);
        M[2][u] = fma(yl, l23.x, M[2][u]), M[3][u] = fma(yl, l23.y, M[3][u]);
        M[4][u] = fma(yl, l45.x, M[4][u]), M[5][u] = fma(yl, l45.y, M[5][u]);
        M[0][u] = fma(yh, h01.x, M[0][u]), M[1][u] = fma(yh, h01.y, M[1][u]);
        M[2][u] = fma(yh, h23.x, M[2][u]), M[3][u] = fma(yh, h23.y, M[3][u]);
        M[4][u] = fma(yh, h45.x, M[4][u]), M[5][u] = fma(yh, h45.y, M[5][u]);
    }
}

template <int P>
__device__ __forceinline__ void thermo_finish(const double (&M)[6][P], const double (&Ti)[P], double (&cp)[P], double (&h)[P])
{
#pragma unroll
    for (int u = 0; u < P; ++u) {
        const double T = Ti[u];
        double c = fma(T, M[4][u], M[3][u]);
        c = fma(T, c, M[2][u]);
        c = fma(T, c, M[1][u]);
        c = fma(T, c, M[0][u]);
        cp[u] = c * CRF_R_GAS;
        double e = fma(T, M[4][u] * 0.2, M[3][u] * 0.25);
        e = fma(T, e, M[2][u] * (1.0 / 3.0));
        e = fma(T, e, M[1][u] * 0.5);
        e = fma(T, e, M[0][u]);
        h[u] = fma(T, e, M[5][u]) * CRF_R_GAS;  // R T (e + M_5 / T)
    }
}

template <bool BOTH>
__global__ void __launch_bounds__(TB, TH_MINB) thermo_kernel(DevTables m, const double *__restrict__ T,
                                                       const double *__restrict__ Y, int64_t n,
                                                       double *__restrict__ cp, double *__restrict__ h)
{
    extern __shared__ __align__(16) double sm[];
    const int Ns = m.Ns;
    for (int idx = threadIdx.x; idx < TH_STRIDE * Ns; idx += TB) sm[idx] = __ldg(m.thermo_tab + idx);
    __syncthreads();
    const bool vec = (n & 1) == 0;
    const int64_t npair = (n + 1) >> 1;
    for (int64_t j = (int64_t)blockIdx.x * TB + threadIdx.x; j < npair; j += (int64_t)gridDim.x * TB) {
        const int64_t i = 2 * j;
        if (vec) {
            const double2 t2 = *reinterpret_cast<const double2 *>(T + i);
            const double Ti[2] = {t2.x, t2.y};
            const long long Tb[2] = {__double_as_longlong(t2.x), __double_as_longlong(t2.y)};
            double M[6][2];
#pragma unroll
            for (int c = 0; c < 6; ++c) M[c][0] = M[c][1] = 0.0;
            int k = 0;
            for (; k + TH_UNROLL <= Ns; k += TH_UNROLL) {
                double2 y4[TH_UNROLL];
#pragma unroll
                for (int q = 0; q < TH_UNROLL; ++q) y4[q] = *reinterpret_cast<const double2 *>(Y + (int64_t)(k + q) * n + i);
#pragma unroll
                for (int q = 0; q < TH_UNROLL; ++q) {
                    const double y[2] = {y4[q].x, y4[q].y};
                    if (BOTH)
                        thermo_species_step_both<2>(sm, k + q, y, Tb, M);
                    else
                        thermo_species_step<2>(sm, k + q, y, Tb, M);
                }
            }
            for (; k < Ns; ++k) {
                const double2 yy = *reinterpret_cast<const double2 *>(Y + (int64_t)k * n + i);
                const double y[2] = {yy.x, yy.y};
                if (BOTH)
                    thermo_species_step_both<2>(sm, k, y, Tb, M);
                else
                    thermo_species_step<2>(sm, k, y, Tb, M);
            }
            double c2[2], h2[2];
            thermo_finish<2>(M, Ti, c2, h2);
            *reinterpret_cast<double2 *>(cp + i) = make_double2(c2[0], c2[1]);
            *reinterpret_cast<double2 *>(h + i) = make_double2(h2[0], h2[1]);
        } else {
            for (int64_t ii = i; ii < n && ii < i + 2; ++ii) {  // odd n: rows are not 16-byte aligned, scalar accesses
                const double Ti[1] = {T[ii]};
                const long long Tb[1] = {__double_as_longlong(Ti[0])};
                double M[6][1];
#pragma unroll
                for (int c = 0; c < 6; ++c) M[c][0] = 0.0;
                for (int k = 0; k < Ns; ++k) {
                    const double y[1] = {Y[(int64_t)k * n + ii]};
                    thermo_species_step<1>(sm, k, y, Tb, M);
                }
                double c1[1], h1[1];
                thermo_finish<1>(M, Ti, c1, h1);
                cp[ii] = c1[0], h[ii] = h1[0];
            }
        }
    }
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

// rho = p Wbar / (R T), Wbar = 1 / sum_k Y_k / W_k (the unfused path of crf_rhs_pointwise)
__global__ void __launch_bounds__(TB) density_kernel(DevTables m, const double *__restrict__ T, const double *__restrict__ p,
                                                     const double *__restrict__ Y, int64_t n, double *__restrict__ rho,
                                                     double *__restrict__ Wbar)
{
    const int64_t i = (int64_t)blockIdx.x * TB + threadIdx.x;
    if (i >= n) return;
    double iw = 0.0;
    for (int k = 0; k < m.Ns; ++k) iw = fma(Y[(int64_t)k * n + i], __ldg(m.rW + k), iw);
    if (Wbar) Wbar[i] = 1.0 / iw;
    if (rho) rho[i] = p[i] / (CRF_R_GAS * T[i] * iw);
}

}  // namespace

cudaError_t launch_density(const DevTables &m, const double *T, const double *p, const double *Y, int64_t n, double *rho,
                           double *Wbar, cudaStream_t st)
{
    density_kernel<<<(unsigned)((n + TB - 1) / TB), TB, 0, st>>>(m, T, p, Y, n, rho, Wbar);
    crf_count_launch();
    return cudaGetLastError();
}

cudaError_t launch_thermo(const DevTables &m, const double *T, const double *Y, int64_t n, double *cp, double *h,
                          cudaStream_t st)
{
    const size_t smem = sizeof(double) * TH_STRIDE * (size_t)m.Ns;
    const int64_t npair = (n + 1) / 2;
    // TH_MINB blocks of 8 warps per SM; a block walks its share of the point pairs (the table is staged once per block)
    const int64_t blocks = std::min<int64_t>((npair + TB - 1) / TB, 148 * TH_MINB * 4);
    if (m.thermo_sets == 2)
        thermo_kernel<true><<<(unsigned)blocks, TB, smem, st>>>(m, T, Y, n, cp, h);
    else
        thermo_kernel<false><<<(unsigned)blocks, TB, smem, st>>>(m, T, Y, n, cp, h);
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
