// rates.cu -- crf_production_rates kernel.
//
// v1 (generic, any Ns): one thread per grid point.  The per-point state the reaction loop
// gathers from -- concentrations C_k and Gibbs functions g_k/(RT) -- lives in shared memory as
// columns [k][thread] (each thread reads only its own column: conflict-free, warp-uniform
// species index).  omega_k is accumulated in the caller's output array (same thread, same
// address: no race).  Reactions are sorted elementary | third-body | falloff, so each of the
// three loops is uniform across the warp.
#include "crf_internal.h"
#include "launch.h"

namespace {

struct RatesShared {
    double *C;  // [Ns][B]
    double *G;  // [Ns][B]
};

// one reversible reaction: rates of progress from k_f, then scatter nu*q into omega
__device__ __forceinline__ void progress_and_scatter(const DevTables &m, int r, double kf, double third,
                                                     const double *sC, const double *sG, int B, int tid,
                                                     double lnc0, double *__restrict__ omega, int64_t n, int64_t i)
{
    const int Nr = m.Nr;
    int a[3], b[3];
#pragma unroll
    for (int s = 0; s < 3; ++s) {
        a[s] = m.reac[s * Nr + r];
        b[s] = m.prod[s * Nr + r];
    }
    double dG = 0.0, Pf = 1.0, Pr = 1.0;
#pragma unroll
    for (int s = 0; s < 3; ++s) {
        if (a[s] >= 0) {
            dG -= sG[a[s] * B + tid];
            Pf *= sC[a[s] * B + tid];
        }
        if (b[s] >= 0) {
            dG += sG[b[s] * B + tid];
            Pr *= sC[b[s] * B + tid];
        }
    }
    // k_r = k_f / K_c,  1/K_c = exp(sum nu g/(RT) - dnu ln(p_ref/(RT)))
    const double kr = kf * exp(dG - m.dnu[r] * lnc0);
    const double q = third * (kf * Pf - kr * Pr);
#pragma unroll
    for (int s = 0; s < 3; ++s) {
        if (a[s] >= 0) omega[(int64_t)a[s] * n + i] -= q;
        if (b[s] >= 0) omega[(int64_t)b[s] * n + i] += q;
    }
}

template <int B>
__global__ void __launch_bounds__(B) rates_generic_kernel(DevTables m, const double *__restrict__ T,
                                                          const double *__restrict__ p, const double *__restrict__ Y,
                                                          int64_t n, double *__restrict__ omega,
                                                          double *__restrict__ qdot)
{
    extern __shared__ double sm[];
    const int Ns = m.Ns, tid = threadIdx.x;
    double *sC = sm, *sG = sm + (size_t)Ns * B;
    const int64_t i = (int64_t)blockIdx.x * B + tid;
    if (i >= n) return;  // no block-wide barrier below
    const double Ti = T[i], pi = p[i];
    const double lnT = log(Ti), rT = 1.0 / Ti;
    // a1: Wbar, rho, C_k
    double invW = 0.0;
    for (int k = 0; k < Ns; ++k) invW = fma(Y[(int64_t)k * n + i], __ldg(m.rW + k), invW);
    const double rho = pi / (CRF_R_GAS * Ti * invW);
    double Csum = 0.0;
    for (int k = 0; k < Ns; ++k) {
        const double c = rho * Y[(int64_t)k * n + i] * __ldg(m.rW + k);
        sC[k * B + tid] = c;
        Csum += c;
        // a2: g_k/(RT)
        const double *gc = m.gc + ((Ti <= __ldg(m.Tmid + k)) ? 0 : 7 * Ns) + k;
        double g = fma(Ti, __ldg(gc + 4 * Ns), __ldg(gc + 3 * Ns));
        g = fma(Ti, g, __ldg(gc + 2 * Ns));
        g = fma(Ti, g, __ldg(gc + Ns));
        g = fma(Ti, g, __ldg(gc + 6 * Ns));
        g = fma(__ldg(gc + 5 * Ns), rT, g);
        g = fma(__ldg(gc), 1.0 - lnT, g);
        sG[k * B + tid] = g;
        omega[(int64_t)k * n + i] = 0.0;
    }
    const double lnc0 = log(m.p_ref / CRF_R_GAS) - lnT;  // ln(p_ref/(R T))
    // a4, a7, a8: elementary reactions
    int r = 0;
    for (; r < m.Ne; ++r) {
        const double kf = exp(fma(__ldg(m.beta + r), lnT, __ldg(m.lnA + r)) - __ldg(m.Ea_R + r) * rT);
        progress_and_scatter(m, r, kf, 1.0, sC, sG, B, tid, lnc0, omega, n, i);
    }
    // a5: third-body reactions, both rates of progress times [M]
    for (int t = 0; t < m.N3; ++t, ++r) {
        double M = Csum;
        for (int e = m.eff_ptr[t]; e < m.eff_ptr[t + 1]; ++e) M = fma(m.eff_val[e], sC[m.eff_idx[e] * B + tid], M);
        const double kf = exp(fma(__ldg(m.beta + r), lnT, __ldg(m.lnA + r)) - __ldg(m.Ea_R + r) * rT);
        progress_and_scatter(m, r, kf, M, sC, sG, B, tid, lnc0, omega, n, i);
    }
    // a6: Troe falloff
    for (int t = 0; t < m.Nt; ++t, ++r) {
        double M = Csum;
        for (int e = m.eff_ptr[m.N3 + t]; e < m.eff_ptr[m.N3 + t + 1]; ++e)
            M = fma(m.eff_val[e], sC[m.eff_idx[e] * B + tid], M);
        const double lnkinf = fma(m.beta[r], lnT, m.lnA[r]) - m.Ea_R[r] * rT;
        const double lnk0 = fma(m.beta0[t], lnT, m.lnA0[t]) - m.Ea0_R[t] * rT;
        const double kinf = exp(lnkinf);
        const double Pr = exp(lnk0 - lnkinf) * M;
        const double al = m.alpha[t];
        const double Fc = (1.0 - al) * exp(-Ti * m.rT3[t]) + al * exp(-Ti * m.rT1[t]) + exp(-m.T2[t] * rT);
        const double lFc = log10(fmax(Fc, 1.0e-300));
        const double lPr = log10(Pr);
        const double c = -0.4 - 0.67 * lFc;
        const double N = 0.75 - 1.27 * lFc;
        const double f1 = (lPr + c) / (N - 0.14 * (lPr + c));
        const double F = exp10(lFc / fma(f1, f1, 1.0));
        const double kf = kinf * (Pr / (1.0 + Pr)) * F;
        progress_and_scatter(m, r, kf, 1.0, sC, sG, B, tid, lnc0, omega, n, i);
    }
    // a9: qdot = -sum_k h_k omega_k
    double qd = 0.0;
    for (int k = 0; k < Ns; ++k) {
        const double *d = m.hc + ((Ti <= __ldg(m.Tmid + k)) ? 0 : 6 * Ns) + k;
        double hk = fma(Ti, __ldg(d + 4 * Ns), __ldg(d + 3 * Ns));
        hk = fma(Ti, hk, __ldg(d + 2 * Ns));
        hk = fma(Ti, hk, __ldg(d + Ns));
        hk = fma(Ti, hk, __ldg(d));
        hk = fma(__ldg(d + 5 * Ns), rT, hk);
        qd = fma(-hk, omega[(int64_t)k * n + i], qd);
    }
    qdot[i] = qd * (CRF_R_GAS * Ti);
}

template <int B>
cudaError_t launch_b(const DevTables &m, const double *T, const double *p, const double *Y, int64_t n,
                     double *omega, double *qdot, cudaStream_t st)
{
    const size_t smem = sizeof(double) * 2 * (size_t)m.Ns * B;
    cudaError_t e = cudaFuncSetAttribute(rates_generic_kernel<B>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                         (int)smem);
    if (e != cudaSuccess) return e;
    rates_generic_kernel<B><<<(unsigned)((n + B - 1) / B), B, smem, st>>>(m, T, p, Y, n, omega, qdot);
    crf_count_launch();
    return cudaGetLastError();
}

}  // namespace

size_t rates_dynamic_smem(const DevTables &m)
{
    if (m.rs.W > 0) return rates_smem_dynamic_smem(m);
    if (m.rg.W > 0) return rates_group_dynamic_smem(m);
    if (m.rp.W > 0) return rates_staged_dynamic_smem(m);
    const size_t per_thread = sizeof(double) * 2 * (size_t)m.Ns;
    return per_thread * (per_thread * 128 <= 100 * 1024 ? 128 : (per_thread * 64 <= 200 * 1024 ? 64 : 32));
}

cudaError_t launch_rates(const DevTables &m, const double *T, const double *p, const double *Y, int64_t n,
                         double *omega, double *qdot, cudaStream_t st)
{
    if (m.rs.W > 0) return launch_rates_smem(m, T, p, Y, n, omega, qdot, st);
    if (m.rg.W > 0) return launch_rates_group(m, rates_io(T, p, Y, omega, qdot), n, st);
    if (m.rp.W > 0) return launch_rates_staged(m, T, p, Y, n, omega, qdot, st);
    const size_t per_thread = sizeof(double) * 2 * (size_t)m.Ns;
    const size_t budget = 100 * 1024;  // two blocks per SM
    if (per_thread * 128 <= budget) return launch_b<128>(m, T, p, Y, n, omega, qdot, st);
    if (per_thread * 64 <= 2 * budget) return launch_b<64>(m, T, p, Y, n, omega, qdot, st);
    return launch_b<32>(m, T, p, Y, n, omega, qdot, st);
}
