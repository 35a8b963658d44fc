// transport_small.cu -- crf_mix_transport for small mechanisms, 2 <= Ns <= 16 (
// the paper's own workload is of this size: 9 species).
//
// One thread per grid point, the whole per-point state in registers (Z_k, 1/a_k, the Wilke right-hand sides and
// the diffusion sums S_k: 5 Ns doubles), every loop fully unrolled on the template parameter NS.  The mechanism's
// transport tables (< 8 KB) are copied to shared memory once per block; lanes are points, so every coefficient
// is a warp-uniform (broadcast) shared-memory load.  Arithmetic as in transport_tiled.cu: each unordered pair once,
// 1/D_jk = 2^(cubic(ln T)) with the 64-entry table, Wilke expanded into three FMAs per ordered pair, Newton
// reciprocals, rho D_km = p_ref (1 - Y_k)/(R T S_k).
#include "crf_internal.h"
#include "fastmath.cuh"
#include "launch.h"

namespace {

using crf::exp2_poly9;
using crf::exp2_tab64;
using crf::rcp_newton;

__constant__ double kTab64[64] = CRF_EXP2_TAB64;

__device__ __forceinline__ double cubic_s(const double *c, double x)
{
    const double2 lo = *reinterpret_cast<const double2 *>(c), hi = *reinterpret_cast<const double2 *>(c + 2);
    return fma(x, fma(x, fma(x, hi.y, hi.x), lo.y), lo.x);
}

constexpr int TBS = 128;

template <int NS>
__global__ void __launch_bounds__(TBS) transport_small_kernel(DevTables m, const double *__restrict__ T,
                                                              const double *__restrict__ Y, int64_t n,
                                                              double *__restrict__ mu, double *__restrict__ lambda,
                                                              double *__restrict__ rhoD)
{
    extern __shared__ double2 sm2[];
    double *tb = reinterpret_cast<double *>(sm2);  // the mechanism's table, then the exp2 table
    const int ntab = m.tp.small_n;
    double *tab64 = tb + ntab;
    for (int i = threadIdx.x; i < ntab; i += TBS) tb[i] = __ldg(m.tp.small + i);
    for (int i = threadIdx.x; i < 64; i += TBS) tab64[i] = kTab64[i];
    __syncthreads();
    const double *sp = tb, *dd = tb + 12 * NS, *cw = dd + 4 * NS, *pc = cw + ((NS * NS + 1) & ~1);  // 16-byte aligned

    const int64_t i = (int64_t)blockIdx.x * TBS + threadIdx.x;
    if (i >= n) return;
    const double Ti = T[i];
    const double L = log(Ti);

    // ---- a1, a10, a12
    double y[NS], z[NS], r[NS], u1[NS], u2[NS];
#pragma unroll
    for (int k = 0; k < NS; ++k) y[k] = Y[(int64_t)k * n + i];
    double iw = 0.0, sum_a = 0.0, sum_h = 0.0;
#pragma unroll
    for (int k = 0; k < NS; ++k) {
        z[k] = y[k] * sp[12 * k + 10];
        r[k] = exp2_poly9(cubic_s(sp + 12 * k, L)) * sp[12 * k + 8];  // 1/a_k = W_k^(1/4)/sqrt(mu_k)
        const double lam = exp2_poly9(cubic_s(sp + 12 * k + 4, L));
        iw += z[k];
        sum_a = fma(z[k], lam, sum_a);
        sum_h = fma(z[k], rcp_newton(lam), sum_h);
        u1[k] = z[k] * r[k];
        u2[k] = u1[k] * r[k];
    }
    lambda[i] = 0.5 * (sum_a / iw + iw / sum_h);

    // ---- a11: Wilke, sum_j Z_j Phi_kj = A_k + 2 a_k B_k + a_k^2 C_k
    double mu_mix = 0.0;
#pragma unroll
    for (int k = 0; k < NS; ++k) {
        double A = 0.0, B = 0.0, C = 0.0;
#pragma unroll
        for (int j = 0; j < NS; ++j) {
            const double c = cw[k * NS + j];
            A = fma(c, z[j], A);
            B = fma(c, u1[j], B);
            C = fma(c, u2[j], C);
        }
        const double ak = rcp_newton(r[k]);
        const double ak2 = ak * ak;
        const double den = fma(ak2, C, fma(ak + ak, B, A));
        mu_mix = fma(z[k] * (ak2 * sp[12 * k + 9]), rcp_newton(den), mu_mix);
    }
    mu[i] = mu_mix;

    // ---- a13: each unordered pair once
    double S[NS];
#pragma unroll
    for (int k = 0; k < NS; ++k) S[k] = 0.0;
    int q = 0;
#pragma unroll
    for (int j = 0; j < NS; ++j) {
#pragma unroll
        for (int k = j + 1; k < NS; ++k, ++q) {
            const double e = exp2_tab64(cubic_s(pc + 4 * q, L), tab64);
            S[j] = fma(z[k], e, S[j]);
            S[k] = fma(z[j], e, S[k]);
        }
    }
    const double f = m.p_ref / (CRF_R_GAS * Ti);
#pragma unroll
    for (int k = 0; k < NS; ++k) {
        double v;
        if (S[k] == 0.0)  // pure species: rho D_kk = Wbar p_ref D_kk(p_ref)/(R T)
            v = f / iw * exp(cubic_s(dd + 4 * k, L));
        else
            v = f * (1.0 - y[k]) * rcp_newton(S[k]);
        rhoD[(int64_t)k * n + i] = v;
    }
}

template <int NS>
cudaError_t launch_ns(const DevTables &m, const double *T, const double *Y, int64_t n, double *mu, double *lambda,
                      double *rhoD, cudaStream_t st)
{
    const size_t smem = transport_small_dynamic_smem(m);
    transport_small_kernel<NS><<<(unsigned)((n + TBS - 1) / TBS), TBS, smem, st>>>(m, T, Y, n, mu, lambda, rhoD);
    crf_count_launch();
    return cudaGetLastError();
}

}  // namespace

size_t transport_small_dynamic_smem(const DevTables &m) { return sizeof(double) * ((size_t)m.tp.small_n + 64); }

cudaError_t launch_transport_small(const DevTables &m, const double *T, const double *Y, int64_t n, double *mu,
                                   double *lambda, double *rhoD, cudaStream_t st)
{
    switch (m.Ns) {
#define CRF_CASE(N) \
    case N: return launch_ns<N>(m, T, Y, n, mu, lambda, rhoD, st);
        CRF_CASE(2) CRF_CASE(3) CRF_CASE(4) CRF_CASE(5) CRF_CASE(6) CRF_CASE(7) CRF_CASE(8) CRF_CASE(9)
        CRF_CASE(10) CRF_CASE(11) CRF_CASE(12) CRF_CASE(13) CRF_CASE(14) CRF_CASE(15) CRF_CASE(16)
#undef CRF_CASE
    default: return cudaErrorInvalidValue;
    }
}
