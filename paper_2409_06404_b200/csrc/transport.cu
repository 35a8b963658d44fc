// transport.cu -- crf_mix_transport kernel.
//
// v1 (generic, any Ns): one thread per grid point; the per-point vectors (mole fractions X_k,
// the Wilke factors a_k = sqrt(mu_k) W_k^(-1/4) and 1/a_k, and the diffusion sums S_k) live in
// shared memory as columns [k][thread].  The binary-pair loop visits each unordered pair once:
// e = exp(-cubic(ln T)) = 1/D_jk(p_ref), S_k += X_j e, S_j += X_k e.  The pressure cancels in
// rho D_km analytically (rho ~ p, D ~ 1/p) and is only read for nothing else.
#include "crf_internal.h"
#include "launch.h"

namespace {

__device__ __forceinline__ double cubic(const double *__restrict__ c, int stride, double x)
{
    double v = fma(x, __ldg(c + 3 * stride), __ldg(c + 2 * stride));
    v = fma(x, v, __ldg(c + stride));
    return fma(x, v, __ldg(c));
}

template <int B>
__global__ void __launch_bounds__(B) transport_generic_kernel(DevTables m, const double *__restrict__ T,
                                                              const double *__restrict__ Y, int64_t n,
                                                              double *__restrict__ mu, double *__restrict__ lambda,
                                                              double *__restrict__ rhoD)
{
    extern __shared__ double sm[];
    const int Ns = m.Ns, tid = threadIdx.x;
    double *sX = sm, *sA = sm + (size_t)Ns * B, *sRA = sm + 2 * (size_t)Ns * B, *sS = sm + 3 * (size_t)Ns * B;
    const int64_t i = (int64_t)blockIdx.x * B + tid;
    if (i >= n) return;
    const double Ti = T[i];
    const double lnT = log(Ti);
    double invW = 0.0;
    for (int k = 0; k < Ns; ++k) invW = fma(Y[(int64_t)k * n + i], __ldg(m.rW + k), invW);
    const double Wbar = 1.0 / invW;
    // a10, a12: species fits, conductivity sums, Wilke factors
    double sum_a = 0.0, sum_h = 0.0;
    for (int k = 0; k < Ns; ++k) {
        const double x = Y[(int64_t)k * n + i] * Wbar * __ldg(m.rW + k);
        sX[k * B + tid] = x;
        sS[k * B + tid] = 0.0;
        const double muk = exp(cubic(m.mu_c + k, Ns, lnT));
        const double lamk = exp(cubic(m.lam_c + k, Ns, lnT));
        sum_a = fma(x, lamk, sum_a);
        sum_h += x / lamk;
        const double a = sqrt(muk) * __ldg(m.wq + k);
        sA[k * B + tid] = a;
        sRA[k * B + tid] = 1.0 / a;
    }
    lambda[i] = 0.5 * (sum_a + 1.0 / sum_h);
    // a11: Wilke.  Phi_kj = c_kj (1 + a_k / a_j)^2
    double mu_mix = 0.0;
    for (int k = 0; k < Ns; ++k) {
        const double ak = sA[k * B + tid];
        double den = 0.0;
        for (int j = 0; j < Ns; ++j) {
            const double t = fma(ak, sRA[j * B + tid], 1.0);
            den = fma(sX[j * B + tid] * __ldg(m.wilke_c + k * Ns + j), t * t, den);
        }
        const double muk = exp(cubic(m.mu_c + k, Ns, lnT));
        mu_mix += sX[k * B + tid] * muk / den;
    }
    mu[i] = mu_mix;
    // a13: mixture-averaged diffusion, unordered pairs
    for (int j = 0; j < Ns; ++j) {
        const double xj = sX[j * B + tid];
        double sj = 0.0;
        const double *c = m.nDc + 4 * (size_t)crf_pair_index(j, j + 1, Ns);
        for (int k = j + 1; k < Ns; ++k, c += 4) {
            double v = fma(lnT, __ldg(c + 3), __ldg(c + 2));
            v = fma(lnT, v, __ldg(c + 1));
            const double e = exp(fma(lnT, v, __ldg(c)));
            sj = fma(sX[k * B + tid], e, sj);
            sS[k * B + tid] = fma(xj, e, sS[k * B + tid]);
        }
        sS[j * B + tid] += sj;
    }
    // rho D_km = (Wbar p_ref/(R T)) (1 - Y_k)/S_k ; pure species: (Wbar p_ref/(R T)) D_kk(p_ref)
    const double f = Wbar * m.p_ref / (CRF_R_GAS * Ti);
    for (int k = 0; k < Ns; ++k) {
        const double s = sS[k * B + tid];
        double v;
        if (s == 0.0) {
            const double *c = m.nDc + 4 * (size_t)crf_pair_index(k, k, Ns);
            double w = fma(lnT, __ldg(c + 3), __ldg(c + 2));
            w = fma(lnT, w, __ldg(c + 1));
            v = f * exp(-fma(lnT, w, __ldg(c)));
        } else {
            v = f * (1.0 - Y[(int64_t)k * n + i]) / s;
        }
        rhoD[(int64_t)k * n + i] = v;
    }
}

template <int B>
cudaError_t launch_b(const DevTables &m, const double *T, const double *Y, int64_t n, double *mu, double *lambda,
                     double *rhoD, cudaStream_t st)
{
    const size_t smem = sizeof(double) * 4 * (size_t)m.Ns * B;
    cudaError_t e = cudaFuncSetAttribute(transport_generic_kernel<B>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                         (int)smem);
    if (e != cudaSuccess) return e;
    transport_generic_kernel<B><<<(unsigned)((n + B - 1) / B), B, smem, st>>>(m, T, Y, n, mu, lambda, rhoD);
    crf_count_launch();
    return cudaGetLastError();
}

}  // namespace

size_t transport_dynamic_smem(const DevTables &m)
{
    if (m.tp.W > 0) return transport_tiled_dynamic_smem(m);
    if (m.tp.small_n > 0) return transport_small_dynamic_smem(m);
    const size_t per_thread = sizeof(double) * 4 * (size_t)m.Ns;
    return per_thread * (per_thread * 128 <= 100 * 1024 ? 128 : (per_thread * 64 <= 200 * 1024 ? 64 : 32));
}

cudaError_t launch_transport(const DevTables &m, const double *T, const double *p, const double *Y, int64_t n,
                             double *mu, double *lambda, double *rhoD, cudaStream_t st)
{
    (void)p;
    if (m.tp.W > 0) return launch_transport_tiled(m, T, Y, n, mu, lambda, rhoD, st);
    if (m.tp.small_n > 0) return launch_transport_small(m, T, Y, n, mu, lambda, rhoD, st);
    const size_t per_thread = sizeof(double) * 4 * (size_t)m.Ns;
    const size_t budget = 100 * 1024;
    if (per_thread * 128 <= budget) return launch_b<128>(m, T, Y, n, mu, lambda, rhoD, st);
    if (per_thread * 64 <= 2 * budget) return launch_b<64>(m, T, Y, n, mu, lambda, rhoD, st);
    return launch_b<32>(m, T, Y, n, mu, lambda, rhoD, st);
}
