// rates_staged.cu -- crf_production_rates: W warps share 32 grid
// points (lane = point), reactions and species are dealt to the warps in two alternating stages.
//
// Why this shape.  Per reaction the work is two exponentials (k_f and k_f/K_c) around eight gathers
// of per-point species state (C_k and g_k/RT of the reactants and products) and four scatters into
// omega_k.  With lanes = points every coefficient is a warp-uniform load.  The state of a point
// (C_k, g_k) lives in shared memory as [species][lane] rows of double2 (one conflict-free LDS.128 per
// gather).  Scattering nu*q into omega rows would need read-modify-write traffic and atomics between
// the warps; instead
//   reaction stage: the warps split the reactions of a chunk (<= Rc), each writes q_r to sQ[r][lane];
//   species stage:  the warps split the SPECIES; each owned species sums nu_kr q_r over its incidence
//                   list of the chunk into a REGISTER accumulator (the species loop is unrolled, so
//                   omega of up to 32 owned species per warp stays in registers for the whole kernel).
// omega never touches shared memory; it is stored once, coalesced, with qdot = -sum_k h_k omega_k.
// Exponentials are 2^y (fastmath.cuh) with log2(e) folded into lnA, beta, Ea/R and the NASA g sets.
// Concentrations stay linear (products, not sums of logarithms): exact zeros and negative mass
// fractions behave as in the definition.
//
// Reactions are grouped into chunks of one kind (elementary | third body | Troe falloff) and one shape
// (at most two reactants and two products: four gathers, empty slots read the dummy species C = 1,
// g = 0; anything else: six gathers).
#include "crf_internal.h"
#include "fastmath.cuh"
#include "launch.h"

namespace {

__device__ __forceinline__ double exp2_clamped(double y) { return crf::exp2_clamped<9>(y); }  // (fastmath.cuh)

struct PointCtx {
    double L, rT, lc02;  // ln T, 1/T, log2(e) ln(p_ref/(R T))
    double Csum;         // p/(R T)
    double Ti;
};

__device__ __forceinline__ double2 lds2(const char *sCG, int off, int lane)
{
    return *reinterpret_cast<const double2 *>(sCG + off + lane * 16);
}

// rate of progress of one reaction, without the third-body factor; y_f = log2 k_f is passed in
template <bool GENERIC>
__device__ __forceinline__ double progress(const char *sCG, int lane, const int4 s0, const int4 s1, double yf, double kf,
                                           double dnu, const PointCtx &c)
{
    const double2 a0 = lds2(sCG, s0.x, lane), a1 = lds2(sCG, s0.y, lane), b0 = lds2(sCG, s0.z, lane),
                  b1 = lds2(sCG, s0.w, lane);
    double dg = (b0.y + b1.y) - (a0.y + a1.y);
    double Pf = a0.x * a1.x, Pr = b0.x * b1.x;
    if (GENERIC) {
        const double2 a2 = lds2(sCG, s1.x, lane), b2 = lds2(sCG, s1.y, lane);
        dg += b2.y - a2.y;
        Pf *= a2.x;
        Pr *= b2.x;
    }
    // k_r = k_f / K_c,  log2(1/K_c) = sum nu g2 - dnu log2(e) ln(p_ref/(RT))
    const double kr = exp2_clamped(yf + fma(-dnu, c.lc02, dg));
    return fma(-kr, Pr, kf * Pf);
}

__device__ __forceinline__ double third_body(const DevTables &m, const char *sCG, int lane, int row, double Csum)
{
    double M = Csum;
    const int e1 = __ldg(m.eff_ptr + row + 1);
    for (int e = __ldg(m.eff_ptr + row); e < e1; ++e)
        M = fma(__ldg(m.eff_val + e), lds2(sCG, (int)__ldg(m.eff_idx + e) * 512, lane).x, M);
    return M;
}

template <int KIND, bool GENERIC>
__device__ __forceinline__ double reaction_q(const DevTables &m, const char *sCG, int lane, int r, const PointCtx &c)
{
    const RatesPlan &rp = m.rp;
    const double2 c01 = __ldg(reinterpret_cast<const double2 *>(rp.rc + 4 * (size_t)r));
    const double2 c23 = __ldg(reinterpret_cast<const double2 *>(rp.rc + 4 * (size_t)r) + 1);
    const int4 s0 = __ldg(rp.rs + 2 * (size_t)r), s1 = __ldg(rp.rs + 2 * (size_t)r + 1);
    const double yinf = fma(c01.y, c.L, fma(c23.x, c.rT, c01.x));  // log2 k (high-pressure limit for falloff)
    if (KIND == 0) return progress<GENERIC>(sCG, lane, s0, s1, yinf, exp2_clamped(yinf), c23.y, c);
    const double M = third_body(m, sCG, lane, s1.z, c.Csum);
    if (KIND == 1) return M * progress<GENERIC>(sCG, lane, s0, s1, yinf, exp2_clamped(yinf), c23.y, c);
    // Troe falloff
    const double *tr = rp.troe + 8 * (size_t)s1.w;
    const double2 t01 = __ldg(reinterpret_cast<const double2 *>(tr)), t23 = __ldg(reinterpret_cast<const double2 *>(tr) + 1),
                  t45 = __ldg(reinterpret_cast<const double2 *>(tr) + 2), t67 = __ldg(reinterpret_cast<const double2 *>(tr) + 3);
    const double y0 = fma(t01.y, c.L, fma(t23.x, c.rT, t01.x));
    const double Pr = exp2_clamped(y0 - yinf) * M;
    const double al = t23.y;
    // (arguments clamped before the range reduction: T3 = 1e-30, T2 = 1e30 or inf switch a term off, rates_smem.cu)
    const double Fc = fma(1.0 - al, exp2_clamped(fmax(c.Ti * t45.x, -1022.0)),
                          fma(al, exp2_clamped(fmax(c.Ti * t45.y, -1022.0)), exp2_clamped(fmax(t67.x * c.rT, -1022.0))));
    const double lFc = log10(fmax(Fc, 1.0e-300));
    const double lPr = log10(Pr);
    const double cc = -0.4 - 0.67 * lFc;
    const double N = 0.75 - 1.27 * lFc;
    const double f1 = (lPr + cc) / (N - 0.14 * (lPr + cc));
    const double F = exp10(lFc / fma(f1, f1, 1.0));
    const double kf = exp2_clamped(yinf) * (Pr / (1.0 + Pr)) * F;
    // progress() wants log2 k_f for the reverse constant: k_r = k_f 2^(...) is formed from k_f directly here
    const double2 a0 = lds2(sCG, s0.x, lane), a1 = lds2(sCG, s0.y, lane), b0 = lds2(sCG, s0.z, lane),
                  b1 = lds2(sCG, s0.w, lane);
    double dg = (b0.y + b1.y) - (a0.y + a1.y);
    double Pf = a0.x * a1.x, Pb = b0.x * b1.x;
    if (GENERIC) {
        const double2 a2 = lds2(sCG, s1.x, lane), b2 = lds2(sCG, s1.y, lane);
        dg += b2.y - a2.y;
        Pf *= a2.x;
        Pb *= b2.x;
    }
    const double kr = kf * exp2_clamped(fma(-c23.y, c.lc02, dg));
    return fma(-kr, Pb, kf * Pf);
}

template <int W, int KIND, bool GENERIC>
__device__ __forceinline__ void reaction_stage(const DevTables &m, const char *sCG, double *sQ, int lane, int warp,
                                               int first, int count, const PointCtx &c)
{
    // two reactions per trip: independent chains for the scheduler
    int rl = warp;
    for (; rl + W < count; rl += 2 * W) {
        const double q0 = reaction_q<KIND, GENERIC>(m, sCG, lane, first + rl, c);
        const double q1 = reaction_q<KIND, GENERIC>(m, sCG, lane, first + rl + W, c);
        sQ[rl * 32 + lane] = q0;
        sQ[(rl + W) * 32 + lane] = q1;
    }
    if (rl < count) sQ[rl * 32 + lane] = reaction_q<KIND, GENERIC>(m, sCG, lane, first + rl, c);
}

template <int W, int MAXOWN>
__global__ void __launch_bounds__(32 * W, 12 / W)
    rates_staged_kernel(DevTables m, const double *__restrict__ T, const double *__restrict__ p,
                        const double *__restrict__ Y, int64_t n, double *__restrict__ omega, double *__restrict__ qdot)
{
    extern __shared__ double2 sm2[];
    const RatesPlan &rp = m.rp;
    const int Ns = m.Ns;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    double2 *sCGd = sm2;                                          // [Ns + 1][32] (C_k, log2(e) g_k/(RT)); row Ns = (1, 0)
    double *sQ = reinterpret_cast<double *>(sm2 + (size_t)(Ns + 1) * 32);  // [Rc][32]
    double *sred = sQ + (size_t)rp.Rc * 32;                        // [2][W][32]
    const char *sCG = reinterpret_cast<const char *>(sCGd);

    const int64_t i = (int64_t)blockIdx.x * 32 + lane;
    const bool valid = i < n;
    const int64_t ic = valid ? i : n - 1;
    PointCtx c;
    c.Ti = T[ic];
    const double pi = p[ic];
    c.L = log(c.Ti);
    c.rT = 1.0 / c.Ti;
    c.lc02 = crf::kLog2e * (log(m.p_ref / CRF_R_GAS) - c.L);
    c.Csum = pi * c.rT * (1.0 / CRF_R_GAS);
    const double oml = 1.0 - c.L;

    // ---- a1, a2: Z_k = Y_k/W_k and g_k; warp w owns species w, w+W, ...
    double invW = 0.0;
    for (int k = warp; k < Ns; k += W) {
        const double *g = rp.gco + 16 * (size_t)k;
        const double z = Y[(int64_t)k * n + ic] * __ldg(g + 15);
        invW += z;
        const double *a = g + ((c.Ti <= __ldg(g + 7)) ? 0 : 8);
        double v = fma(c.Ti, __ldg(a + 4), __ldg(a + 3));
        v = fma(c.Ti, v, __ldg(a + 2));
        v = fma(c.Ti, v, __ldg(a + 1));
        v = fma(c.Ti, v, __ldg(a + 6));
        v = fma(__ldg(a + 5), c.rT, v);
        v = fma(__ldg(a), oml, v);
        sCGd[k * 32 + lane] = make_double2(z, v);
    }
    if (warp == 0) sCGd[Ns * 32 + lane] = make_double2(1.0, 0.0);
    sred[warp * 32 + lane] = invW;
    __syncthreads();
    invW = 0.0;
#pragma unroll
    for (int w = 0; w < W; ++w) invW += sred[w * 32 + lane];
    const double rho = pi / (CRF_R_GAS * c.Ti * invW);
    for (int k = warp; k < Ns; k += W) sCGd[k * 32 + lane].x *= rho;  // C_k = rho Y_k / W_k
    __syncthreads();

    double om[MAXOWN];
#pragma unroll
    for (int s = 0; s < MAXOWN; ++s) om[s] = 0.0;

    for (int ci = 0; ci < rp.n_chunks; ++ci) {
        const int4 ch = __ldg(rp.chunk + ci);
        switch (ch.x) {
        case 0: reaction_stage<W, 0, false>(m, sCG, sQ, lane, warp, ch.y, ch.z, c); break;
        case 1: reaction_stage<W, 1, false>(m, sCG, sQ, lane, warp, ch.y, ch.z, c); break;
        case 2: reaction_stage<W, 2, false>(m, sCG, sQ, lane, warp, ch.y, ch.z, c); break;
        case 4: reaction_stage<W, 0, true>(m, sCG, sQ, lane, warp, ch.y, ch.z, c); break;
        case 5: reaction_stage<W, 1, true>(m, sCG, sQ, lane, warp, ch.y, ch.z, c); break;
        default: reaction_stage<W, 2, true>(m, sCG, sQ, lane, warp, ch.y, ch.z, c); break;
        }
        __syncthreads();
        const int *ptr = rp.inc_ptr + (size_t)ci * (Ns + 1);
        const char *sQb = reinterpret_cast<const char *>(sQ) + lane * 8;
#pragma unroll
        for (int s = 0; s < MAXOWN; ++s) {
            const int k = warp + W * s;
            if (k < Ns) {
                const int e1 = __ldg(ptr + k + 1);
                double acc = om[s];
                for (int e = __ldg(ptr + k); e < e1; ++e) {
                    const double2 en = __ldg(rp.inc + e);
                    acc = fma(en.x, *reinterpret_cast<const double *>(sQb + __double2loint(en.y)), acc);
                }
                om[s] = acc;
            }
        }
        __syncthreads();
    }

    // ---- store omega; a9: qdot = -sum_k h_k omega_k
    double qd = 0.0;
#pragma unroll
    for (int s = 0; s < MAXOWN; ++s) {
        const int k = warp + W * s;
        if (k < Ns) {
            const double *h = rp.hco + 16 * (size_t)k;
            const double *a = h + ((c.Ti <= __ldg(h + 7)) ? 0 : 8);
            double v = fma(c.Ti, __ldg(a + 4), __ldg(a + 3));
            v = fma(c.Ti, v, __ldg(a + 2));
            v = fma(c.Ti, v, __ldg(a + 1));
            v = fma(c.Ti, v, __ldg(a));
            v = fma(__ldg(a + 5), c.rT, v);
            qd = fma(-v, om[s], qd);
            if (valid) omega[(int64_t)k * n + i] = om[s];
        }
    }
    sred[(W + warp) * 32 + lane] = qd;
    __syncthreads();
    if (warp == 0 && valid) {
        double q = 0.0;
#pragma unroll
        for (int w = 0; w < W; ++w) q += sred[(W + w) * 32 + lane];
        qdot[i] = q * (CRF_R_GAS * c.Ti);
    }
}

template <int W, int MAXOWN>
cudaError_t launch_wm(const DevTables &m, const double *T, const double *p, const double *Y, int64_t n, double *omega,
                      double *qdot, cudaStream_t st)
{
    const size_t smem = rates_staged_dynamic_smem(m);
    cudaError_t e = cudaFuncSetAttribute(rates_staged_kernel<W, MAXOWN>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                         (int)smem);
    if (e != cudaSuccess) return e;
    rates_staged_kernel<W, MAXOWN><<<(unsigned)((n + 31) / 32), 32 * W, smem, st>>>(m, T, p, Y, n, omega, qdot);
    crf_count_launch();
    return cudaGetLastError();
}

template <int W>
cudaError_t launch_w(const DevTables &m, const double *T, const double *p, const double *Y, int64_t n, double *omega,
                     double *qdot, cudaStream_t st)
{
    const int own = (m.Ns + W - 1) / W;
    if (own <= 8) return launch_wm<W, 8>(m, T, p, Y, n, omega, qdot, st);
    if (own <= 16) return launch_wm<W, 16>(m, T, p, Y, n, omega, qdot, st);
    return launch_wm<W, 32>(m, T, p, Y, n, omega, qdot, st);
}

}  // namespace

size_t rates_staged_dynamic_smem(const DevTables &m)
{
    return sizeof(double) * (2 * 32 * (size_t)(m.Ns + 1) + 32 * (size_t)m.rp.Rc + 2 * (size_t)m.rp.W * 32);
}

cudaError_t launch_rates_staged(const DevTables &m, const double *T, const double *p, const double *Y, int64_t n,
                                double *omega, double *qdot, cudaStream_t st)
{
    switch (m.rp.W) {
    case 1: return launch_w<1>(m, T, p, Y, n, omega, qdot, st);
    case 2: return launch_w<2>(m, T, p, Y, n, omega, qdot, st);
    case 4: return launch_w<4>(m, T, p, Y, n, omega, qdot, st);
    default: return cudaErrorInvalidValue;
    }
}
