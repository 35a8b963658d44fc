// fastmath.cuh -- the one transcendental the hot loops are made of: 2^y on the FP64 pipe.
//
// The pair loop of crf_mix_transport and the reaction loop of crf_production_rates spend
// three quarters of their FP64 instructions in exp().  libdevice's exp() costs 14 DFMA + 1 DADD
// and is accurate to < 1 ulp; the tolerances of this path (1e-12 relative for transport, 1e-10
// of the gross rate for omega) allow a shorter evaluation:
//
//   y  = x * log2(e) is folded into the table coefficients on the host, so the kernels evaluate
//        2^y directly;
//   k  = rint(y) by the magic-number add, f = y - k in [-1/2, 1/2]              (3 DADD)
//   2^f = degree-9 polynomial, Chebyshev-node interpolant, relative error 1.9e-14  (9 DFMA)
//   2^k by an integer add into the exponent field                               (1 IADD)
//
// Domain: |y| < 1000 (no overflow/underflow/NaN handling).  y = -inf (an exact zero
// concentration in log space) is not supported; callers that can see it use exp().
#pragma once

namespace crf {

__device__ __forceinline__ double exp2_poly9(double y)
{
    const double magic = 6755399441055744.0;  // 1.5 * 2^52
    const double t = __dadd_rn(y, magic);
    const int k = __double2loint(t);
    const double f = __dsub_rn(y, __dsub_rn(t, magic));
    double p = 0x1.b6571de2f2351p-24;
    p = fma(p, f, 0x1.63ef969a64d3cp-20);
    p = fma(p, f, 0x1.ffcb76789860fp-17);
    p = fma(p, f, 0x1.43088e257f341p-13);
    p = fma(p, f, 0x1.5d87fe908f88ap-10);
    p = fma(p, f, 0x1.3b2ab72b175eep-7);
    p = fma(p, f, 0x1.c6b08d7044119p-5);
    p = fma(p, f, 0x1.ebfbdff8149f2p-3);
    p = fma(p, f, 0x1.62e42fefa39f7p-1);
    p = fma(p, f, 0x1.000000000003dp+0);
    return __hiloint2double(__double2hiint(p) + (k << 20), __double2loint(p));
}

// 2^y with a 16-entry table: y = k + j/16 + f, |f| <= 1/32; 2^y = 2^k T[j] p5(f).  3 DADD + 5 DFMA + 1 DMUL
// (9 FP64 instructions instead of 12) and one per-lane shared-memory load; relative error 4.7e-15
// (degree-5 Chebyshev-node interpolant of 2^f on [-1/32, 1/32]).  tab: the table kExp2Tab16 copied to shared
// memory (16 doubles = 32 banks: lanes reading different entries do not conflict).  Domain as exp2_poly9.
__device__ __forceinline__ double exp2_tab16(double y, const double *tab)
{
    const double magic = 422212465065984.0;  // 1.5 * 2^48: the sum is rounded to a multiple of 1/16
    const double t = __dadd_rn(y, magic);
    const int n = __double2loint(t);  // round(16 y)
    const double f = __dsub_rn(y, __dsub_rn(t, magic));
    double p = 0x1.5d897e525c216p-10;
    p = fma(p, f, 0x1.3b2c9b8a6caeap-7);
    p = fma(p, f, 0x1.c6b08d6f2a289p-5);
    p = fma(p, f, 0x1.ebfbdff555824p-3);
    p = fma(p, f, 0x1.62e42fefa39f3p-1);
    p = fma(p, f, 0x1.0000000000014p+0);
    p *= tab[n & 15];
    return __hiloint2double(__double2hiint(p) + ((n >> 4) << 20), __double2loint(p));
}

#define CRF_EXP2_TAB16                                                                                           \
    {0x1.0000000000000p+0, 0x1.0b5586cf9890fp+0, 0x1.172b83c7d517bp+0, 0x1.2387a6e756238p+0, 0x1.306fe0a31b715p+0, \
     0x1.3dea64c123422p+0, 0x1.4bfdad5362a27p+0, 0x1.5ab07dd485429p+0, 0x1.6a09e667f3bcdp+0, 0x1.7a11473eb0187p+0, \
     0x1.8ace5422aa0dbp+0, 0x1.9c49182a3f090p+0, 0x1.ae89f995ad3adp+0, 0x1.c199bdd85529cp+0, 0x1.d5818dcfba487p+0, \
     0x1.ea4afa2a490dap+0}

// 1/x for normal x: MUFU.RCP64H seed (relative error < 2^-20) and one cubic Newton step (error ~ 2^-60 + rounding)
__device__ __forceinline__ double rcp_newton(double x)
{
    double y;
    asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(x));
    const double e = fma(-x, y, 1.0);
    return fma(y, fma(e, e, e), y);
}

constexpr double kLog2e = 1.4426950408889634074;

}  // namespace crf
