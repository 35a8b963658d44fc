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

// 2^y with a 64-entry table: y = k + j/64 + f, |f| <= 1/128; 2^y = 2^k T[j] p4(f).  3 DADD + 4 DFMA + 1 DMUL
// (8 FP64 instructions) and one per-lane shared-memory load; relative error 2.5e-15 (degree-4 Chebyshev-node
// interpolant of 2^f on [-1/128, 1/128]).  tab: the table CRF_EXP2_TAB64 copied to shared memory.
__device__ __forceinline__ double exp2_tab64(double y, const double *tab)
{
    const double magic = 105553116266496.0;  // 1.5 * 2^46: the sum is rounded to a multiple of 1/64
    const double t = __dadd_rn(y, magic);
    const int n = __double2loint(t);  // round(64 y)
    const double f = __dsub_rn(y, __dsub_rn(t, magic));
    double p = 0x1.3b2ad0385b409p-7;
    p = fma(p, f, 0x1.c6b0c40d8c4e9p-5);
    p = fma(p, f, 0x1.ebfbdff82ac52p-3);
    p = fma(p, f, 0x1.62e42fefa0352p-1);
    p = fma(p, f, 1.0);
    p *= tab[n & 63];
    return __hiloint2double(__double2hiint(p) + ((n >> 6) << 20), __double2loint(p));
}

#define CRF_EXP2_TAB64 \
    {0x1.0000000000000p+0, 0x1.02c9a3e778061p+0, 0x1.059b0d3158574p+0, 0x1.0874518759bc8p+0, \
     0x1.0b5586cf9890fp+0, 0x1.0e3ec32d3d1a2p+0, 0x1.11301d0125b51p+0, 0x1.1429aaea92de0p+0, \
     0x1.172b83c7d517bp+0, 0x1.1a35beb6fcb75p+0, 0x1.1d4873168b9aap+0, 0x1.2063b88628cd6p+0, \
     0x1.2387a6e756238p+0, 0x1.26b4565e27cddp+0, 0x1.29e9df51fdee1p+0, 0x1.2d285a6e4030bp+0, \
     0x1.306fe0a31b715p+0, 0x1.33c08b26416ffp+0, 0x1.371a7373aa9cbp+0, 0x1.3a7db34e59ff7p+0, \
     0x1.3dea64c123422p+0, 0x1.4160a21f72e2ap+0, 0x1.44e086061892dp+0, 0x1.486a2b5c13cd0p+0, \
     0x1.4bfdad5362a27p+0, 0x1.4f9b2769d2ca7p+0, 0x1.5342b569d4f82p+0, 0x1.56f4736b527dap+0, \
     0x1.5ab07dd485429p+0, 0x1.5e76f15ad2148p+0, 0x1.6247eb03a5585p+0, 0x1.6623882552225p+0, \
     0x1.6a09e667f3bcdp+0, 0x1.6dfb23c651a2fp+0, 0x1.71f75e8ec5f74p+0, 0x1.75feb564267c9p+0, \
     0x1.7a11473eb0187p+0, 0x1.7e2f336cf4e62p+0, 0x1.82589994cce13p+0, 0x1.868d99b4492edp+0, \
     0x1.8ace5422aa0dbp+0, 0x1.8f1ae99157736p+0, 0x1.93737b0cdc5e5p+0, 0x1.97d829fde4e50p+0, \
     0x1.9c49182a3f090p+0, 0x1.a0c667b5de565p+0, 0x1.a5503b23e255dp+0, 0x1.a9e6b5579fdbfp+0, \
     0x1.ae89f995ad3adp+0, 0x1.b33a2b84f15fbp+0, 0x1.b7f76f2fb5e47p+0, 0x1.bcc1e904bc1d2p+0, \
     0x1.c199bdd85529cp+0, 0x1.c67f12e57d14bp+0, 0x1.cb720dcef9069p+0, 0x1.d072d4a07897cp+0, \
     0x1.d5818dcfba487p+0, 0x1.da9e603db3285p+0, 0x1.dfc97337b9b5fp+0, 0x1.e502ee78b3ff6p+0, \
     0x1.ea4afa2a490dap+0, 0x1.efa1bee615a27p+0, 0x1.f50765b6e4540p+0, 0x1.fa7c1819e90d8p+0}

// 1/x for normal x: MUFU.RCP64H seed (relative error < 2^-20) and one cubic Newton step (error ~ 2^-60 + rounding)
__device__ __forceinline__ double rcp_newton(double x)
{
    double y;
    asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(x));
    const double e = fma(-x, y, 1.0);
    return fma(y, fma(e, e, e), y);
}

constexpr double kLog2e = 1.4426950408889634074;

// ---- the transcendentals of the production-rates kernels (rates_group.cu, rates_smem.cu, rates_staged.cu) -------------
// Coefficients in constant memory: the FP64 instructions take them as constant-bank operands instead of occupying (and
// re-materialising) registers.  (static: every translation unit that includes this header gets its own copy)
// 2^f on [-1/2, 1/2]: degree 8 (Chebyshev-node interpolant, relative error 1.06e-12) and degree 9 (1.9e-14)
static __constant__ double kExp2P8[9] = {0x1.0000000000000p+0,  0x1.62e42fef84cf0p-1,  0x1.ebfbdff823cedp-3,
                                         0x1.c6b08dd6fd234p-5,  0x1.3b2ab7181b755p-7,  0x1.5d8745a728441p-10,
                                         0x1.4308ac85aa947p-13, 0x1.00dc4a532fb8ep-16, 0x1.63d136366db24p-20};
static __constant__ double kExp2P9[10] = {0x1.000000000003dp+0,  0x1.62e42fefa39f7p-1,  0x1.ebfbdff8149f2p-3,
                                          0x1.c6b08d7044119p-5,  0x1.3b2ab72b175eep-7,  0x1.5d87fe908f88ap-10,
                                          0x1.43088e257f341p-13, 0x1.ffcb76789860fp-17, 0x1.63ef969a64d3cp-20,
                                          0x1.b6571de2f2351p-24};
static __constant__ double kAtanhOdd[9] = {1.0,        1.0 / 3.0,  1.0 / 5.0,  1.0 / 7.0, 1.0 / 9.0,
                                           1.0 / 11.0, 1.0 / 13.0, 1.0 / 15.0, 1.0 / 17.0};

// 2^y by the degree-DEG polynomial (8 or 9), the exponent clamped from below: an underflowing rate constant becomes a
// negligible number instead of wrapping into the sign bit.  |y| < 2^31 (callers clamp arguments that can be
// arbitrarily large before the range reduction).
template <int DEG>
__device__ __forceinline__ double exp2_clamped(double y)
{
    static_assert(DEG == 8 || DEG == 9, "degree 8 or 9");
    const double magic = 6755399441055744.0;  // 1.5 * 2^52
    const double t = __dadd_rn(y, magic);
    const int k = max(__double2loint(t), -1000);
    const double f = __dsub_rn(y, __dsub_rn(t, magic));
    double p = DEG == 8 ? kExp2P8[8] : kExp2P9[9];
#pragma unroll
    for (int i = DEG - 1; i >= 0; --i) p = fma(p, f, DEG == 8 ? kExp2P8[i] : kExp2P9[i]);
    return __hiloint2double(__double2hiint(p) + (k << 20), __double2loint(p));
}

// log2(x) for normal x > 0, branch-free: x = 2^e m, m in [sqrt(1/2), sqrt(2)), ln m = 2 atanh((m-1)/(m+1)), the odd
// series truncated after TERMS terms (|s| <= 0.172: 7 terms = absolute error 2e-12, 9 terms = 3e-15)
template <int TERMS>
__device__ __forceinline__ double log2_atanh(double x)
{
    static_assert(TERMS >= 2 && TERMS <= 9, "2..9 terms");
    int hi = __double2hiint(x);
    const int e = (hi - 0x3fe6a09e) >> 20;
    hi -= e << 20;
    const double m = __hiloint2double(hi, __double2loint(x));
    const double s = (m - 1.0) * rcp_newton(m + 1.0);
    const double z = s * s;
    double p = kAtanhOdd[TERMS - 1];
#pragma unroll
    for (int i = TERMS - 2; i >= 0; --i) p = fma(p, z, kAtanhOdd[i]);
    return fma(s * (2.0 * kLog2e), p, (double)e);
}

}  // namespace crf
