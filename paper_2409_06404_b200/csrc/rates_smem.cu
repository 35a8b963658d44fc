// rates_smem.cu -- crf_production_rates for SMALL mechanisms: one thread per grid
// point (plan_rates_smem.cu admits Ns <= 12 by default, up to 24 on request); larger mechanisms run rates_group.cu.
//
// Per point and species the thread keeps (C_k, d_k), d_k = (p_ref/RT) exp(-g_k/RT), as a column in shared memory.
//
//   k_f        = 2^(log2e lnA + log2e beta ln T - log2e Ea/(R T))                 one exponential per reaction
//   1/K_c      = prod_reactants d / prod_products d                               (K_c = exp(-sum nu g/RT) (p_ref/RT)^dnu)
//   q          = k_f [M] (prod_reactants C - (1/K_c) prod_products C)
//
// i.e. the second exponential of a reversible reaction is replaced by two multiplications and one
// reciprocal (MUFU seed + one cubic Newton step); the exponentials of g_k are taken once per species and
// point.  crf_mech_create admits this form only if numerator, denominator and quotient stay inside the
// double range for every T in [250, 5000] K (plan_rates_smem.cu), otherwise rates_staged.cu runs.
//
// Reactions are cut into chunks of one kind (elementary | third body | Troe falloff; two or three species per side);
// all chunk blocks (48-byte reaction records, third-body lists, Troe sets) are resident in shared memory.
// Troe falloff is evaluated in base 2 (log2 F = log2 F_cent / (1 + f1^2)) with a branch-free logarithm.
#include <algorithm>

#include "crf_internal.h"
#include "fastmath.cuh"
#include "launch.h"
#include "tmem.cuh"

namespace {

// the transcendentals (fastmath.cuh): 2^y by the degree-9 polynomial, Newton reciprocal, atanh-series log2 (9 terms)
__device__ __forceinline__ double exp2c(double y) { return crf::exp2_clamped<9>(y); }
__device__ __forceinline__ double rcp_fast(double x) { return crf::rcp_newton(x); }
__device__ __forceinline__ double log2_fast(double x) { return crf::log2_atanh<9>(x); }

template <int PPL>
struct Ctx {
    double T[PPL], L[PPL], rT[PPL];  // T, ln T, 1/T
    double Csum[PPL];                // p/(R T)
};

__device__ __forceinline__ double2 lds2(const char *p) { return *reinterpret_cast<const double2 *>(p); }
__device__ __forceinline__ uint4 ldsu4(const char *p) { return *reinterpret_cast<const uint4 *>(p); }

// q of one reaction at the PPL points of this lane.  rec: the 48-byte record; tr: its Troe set (kind 2);
// sL: the (C, d) state at this lane (row offsets come from the record; point u is 512 u bytes further).
// TM: the (C, d) pairs live in tensor memory (PPL = 1; tmq = this warp's quadrant address; pair k at column 4 k = row offset / 512).
template <int KIND, bool GENERIC, int PPL, bool TM = false>
__device__ __forceinline__ void reaction_q(const char *blk, const char *rec, const char *tr, const char *sL,
                                           const Ctx<PPL> &c, double (&q)[PPL], unsigned tmq = 0u)
{
    const double2 A = lds2(rec);        // log2e lnA, log2e beta
    const double2 Ex = lds2(rec + 16);  // -log2e Ea/R, (x0, x1)
    const uint4 S = ldsu4(rec + 32);    // a0, a1, b0, b1
    const unsigned x0 = (unsigned)__double2loint(Ex.y), x1 = (unsigned)__double2hiint(Ex.y);
    double M[PPL];
    if (KIND != 0) {
#pragma unroll
        for (int u = 0; u < PPL; ++u) M[u] = c.Csum[u];
        const char *e = blk + x0, *e1 = e + 16 * x1;
        for (; e < e1; e += 16) {
            const uint4 en = ldsu4(e);
            const double coef = __hiloint2double((int)en.y, (int)en.x);
#pragma unroll
            for (int u = 0; u < PPL; ++u) {
                double Ck;
                if (TM) {
                    crf::TmRow<1> r;
                    crf::tm_ld<1>(tmq + (en.z >> 9), r);
                    crf::tm_wait1<1>(r);
                    Ck = crf::tm_one(r);
                } else {
                    Ck = lds2(sL + en.z + 512 * u).x;
                }
                M[u] = fma(coef, Ck, M[u]);
            }
        }
    }
#pragma unroll
    for (int u = 0; u < PPL; ++u) {
        const char *s = sL + 512 * u;
        const double yinf = fma(A.y, c.L[u], fma(Ex.x, c.rT[u], A.x));  // log2 k_f (high-pressure limit)
        double2 a0, a1, b0, b1;
        if (TM) {
            crf::TmRow<2> r0, r1, r2, r3;
            crf::tm_ld<2>(tmq + (S.x >> 9), r0), crf::tm_ld<2>(tmq + (S.y >> 9), r1);
            crf::tm_ld<2>(tmq + (S.z >> 9), r2), crf::tm_ld<2>(tmq + (S.w >> 9), r3);
            crf::tm_wait4(r0, r1, r2, r3);
            a0 = crf::tm_pair(r0), a1 = crf::tm_pair(r1), b0 = crf::tm_pair(r2), b1 = crf::tm_pair(r3);
        } else {
            a0 = lds2(s + S.x), a1 = lds2(s + S.y), b0 = lds2(s + S.z), b1 = lds2(s + S.w);
        }
        double Pf = a0.x * a1.x, Pr = b0.x * b1.x, num = a0.y * a1.y, den = b0.y * b1.y;
        if (GENERIC) {
            double2 a2, b2;
            if (TM) {
                crf::TmRow<2> r0, r1;
                crf::tm_ld<2>(tmq + (x0 >> 9), r0), crf::tm_ld<2>(tmq + (x1 >> 9), r1);
                crf::tm_wait1<2>(r0), crf::tm_wait1<2>(r1);
                a2 = crf::tm_pair(r0), b2 = crf::tm_pair(r1);
            } else {
                a2 = lds2(s + x0), b2 = lds2(s + x1);
            }
            Pf *= a2.x, Pr *= b2.x, num *= a2.y, den *= b2.y;
        }
        // 1/K_c = num/den with the MUFU seed and ONE Newton step (relative error 2^-40: the tolerance of omega is
        // 1e-10 of the gross rate); net = prod C_reactants - prod C_products / K_c
        double ry;
        asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(ry) : "d"(den));
        const double t0 = num * ry;
        const double net = fma(-fma(t0, fma(-den, ry, 1.0), t0), Pr, Pf);
        if (KIND == 0) q[u] = exp2c(yinf) * net;
        if (KIND == 1) q[u] = exp2c(yinf) * M[u] * net;
        if (KIND == 2) {
            // Troe falloff in base 2
            const double2 t01 = lds2(tr), t23 = lds2(tr + 16), t45 = lds2(tr + 32), t67 = lds2(tr + 48);
            const double y0 = fma(t01.y, c.L[u], fma(t23.x, c.rT[u], t01.x));
            const double l2Pr = (y0 - yinf) + log2_fast(fmax(M[u], 1.0e-300));  // log2(k_0 [M] / k_inf)
            const double al = t23.y;
            // (the arguments are clamped BEFORE the range reduction: Chemkin-style switched-off terms, T3 = 1e-30 or
            // T2 = 1e30 / inf, give arguments of -1e33 or -inf, whose integer part has no meaning as an exponent)
            const double Fc = fma(1.0 - al, exp2c(fmax(c.T[u] * t45.x, -1022.0)),
                                  fma(al, exp2c(fmax(c.T[u] * t45.y, -1022.0)), exp2c(fmax(t67.x * c.rT[u], -1022.0))));
            const double l2Fc = log2_fast(fmax(Fc, 1.0e-300));
            const double l10_2 = 0.30102999566398119521;
            const double lFc = l10_2 * l2Fc;
            const double x = fma(l10_2, l2Pr, fma(-0.67, lFc, -0.4));  // log10 P_r + c
            const double f1 = x * rcp_fast(fma(-0.14, x, fma(-1.27, lFc, 0.75)));
            const double l2F = l2Fc * rcp_fast(fma(f1, f1, 1.0));
            const double Pred = exp2c(l2Pr);
            q[u] = exp2c(yinf + l2F) * (Pred * rcp_fast(1.0 + Pred)) * net;
        }
    }
}

// ---------------------------------------------------------------------------------------------------------------
// Small mechanisms (plan W = 1, PPL = 4): one THREAD per point, 128 points per block.  The (C, d) state and the
// omega accumulators are per-thread columns in shared memory (row stride 128 x 16 and 128 x 8 bytes), every chunk
// block is resident, each thread walks all reactions and scatters q into its own omega column: no incidence
// lists, no q buffer and no barrier after the tables have landed; the SM holds 12-28 warps.
constexpr int RT_B = 128;

__device__ __forceinline__ void scatter_q(char *om, const char *rec, double q, bool generic)
{
    const uint4 S = ldsu4(rec + 32);  // state row offsets (stride 2048) -> omega rows (stride 1024)
    if (!generic && S.x != S.y && S.z != S.w && S.x != S.z && S.x != S.w && S.y != S.z && S.y != S.w) {
        // four distinct rows (a warp-uniform test): the four loads go out together, then the four stores
        double *r0 = reinterpret_cast<double *>(om + (S.x >> 1)), *r1 = reinterpret_cast<double *>(om + (S.y >> 1));
        double *r2 = reinterpret_cast<double *>(om + (S.z >> 1)), *r3 = reinterpret_cast<double *>(om + (S.w >> 1));
        const double v0 = *r0, v1 = *r1, v2 = *r2, v3 = *r3;
        *r0 = v0 - q, *r1 = v1 - q, *r2 = v2 + q, *r3 = v3 + q;
        return;
    }
    *reinterpret_cast<double *>(om + (S.x >> 1)) -= q;
    *reinterpret_cast<double *>(om + (S.y >> 1)) -= q;
    *reinterpret_cast<double *>(om + (S.z >> 1)) += q;
    *reinterpret_cast<double *>(om + (S.w >> 1)) += q;
    if (generic) {
        const uint2 X = *reinterpret_cast<const uint2 *>(rec + 24);
        *reinterpret_cast<double *>(om + (X.x >> 1)) -= q;
        *reinterpret_cast<double *>(om + (X.y >> 1)) += q;
    }
}

template <int KIND, bool GENERIC>
__device__ __forceinline__ void thread_chunk(const char *blk, int count, int o_troe, const char *sL, char *om, const Ctx<1> &c)
{
    constexpr int NR = 4;  // independent reactions per trip
    int rl = 0;
    for (; rl + NR - 1 < count; rl += NR) {
        double q[NR][1];
#pragma unroll
        for (int v = 0; v < NR; ++v)
            reaction_q<KIND, GENERIC, 1>(blk, blk + 48 * (rl + v), blk + o_troe + 64 * (rl + v), sL, c, q[v]);
#pragma unroll
        for (int v = 0; v < NR; ++v) scatter_q(om, blk + 48 * (rl + v), q[v][0], GENERIC);
    }
    for (; rl < count; ++rl) {
        double q0[1];
        reaction_q<KIND, GENERIC, 1>(blk, blk + 48 * rl, blk + o_troe + 64 * rl, sL, c, q0);
        scatter_q(om, blk + 48 * rl, q0[0], GENERIC);
    }
}

__global__ void __launch_bounds__(RT_B) rates_thread_kernel(DevTables m, const double *__restrict__ T,
                                                            const double *__restrict__ p, const double *__restrict__ Y,
                                                            int64_t n, double *__restrict__ omega, double *__restrict__ qdot)
{
    extern __shared__ double2 sm2[];
    const RatesSmemPlan &rs = m.rs;
    const int Ns = m.Ns, tid = threadIdx.x;
    char *sCD = reinterpret_cast<char *>(sm2);        // [Ns + 1][128] (C_k, d_k); row Ns = (1, 1)
    char *sOm = sCD + (size_t)(Ns + 1) * 2048;        // [Ns + 1][128] omega_k; row Ns collects the empty slots
    char *sTab = sOm + (size_t)(Ns + 1) * 1024;       // the chunk blocks
    char *sGH = sTab + rs.stage_bytes;                // g/(RT) sets [Ns][128 B], then h/(RT) sets [Ns][128 B]
    for (int o = tid * 16; o < rs.stage_bytes; o += RT_B * 16)
        *reinterpret_cast<uint4 *>(sTab + o) = __ldg(reinterpret_cast<const uint4 *>(rs.stage + o));
    for (int o = tid * 16; o < 128 * Ns; o += RT_B * 16) {
        *reinterpret_cast<uint4 *>(sGH + o) = __ldg(reinterpret_cast<const uint4 *>(reinterpret_cast<const char *>(rs.gco) + o));
        *reinterpret_cast<uint4 *>(sGH + 128 * Ns + o) =
            __ldg(reinterpret_cast<const uint4 *>(reinterpret_cast<const char *>(rs.hco) + o));
    }
    char *sL = sCD + tid * 16, *om = sOm + tid * 8;

    const int64_t i = (int64_t)blockIdx.x * RT_B + tid;
    const int64_t ic = i < n ? i : n - 1;  // threads past the end recompute the last point and store nothing
    Ctx<1> c;
    c.T[0] = T[ic];
    const double pi = p[ic], Tu = c.T[0];
    c.L[0] = log(Tu);
    c.rT[0] = 1.0 / Tu;
    const double lc02 = crf::kLog2e * (log(m.p_ref / CRF_R_GAS) - c.L[0]);
    c.Csum[0] = pi * c.rT[0] * (1.0 / CRF_R_GAS);
    const double oml = 1.0 - c.L[0];

    __syncthreads();  // the tables have landed (the state and omega columns are private to the thread)
    double invW = 0.0;
    for (int k0 = 0; k0 < Ns; k0 += 4) {
      double y4[4];
#pragma unroll
      for (int j = 0; j < 4; ++j) y4[j] = Y[(int64_t)min(k0 + j, Ns - 1) * n + ic];  // four row loads in flight
#pragma unroll
      for (int j = 0; j < 4; ++j) {
        const int k = k0 + j;
        if (k >= Ns) break;
        const double2 *g = reinterpret_cast<const double2 *>(sGH) + 8 * k;
        const double2 l01 = g[0], l23 = g[1], l45 = g[2], l6t = g[3];
        const double2 h01 = g[4], h23 = g[5], h45 = g[6], h6w = g[7];
        const double y = y4[j];
        double lo = fma(Tu, l45.x, l23.y);
        lo = fma(Tu, lo, l23.x);
        lo = fma(Tu, lo, l01.y);
        lo = fma(Tu, lo, l6t.x);
        lo = fma(l45.y, c.rT[0], lo);
        lo = fma(l01.x, oml, lo);
        double hi = fma(Tu, h45.x, h23.y);
        hi = fma(Tu, hi, h23.x);
        hi = fma(Tu, hi, h01.y);
        hi = fma(Tu, hi, h6w.x);
        hi = fma(h45.y, c.rT[0], hi);
        hi = fma(h01.x, oml, hi);
        const double g2 = Tu <= l6t.y ? lo : hi;
        const double z = y * h6w.y;
        invW += z;
        *reinterpret_cast<double2 *>(sL + (size_t)k * 2048) = make_double2(z, exp2c(lc02 - g2));
        *reinterpret_cast<double *>(om + (size_t)k * 1024) = 0.0;
      }
    }
    *reinterpret_cast<double2 *>(sL + (size_t)Ns * 2048) = make_double2(1.0, 1.0);
    *reinterpret_cast<double *>(om + (size_t)Ns * 1024) = 0.0;
    const double rho = pi / (CRF_R_GAS * Tu * invW);
    for (int k = 0; k < Ns; ++k) *reinterpret_cast<double *>(sL + (size_t)k * 2048) *= rho;  // C_k

    for (int ci = 0; ci < rs.n_chunks; ++ci) {
        const int4 ch = __ldg(rs.chunk + ci);
        const char *blk = sTab + ch.z;
        const int count = ch.y, o_troe = 48 * count + 32;  // one slot row (W = 1, maxown = 4) follows the records
        switch (ch.x) {
        case 0: thread_chunk<0, false>(blk, count, o_troe, sL, om, c); break;
        case 1: thread_chunk<1, false>(blk, count, o_troe, sL, om, c); break;
        case 2: thread_chunk<2, false>(blk, count, o_troe, sL, om, c); break;
        default: thread_chunk<0, true>(blk, count, o_troe, sL, om, c); break;
        }
    }

    // ---- store omega; a9: qdot = -sum_k h_k omega_k
    double qd = 0.0;
    for (int k = 0; k < Ns; ++k) {
        const double2 *h = reinterpret_cast<const double2 *>(sGH + 128 * Ns) + 8 * k;
        const double2 l01 = h[0], l23 = h[1], l45 = h[2], l6t = h[3];
        const double2 h01 = h[4], h23 = h[5], h45 = h[6];
        double lo = fma(Tu, l45.x, l23.y);
        lo = fma(Tu, lo, l23.x);
        lo = fma(Tu, lo, l01.y);
        lo = fma(Tu, lo, l01.x);
        lo = fma(l45.y, c.rT[0], lo);
        double hi = fma(Tu, h45.x, h23.y);
        hi = fma(Tu, hi, h23.x);
        hi = fma(Tu, hi, h01.y);
        hi = fma(Tu, hi, h01.x);
        hi = fma(h45.y, c.rT[0], hi);
        const double w = *reinterpret_cast<const double *>(om + (size_t)k * 1024);
        qd = fma(-(Tu <= l6t.y ? lo : hi), w, qd);
        if (i < n) omega[(int64_t)k * n + i] = w;
    }
    if (i < n) qdot[i] = qd * (CRF_R_GAS * Tu);
}

// ---------------------------------------------------------------------------------------------------------------
// The same kernel with the per-thread state in TENSOR MEMORY (tmem.cuh): the (C, d) pair of species k in columns
// 4 k .. 4 k + 3 of the thread's lane, omega_k in columns 4 (Ns + 1) + 2 k.  ncu showed the shared-memory version
// bound by the shared-memory pipe (90 % of its wavefronts on C2): every state access there is a non-broadcast 64- or
// 128-bit access per lane.  Tensor memory is indexed by a warp-uniform column (the species of the reaction) and has its
// own data path; shared memory keeps only the mechanism's tables (broadcast reads).
__device__ __forceinline__ void scatter_q_tm(unsigned tom, const char *rec, double q, bool generic)
{
    const uint4 S = ldsu4(rec + 32);  // state row offsets (stride 2048) -> omega columns (2 per species)
    const unsigned c0 = tom + (S.x >> 10), c1 = tom + (S.y >> 10), c2 = tom + (S.z >> 10), c3 = tom + (S.w >> 10);
    if (!generic && S.x != S.y && S.z != S.w && S.x != S.z && S.x != S.w && S.y != S.z && S.y != S.w) {
        // four distinct species (a warp-uniform test): the four loads go out together, then the four stores
        crf::TmRow<1> r0, r1, r2, r3;
        crf::tm_ld<1>(c0, r0), crf::tm_ld<1>(c1, r1), crf::tm_ld<1>(c2, r2), crf::tm_ld<1>(c3, r3);
        crf::tm_wait4(r0, r1, r2, r3);
        const double v0[1] = {crf::tm_one(r0) - q}, v1[1] = {crf::tm_one(r1) - q}, v2[1] = {crf::tm_one(r2) + q},
                     v3[1] = {crf::tm_one(r3) + q};
        crf::tm_st<1>(c0, v0), crf::tm_st<1>(c1, v1), crf::tm_st<1>(c2, v2), crf::tm_st<1>(c3, v3);
        return;
    }
    auto add = [&](unsigned col, double dq) {  // (a species listed twice: the updates must follow one another)
        crf::TmRow<1> r;
        crf::tm_ld<1>(col, r);
        crf::tm_wait1<1>(r);
        const double v[1] = {crf::tm_one(r) + dq};
        crf::tm_st<1>(col, v);
        crf::tm_wait_st();
    };
    add(c0, -q), add(c1, -q), add(c2, q), add(c3, q);
    if (generic) {
        const uint2 X = *reinterpret_cast<const uint2 *>(rec + 24);
        add(tom + (X.x >> 10), -q), add(tom + (X.y >> 10), q);
    }
}

template <int KIND, bool GENERIC>
__device__ __forceinline__ void thread_chunk_tm(const char *blk, int count, int o_troe, unsigned tmq, unsigned tom, const Ctx<1> &c)
{
    constexpr int NR = 2;  // independent reactions per trip (1, 3, 4 measured: no difference)
    int rl = 0;
    for (; rl + NR - 1 < count; rl += NR) {
        double q[NR][1];
#pragma unroll
        for (int v = 0; v < NR; ++v)
            reaction_q<KIND, GENERIC, 1, true>(blk, blk + 48 * (rl + v), blk + o_troe + 64 * (rl + v), nullptr, c, q[v], tmq);
#pragma unroll
        for (int v = 0; v < NR; ++v) {
            scatter_q_tm(tom, blk + 48 * (rl + v), q[v][0], GENERIC);
            crf::tm_wait_st();  // (the next reaction may update the same species)
        }
    }
    for (; rl < count; ++rl) {
        double q0[1];
        reaction_q<KIND, GENERIC, 1, true>(blk, blk + 48 * rl, blk + o_troe + 64 * rl, nullptr, c, q0, tmq);
        scatter_q_tm(tom, blk + 48 * rl, q0[0], GENERIC);
        crf::tm_wait_st();
    }
}

// MODE (RatesIO.mode; 3 = mode 0 with the by-products of crf_rhs_pointwise): in modes 1 and 2 the thread evaluates the
// two states of its grid point one after the other (the tables are staged once, the tensor-memory columns are reused).
template <int MODE>
__global__ void __launch_bounds__(RT_B) rates_thread_tm_kernel(DevTables m, RatesIO io, int64_t n, unsigned tm_cols)
{
    extern __shared__ double2 sm2[];
    __shared__ unsigned sTmBase;
    const RatesSmemPlan &rs = m.rs;
    const int Ns = m.Ns, tid = threadIdx.x, warp = tid >> 5;
    char *sTab = reinterpret_cast<char *>(sm2);  // the chunk blocks
    char *sGH = sTab + rs.stage_bytes;            // g/(RT) sets [Ns][128 B], then h/(RT) sets [Ns][128 B]
    if (warp == 0) crf::tm_alloc(&sTmBase, tm_cols);
    for (int o = tid * 16; o < rs.stage_bytes; o += RT_B * 16)
        *reinterpret_cast<uint4 *>(sTab + o) = __ldg(reinterpret_cast<const uint4 *>(rs.stage + o));
    for (int o = tid * 16; o < 128 * Ns; o += RT_B * 16) {
        *reinterpret_cast<uint4 *>(sGH + o) = __ldg(reinterpret_cast<const uint4 *>(reinterpret_cast<const char *>(rs.gco) + o));
        *reinterpret_cast<uint4 *>(sGH + 128 * Ns + o) =
            __ldg(reinterpret_cast<const uint4 *>(reinterpret_cast<const char *>(rs.hco) + o));
    }
    const int64_t i = (int64_t)blockIdx.x * RT_B + tid;
    const int64_t ic = i < n ? i : n - 1;  // threads past the end recompute the last point and store nothing
    crf::tm_fence_before_sync();
    __syncthreads();  // the tables have landed, the tensor-memory columns are allocated
    crf::tm_fence_after_sync();
    const unsigned tmq = crf::tm_quadrant(sTmBase, warp);
    constexpr int NSTATE = (MODE == 1 || MODE == 2) ? 2 : 1;
    const double zero[1] = {0.0};

#pragma unroll 1
    for (int st = 0; st < NSTATE; ++st) {
        const unsigned tom = tmq + 4u * (Ns + 1);  // omega of this state (the columns are reused by the second state)
        // the state: mode 1 = the second set of arrays, mode 2 = perturbed in place (multiply, then add: one rounding each)
        auto in = [&](const double *a, const double *b, double sg, int64_t idx) {
            if (MODE == 4) return __dadd_rn(a[idx], __dmul_rn(sg, b[idx]));  // (the perturbed state only: the base is given)
            if (st == 0 || MODE == 0 || MODE == 3) return a[idx];
            return MODE == 1 ? b[idx] : __dadd_rn(a[idx], __dmul_rn(sg, b[idx]));
        };
        Ctx<1> c;
        c.T[0] = in(io.T, io.T2, io.sigma, ic);
        const double pi = in(io.p, io.p2, io.sigma_p, ic), Tu = c.T[0];
        c.L[0] = log(Tu);
        c.rT[0] = 1.0 / Tu;
        const double lc02 = crf::kLog2e * (log(m.p_ref / CRF_R_GAS) - c.L[0]);
        c.Csum[0] = pi * c.rT[0] * (1.0 / CRF_R_GAS);
        const double oml = 1.0 - c.L[0];

        double invW = 0.0;
        for (int k0 = 0; k0 < Ns; k0 += 4) {
            double y4[4];
#pragma unroll
            for (int j = 0; j < 4; ++j) {  // four row loads in flight
                const int64_t idx = (int64_t)min(k0 + j, Ns - 1) * n + ic;
                y4[j] = in(io.Y, io.Y2, io.sigma, idx);
            }
#pragma unroll
            for (int j = 0; j < 4; ++j) {
                const int k = k0 + j;
                if (k >= Ns) break;
                const double2 *g = reinterpret_cast<const double2 *>(sGH) + 8 * k;
                const double2 *gs = g + (Tu <= g[3].y ? 0 : 4);
                const double2 c01 = gs[0], c23 = gs[1], c45 = gs[2];
                double g2 = fma(Tu, c45.x, c23.y);
                g2 = fma(Tu, g2, c23.x);
                g2 = fma(Tu, g2, c01.y);
                g2 = fma(Tu, g2, gs[3].x);
                g2 = fma(c45.y, c.rT[0], g2);
                g2 = fma(c01.x, oml, g2);
                const double z = y4[j] * g[7].y;
                invW += z;
                const double zd[2] = {z, exp2c(lc02 - g2)};
                crf::tm_st<2>(tmq + 4u * k, zd);
                crf::tm_st<1>(tom + 2u * k, zero);
            }
        }
        const double one[2] = {1.0, 1.0};
        crf::tm_st<2>(tmq + 4u * Ns, one);
        crf::tm_st<1>(tom + 2u * Ns, zero);
        crf::tm_wait_st();
        const double rho = pi / (CRF_R_GAS * Tu * invW);
        for (int k = 0; k < Ns; ++k) {  // C_k = rho Z_k
            crf::TmRow<1> r;
            crf::tm_ld<1>(tmq + 4u * k, r);
            crf::tm_wait1<1>(r);
            const double v[1] = {crf::tm_one(r) * rho};
            crf::tm_st<1>(tmq + 4u * k, v);
        }
        crf::tm_wait_st();
        if (MODE == 3 && i < n) {  // by-products of crf_rhs_pointwise (Eq. 1d)
            if (io.rho) io.rho[i] = rho;
            if (io.Wbar) io.Wbar[i] = 1.0 / invW;
        }

        for (int ci = 0; ci < rs.n_chunks; ++ci) {
            const int4 ch = __ldg(rs.chunk + ci);
            const char *blk = sTab + ch.z;
            const int count = ch.y, o_troe = 48 * count + 32;  // one slot row (W = 1, maxown = 4) follows the records
            switch (ch.x) {
            case 0: thread_chunk_tm<0, false>(blk, count, o_troe, tmq, tom, c); break;
            case 1: thread_chunk_tm<1, false>(blk, count, o_troe, tmq, tom, c); break;
            case 2: thread_chunk_tm<2, false>(blk, count, o_troe, tmq, tom, c); break;
            default: thread_chunk_tm<0, true>(blk, count, o_troe, tmq, tom, c); break;
            }
        }

        // ---- omega of this state; a9: qdot = -sum_k h_k omega_k; mode 2, second state: the difference quotients
        double qd = 0.0, cpm = 0.0, hm = 0.0;
        for (int k = 0; k < Ns; ++k) {
            const double2 *h = reinterpret_cast<const double2 *>(sGH + 128 * Ns) + 8 * k;
            const double2 *hs = h + (Tu <= h[3].y ? 0 : 4);
            const double2 c01 = hs[0], c23 = hs[1], c45 = hs[2];
            double hk = fma(Tu, c45.x, c23.y);
            hk = fma(Tu, hk, c23.x);
            hk = fma(Tu, hk, c01.y);
            hk = fma(Tu, hk, c01.x);
            hk = fma(c45.y, c.rT[0], hk);
            crf::TmRow<1> r;
            crf::tm_ld<1>(tom + 2u * k, r);
            crf::tm_wait1<1>(r);
            const double w = crf::tm_one(r);
            qd = fma(-hk, w, qd);
            if (i < n) {
                const int64_t o = (int64_t)k * n + i;
                // (mode 2: omega of the base state waits in global memory, in `omega` if the caller wants it, else in the
                // quotient's own row, and is read back by the same thread when the second state is done)
                double *base = MODE == 2 && !io.omega ? io.omega2 : io.omega;
                if (MODE == 4)
                    io.omega2[o] = __dmul_rn(__dsub_rn(w, io.omega[o]), io.inv_sigma);
                else if (st == 0)
                    base[o] = w;
                else if (MODE == 1)
                    io.omega2[o] = w;
                else
                    io.omega2[o] = __dmul_rn(__dsub_rn(w, base[o]), io.inv_sigma);
            }
            if (MODE == 3 && (io.cp || io.h || io.cpk)) {
                // c_pk/R from the h/(RT) set (a_i = (i + 1) c_i); the mixture sums take Z_k = C_k / rho from the Y row again
                double v = fma(Tu, 5.0 * c45.x, 4.0 * c23.y);
                v = fma(Tu, v, 3.0 * c23.x);
                v = fma(Tu, v, 2.0 * c01.y);
                v = fma(Tu, v, c01.x);
                const double zk = io.Y[(int64_t)k * n + ic] * h[7].y;
                cpm = fma(zk, v, cpm);
                hm = fma(zk, hk, hm);
                if (io.cpk && i < n) io.cpk[(int64_t)k * n + i] = v * CRF_R_GAS;
            }
        }
        if (i < n) {
            const double q = qd * (CRF_R_GAS * Tu);
            double *base = MODE == 2 && !io.qdot ? io.qdot2 : io.qdot;
            if (MODE == 4) {
                io.qdot2[i] = __dmul_rn(__dsub_rn(q, io.qdot[i]), io.inv_sigma);
            } else if (st == 0) {
                base[i] = q;
                if (MODE == 3 && io.cp) io.cp[i] = cpm * CRF_R_GAS;
                if (MODE == 3 && io.h) io.h[i] = hm * (CRF_R_GAS * Tu);
            } else if (MODE == 1) {
                io.qdot2[i] = q;
            } else {
                io.qdot2[i] = __dmul_rn(__dsub_rn(q, base[i]), io.inv_sigma);
            }
        }
    }
    __syncthreads();
    if (warp == 0) crf::tm_dealloc(sTmBase, tm_cols);
}

// columns: the (C, d) pairs 4 (Ns + 1), omega 2 (Ns + 1)
cudaError_t launch_thread_tm(const DevTables &m, const RatesIO &io, int64_t n, cudaStream_t st)
{
    unsigned cols = 32;
    while ((int)cols < 6 * (m.Ns + 1)) cols *= 2;
    if (cols > 512) return cudaErrorInvalidValue;
    // tables in shared memory, padded so that no more blocks are resident on an SM than the 512 columns hold
    const size_t tables = (size_t)m.rs.stage_bytes + 256 * (size_t)m.Ns;
    const size_t smem = std::max(tables, (size_t)(227 * 1024) / (512 / cols) - 2048);
    const bool emit = io.cp || io.h || io.cpk || io.rho || io.Wbar;
    void (*kernel)(DevTables, RatesIO, int64_t, unsigned) = rates_thread_tm_kernel<0>;
    if (io.mode == 0 && emit) kernel = rates_thread_tm_kernel<3>;
    if (io.mode == 1) kernel = rates_thread_tm_kernel<1>;
    if (io.mode == 2) kernel = rates_thread_tm_kernel<2>;
    if (io.mode == 4) kernel = rates_thread_tm_kernel<4>;
    cudaError_t e = cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
    kernel<<<(unsigned)((n + RT_B - 1) / RT_B), RT_B, smem, st>>>(m, io, n, cols);
    crf_count_launch();
    return cudaGetLastError();
}

cudaError_t launch_thread(const DevTables &m, const double *T, const double *p, const double *Y, int64_t n, double *omega,
                          double *qdot, cudaStream_t st)
{
    const size_t smem = rates_smem_dynamic_smem(m);
    cudaError_t e = cudaFuncSetAttribute(rates_thread_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
    rates_thread_kernel<<<(unsigned)((n + RT_B - 1) / RT_B), RT_B, smem, st>>>(m, T, p, Y, n, omega, qdot);
    crf_count_launch();
    return cudaGetLastError();
}

}  // namespace

size_t rates_smem_dynamic_smem(const DevTables &m)
{
    // state + omega columns, all chunk blocks, g and h sets
    return (size_t)(m.Ns + 1) * (2048 + 1024) + (size_t)m.rs.stage_bytes + 256 * (size_t)m.Ns;
}

cudaError_t launch_rates_smem(const DevTables &m, const double *T, const double *p, const double *Y, int64_t n,
                              double *omega, double *qdot, cudaStream_t st)
{
    if (m.rs.W != 1 || m.rs.PPL != 4) return cudaErrorInvalidValue;
    if (m.rs.tmem) return launch_thread_tm(m, rates_io(T, p, Y, omega, qdot), n, st);
    return launch_thread(m, T, p, Y, n, omega, qdot, st);
}

// the pair / difference-quotient / by-product calls on a small mechanism: the tensor-memory thread kernel, if the plan has it
bool rates_thread_tm_serves(const DevTables &m, const RatesIO &io)
{
    (void)io;
    return m.rs.W == 1 && m.rs.PPL == 4 && m.rs.tmem && 6 * (m.Ns + 1) <= 512;
}
cudaError_t launch_rates_thread_io(const DevTables &m, const RatesIO &io, int64_t n, cudaStream_t st)
{
    return launch_thread_tm(m, io, n, st);
}
