// rates_group.cu -- crf_production_rates, the kernel the library uses whenever the
// mechanism admits its plan (plan_rates_group.cu); rates_staged.cu (log-space K_c) and rates.cu are the fall-backs.
//
// Shape.  W warps share a group of 32 PPL grid points (lane = point, PPL points per lane), so every mechanism
// coefficient is a warp-uniform shared-memory load.  ncu (profiles/r02_rates_c5.md) shows the kernel bound by two
// resources at once, the issue port (FP64 instructions hold it for two cycles) and the shared-memory pipe (one
// 128-byte wavefront per cycle per SM), so the FP64 instructions and the shared-memory bytes per reaction are both kept
// as low as the method allows, and part of the state lives in TENSOR MEMORY, which has its own read path:
//
//   activity form   per point and species the block keeps d_k = (p_ref/RT) exp(-g_k/RT) and u_k = C_k / d_k.
//                   With K_c = prod_products d / prod_reactants d, k_r = k_f / K_c and
//                   C_k = u_k d_k the rate of progress of step 8 becomes
//                       q = k_f prod_reactants d_a (prod_reactants u_a - prod_products u_b) [M]
//                   one exponential (k_f) per reaction, no division, and the product side needs u only.
//                   crf_mech_create admits this form only if every factor stays a normal double for
//                   250 K <= T <= 5000 K (plan_rates_group.cu).
//   U in TMEM       (TM = true, Ns <= 127 at two points per lane) the u rows, four of the six state rows a reaction
//                   reads, live in tensor memory: lane = grid point pair, 2 PPL columns per species, read with
//                   tcgen05.ld.32x32b (a warp reads the lanes of its own quadrant, so the prologue replicates U into the
//                   quadrants of all warps); only the d rows, the q buffer and the chunk tables use shared memory.
//   pair layout     the PPL = 2 points of a lane are adjacent in every row: one 128-bit access serves both.
//   reaction stage  the reactions are cut into a few chunks; a chunk's reactions are dealt to the warps balanced by
//                   cost (a falloff reaction costs six elementary ones), q_r -> q buffer.
//   species stage   every species is owned by one warp (balanced by incidence count); the owner sums q_r over the
//                   chunk's plus list and minus list of the species (4-byte entries = q row offsets, read two at a time,
//                   lists padded to even length with the zero row) into register accumulators that live for the whole
//                   kernel: omega never touches shared memory.
//   staging         a chunk's tables (records, Troe sets, third-body lists, incidence lists) are one contiguous block,
//                   copied global -> shared by ONE bulk copy (cp.async.bulk, completion on an mbarrier) issued by one
//                   thread while the previous chunk is evaluated.
// Troe falloff is evaluated in base 2 (log2 F = log2 F_cent / (1 + f1^2)) with a branch-free logarithm.
// Accuracy: 2^y by a degree-8 polynomial (relative error 1.1e-12), sized to the tolerance of omega and qdot
// (1e-10 of the gross rate, BASELINE.json north_star), not to 1 ulp.
#include "crf_internal.h"
#include "fastmath.cuh"
#include "launch.h"
#include "row_io.cuh"
#include "tmem.cuh"

namespace {

// the transcendentals (fastmath.cuh): 2^y by the degree-8 polynomial (1.1e-12), Newton reciprocal, atanh-series log2
__device__ __forceinline__ double exp2r(double y) { return crf::exp2_clamped<8>(y); }
__device__ __forceinline__ double rcp_fast(double x) { return crf::rcp_newton(x); }
__device__ __forceinline__ double log2_fast(double x) { return crf::log2_atanh<7>(x); }

// ---- rows: [lane][PPL] doubles; a lane's PPL points are adjacent -------------------------------------------------
template <int PPL>
__device__ __forceinline__ void ld_row(const char *p, double (&v)[PPL])
{
    if (PPL == 2) {
        const double2 t = *reinterpret_cast<const double2 *>(p);
        v[0] = t.x, v[PPL - 1] = t.y;
    } else {
        v[0] = *reinterpret_cast<const double *>(p);
    }
}
template <int PPL>
__device__ __forceinline__ void st_row(char *p, const double (&v)[PPL])
{
    if (PPL == 2)
        *reinterpret_cast<double2 *>(p) = make_double2(v[0], v[PPL - 1]);
    else
        *reinterpret_cast<double *>(p) = v[0];
}
__device__ __forceinline__ uint4 ldsu4(const char *p) { return *reinterpret_cast<const uint4 *>(p); }
__device__ __forceinline__ uint2 ldsu2(const char *p) { return *reinterpret_cast<const uint2 *>(p); }
__device__ __forceinline__ double2 lds2(const char *p) { return *reinterpret_cast<const double2 *>(p); }

using crf::load_row;
using crf::store_row;

// input row of the lane: MODE 0 the PPL adjacent points of `a`; MODE 1 (a[i], b[i]); MODE 2 (a[i], a[i] + sigma b[i]),
// one rounding per operation so that the perturbed state is the one a host forms; MODE 4: the PPL adjacent points of
// a + sigma b (the perturbed state only: the base values of the quotient are given)
template <int PPL, int MODE>
__device__ __forceinline__ void in_row(const RatesIO &io, const double *__restrict__ a, const double *__restrict__ b,
                                       double sigma, int64_t i0, int64_t n, bool vec, double (&v)[PPL])
{
    if (MODE == 0) {
        load_row<PPL>(a, i0, n, vec, v);
        return;
    }
    if (MODE == 4) {
        double vb[PPL];
        load_row<PPL>(a, i0, n, vec, v);
        load_row<PPL>(b, i0, n, vec, vb);
#pragma unroll
        for (int u = 0; u < PPL; ++u) v[u] = __dadd_rn(v[u], __dmul_rn(sigma, vb[u]));
        return;
    }
    const int64_t i = min(i0, n - 1);
    const double va = a[i], vb = b[i];
    v[0] = va;
    v[PPL - 1] = MODE == 1 ? vb : __dadd_rn(va, __dmul_rn(sigma, vb));
}
// output rows: MODE 0 -> a; MODE 1: v[0] -> a, v[1] -> b; MODE 2: v[0] -> a (if given), (v[1] - v[0]) (1/sigma) -> b;
// MODE 4: (v - a) (1/sigma) -> b, a holding the base values (read only)
template <int PPL, int MODE>
__device__ __forceinline__ void out_rows(const RatesIO &io, double *__restrict__ a, double *__restrict__ b, int64_t off,
                                         int64_t i0, int64_t n, bool vec, const double (&v)[PPL])
{
    if (MODE == 0) {
        store_row<PPL>(a + off, i0, n, vec, v);
        return;
    }
    if (MODE == 4) {
        double base[PPL], o[PPL];
        load_row<PPL>(a + off, i0, n, vec, base);
#pragma unroll
        for (int u = 0; u < PPL; ++u) o[u] = __dmul_rn(__dsub_rn(v[u], base[u]), io.inv_sigma);
        store_row<PPL>(b + off, i0, n, vec, o);
        return;
    }
    if (i0 >= n) return;
    if (a) a[off + i0] = v[0];
    b[off + i0] = MODE == 1 ? v[PPL - 1] : __dmul_rn(__dsub_rn(v[PPL - 1], v[0]), io.inv_sigma);
}

// ---- bulk copy global -> shared with mbarrier completion (TMA, non-tensor form) ------------------------------------
__device__ __forceinline__ unsigned smem_u32(const void *p) { return (unsigned)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(uint64_t *bar, unsigned count)
{
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count) : "memory");
}
__device__ __forceinline__ void bulk_load(void *dst, const void *src, unsigned bytes, uint64_t *bar)
{
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(smem_u32(dst)),
                 "l"(src), "r"(bytes), "r"(smem_u32(bar))
                 : "memory");
}
__device__ __forceinline__ void mbar_wait(uint64_t *bar, unsigned parity)
{
    asm volatile(
        "{\n"
        ".reg .pred P1;\n"
        "WAIT_%=:\n"
        "mbarrier.try_wait.parity.shared::cta.b64 P1, [%0], %1;\n"
        "@P1 bra DONE_%=;\n"
        "bra WAIT_%=;\n"
        "DONE_%=:\n"
        "}\n" ::"r"(smem_u32(bar)),
        "r"(parity)
        : "memory");
}

using crf::TmRow;
using crf::tm_get;
using crf::tm_ld;
using crf::tm_st;
using crf::tm_wait1;

// the u row of one species: from tensor memory (h = column) or from shared memory (h = byte offset in the state)
template <bool TM, int PPL>
struct URow {
    TmRow<PPL> t;
    double v[PPL];
    __device__ __forceinline__ void load(const char *sl, unsigned tmq, unsigned h)
    {
        if (TM)
            tm_ld<PPL>(tmq + h, t);
        else
            ld_row<PPL>(sl + h, v);
    }
    __device__ __forceinline__ void get(double (&o)[PPL])
    {
        if (TM) {
            tm_get<PPL>(t, o);
        } else {
#pragma unroll
            for (int u = 0; u < PPL; ++u) o[u] = v[u];
        }
    }
};
// one wait for up to six rows in flight (a wait covers every earlier load of the thread; the operands order the uses)
template <bool TM, int PPL>
__device__ __forceinline__ void u_wait(URow<TM, PPL> &a, URow<TM, PPL> &b, URow<TM, PPL> &c, URow<TM, PPL> &d)
{
    if (!TM) return;
    if (PPL == 2)
        asm volatile("tcgen05.wait::ld.sync.aligned;"
                     : "+r"(a.t.r[0]), "+r"(a.t.r[1]), "+r"(a.t.r[2 * PPL - 2]), "+r"(a.t.r[2 * PPL - 1]), "+r"(b.t.r[0]),
                       "+r"(b.t.r[1]), "+r"(b.t.r[2 * PPL - 2]), "+r"(b.t.r[2 * PPL - 1]), "+r"(c.t.r[0]), "+r"(c.t.r[1]),
                       "+r"(c.t.r[2 * PPL - 2]), "+r"(c.t.r[2 * PPL - 1]), "+r"(d.t.r[0]), "+r"(d.t.r[1]),
                       "+r"(d.t.r[2 * PPL - 2]), "+r"(d.t.r[2 * PPL - 1]));
    else
        asm volatile("tcgen05.wait::ld.sync.aligned;"
                     : "+r"(a.t.r[0]), "+r"(a.t.r[1]), "+r"(b.t.r[0]), "+r"(b.t.r[1]), "+r"(c.t.r[0]), "+r"(c.t.r[1]),
                       "+r"(d.t.r[0]), "+r"(d.t.r[1]));
}

template <int PPL>
struct Ctx {
    double T[PPL], L[PPL], rT[PPL];  // T, ln T, 1/T
    double Csum[PPL];                // p/(R T)
};

// q of one reaction at the PPL points of this lane.  rec: the 64-byte record; tr: its Troe set (kind 2); blk: the chunk
// block (third-body lists); sl: the shared-memory state at this lane (d rows; the u rows too unless TM); tmq: the
// tensor-memory address of this warp's quadrant.
template <int KIND, bool GENERIC, int PPL, bool TM>
__device__ __forceinline__ void reaction_q(const char *blk, const char *rec, const char *tr, const char *sl, unsigned tmq,
                                           const Ctx<PPL> &c, double (&q)[PPL])
{
    const double2 A = lds2(rec);        // log2e lnA, log2e beta
    const double2 Ex = lds2(rec + 16);  // -log2e Ea/R, (b0u, b1u)
    const uint4 S = ldsu4(rec + 32);    // a0d, a1d, a0u, a1u
    const unsigned b0u = (unsigned)__double2loint(Ex.y), b1u = (unsigned)__double2hiint(Ex.y);
    URow<TM, PPL> Ua0, Ua1, Ub0, Ub1;
    Ua0.load(sl, tmq, S.z), Ua1.load(sl, tmq, S.w), Ub0.load(sl, tmq, b0u), Ub1.load(sl, tmq, b1u);
    double da0[PPL], da1[PPL];
    ld_row<PPL>(sl + S.x, da0), ld_row<PPL>(sl + S.y, da1);
    uint4 X = make_uint4(0, 0, 0, 0);  // x0, x1, x0u, x1u
    if (KIND != 0 || GENERIC) X = ldsu4(rec + 48);
    u_wait<TM, PPL>(Ua0, Ua1, Ub0, Ub1);
    double ua0[PPL], ua1[PPL], ub0[PPL], ub1[PPL];
    Ua0.get(ua0), Ua1.get(ua1), Ub0.get(ub0), Ub1.get(ub1);
    double M[PPL];
    if (KIND != 0) {
#pragma unroll
        for (int u = 0; u < PPL; ++u) M[u] = c.Csum[u];
        const char *e = blk + X.x, *e1 = e + 16 * X.y;
        for (; e < e1; e += 16) {
            const uint4 en = ldsu4(e);  // f64 efficiency - 1, u32 d row, u32 u handle
            const double coef = __hiloint2double((int)en.y, (int)en.x);
            URow<TM, PPL> Uk;
            Uk.load(sl, tmq, en.w);
            double uu[PPL], dd[PPL];
            ld_row<PPL>(sl + en.z, dd);
            if (TM) tm_wait1<PPL>(Uk.t);
            Uk.get(uu);
#pragma unroll
            for (int u = 0; u < PPL; ++u) M[u] = fma(coef, uu[u] * dd[u], M[u]);  // C_k = u_k d_k
        }
    }
    double ua2[PPL], da2[PPL], ub2[PPL];
    if (GENERIC) {
        URow<TM, PPL> Ua2, Ub2;
        Ua2.load(sl, tmq, X.z), Ub2.load(sl, tmq, X.w);
        ld_row<PPL>(sl + X.x, da2);
        if (TM) tm_wait1<PPL>(Ua2.t), tm_wait1<PPL>(Ub2.t);
        Ua2.get(ua2), Ub2.get(ub2);
    }
#pragma unroll
    for (int u = 0; u < PPL; ++u) {
        const double yinf = fma(A.y, c.L[u], fma(Ex.x, c.rT[u], A.x));  // log2 k_f (high-pressure limit)
        double dd = da0[u] * da1[u], pb = ub0[u] * ub1[u], net;
        if (GENERIC) {
            dd *= da2[u], pb *= ub2[u];
            net = fma(ua0[u] * ua1[u], ua2[u], -pb);
        } else {
            net = fma(ua0[u], ua1[u], -pb);
        }
        if (KIND == 0) q[u] = (exp2r(yinf) * dd) * net;
        if (KIND == 1) q[u] = (exp2r(yinf) * dd) * (M[u] * net);
        if (KIND == 2) {
            // Troe falloff in base 2
            const double2 t01 = lds2(tr), t23 = lds2(tr + 16), t45 = lds2(tr + 32), t67 = lds2(tr + 48);
            const double y0 = fma(t01.y, c.L[u], fma(t23.x, c.rT[u], t01.x));
            const double l2Pr = (y0 - yinf) + log2_fast(fmax(M[u], 1.0e-300));  // log2(k_0 [M] / k_inf)
            const double al = t23.y;
            // (the arguments are clamped BEFORE the range reduction: Chemkin-style switched-off terms, T3 = 1e-30 or
            // T2 = 1e30 / inf, give arguments of -1e33 or -inf, whose integer part has no meaning as an exponent)
            const double Fc = fma(1.0 - al, exp2r(fmax(c.T[u] * t45.x, -1022.0)),
                                  fma(al, exp2r(fmax(c.T[u] * t45.y, -1022.0)), exp2r(fmax(t67.x * c.rT[u], -1022.0))));
            const double l2Fc = log2_fast(fmax(Fc, 1.0e-300));
            const double l10_2 = 0.30102999566398119521;
            const double lFc = l10_2 * l2Fc;
            const double x = fma(l10_2, l2Pr, fma(-0.67, lFc, -0.4));  // log10 P_r + c
            const double f1 = x * rcp_fast(fma(-0.14, x, fma(-1.27, lFc, 0.75)));
            const double l2F = l2Fc * rcp_fast(fma(f1, f1, 1.0));
            const double Pred = exp2r(l2Pr);
            q[u] = (exp2r(yinf + l2F) * dd) * ((Pred * rcp_fast(1.0 + Pred)) * net);
        }
    }
}

template <int KIND, bool GENERIC, int PPL, bool TM>
__device__ __forceinline__ void reaction_loop(const char *blk, const char *&rec, const char *&tr, char *&qp, int count,
                                              const char *sl, unsigned tmq, const Ctx<PPL> &c)
{
    constexpr int RB = 256 * PPL;
#pragma unroll 1
    for (int i = 0; i < count; ++i) {
        double q[PPL];
        reaction_q<KIND, GENERIC, PPL, TM>(blk, rec, tr, sl, tmq, c, q);
        st_row<PPL>(qp, q);
        rec += 64, qp += RB;
        if (KIND == 2) tr += 64;
    }
}

// om (+/-)= q[row a] + q[row b]
template <int PPL, bool PLUS>
__device__ __forceinline__ void gather2(uint2 en, const char *sQl, double (&om)[PPL])
{
    double qa[PPL], qb[PPL];
    ld_row<PPL>(sQl + en.x, qa), ld_row<PPL>(sQl + en.y, qb);
#pragma unroll
    for (int u = 0; u < PPL; ++u) om[u] = PLUS ? (om[u] + qa[u]) + qb[u] : (om[u] - qa[u]) - qb[u];
}
// one list [e, end): 8-byte aligned, even length
template <int PPL, bool PLUS>
__device__ __forceinline__ void gather_list(const char *blk, unsigned &e, unsigned end, const char *sQl, double (&om)[PPL])
{
#pragma unroll 1
    for (; e < end; e += 8) gather2<PPL, PLUS>(ldsu2(blk + e), sQl, om);
}

// g/(RT) set (log2 e folded in) or h/(RT) set of one species at one point: 7 (6) Horner coefficients of the range T is in,
// read with a per-lane address (the two ranges are 64 bytes apart: lanes in different ranges hit different banks)
template <bool GIBBS>
__device__ __forceinline__ double nasa_eval(const double2 *set, double Tu, double rTu, double omL, double Tmid)
{
    const double2 *g = set + (Tu <= Tmid ? 0 : 4);
    const double2 c01 = g[0], c23 = g[1], c45 = g[2];
    double v = fma(Tu, c45.x, c23.y);
    v = fma(Tu, v, c23.x);
    v = fma(Tu, v, c01.y);
    if (GIBBS) {
        v = fma(Tu, v, g[3].x);
        v = fma(c45.y, rTu, v);
        return fma(c01.x, omL, v);  // c0 (1 - ln T)
    }
    v = fma(Tu, v, c01.x);
    return fma(c45.y, rTu, v);
}

// MODE 0: crf_production_rates; 1, 2: the pair / difference-quotient calls (RatesIO.mode); 3: mode 0 with the by-products
// of crf_rhs_pointwise.  Separate instances: the code of one call does not cost another a register or a branch.
template <int W, int PPL, int MAXOWN, bool TM, int MODE>
__global__ void __launch_bounds__(32 * W, 16 / W)
    rates_group_kernel(DevTables m, RatesIO io, int64_t n)
{
    extern __shared__ double2 sm2[];
    __shared__ uint64_t mbar[2];
    __shared__ int4 sChunk[64];
    __shared__ unsigned sTmBase;
    const RatesGroupPlan &rg = m.rg;
    constexpr int RB = 256 * PPL, LB = 8 * PPL;
    const int Ns = m.Ns;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    // state rows: TM: [Ns + 1] d rows; otherwise [Ns + 1] d rows then [Ns + 1] u rows; row Ns = 1 (the dummy species)
    char *sS = reinterpret_cast<char *>(sm2);
    char *sQ = sS + (size_t)(Ns + 1) * (TM ? 1 : 2) * RB;  // [q_rows][RB] q_r (row Rc = 0); prologue scratch
    char *sStage = sQ + (size_t)rg.q_rows * RB;            // [2][stage_bytes]
    char *sl = sS + lane * LB;
    char *sQl = sQ + lane * LB;
    const int sb = rg.stage_bytes, nch = rg.n_chunks;

    if (threadIdx.x == 0) {
        mbar_init(&mbar[0], 1);
        mbar_init(&mbar[1], 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    if (TM && warp == 0) {
        asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(smem_u32(&sTmBase)),
                     "r"((unsigned)rg.tm_cols)
                     : "memory");
        asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
    }
    for (int ci = threadIdx.x; ci < nch && ci < 64; ci += 32 * W) sChunk[ci] = __ldg(rg.chunk + ci);
    if (TM) asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
    __syncthreads();
    if (TM) asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
    if (threadIdx.x == 0) {
        // chunk 0 -> buffer 0; buffer 1 is free until chunk 1 is prefetched: it carries the g/(RT) sets for the prologue
        bulk_load(sStage, rg.stage + sChunk[0].x, (unsigned)sChunk[0].y, &mbar[0]);
        bulk_load(sStage + sb, rg.gco, 128u * Ns, &mbar[1]);
    }
    const unsigned tmq = TM ? sTmBase + (((unsigned)(warp & 3) * 32u) << 16) : 0u;

    // mode 0: the lane's PPL points are adjacent grid points; modes 1, 2 (PPL = 2): the lane's two "points" are the two
    // states of ONE grid point, so tables, records and lists are read once for both evaluations
    constexpr int mode = MODE == 3 ? 0 : MODE;
    constexpr bool EXT = MODE == 3;
    const int64_t i0 = ((int64_t)blockIdx.x * 32 + lane) * (mode == 0 || mode == 4 ? PPL : 1);
    const bool vec = (n & 1) == 0;
    Ctx<PPL> c;
    double pi[PPL];
    in_row<PPL, mode>(io, io.T, io.T2, io.sigma, i0, n, vec, c.T);
    in_row<PPL, mode>(io, io.p, io.p2, io.sigma_p, i0, n, vec, pi);
    // ---- a1: Z_k = Y_k / W_k; warp w takes species w, w + W, ...: all row loads of the warp are in flight together
    double z[MAXOWN][PPL];
#pragma unroll
    for (int s = 0; s < MAXOWN; ++s) {
        const int k = warp + W * s;
        if (k < Ns) in_row<PPL, mode>(io, io.Y + (int64_t)k * n, io.Y2 + (int64_t)k * n, io.sigma, i0, n, vec, z[s]);
    }
    double lc02[PPL], omL[PPL];
#pragma unroll
    for (int u = 0; u < PPL; ++u) {
        c.L[u] = log(c.T[u]);
        c.rT[u] = 1.0 / c.T[u];
        lc02[u] = fma(-crf::kLog2e, c.L[u], rg.log2_c0);  // log2(p_ref/(R T))
        omL[u] = 1.0 - c.L[u];
        c.Csum[u] = pi[u] * c.rT[u] * (1.0 / CRF_R_GAS);
    }
    mbar_wait(&mbar[1], 0);
    const double2 *sG = reinterpret_cast<const double2 *>(sStage + sb);
    double invW[PPL];
#pragma unroll
    for (int u = 0; u < PPL; ++u) invW[u] = 0.0;
#pragma unroll
    for (int s = 0; s < MAXOWN; ++s) {
        const int k = warp + W * s;
        if (k < Ns) {
            const double rW = sG[8 * k + 7].y;
#pragma unroll
            for (int u = 0; u < PPL; ++u) {
                z[s][u] *= rW;
                invW[u] += z[s][u];
            }
        }
    }
    double *sred = reinterpret_cast<double *>(sQ);  // rows [0, W): [W][PPL][32] reduction scratch, outside the chunk loop
    char *sUtmp = sQ + (size_t)W * RB;               // TM: rows [W, W + Ns + 1): the u rows on their way to tensor memory
#pragma unroll
    for (int u = 0; u < PPL; ++u) sred[(warp * PPL + u) * 32 + lane] = invW[u];
    __syncthreads();
    double rho[PPL];
#pragma unroll
    for (int u = 0; u < PPL; ++u) {
        double s = 0.0;
#pragma unroll
        for (int w = 0; w < W; ++w) s += sred[(w * PPL + u) * 32 + lane];
        rho[u] = pi[u] / (CRF_R_GAS * c.T[u] * s);
        invW[u] = s;
    }
    if (EXT && warp == 0 && mode == 0 && (io.rho || io.Wbar)) {  // by-products of crf_rhs_pointwise (Eq. 1d)
        double wb[PPL];
#pragma unroll
        for (int u = 0; u < PPL; ++u) wb[u] = 1.0 / invW[u];
        if (io.rho) store_row<PPL>(io.rho, i0, n, vec, rho);
        if (io.Wbar) store_row<PPL>(io.Wbar, i0, n, vec, wb);
    }
    // ---- a2: d_k = 2^(log2(p_ref/RT) - log2e g_k/RT), u_k = rho Z_k / d_k
    char *uDst = (TM ? sUtmp : sS + (size_t)(Ns + 1) * RB) + lane * LB;
#pragma unroll
    for (int s = 0; s < MAXOWN; ++s) {
        const int k = warp + W * s;
        if (k >= Ns) continue;
        const double2 *g = sG + 8 * k;
        const double Tmid = g[3].y;
        double uu[PPL], dd[PPL];
#pragma unroll
        for (int u = 0; u < PPL; ++u) {
            const double g2 = nasa_eval<true>(g, c.T[u], c.rT[u], omL[u], Tmid);
            dd[u] = exp2r(lc02[u] - g2);
            uu[u] = (rho[u] * z[s][u]) * rcp_fast(dd[u]);
        }
        st_row<PPL>(uDst + (size_t)k * RB, uu);
        st_row<PPL>(sl + (size_t)k * RB, dd);
    }
    if (warp == 0) {
        double one[PPL];
#pragma unroll
        for (int u = 0; u < PPL; ++u) one[u] = 1.0;
        st_row<PPL>(uDst + (size_t)Ns * RB, one);
        st_row<PPL>(sl + (size_t)Ns * RB, one);
    }
    __syncthreads();  // the state is complete; everyone is done with the g sets and the reduction scratch
    if (TM) {
        // every quadrant gets the whole of U: the W/4 warps of a quadrant split the rows
        for (int k = warp >> 2; k <= Ns; k += W / 4) {
            double uu[PPL];
            ld_row<PPL>(sUtmp + (size_t)k * RB + lane * LB, uu);
            tm_st<PPL>(tmq + (unsigned)(2 * PPL * k), uu);
        }
        asm volatile("tcgen05.wait::st.sync.aligned;" ::: "memory");
        asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
        __syncthreads();
        asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
    }
    if (warp == W - 1) {  // the zero row the padded incidence lists point at
        double zero[PPL];
#pragma unroll
        for (int u = 0; u < PPL; ++u) zero[u] = 0.0;
        st_row<PPL>(sQl + (size_t)rg.Rc * RB, zero);
    }

    double om[MAXOWN][PPL];
#pragma unroll
    for (int s = 0; s < MAXOWN; ++s)
#pragma unroll
        for (int u = 0; u < PPL; ++u) om[s][u] = 0.0;

    for (int ci = 0; ci < nch; ++ci) {
        const char *blk = sStage + (size_t)(ci & 1) * sb;
        if (threadIdx.x == 0) {
            char *dst = sStage + (size_t)((ci + 1) & 1) * sb;
            if (ci + 1 < nch)
                bulk_load(dst, rg.stage + sChunk[ci + 1].x, (unsigned)sChunk[ci + 1].y, &mbar[(ci + 1) & 1]);
            else  // behind the last chunk: the h/(RT) sets for the epilogue
                bulk_load(dst, rg.hco, 128u * Ns, &mbar[(ci + 1) & 1]);
        }
        mbar_wait(&mbar[ci & 1], (unsigned)((ci >> 1) + (ci & 1)) & 1u);
        {
            const uint4 hw = ldsu4(blk + 32 * warp);  // records, first q row, slot table, Troe sets
            const uint2 cn = ldsu2(blk + 32 * warp + 16);
            const char *rec = blk + hw.x, *tr = blk + hw.w;
            char *qp = sQl + hw.y;
            reaction_loop<0, false, PPL, TM>(blk, rec, tr, qp, (int)(cn.x & 0xffffu), sl, tmq, c);
            if (cn.x >> 16) reaction_loop<0, true, PPL, TM>(blk, rec, tr, qp, (int)(cn.x >> 16), sl, tmq, c);
            if (cn.y & 0xffffu) reaction_loop<1, false, PPL, TM>(blk, rec, tr, qp, (int)(cn.y & 0xffffu), sl, tmq, c);
            if (cn.y >> 16) reaction_loop<2, false, PPL, TM>(blk, rec, tr, qp, (int)(cn.y >> 16), sl, tmq, c);
            __syncthreads();
            // ---- species stage: the warp's lists are contiguous: plus list of slot 0, minus list of slot 0, plus list of
            // slot 1, ...; each 8-byte aligned and of even length; the table holds where each ends
            const char *tab = blk + hw.z;
            unsigned e = *reinterpret_cast<const unsigned *>(tab + 8 * MAXOWN);
#pragma unroll
            for (int s2 = 0; s2 < MAXOWN; s2 += 2) {
                const uint4 ends = ldsu4(tab + 8 * s2);  // endP[s2], endM[s2], endP[s2 + 1], endM[s2 + 1]
                gather_list<PPL, true>(blk, e, ends.x, sQl, om[s2]);
                gather_list<PPL, false>(blk, e, ends.y, sQl, om[s2]);
                gather_list<PPL, true>(blk, e, ends.z, sQl, om[s2 + 1]);
                gather_list<PPL, false>(blk, e, ends.w, sQl, om[s2 + 1]);
            }
        }
        __syncthreads();
    }

    // ---- store omega; a9: qdot = -sum_k h_k omega_k
    mbar_wait(&mbar[nch & 1], (unsigned)((nch >> 1) + (nch & 1)) & 1u);
    const double2 *sH = reinterpret_cast<const double2 *>(sStage + (size_t)(nch & 1) * sb);
    const bool emit = EXT && mode == 0 && (io.cp || io.h || io.cpk);
    double qd[PPL], cpm[PPL], hm[PPL];
#pragma unroll
    for (int u = 0; u < PPL; ++u) qd[u] = cpm[u] = hm[u] = 0.0;
    if (mode == 4) {  // the quotient against given base values: their rows are read in one batch, then om -> (om - base) / sigma
        double base[MAXOWN][PPL];
#pragma unroll
        for (int s = 0; s < MAXOWN; ++s) {
            const int k = __ldg(rg.own + warp * MAXOWN + s);
            load_row<PPL>(io.omega + (int64_t)max(k, 0) * n, i0, n, vec, base[s]);
        }
#pragma unroll
        for (int s = 0; s < MAXOWN; ++s)
#pragma unroll
            for (int u = 0; u < PPL; ++u) base[s][u] = __dmul_rn(__dsub_rn(om[s][u], base[s][u]), io.inv_sigma);
#pragma unroll
        for (int s = 0; s < MAXOWN; ++s) {
            const int k = __ldg(rg.own + warp * MAXOWN + s);
            if (k >= 0) store_row<PPL>(io.omega2 + (int64_t)k * n, i0, n, vec, base[s]);
        }
    }
#pragma unroll
    for (int s = 0; s < MAXOWN; ++s) {
        const int k = __ldg(rg.own + warp * MAXOWN + s);
        if (k >= 0) {
            const double2 *h = sH + 8 * k;
            const double Tmid = h[3].y;
            double hk[PPL];
#pragma unroll
            for (int u = 0; u < PPL; ++u) {
                hk[u] = nasa_eval<false>(h, c.T[u], c.rT[u], 0.0, Tmid);
                qd[u] = fma(-hk[u], om[s][u], qd[u]);
            }
            if (mode != 4) out_rows<PPL, mode>(io, io.omega, io.omega2, (int64_t)k * n, i0, n, vec, om[s]);
            if (emit) {
                // crf_rhs_pointwise: c_pk/R from the h/(RT) set (a_i = (i + 1) c_i), mixture c_p and h; the Y row is
                // read again (it was consumed by the species this warp handled in the prologue, not the ones it owns)
                double y[PPL], cpk[PPL];
                load_row<PPL>(io.Y + (int64_t)k * n, i0, n, vec, y);
                const double rW = h[7].y;
#pragma unroll
                for (int u = 0; u < PPL; ++u) {
                    const double2 *g = h + (c.T[u] <= Tmid ? 0 : 4);
                    const double2 c01 = g[0], c23 = g[1], c45 = g[2];
                    double v = fma(c.T[u], 5.0 * c45.x, 4.0 * c23.y);
                    v = fma(c.T[u], v, 3.0 * c23.x);
                    v = fma(c.T[u], v, 2.0 * c01.y);
                    v = fma(c.T[u], v, c01.x);
                    const double zk = y[u] * rW;
                    cpm[u] = fma(zk, v, cpm[u]);
                    hm[u] = fma(zk, hk[u], hm[u]);
                    cpk[u] = v * CRF_R_GAS;
                }
                if (io.cpk) store_row<PPL>(io.cpk + (int64_t)k * n, i0, n, vec, cpk);
            }
        }
    }
    // block-wide sums of qdot (and c_p, h): [3][W][PPL][32] in the q buffer
#pragma unroll
    for (int u = 0; u < PPL; ++u) {
        sred[(warp * PPL + u) * 32 + lane] = qd[u];
        if (emit) {
            sred[((W + warp) * PPL + u) * 32 + lane] = cpm[u];
            sred[((2 * W + warp) * PPL + u) * 32 + lane] = hm[u];
        }
    }
    __syncthreads();
    if (warp == 0) {
        double out[PPL];
#pragma unroll
        for (int u = 0; u < PPL; ++u) {
            double s = 0.0;
#pragma unroll
            for (int w = 0; w < W; ++w) s += sred[(w * PPL + u) * 32 + lane];
            out[u] = s * (CRF_R_GAS * c.T[u]);
        }
        out_rows<PPL, mode>(io, io.qdot, io.qdot2, 0, i0, n, vec, out);
        if (TM)
            asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(sTmBase), "r"((unsigned)rg.tm_cols)
                         : "memory");
    }
    if (warp == 1 && emit) {
        double oc[PPL], oh[PPL];
#pragma unroll
        for (int u = 0; u < PPL; ++u) {
            double sc = 0.0, sh = 0.0;
#pragma unroll
            for (int w = 0; w < W; ++w) {
                sc += sred[((W + w) * PPL + u) * 32 + lane];
                sh += sred[((2 * W + w) * PPL + u) * 32 + lane];
            }
            oc[u] = sc * CRF_R_GAS;
            oh[u] = sh * (CRF_R_GAS * c.T[u]);
        }
        if (io.cp) store_row<PPL>(io.cp, i0, n, vec, oc);
        if (io.h) store_row<PPL>(io.h, i0, n, vec, oh);
    }
}

template <int W, int PPL, int MAXOWN, bool TM>
cudaError_t launch_k(const DevTables &m, const RatesIO &io, int64_t n, cudaStream_t st)
{
    const size_t smem = rates_group_dynamic_smem(m);
    const bool emit = io.cp || io.h || io.cpk || io.rho || io.Wbar;
    void (*kernel)(DevTables, RatesIO, int64_t) = rates_group_kernel<W, PPL, MAXOWN, TM, 0>;
    if (io.mode == 0 && emit) kernel = rates_group_kernel<W, PPL, MAXOWN, TM, 3>;
    if (io.mode == 4) kernel = rates_group_kernel<W, PPL, MAXOWN, TM, 4>;
    if (io.mode == 1 || io.mode == 2) {
        if (PPL != 2) return cudaErrorInvalidValue;
        // (instantiated for two points per lane only)
        kernel = io.mode == 1 ? rates_group_kernel<W, 2, MAXOWN, TM, 1> : rates_group_kernel<W, 2, MAXOWN, TM, 2>;
    }
    cudaError_t e = cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
    const int64_t per_block = io.mode == 0 || io.mode == 4 ? 32 * PPL : 32;
    kernel<<<(unsigned)((n + per_block - 1) / per_block), 32 * W, smem, st>>>(m, io, n);
    crf_count_launch();
    return cudaGetLastError();
}

template <int W, int PPL>
cudaError_t launch_wp(const DevTables &m, const RatesIO &io, int64_t n, cudaStream_t st)
{
    switch (m.rg.maxown * 2 + (m.rg.tm_cols > 0)) {
    case 8: return launch_k<W, PPL, 4, false>(m, io, n, st);
    case 9: return launch_k<W, PPL, 4, true>(m, io, n, st);
    case 16: return launch_k<W, PPL, 8, false>(m, io, n, st);
    case 17: return launch_k<W, PPL, 8, true>(m, io, n, st);
    case 32: return launch_k<W, PPL, 16, false>(m, io, n, st);
    case 33: return launch_k<W, PPL, 16, true>(m, io, n, st);
    default: return cudaErrorInvalidValue;
    }
}

}  // namespace

size_t rates_group_dynamic_smem(const DevTables &m)
{
    const RatesGroupPlan &rg = m.rg;
    const size_t rb = 256 * (size_t)rg.PPL;
    return (size_t)(m.Ns + 1) * (rg.tm_cols > 0 ? 1 : 2) * rb + (size_t)rg.q_rows * rb + 2 * (size_t)rg.stage_bytes;
}

// io.mode 1 and 2 need a plan with two points per lane (the two states of a grid point share a lane)
cudaError_t launch_rates_group(const DevTables &m, const RatesIO &io, int64_t n, cudaStream_t st)
{
    if ((io.mode == 1 || io.mode == 2) && m.rg.PPL != 2) return cudaErrorInvalidValue;
    switch (m.rg.W * 10 + m.rg.PPL) {
    case 41: return launch_wp<4, 1>(m, io, n, st);
    case 42: return launch_wp<4, 2>(m, io, n, st);
    case 81: return launch_wp<8, 1>(m, io, n, st);
    case 82: return launch_wp<8, 2>(m, io, n, st);
    case 161: return launch_wp<16, 1>(m, io, n, st);
    case 162: return launch_wp<16, 2>(m, io, n, st);
    default: return cudaErrorInvalidValue;
    }
}
