// transport_tiled.cu -- crf_mix_transport for mechanisms too large for registers (SURVEY 8(a) rows
// a1, a10-a13): W warps share 32 grid points (lane = point).
//
// Why this shape.  The path is FP64-ALU bound: per point Ns(Ns-1)/2 exponentials (1/D_jk) and Ns^2
// Wilke terms against 16(Ns+2) bytes of HBM traffic.  Lanes are points so that every mechanism
// coefficient is a warp-uniform load (one 32-byte record serves 32 points).  The per-point state
// (Z_k = Y_k/W_k and the diffusion sums S_k, 2 Ns doubles) does not fit in registers at Ns = 118, and
// at one thread per point it would leave 3 warps per SM; so the state lives in shared memory as
// [species][lane] columns (conflict-free, 2 wavefronts per access) and W warps work on the SAME 32
// points: the pair triangle is cut into 8x8 species tiles, a tile is evaluated entirely in registers
// (Z_j[8], Z_k[8], S_j[8], S_k[8] -> 64 independent exp chains of ILP), and tiles are dealt to the
// warps in rounds whose tiles touch disjoint species blocks, so the shared S rows are updated without
// atomics; one __syncthreads per round (round-robin tournament over the blocks, plan_transport.cu).  A round's
// coefficients are copied global -> shared with cp.async while the previous round is evaluated, so the pair
// loop reads every coefficient as a warp-uniform shared-memory load.  A lane may carry PPL = 2 adjacent
// points: each coefficient load then serves two points.  Each unordered pair is evaluated once:
// e = 1/D_jk(p_ref) = 2^(cubic(ln T)) with -log2(e) folded into the table, S_j += Z_k e, S_k += Z_j e.
//
// Wilke: Phi_kj = c_kj (1 + a_k/a_j)^2, a_k = sqrt(mu_k) W_k^(-1/4), expanded so that the O(Ns^2) part is
// three FMAs per ordered pair:  sum_j Z_j Phi_kj = A_k + 2 a_k B_k + a_k^2 C_k,
// (A,B,C)_k = sum_j c_kj (Z_j, Z_j/a_j, Z_j/a_j^2)   (all terms positive: no cancellation).
//
// rho D_km needs neither rho nor p nor Wbar: rho D_km = p_ref (1 - Y_k) / (R T sum_{j!=k} Z_j/D_jk(p_ref)).
#include "crf_internal.h"
#include "fastmath.cuh"
#include "launch.h"
#include "row_io.cuh"

namespace {

using crf::exp2_poly9;
using crf::exp2_tab64;

__constant__ double kExp2Tab64[64] = CRF_EXP2_TAB64;

__device__ __forceinline__ double cubic4(const double *__restrict__ c, double x)
{
    const double2 lo = __ldg(reinterpret_cast<const double2 *>(c));
    const double2 hi = __ldg(reinterpret_cast<const double2 *>(c) + 1);
    return fma(x, fma(x, fma(x, hi.y, hi.x), lo.y), lo.x);
}

// state rows: [species][PPL][32] doubles; sZl / sSl point at this lane's column
#define ROW(k, u) (((k) * PPL + (u)) * 32)

// off-diagonal tile: species blocks jb < kb of TS species each, TS^2 pairs; cf: the tile's coefficients in shared memory
template <int PPL, int TS>
__device__ __forceinline__ void tile_offdiag(const double2 *cf, const double (&L)[PPL], const double *sZl, double *sSl,
                                             int jb, int kb, const double *tab)
{
    double zj[PPL][TS], zk[PPL][TS], sj[PPL][TS], sk[PPL][TS];
#pragma unroll
    for (int u = 0; u < PPL; ++u)
#pragma unroll
        for (int a = 0; a < TS; ++a) {
            zj[u][a] = sZl[ROW(TS * jb + a, u)];
            zk[u][a] = sZl[ROW(TS * kb + a, u)];
            sj[u][a] = 0.0;
            sk[u][a] = 0.0;
        }
#pragma unroll
    for (int a = 0; a < TS; ++a) {
#pragma unroll
        for (int b = 0; b < TS; ++b) {
            const double2 lo = cf[2 * (TS * a + b)], hi = cf[2 * (TS * a + b) + 1];
#pragma unroll
            for (int u = 0; u < PPL; ++u) {
                const double e = exp2_tab64(fma(L[u], fma(L[u], fma(L[u], hi.y, hi.x), lo.y), lo.x), tab);
                sj[u][a] = fma(zk[u][b], e, sj[u][a]);
                sk[u][b] = fma(zj[u][a], e, sk[u][b]);
            }
        }
    }
#pragma unroll
    for (int u = 0; u < PPL; ++u)
#pragma unroll
        for (int a = 0; a < TS; ++a) {
            sSl[ROW(TS * jb + a, u)] += sj[u][a];
            sSl[ROW(TS * kb + a, u)] += sk[u][a];
        }
}

// diagonal tile: pairs a < b inside block jb, TS (TS - 1) / 2 pairs
template <int PPL, int TS>
__device__ __forceinline__ void tile_diag(const double2 *cf, const double (&L)[PPL], const double *sZl, double *sSl, int jb,
                                          const double *tab)
{
    double z[PPL][TS], s[PPL][TS];
#pragma unroll
    for (int u = 0; u < PPL; ++u)
#pragma unroll
        for (int a = 0; a < TS; ++a) {
            z[u][a] = sZl[ROW(TS * jb + a, u)];
            s[u][a] = 0.0;
        }
    int q = 0;
#pragma unroll
    for (int a = 0; a < TS; ++a) {
#pragma unroll
        for (int b = a + 1; b < TS; ++b, ++q) {
            const double2 lo = cf[2 * q], hi = cf[2 * q + 1];
#pragma unroll
            for (int u = 0; u < PPL; ++u) {
                const double e = exp2_tab64(fma(L[u], fma(L[u], fma(L[u], hi.y, hi.x), lo.y), lo.x), tab);
                s[u][a] = fma(z[u][b], e, s[u][a]);
                s[u][b] = fma(z[u][a], e, s[u][b]);
            }
        }
    }
#pragma unroll
    for (int u = 0; u < PPL; ++u)
#pragma unroll
        for (int a = 0; a < TS; ++a) sSl[ROW(TS * jb + a, u)] += s[u][a];
}

__device__ __forceinline__ void stage_async(unsigned char *dst, const unsigned char *src, int bytes, int tid, int nthreads)
{
    for (int o = tid * 16; o < bytes; o += nthreads * 16) {
        const unsigned d = (unsigned)__cvta_generic_to_shared(dst + o);
        asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(d), "l"(src + o) : "memory");
    }
    asm volatile("cp.async.commit_group;" ::: "memory");
}
__device__ __forceinline__ void stage_wait() { asm volatile("cp.async.wait_all;" ::: "memory"); }

using crf::load_row;
using crf::store_row;

template <int W, int PPL, int TS>
__global__ void __launch_bounds__(32 * W, 16 / (W * PPL))
    transport_tiled_kernel(DevTables m, const double *__restrict__ T, const double *__restrict__ Y, int64_t n,
                           double *__restrict__ mu, double *__restrict__ lambda, double *__restrict__ rhoD)
{
    extern __shared__ double2 sm2[];
    __shared__ double sTab[64];
    for (int i = threadIdx.x; i < 64; i += 32 * W) sTab[i] = kExp2Tab64[i];
    double *sm = reinterpret_cast<double *>(sm2);
    const TransportPlan &tp = m.tp;
    const int Ns = m.Ns, NsP = tp.NsP, nb = tp.nb;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    double *sZ = sm;                             // [NsP][PPL][32]  Z_k = Y_k / W_k
    double *sS = sZ + (size_t)NsP * PPL * 32;    // [NsP][PPL][32]  1/a_k during the Wilke phase, then the diffusion sums
    double *sred = sS + (size_t)NsP * PPL * 32;  // [4][W][PPL][32] partial sums of the warps
    unsigned char *sStage = reinterpret_cast<unsigned char *>(sred + 4 * W * PPL * 32);  // [2][stage_bytes]
    const double *sZl = sZ + lane;
    double *sSl = sS + lane;

    int4 cur = __ldg(tp.rounds);  // descriptor of the block being staged / used; later ones come with the blocks
    stage_async(sStage, tp.pair_coef + cur.x, cur.y, threadIdx.x, 32 * W);
    constexpr int HDR = (16 + 8 * W + 15) / 16 * 16;

    const int64_t i0 = ((int64_t)blockIdx.x * 32 + lane) * PPL;
    const bool vec = (n & 1) == 0;
    double Ti[PPL], L[PPL];
    load_row<PPL>(T, i0, n, vec, Ti);
#pragma unroll
    for (int u = 0; u < PPL; ++u) L[u] = log(Ti[u]);

    // ---- a1, a10, a12: Z_k, species fits, conductivity sums; warp w takes species w, w+W, ...
    double invW[PPL], sum_a[PPL], sum_h[PPL];
#pragma unroll
    for (int u = 0; u < PPL; ++u) invW[u] = sum_a[u] = sum_h[u] = 0.0;
    // (groups of G species: the G row loads are in flight together)
    constexpr int G = 8 / PPL;
    for (int k0 = warp; k0 < NsP; k0 += G * W) {
        double y[G][PPL];
#pragma unroll
        for (int g = 0; g < G; ++g) {
            const int k = k0 + g * W;
            if (k < Ns) {
                load_row<PPL>(Y + (int64_t)k * n, i0, n, vec, y[g]);
            } else {
#pragma unroll
                for (int u = 0; u < PPL; ++u) y[g][u] = 0.0;
            }
        }
#pragma unroll
        for (int g = 0; g < G; ++g) {
            const int k = k0 + g * W;
            if (k < NsP) {
                const double *sp = tp.sp + 12 * k;  // padded rows are all zero: z = 0, r = 0
                const double rW = __ldg(sp + 10), w4 = __ldg(sp + 8);
#pragma unroll
                for (int u = 0; u < PPL; ++u) {
                    const double z = y[g][u] * rW;
                    const double r = exp2_poly9(cubic4(sp, L[u])) * w4;   // 1/a_k = W_k^(1/4) / sqrt(mu_k)
                    const double lam = exp2_poly9(cubic4(sp + 4, L[u]));  // lambda_k
                    invW[u] += z;
                    sum_a[u] = fma(z, lam, sum_a[u]);
                    sum_h[u] = fma(z, crf::rcp_newton(lam), sum_h[u]);
                    sZ[ROW(k, u) + lane] = z;
                    sS[ROW(k, u) + lane] = r;
                }
            }
        }
    }
#pragma unroll
    for (int u = 0; u < PPL; ++u) {
        sred[((0 * W + warp) * PPL + u) * 32 + lane] = invW[u];
        sred[((1 * W + warp) * PPL + u) * 32 + lane] = sum_a[u];
        sred[((2 * W + warp) * PPL + u) * 32 + lane] = sum_h[u];
    }

    // ---- a11: Wilke.  Pass ps gives warp w the row block I = ps W + w; the c_kj of a pass arrive in panels of
    // column blocks (stage blocks, plan_transport.cu); the block after the last panel is pair round 0.
    double mu_p[PPL];
#pragma unroll
    for (int u = 0; u < PPL; ++u) mu_p[u] = 0.0;
    const int nwk = tp.n_wilke;
    {
        double A[PPL][TS], B[PPL][TS], C[PPL][TS];
        for (int s = 0; s < nwk; ++s) {
            stage_wait();
            __syncthreads();  // block s has landed; everyone is done with block s - 1
            const unsigned char *blk = sStage + (size_t)(s & 1) * tp.stage_bytes;
            const int4 ds = cur;
            cur = *reinterpret_cast<const int4 *>(blk);
            stage_async(sStage + (size_t)((s + 1) & 1) * tp.stage_bytes, tp.pair_coef + cur.x, cur.y, threadIdx.x, 32 * W);
            const int J0 = ds.z & 0xff, I = ((ds.z >> 8) & 0xff) * W + warp, nJ = ds.w;
            if (I >= nb) continue;
            if (ds.z & (1 << 16)) {
#pragma unroll
                for (int u = 0; u < PPL; ++u)
#pragma unroll
                    for (int a = 0; a < TS; ++a) A[u][a] = B[u][a] = C[u][a] = 0.0;
            }
            // row length of the slab: the nJ column blocks, rounded up to whole groups of four columns (zero coefficients)
            const int ld = TS == 8 ? 8 * nJ : (TS * nJ + 3) & ~3;
            const double *cw = reinterpret_cast<const double *>(blk + HDR) + warp * TS * ld;
            // four columns at a time: 12 right-hand-side values in registers leave room for the compiler to
            // keep several coefficient loads in flight
            for (int j4 = 0; j4 < (TS == 8 ? 2 * nJ : ld >> 2); ++j4) {
#pragma unroll
                for (int u = 0; u < PPL; ++u) {
                    double u0[4], u1[4], u2[4];
#pragma unroll
                    for (int b = 0; b < 4; ++b) {
                        u0[b] = sZl[ROW(TS * J0 + 4 * j4 + b, u)];
                        const double r = sSl[ROW(TS * J0 + 4 * j4 + b, u)];
                        u1[b] = u0[b] * r;
                        u2[b] = u1[b] * r;
                    }
#pragma unroll
                    for (int a = 0; a < TS; ++a) {
                        const double2 c01 = *reinterpret_cast<const double2 *>(cw + a * ld + 4 * j4);
                        const double2 c23 = *reinterpret_cast<const double2 *>(cw + a * ld + 4 * j4 + 2);
                        A[u][a] = fma(c01.x, u0[0], A[u][a]);
                        B[u][a] = fma(c01.x, u1[0], B[u][a]);
                        C[u][a] = fma(c01.x, u2[0], C[u][a]);
                        A[u][a] = fma(c01.y, u0[1], A[u][a]);
                        B[u][a] = fma(c01.y, u1[1], B[u][a]);
                        C[u][a] = fma(c01.y, u2[1], C[u][a]);
                        A[u][a] = fma(c23.x, u0[2], A[u][a]);
                        B[u][a] = fma(c23.x, u1[2], B[u][a]);
                        C[u][a] = fma(c23.x, u2[2], C[u][a]);
                        A[u][a] = fma(c23.y, u0[3], A[u][a]);
                        B[u][a] = fma(c23.y, u1[3], B[u][a]);
                        C[u][a] = fma(c23.y, u2[3], C[u][a]);
                    }
                }
            }
            if (ds.z & (1 << 17)) {
#pragma unroll
                for (int a = 0; a < TS; ++a) {
                    const int k = TS * I + a;
                    if (k < Ns) {
                        const double wk = __ldg(tp.sp + 12 * k + 9);
#pragma unroll
                        for (int u = 0; u < PPL; ++u) {
                            const double ak = crf::rcp_newton(sSl[ROW(k, u)]);
                            const double ak2 = ak * ak;
                            const double den = fma(ak2, C[u][a], fma(ak + ak, B[u][a], A[u][a]));
                            mu_p[u] = fma(sZl[ROW(k, u)] * (ak2 * wk), crf::rcp_newton(den), mu_p[u]);
                        }
                    }
                }
            }
        }
    }
#pragma unroll
    for (int u = 0; u < PPL; ++u) sred[((3 * W + warp) * PPL + u) * 32 + lane] = mu_p[u];
    __syncthreads();  // every warp is done reading 1/a_k
    for (int k = warp; k < NsP; k += W)
#pragma unroll
        for (int u = 0; u < PPL; ++u) sS[ROW(k, u) + lane] = 0.0;
    double iw[PPL];
#pragma unroll
    for (int u = 0; u < PPL; ++u) {
        iw[u] = 0.0;
#pragma unroll
        for (int w = 0; w < W; ++w) iw[u] += sred[((0 * W + w) * PPL + u) * 32 + lane];
    }
    if (warp == 0) {
        double lam_o[PPL], mu_o[PPL];
#pragma unroll
        for (int u = 0; u < PPL; ++u) {
            double sa = 0.0, sh = 0.0, mm = 0.0;
#pragma unroll
            for (int w = 0; w < W; ++w) {
                sa += sred[((1 * W + w) * PPL + u) * 32 + lane];
                sh += sred[((2 * W + w) * PPL + u) * 32 + lane];
                mm += sred[((3 * W + w) * PPL + u) * 32 + lane];
            }
            // lambda = (sum X lambda_k + 1/sum X/lambda_k)/2 with X = Z Wbar = Z / iw ; mu: Wbar cancels
            lam_o[u] = 0.5 * (sa / iw[u] + iw[u] / sh);
            mu_o[u] = mm;
        }
        store_row<PPL>(lambda, i0, n, vec, lam_o);
        store_row<PPL>(mu, i0, n, vec, mu_o);
    }
    stage_wait();
    __syncthreads();

    // ---- a13: binary pairs, tiles in rounds; round rd+1 is staged while round rd is evaluated
    const int nrd = tp.n_rounds;
    for (int rd = 0; rd < nrd; ++rd) {
        const unsigned char *blk = sStage + (size_t)((nwk + rd) & 1) * tp.stage_bytes;
        if (rd + 1 < nrd) {
            const int4 r1 = *reinterpret_cast<const int4 *>(blk);
            stage_async(sStage + (size_t)((nwk + rd + 1) & 1) * tp.stage_bytes, tp.pair_coef + r1.x, r1.y, threadIdx.x, 32 * W);
        }
        const int2 d = *reinterpret_cast<const int2 *>(blk + 16 + 8 * warp);
        const int kind = d.x & 0xff, jb = (d.x >> 8) & 0xff, kb = (d.x >> 16) & 0xff;
        const double2 *cf = reinterpret_cast<const double2 *>(blk + d.y);
        if (kind == 1)
            tile_offdiag<PPL, TS>(cf, L, sZl, sSl, jb, kb, sTab);
        else if (kind == 2)
            tile_diag<PPL, TS>(cf, L, sZl, sSl, jb, sTab);
        stage_wait();
        __syncthreads();
    }

    // ---- rho D_km = p_ref (1 - Y_k) / (R T S_k); pure species: rho D_kk = Wbar p_ref D_kk(p_ref) / (R T)
    double f[PPL];
#pragma unroll
    for (int u = 0; u < PPL; ++u) f[u] = m.p_ref / (CRF_R_GAS * Ti[u]);
    for (int k0 = warp; k0 < Ns; k0 += G * W) {
        double y[G][PPL];
#pragma unroll
        for (int g = 0; g < G; ++g)
            if (k0 + g * W < Ns) load_row<PPL>(Y + (int64_t)(k0 + g * W) * n, i0, n, vec, y[g]);
#pragma unroll
        for (int g = 0; g < G; ++g) {
            const int k = k0 + g * W;
            if (k < Ns) {
                double v[PPL];
#pragma unroll
                for (int u = 0; u < PPL; ++u) {
                    const double s = sS[ROW(k, u) + lane];
                    if (s == 0.0)
                        v[u] = f[u] / iw[u] * exp(cubic4(tp.Ddiag + 4 * k, L[u]));
                    else
                        v[u] = f[u] * (1.0 - y[g][u]) * crf::rcp_newton(s);
                }
                store_row<PPL>(rhoD + (int64_t)k * n, i0, n, vec, v);
            }
        }
    }
}

template <int W, int PPL, int TS>
cudaError_t launch_w2(const DevTables &m, const double *T, const double *Y, int64_t n, double *mu, double *lambda,
                     double *rhoD, cudaStream_t st)
{
    const size_t smem = transport_tiled_dynamic_smem(m);
    cudaError_t e = cudaFuncSetAttribute(transport_tiled_kernel<W, PPL, TS>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                         (int)smem);
    if (e != cudaSuccess) return e;
    const int64_t per_block = 32 * PPL;
    transport_tiled_kernel<W, PPL, TS><<<(unsigned)((n + per_block - 1) / per_block), 32 * W, smem, st>>>(m, T, Y, n, mu,
                                                                                                     lambda, rhoD);
    crf_count_launch();
    return cudaGetLastError();
}

template <int W, int PPL>
cudaError_t launch_w(const DevTables &m, const double *T, const double *Y, int64_t n, double *mu, double *lambda,
                     double *rhoD, cudaStream_t st)
{
    return m.tp.TS == 7 ? launch_w2<W, PPL, 7>(m, T, Y, n, mu, lambda, rhoD, st) : launch_w2<W, PPL, 8>(m, T, Y, n, mu, lambda, rhoD, st);
}

}  // namespace

size_t transport_tiled_dynamic_smem(const DevTables &m)
{
    return sizeof(double) * ((size_t)2 * m.tp.NsP + 4 * (size_t)m.tp.W) * m.tp.PPL * 32 + 2 * (size_t)m.tp.stage_bytes;
}

cudaError_t launch_transport_tiled(const DevTables &m, const double *T, const double *Y, int64_t n, double *mu,
                                   double *lambda, double *rhoD, cudaStream_t st)
{
    switch (m.tp.W * 10 + m.tp.PPL) {
    case 11: return launch_w<1, 1>(m, T, Y, n, mu, lambda, rhoD, st);
    case 21: return launch_w<2, 1>(m, T, Y, n, mu, lambda, rhoD, st);
    case 41: return launch_w<4, 1>(m, T, Y, n, mu, lambda, rhoD, st);
    case 81: return launch_w<8, 1>(m, T, Y, n, mu, lambda, rhoD, st);
    case 12: return launch_w<1, 2>(m, T, Y, n, mu, lambda, rhoD, st);
    case 22: return launch_w<2, 2>(m, T, Y, n, mu, lambda, rhoD, st);
    case 42: return launch_w<4, 2>(m, T, Y, n, mu, lambda, rhoD, st);
    case 82: return launch_w<8, 2>(m, T, Y, n, mu, lambda, rhoD, st);
    default: return cudaErrorInvalidValue;
    }
}
