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
// atomics; one __syncthreads per round.  Each unordered pair is evaluated once:
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

namespace {

using crf::exp2_poly9;

__device__ __forceinline__ double cubic4(const double *__restrict__ c, double x)
{
    const double2 lo = __ldg(reinterpret_cast<const double2 *>(c));
    const double2 hi = __ldg(reinterpret_cast<const double2 *>(c) + 1);
    return fma(x, fma(x, fma(x, hi.y, hi.x), lo.y), lo.x);
}

// off-diagonal tile: species blocks jb < kb, 64 pairs
__device__ __forceinline__ void tile_offdiag(const double *__restrict__ cf, double L, const double *sZ, double *sS,
                                             int jb, int kb, int lane)
{
    double zj[8], zk[8], sj[8], sk[8];
#pragma unroll
    for (int a = 0; a < 8; ++a) {
        zj[a] = sZ[(8 * jb + a) * 32 + lane];
        zk[a] = sZ[(8 * kb + a) * 32 + lane];
        sj[a] = 0.0;
        sk[a] = 0.0;
    }
#pragma unroll
    for (int a = 0; a < 8; ++a) {
#pragma unroll
        for (int b = 0; b < 8; ++b) {
            const double e = exp2_poly9(cubic4(cf + 4 * (8 * a + b), L));
            sj[a] = fma(zk[b], e, sj[a]);
            sk[b] = fma(zj[a], e, sk[b]);
        }
    }
#pragma unroll
    for (int a = 0; a < 8; ++a) {
        sS[(8 * jb + a) * 32 + lane] += sj[a];
        sS[(8 * kb + a) * 32 + lane] += sk[a];
    }
}

// diagonal tile: pairs a < b inside block jb, 28 pairs
__device__ __forceinline__ void tile_diag(const double *__restrict__ cf, double L, const double *sZ, double *sS, int jb,
                                          int lane)
{
    double z[8], s[8];
#pragma unroll
    for (int a = 0; a < 8; ++a) {
        z[a] = sZ[(8 * jb + a) * 32 + lane];
        s[a] = 0.0;
    }
    int q = 0;
#pragma unroll
    for (int a = 0; a < 8; ++a) {
#pragma unroll
        for (int b = a + 1; b < 8; ++b, ++q) {
            const double e = exp2_poly9(cubic4(cf + 4 * q, L));
            s[a] = fma(z[b], e, s[a]);
            s[b] = fma(z[a], e, s[b]);
        }
    }
#pragma unroll
    for (int a = 0; a < 8; ++a) sS[(8 * jb + a) * 32 + lane] += s[a];
}

template <int W>
__global__ void __launch_bounds__(32 * W, 12 / W)
    transport_tiled_kernel(DevTables m, const double *__restrict__ T, const double *__restrict__ Y, int64_t n,
                           double *__restrict__ mu, double *__restrict__ lambda, double *__restrict__ rhoD)
{
    extern __shared__ double sm[];
    const TransportPlan &tp = m.tp;
    const int Ns = m.Ns, NsP = tp.NsP, nb = tp.nb;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    double *sZ = sm;                     // [NsP][32]  Z_k = Y_k / W_k
    double *sS = sm + (size_t)NsP * 32;  // [NsP][32]  1/a_k during the Wilke phase, then the diffusion sums
    double *sred = sS + (size_t)NsP * 32;  // [4][W][32] partial sums of the warps

    const int64_t i = (int64_t)blockIdx.x * 32 + lane;
    const bool valid = i < n;
    const int64_t ic = valid ? i : n - 1;  // lanes past the end recompute the last point and store nothing
    const double Ti = T[ic];
    const double L = log(Ti);

    // ---- a1, a10, a12: Z_k, species fits, conductivity sums; warp w takes species w, w+W, ...
    double invW = 0.0, sum_a = 0.0, sum_h = 0.0;
    for (int k = warp; k < NsP; k += W) {
        double z = 0.0, r = 0.0;
        if (k < Ns) {
            const double *sp = tp.sp + 12 * k;
            z = Y[(int64_t)k * n + ic] * __ldg(sp + 10);
            const double smu = exp(cubic4(sp, L));       // sqrt(mu_k)
            const double lam = exp(cubic4(sp + 4, L));   // lambda_k
            r = 1.0 / (smu * __ldg(sp + 8));             // 1/a_k
            invW += z;
            sum_a = fma(z, lam, sum_a);
            sum_h += z / lam;
        }
        sZ[k * 32 + lane] = z;
        sS[k * 32 + lane] = r;
    }
    sred[(0 * W + warp) * 32 + lane] = invW;
    sred[(1 * W + warp) * 32 + lane] = sum_a;
    sred[(2 * W + warp) * 32 + lane] = sum_h;
    __syncthreads();

    // ---- a11: Wilke, row blocks dealt to the warps
    double mu_p = 0.0;
    for (int I = warp; I < nb; I += W) {
        double A[8], B[8], C[8];
#pragma unroll
        for (int a = 0; a < 8; ++a) A[a] = B[a] = C[a] = 0.0;
        for (int J = 0; J < nb; ++J) {
            double u0[8], u1[8], u2[8];
#pragma unroll
            for (int b = 0; b < 8; ++b) {
                u0[b] = sZ[(8 * J + b) * 32 + lane];
                const double r = sS[(8 * J + b) * 32 + lane];
                u1[b] = u0[b] * r;
                u2[b] = u1[b] * r;
            }
            const double *c = tp.wilke_cP + (size_t)(8 * I) * NsP + 8 * J;
#pragma unroll
            for (int a = 0; a < 8; ++a) {
#pragma unroll
                for (int b = 0; b < 8; b += 2) {
                    const double2 cc = __ldg(reinterpret_cast<const double2 *>(c + (size_t)a * NsP + b));
                    A[a] = fma(cc.x, u0[b], A[a]);
                    B[a] = fma(cc.x, u1[b], B[a]);
                    C[a] = fma(cc.x, u2[b], C[a]);
                    A[a] = fma(cc.y, u0[b + 1], A[a]);
                    B[a] = fma(cc.y, u1[b + 1], B[a]);
                    C[a] = fma(cc.y, u2[b + 1], C[a]);
                }
            }
        }
#pragma unroll
        for (int a = 0; a < 8; ++a) {
            const int k = 8 * I + a;
            if (k < Ns) {
                const double ak = 1.0 / sS[k * 32 + lane];
                const double ak2 = ak * ak;
                const double den = fma(ak2, C[a], fma(ak + ak, B[a], A[a]));
                mu_p += sZ[k * 32 + lane] * (ak2 * __ldg(tp.sp + 12 * k + 9)) / den;
            }
        }
    }
    sred[(3 * W + warp) * 32 + lane] = mu_p;
    __syncthreads();  // every warp is done reading 1/a_k
    for (int k = warp; k < NsP; k += W) sS[k * 32 + lane] = 0.0;
    if (warp == 0 && valid) {
        double iw = 0.0, sa = 0.0, sh = 0.0, mm = 0.0;
#pragma unroll
        for (int w = 0; w < W; ++w) {
            iw += sred[(0 * W + w) * 32 + lane];
            sa += sred[(1 * W + w) * 32 + lane];
            sh += sred[(2 * W + w) * 32 + lane];
            mm += sred[(3 * W + w) * 32 + lane];
        }
        // lambda = (sum X lambda_k + 1/sum X/lambda_k)/2 with X = Z Wbar = Z / iw ; mu: Wbar cancels
        lambda[i] = 0.5 * (sa / iw + iw / sh);
        mu[i] = mm;
    }
    __syncthreads();

    // ---- a13: binary pairs, tiles in rounds
    for (int rd = 0; rd < tp.n_rounds; ++rd) {
        const int2 d = __ldg(tp.sched + rd * W + warp);
        const int kind = d.x & 0xff, jb = (d.x >> 8) & 0xff, kb = (d.x >> 16) & 0xff;
        const double *cf = tp.pair_coef + d.y;
        if (kind == 1)
            tile_offdiag(cf, L, sZ, sS, jb, kb, lane);
        else if (kind == 2)
            tile_diag(cf, L, sZ, sS, jb, lane);
        if (W > 1) __syncthreads();
    }

    // ---- rho D_km = p_ref (1 - Y_k) / (R T S_k); pure species: rho D_kk = Wbar p_ref D_kk(p_ref) / (R T)
    const double f = m.p_ref / (CRF_R_GAS * Ti);
    double iw = 0.0;
#pragma unroll
    for (int w = 0; w < W; ++w) iw += sred[(0 * W + w) * 32 + lane];
    for (int k = warp; k < Ns; k += W) {
        const double s = sS[k * 32 + lane];
        double v;
        if (s == 0.0)
            v = f / iw * exp(cubic4(tp.Ddiag + 4 * k, L));
        else
            v = f * (1.0 - Y[(int64_t)k * n + ic]) / s;
        if (valid) rhoD[(int64_t)k * n + i] = v;
    }
}

template <int W>
cudaError_t launch_w(const DevTables &m, const double *T, const double *Y, int64_t n, double *mu, double *lambda,
                     double *rhoD, cudaStream_t st)
{
    const size_t smem = sizeof(double) * ((size_t)2 * m.tp.NsP * 32 + 4 * W * 32);
    cudaError_t e = cudaFuncSetAttribute(transport_tiled_kernel<W>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                         (int)smem);
    if (e != cudaSuccess) return e;
    transport_tiled_kernel<W><<<(unsigned)((n + 31) / 32), 32 * W, smem, st>>>(m, T, Y, n, mu, lambda, rhoD);
    crf_count_launch();
    return cudaGetLastError();
}

}  // namespace

cudaError_t launch_transport_tiled(const DevTables &m, const double *T, const double *Y, int64_t n, double *mu,
                                   double *lambda, double *rhoD, cudaStream_t st)
{
    switch (m.tp.W) {
    case 1: return launch_w<1>(m, T, Y, n, mu, lambda, rhoD, st);
    case 2: return launch_w<2>(m, T, Y, n, mu, lambda, rhoD, st);
    case 4: return launch_w<4>(m, T, Y, n, mu, lambda, rhoD, st);
    default: return cudaErrorInvalidValue;
    }
}
