// sem_diffusion.cu -- crf_sem_diffusion: the element-local spectral-element diffusion operator that
// consumes what crf_rhs_pointwise emits (rho D_k, lambda, Wbar): the weak form of -div(rho Y_k V_k) with the
// mixture-averaged diffusion velocity and its correction velocity (Eq. 1a, 2) and of
// div(lambda grad T) (Eq. 1b) on the 8^3 Gauss-Lobatto-Legendre points of order-7 hexahedra (PAPER.md:92,
// 102), affine box elements.  "diffusion" is the most expensive kernel of the paper's right-hand side (28 %,
// PAPER.md:178) and is bound by global memory bandwidth there (987 GB/s on A100).
//
//   X_k = Y_k Wbar / W_k;  f_k = (W_k / Wbar) (rho D_k) grad X_k;  j_k = -f_k + Y_k sum_j f_j
//   dY_k[i] = sum_q w_q |J| grad phi_i . j_k,     dT[i] = -sum_q w_q |J| grad phi_i . lambda grad T
//
// Shape.  One element per block of two warps; the 8 x 8 x 8 derivative contractions along x and y run on the FP64 tensor
// cores (mma.sync.m8n8k4.f64: the one dense contraction of this operator; the fields are held in the MMA accumulator
// layout, details at the kernel), the one along z is a register contraction with constant-bank matrix entries.  The
// correction flux sum_j f_j needs every species before any j_k can be formed: pass 1 accumulates it in registers, pass 2
// recomputes grad X_k (its inputs come back from L2), forms j_k and applies the transposed derivative to the weighted
// flux.  The quadrature nodes, weights and the derivative matrix are computed on the host by the closed forms of the
// Legendre polynomials (Newton iteration for the nodes) and live in constant memory.
#include <cmath>
#include <mutex>

#include "crf_internal.h"
#include "launch.h"

namespace {

constexpr int N = 8, NP = N * N * N;

__constant__ double cD[N * N];  // D[i][m] = l_m'(x_i)
__constant__ double cW[N];      // GLL weights

// Legendre P_p and P_{p-1} at x by the three-term recurrence
void legendre(int p, double x, double &Pp, double &Pm)
{
    double a = 1.0, b = x;
    for (int k = 2; k <= p; ++k) {
        const double c = ((2 * k - 1) * x * b - (k - 1) * a) / k;
        a = b, b = c;
    }
    Pp = b, Pm = a;
}

// GLL nodes (Newton on (1 - x^2) P_p'(x) from the Chebyshev points), weights 2 / (p (p + 1) P_p(x)^2) and the derivative
// matrix D_im = P_p(x_i) / (P_p(x_m) (x_i - x_m)), D_00 = -p (p + 1) / 4 = -D_pp, 0 elsewhere on the diagonal
void gll_tables(double *x, double *w, double *D)
{
    const int p = N - 1;
    const double pi = 3.14159265358979323846;
    double P[N];
    for (int i = 0; i < N; ++i) {
        double xi = -std::cos(pi * i / p);
        for (int it = 0; it < 100; ++it) {
            double Pp, Pm;
            legendre(p, xi, Pp, Pm);
            const double dx = (xi * Pp - Pm) / ((p + 1) * Pp);
            xi -= dx;
            if (std::fabs(dx) < 1e-16) break;
        }
        if (i == 0) xi = -1.0;
        if (i == p) xi = 1.0;
        double Pm;
        legendre(p, xi, P[i], Pm);
        x[i] = xi;
        w[i] = 2.0 / (p * (p + 1) * P[i] * P[i]);
    }
    for (int i = 0; i < N; ++i)
        for (int m = 0; m < N; ++m) {
            if (i != m)
                D[i * N + m] = P[i] / (P[m] * (x[i] - x[m]));
            else
                D[i * N + m] = i == 0 ? -0.25 * p * (p + 1) : (i == p ? 0.25 * p * (p + 1) : 0.0);
        }
}

// ---- the kernel: one element per 64 threads (two warps), the derivative contractions on the FP64 tensor cores -----
// A field of the element is held in the accumulator layout of mma.m8n8k4.f64: at level k (z index) the 8 x 8 matrix
// F_k[j][i] (row j = y index, column i = x index) is spread over the warp, lane (g, t) = (lane / 4, lane % 4) holding
// F_k[g][2 t] and F_k[g][2 t + 1], two adjacent points: one 128-bit access.  Warp w of the block owns levels 4 w .. 4 w + 3.
//   d/dx:  G_k = F_k D^T   A = F_k (from the shared-memory copy, lane reads F_k[g][4 c + t]),  B = D^T: lane constant D[g][4 c + t]
//   d/dy:  G_k = D F_k     A = D:  the same lane constant,                                     B = F_k: lane reads F_k[4 c + t][g]
//   d/dz:  G_k = sum_m D[k][m] F_m   the lane's own points of all levels (shared-memory copy), D as constant-bank operands
// and the transposed matrices for the weak divergence (lane constant D[4 c + t][g]).  Each 8 x 8 x 8 product is two MMAs
// (k = 4 each); an MMA does the work of eight warp-wide DFMAs in one issue slot.
// Slab [level][row][col] of 8 x 8 x 8 doubles with the column PAIRS of rows 2, 3, 6, 7 swapped in halves (pair p of row r at
// p ^ 2 ((r >> 1) & 1)): the 128-bit accesses of a lane's own pair, the 64-bit reads of the A fragments (row g, columns
// 4 c + t) and of the B fragments (rows 4 c + t, column g) are then all free of bank conflicts.
constexpr int LS = 64, SLAB = 8 * LS;
__device__ __forceinline__ int slab_off(int r, int i) { return r * 8 + (((i >> 1) ^ (2 * ((r >> 1) & 1))) << 1) + (i & 1); }

__device__ __forceinline__ void dmma(double &d0, double &d1, double a, double b)
{
    asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0, %1}, {%2}, {%3}, {%0, %1};" : "+d"(d0), "+d"(d1) : "d"(a), "d"(b));
}

struct Lane {
    int own, offA[2], offB[2];  // slab offsets: the lane's pair (g, 2 t); A fragment (g, 4 c + t); B fragment (4 c + t, g)
    double dg[2], dt[2];        // D[g][4 c + t] (gradient), D[4 c + t][g] (weak divergence)
};

// Reference-element gradient at the lane's points of level 4 WI + Q.  s: the slab of the field (all levels); u: the lane's
// own values (levels 4 WI .. 4 WI + 3); up: the other warp's four levels at the same points (read from the slab once per
// species).  The matrix entries of the z-derivative are constant-bank operands (WI, Q are template parameters for that).
template <int WI, int Q>
__device__ __forceinline__ void grad_level(const double *s, const Lane &l, const double2 (&u)[4], const double2 (&up)[4], double2 &gr,
                                           double2 &gs, double2 &gt)
{
    const double *lev = s + (4 * WI + Q) * LS;
    gr = gs = gt = make_double2(0.0, 0.0);
#pragma unroll
    for (int c = 0; c < 2; ++c) {
        dmma(gr.x, gr.y, lev[l.offA[c]], l.dg[c]);
        dmma(gs.x, gs.y, l.dg[c], lev[l.offB[c]]);
    }
#pragma unroll
    for (int m = 0; m < 4; ++m) {
        const double d0 = cD[(4 * WI + Q) * N + 4 * WI + m], d1 = cD[(4 * WI + Q) * N + 4 * (1 - WI) + m];
        gt.x = fma(d0, u[m].x, gt.x), gt.y = fma(d0, u[m].y, gt.y);
        gt.x = fma(d1, up[m].x, gt.x), gt.y = fma(d1, up[m].y, gt.y);
    }
}
template <int Q>
struct Lvl {
    static constexpr int value = Q;
};
template <class F>
__device__ __forceinline__ void for_levels(F &&f)
{
    f(Lvl<0>()), f(Lvl<1>()), f(Lvl<2>()), f(Lvl<3>());
}

// sum_m D[m][i] ax(m, j, k) + sum_m D[m][j] ay(i, m, k) + sum_m D[m][k] az(i, j, m) at the lane's points of its four levels;
// az: the lane's own values, the other warp's from the slab sC
template <int WI>
__device__ __forceinline__ void weak_div(const double *sA, const double *sB, const double *sC, const Lane &l, const double2 (&az)[4],
                                         double2 (&o)[4])
{
    double2 ap[4];
#pragma unroll
    for (int q = 0; q < 4; ++q) ap[q] = *reinterpret_cast<const double2 *>(sC + (4 * (1 - WI) + q) * LS + l.own);
#pragma unroll
    for (int q = 0; q < 4; ++q) {
        const int k = 4 * WI + q;
        o[q] = make_double2(0.0, 0.0);
#pragma unroll
        for (int c = 0; c < 2; ++c) {
            dmma(o[q].x, o[q].y, sA[k * LS + l.offA[c]], l.dt[c]);
            dmma(o[q].x, o[q].y, l.dt[c], sB[k * LS + l.offB[c]]);
        }
#pragma unroll
        for (int m = 0; m < 4; ++m) {
            const double d0 = cD[(4 * WI + m) * N + k], d1 = cD[(4 * (1 - WI) + m) * N + k];
            o[q].x = fma(d0, az[m].x, o[q].x), o[q].y = fma(d0, az[m].y, o[q].y);
            o[q].x = fma(d1, ap[m].x, o[q].x), o[q].y = fma(d1, ap[m].y, o[q].y);
        }
    }
}

// cp.async of 16 bytes (global -> shared); the issuing thread reads them back after cp_wait
__device__ __forceinline__ void cp16(void *dst, const void *src)
{
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"((unsigned)__cvta_generic_to_shared(dst)), "l"(src) : "memory");
}
__device__ __forceinline__ void cp_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
template <int PENDING>
__device__ __forceinline__ void cp_wait()
{
    asm volatile("cp.async.wait_group %0;" ::"n"(PENDING) : "memory");
}

template <int WI>
__device__ __forceinline__ void element(const DevTables &m, double *sm, const double *__restrict__ h3, const double *__restrict__ T,
                                        const double *__restrict__ Wbar, const double *__restrict__ Y, const double *__restrict__ lam,
                                        const double *__restrict__ rhoD, int64_t nel, double *__restrict__ dY, double *__restrict__ dT)
{
    double *sU2 = sm, *sA = sm + 2 * SLAB, *sB = sm + 3 * SLAB, *sC = sm + 4 * SLAB;  // (the field slab is double: one barrier less per species)
    double2 *sStage = reinterpret_cast<double2 *>(sm + 5 * SLAB);  // [2 buffers][2 fields][4 levels x 64 threads] of point pairs
    const int lane = threadIdx.x & 31, g = lane >> 2, t = lane & 3;
    Lane l;
    l.own = slab_off(g, 2 * t);
#pragma unroll
    for (int c = 0; c < 2; ++c) {
        l.offA[c] = slab_off(g, 4 * c + t), l.offB[c] = slab_off(4 * c + t, g);
        l.dg[c] = cD[g * N + 4 * c + t], l.dt[c] = cD[(4 * c + t) * N + g];
    }
    const int64_t e = blockIdx.x, n = nel * NP;
    // the lane's points: (i, j, k) = (2 t + {0, 1}, g, 4 WI + q): global offset of the pair at level q = 0
    const int64_t gbase = e * NP + (4 * WI) * 64 + g * 8 + 2 * t;
    const int sbase = (4 * WI) * LS + l.own;
    auto ld2 = [&](const double *f, int q) { return *reinterpret_cast<const double2 *>(f + gbase + 64 * q); };
    const double hx = h3[3 * e], hy = h3[3 * e + 1], hz = h3[3 * e + 2];
    const double sx = 2.0 / hx, sy = 2.0 / hy, sz = 2.0 / hz, jac = 0.125 * hx * hy * hz;
    // Wbar and 1 / Wbar of the lane's points: shared memory (read back by the same thread for every species)
    double2 *sWb = sStage + 1024 + threadIdx.x;  // [4 levels][64 threads] Wbar, then [4][64] 1 / Wbar
#pragma unroll
    for (int q = 0; q < 4; ++q) {
        const double2 w = ld2(Wbar, q);
        sWb[64 * q] = w;
        sWb[256 + 64 * q] = make_double2(1.0 / w.x, 1.0 / w.y);
    }
    const int Ns = m.Ns;
    // Jobs 0 .. Ns - 1: pass 1; Ns .. 2 Ns - 1: pass 2; 2 Ns: the heat flux.  The two input fields of job + 1 are fetched with
    // cp.async into a stage while job computes (each thread fetches and reads back its own point pairs).
    auto fetch = [&](int job) {
        const int s = job < Ns ? job : 2 * Ns - 1 - job;  // (pass 2 walks the species backwards: the last ones of pass 1 are still in L2)
        const double *a = job == 2 * Ns ? T : Y + (int64_t)s * n, *b = job == 2 * Ns ? lam : rhoD + (int64_t)s * n;
        double2 *dst = sStage + (size_t)(job & 1) * 512 + threadIdx.x;
#pragma unroll
        for (int q = 0; q < 4; ++q) cp16(dst + 64 * q, a + gbase + 64 * q), cp16(dst + 256 + 64 * q, b + gbase + 64 * q);
        cp_commit();
    };
    auto staged = [&](int job, int field, int q) { return sStage[(size_t)(job & 1) * 512 + field * 256 + 64 * q + threadIdx.x]; };
    fetch(0);

    // ---- pass 1: the correction flux sum_k f_k at the lane's points
    double2 fcx[4], fcy[4], fcz[4];
#pragma unroll
    for (int q = 0; q < 4; ++q) fcx[q] = fcy[q] = fcz[q] = make_double2(0.0, 0.0);
    for (int s = 0; s < Ns; ++s) {
        const double Ws = __ldg(m.W + s), rWs = __ldg(m.rW + s);
        fetch(s + 1);
        cp_wait<1>();
        double2 u[4];
#pragma unroll
        for (int q = 0; q < 4; ++q) {
            const double2 y = staged(s, 0, q), w = sWb[64 * q];
            u[q] = make_double2(y.x * w.x * rWs, y.y * w.y * rWs);
        }
        double *sU = sU2 + (s & 1) * SLAB;  // (its previous readers, two species back, passed the barrier of the last species)
#pragma unroll
        for (int q = 0; q < 4; ++q) *reinterpret_cast<double2 *>(sU + sbase + q * LS) = u[q];
        __syncthreads();
        double2 up[4];
#pragma unroll
        for (int q = 0; q < 4; ++q) up[q] = *reinterpret_cast<const double2 *>(sU + (4 * (1 - WI) + q) * LS + l.own);
        for_levels([&](auto Q) {
            constexpr int q = decltype(Q)::value;
            double2 gr, gs, gt;
            grad_level<WI, q>(sU, l, u, up, gr, gs, gt);
            const double2 r = staged(s, 1, q), rw = sWb[256 + 64 * q];
            const double cx = Ws * r.x * rw.x, cy = Ws * r.y * rw.y;
            fcx[q].x = fma(cx * sx, gr.x, fcx[q].x), fcx[q].y = fma(cy * sx, gr.y, fcx[q].y);
            fcy[q].x = fma(cx * sy, gs.x, fcy[q].x), fcy[q].y = fma(cy * sy, gs.y, fcy[q].y);
            fcz[q].x = fma(cx * sz, gt.x, fcz[q].x), fcz[q].y = fma(cy * sz, gt.y, fcz[q].y);
        });
    }

    // ---- pass 2: j_k = -f_k + Y_k sum f and its weak divergence; last: the heat flux
    const double wgx = cW[g] * cW[2 * t] * jac, wgy = cW[g] * cW[2 * t + 1] * jac;  // w_j w_i |J| of the two points
    for (int s = 0; s <= Ns; ++s) {
        const bool heat = s == Ns;
        const int sp = heat ? Ns : Ns - 1 - s;  // the species of this step
        const double Ws = heat ? 1.0 : __ldg(m.W + sp), rWs = heat ? 1.0 : __ldg(m.rW + sp);
        if (!heat) {
            fetch(Ns + s + 1);
            cp_wait<1>();
        } else {
            cp_wait<0>();
        }
        double2 u[4];
#pragma unroll
        for (int q = 0; q < 4; ++q) {
            const double2 y = staged(Ns + s, 0, q), w = sWb[64 * q];
            u[q] = heat ? y : make_double2(y.x * w.x * rWs, y.y * w.y * rWs);
        }
        double *sU = sU2 + ((Ns + s) & 1) * SLAB;
#pragma unroll
        for (int q = 0; q < 4; ++q) *reinterpret_cast<double2 *>(sU + sbase + q * LS) = u[q];
        __syncthreads();  // (also: the previous species is done with sA, sB, sC)
        double2 up[4], az[4];
#pragma unroll
        for (int q = 0; q < 4; ++q) up[q] = *reinterpret_cast<const double2 *>(sU + (4 * (1 - WI) + q) * LS + l.own);
        for_levels([&](auto Q) {
            constexpr int q = decltype(Q)::value;
            double2 gr, gs, gt;
            grad_level<WI, q>(sU, l, u, up, gr, gs, gt);
            const double2 y = staged(Ns + s, 0, q), r = staged(Ns + s, 1, q), rw = sWb[256 + 64 * q];
            const double cx = heat ? r.x : Ws * r.x * rw.x, cy = heat ? r.y : Ws * r.y * rw.y;
            const double yx = heat ? 0.0 : y.x, yy = heat ? 0.0 : y.y;
            const double wk = cW[4 * WI + q];
            // (both: minus the gradient flux; species: plus Y_k times the correction flux), times w_q |J| and the metric
            const double2 ax = make_double2(fma(yx, fcx[q].x, -(cx * sx) * gr.x) * (wgx * wk * sx),
                                            fma(yy, fcx[q].y, -(cy * sx) * gr.y) * (wgy * wk * sx));
            const double2 ay = make_double2(fma(yx, fcy[q].x, -(cx * sy) * gs.x) * (wgx * wk * sy),
                                            fma(yy, fcy[q].y, -(cy * sy) * gs.y) * (wgy * wk * sy));
            az[q] = make_double2(fma(yx, fcz[q].x, -(cx * sz) * gt.x) * (wgx * wk * sz),
                                 fma(yy, fcz[q].y, -(cy * sz) * gt.y) * (wgy * wk * sz));
            *reinterpret_cast<double2 *>(sA + sbase + q * LS) = ax;
            *reinterpret_cast<double2 *>(sB + sbase + q * LS) = ay;
            *reinterpret_cast<double2 *>(sC + sbase + q * LS) = az[q];
        });
        __syncthreads();
        double2 o[4];
        weak_div<WI>(sA, sB, sC, l, az, o);
        double *dst = heat ? dT : dY + (int64_t)sp * n;
#pragma unroll
        for (int q = 0; q < 4; ++q) *reinterpret_cast<double2 *>(dst + gbase + 64 * q) = o[q];
    }
}

// (four blocks per SM at 214 registers: measured against five and six with a register cap, which spill or run slower)
__global__ void __launch_bounds__(64, 4) sem_diffusion_kernel
(DevTables m, const double *__restrict__ h3, const double *__restrict__ T,
                                                           const double *__restrict__ Wbar, const double *__restrict__ Y,
                                                           const double *__restrict__ lam, const double *__restrict__ rhoD,
                                                           int64_t nel, double *__restrict__ dY, double *__restrict__ dT)
{
    __shared__ __align__(16) double sm[5 * SLAB + 2048 + 1024];  // the field; the three components of the weighted flux; the input stage; Wbar, 1 / Wbar
    // (the two warps run the same steps, barriers included, in two instances: the warp index is a compile-time constant)
    if (threadIdx.x < 32)
        element<0>(m, sm, h3, T, Wbar, Y, lam, rhoD, nel, dY, dT);
    else
        element<1>(m, sm, h3, T, Wbar, Y, lam, rhoD, nel, dY, dT);
}

std::mutex g_mu;
bool g_done[64] = {};  // (per device: the constant tables belong to a device's copy of the module)

}  // namespace

cudaError_t launch_sem_diffusion(const DevTables &m, const double *h3, const double *T, const double *Wbar, const double *Y,
                                 const double *lam, const double *rhoD, int64_t nel, double *dY, double *dT, cudaStream_t st)
{
    int dev = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return e;
    {
        std::lock_guard<std::mutex> lock(g_mu);
        if (dev < 0 || dev >= 64) return cudaErrorInvalidDevice;
        if (!g_done[dev]) {
            double x[N], w[N], D[N * N];
            gll_tables(x, w, D);
            if ((e = cudaMemcpyToSymbol(cD, D, sizeof(D))) != cudaSuccess) return e;
            if ((e = cudaMemcpyToSymbol(cW, w, sizeof(w))) != cudaSuccess) return e;
            g_done[dev] = true;
        }
    }
    sem_diffusion_kernel<<<(unsigned)nel, 64, 0, st>>>(m, h3, T, Wbar, Y, lam, rhoD, nel, dY, dT);
    crf_count_launch();
    return cudaGetLastError();
}
