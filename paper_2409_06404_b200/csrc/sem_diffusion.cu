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
// Shape.  One element per 64 threads: thread (i, j) owns the column of nodes (i, j, 0..7) in registers, so the
// derivative along z is a register contraction whose matrix entries are constant-bank operands (loops fully unrolled),
// and the derivatives along x and y read an 8 x 8 x 8 shared-memory copy of the field with the thread's rows of D in
// registers.  The correction flux sum_j f_j needs every species before any j_k can be formed: pass 1 accumulates it
// (kept in shared memory), pass 2 recomputes grad X_k (its inputs come back from L2) and applies the transposed
// derivative to the weighted flux.  The quadrature nodes, weights and the derivative matrix are computed on the host
// by the closed forms of the Legendre polynomials (Newton iteration for the nodes) and live in constant memory.
#include <cmath>
#include <mutex>

#include "crf_internal.h"
#include "launch.h"

namespace {

constexpr int N = 8, NP = N * N * N;
#ifndef SEM_EPB
#define SEM_EPB 2
#endif
#ifndef SEM_MINB
#define SEM_MINB 1
#endif
constexpr int EPB = SEM_EPB;  // elements per block

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

struct Thread {
    double dI[N], dJ[N], tI[N], tJ[N];  // D[i][m], D[j][m], D[m][i], D[m][j]
};

// gradient of the field whose column is u[8] (registers) and whose copy is in sU, at level K: reference-element derivatives
template <int K>
__device__ __forceinline__ void grad_level(const double *sU, const Thread &t, int i, int j, const double (&u)[N], double &gr, double &gs,
                                           double &gt)
{
    double a = 0.0, b = 0.0, c = 0.0;
#pragma unroll
    for (int m = 0; m < N; ++m) {
        a = fma(t.dI[m], sU[K * 64 + j * 8 + m], a);
        b = fma(t.dJ[m], sU[K * 64 + m * 8 + i], b);
        c = fma(cD[K * N + m], u[m], c);
    }
    gr = a, gs = b, gt = c;
}

// out[k] = sum_m D[m][i] ax(m, j, k) + sum_m D[m][j] ay(i, m, k) + sum_m D[m][k] az[m]  (ax, ay in shared memory)
__device__ __forceinline__ void weak_div(const double *sA, const double *sB, const Thread &t, int i, int j, const double (&az)[N],
                                         double (&out)[N])
{
#pragma unroll
    for (int k = 0; k < N; ++k) {
        double a = 0.0;
#pragma unroll
        for (int m = 0; m < N; ++m) {
            a = fma(t.tI[m], sA[k * 64 + j * 8 + m], a);
            a = fma(t.tJ[m], sB[k * 64 + m * 8 + i], a);
            a = fma(cD[m * N + k], az[m], a);
        }
        out[k] = a;
    }
}

template <int K>
struct Level {
    static constexpr int value = K;
};
template <class F>
__device__ __forceinline__ void for_levels(F &&f)
{
    f(Level<0>()), f(Level<1>()), f(Level<2>()), f(Level<3>()), f(Level<4>()), f(Level<5>()), f(Level<6>()), f(Level<7>());
}

// cp.async of one double (global -> shared); the issuing thread reads it back after cp_wait
__device__ __forceinline__ void cp8(double *dst, const double *src)
{
    asm volatile("cp.async.ca.shared.global [%0], [%1], 8;" ::"r"((unsigned)__cvta_generic_to_shared(dst)), "l"(src) : "memory");
}
__device__ __forceinline__ void cp_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
template <int PENDING>
__device__ __forceinline__ void cp_wait()
{
    asm volatile("cp.async.wait_group %0;" ::"n"(PENDING) : "memory");
}

// Jobs 0 .. Ns-1: pass 1 (the correction flux sum_k f_k); jobs Ns .. 2 Ns - 1: pass 2 (j_k, weak divergence);
// job 2 Ns: the heat flux.  The two input fields of job t + 1 are fetched with cp.async into a shared-memory stage
// while job t computes (the kernel is otherwise bound by the latency of these loads: 8 warps per SM).
__global__ void __launch_bounds__(64 * EPB, SEM_MINB) sem_diffusion_kernel(DevTables m, const double *__restrict__ h3,
                                                                 const double *__restrict__ T, const double *__restrict__ Wbar,
                                                                 const double *__restrict__ Y, const double *__restrict__ lam,
                                                                 const double *__restrict__ rhoD, int64_t nel,
                                                                 double *__restrict__ dY, double *__restrict__ dT)
{
    extern __shared__ double sm_dyn[];  // per element: field copy, two flux slabs, correction flux (3), Wbar, 1/Wbar, stage 2 x 2 slabs
    const int le = threadIdx.x >> 6, tid = threadIdx.x & 63, i = tid & 7, j = tid >> 3;
    const int64_t e = (int64_t)blockIdx.x * EPB + le;
    const bool live = e < nel;
    const int64_t ec = live ? e : nel - 1;  // (a block's idle half recomputes the last element and stores nothing)
    const int64_t n = nel * NP, base = ec * NP + tid;
    double *sm0 = sm_dyn + (size_t)le * 12 * NP;
    double *sU = sm0, *sA = sm0 + NP, *sB = sm0 + 2 * NP, *sFx = sm0 + 3 * NP, *sFy = sm0 + 4 * NP, *sFz = sm0 + 5 * NP;
    double *sWb = sm0 + 6 * NP, *sRw = sm0 + 7 * NP, *sStage = sm0 + 8 * NP;  // Wbar, 1 / Wbar; stage [2][2][NP]
    Thread t;
#pragma unroll
    for (int q = 0; q < N; ++q) t.dI[q] = cD[i * N + q], t.dJ[q] = cD[j * N + q];
    const int Ns = m.Ns, njobs = 2 * Ns + 1;

    auto fetch = [&](int job) {  // the two input fields of a job -> stage[job & 1]
        const int s = job < Ns ? job : job - Ns;
        const double *a = job == 2 * Ns ? T : Y + (int64_t)s * n, *b = job == 2 * Ns ? lam : rhoD + (int64_t)s * n;
        double *dst = sStage + (size_t)(job & 1) * 2 * NP;
#pragma unroll
        for (int k = 0; k < N; ++k) cp8(dst + k * 64 + tid, a + base + 64 * k), cp8(dst + NP + k * 64 + tid, b + base + 64 * k);
        cp_commit();
    };
    fetch(0);

    const double hx = h3[3 * ec], hy = h3[3 * ec + 1], hz = h3[3 * ec + 2];
    const double sx = 2.0 / hx, sy = 2.0 / hy, sz = 2.0 / hz, jac = 0.125 * hx * hy * hz;
    // Wbar and 1 / Wbar of the thread's nodes: shared memory (read back by the same thread in every job)
#pragma unroll
    for (int k = 0; k < N; ++k) {
        const double w = Wbar[base + 64 * k];
        sWb[k * 64 + tid] = w;
        sRw[k * 64 + tid] = 1.0 / w;
    }

    // ---- pass 1: the correction flux sum_k f_k
    {
        double fcx[N], fcy[N], fcz[N];
#pragma unroll
        for (int k = 0; k < N; ++k) fcx[k] = fcy[k] = fcz[k] = 0.0;
        for (int job = 0; job < Ns; ++job) {
            fetch(job + 1);
            cp_wait<1>();
            const double Ws = __ldg(m.W + job), rWs = __ldg(m.rW + job);
            const double *st = sStage + (size_t)(job & 1) * 2 * NP;
            double u[N];
#pragma unroll
            for (int k = 0; k < N; ++k) u[k] = st[k * 64 + tid] * sWb[k * 64 + tid] * rWs;
            __syncthreads();  // (the previous job is done with sU)
#pragma unroll
            for (int k = 0; k < N; ++k) sU[k * 64 + tid] = u[k];
            __syncthreads();
            auto level = [&](auto K) {
                constexpr int k = decltype(K)::value;
                double gr, gs, gt;
                grad_level<k>(sU, t, i, j, u, gr, gs, gt);
                const double c = Ws * st[NP + k * 64 + tid] * sRw[k * 64 + tid];
                fcx[k] = fma(c * sx, gr, fcx[k]);
                fcy[k] = fma(c * sy, gs, fcy[k]);
                fcz[k] = fma(c * sz, gt, fcz[k]);
            };
            for_levels(level);
        }
#pragma unroll
        for (int k = 0; k < N; ++k) sFx[k * 64 + tid] = fcx[k], sFy[k * 64 + tid] = fcy[k], sFz[k * 64 + tid] = fcz[k];
    }

    // ---- pass 2: j_k = -f_k + Y_k sum f and its weak divergence; last job: the heat flux
#pragma unroll
    for (int q = 0; q < N; ++q) t.tI[q] = cD[q * N + i], t.tJ[q] = cD[q * N + j];
    const double wij = cW[i] * cW[j] * jac;
    for (int job = Ns; job < njobs; ++job) {
        if (job + 1 < njobs) {
            fetch(job + 1);
            cp_wait<1>();
        } else {
            cp_wait<0>();
        }
        const bool heat = job == 2 * Ns;
        const int s = job - Ns;
        const double Ws = heat ? 1.0 : __ldg(m.W + s), rWs = heat ? 1.0 : __ldg(m.rW + s);
        const double *st = sStage + (size_t)(job & 1) * 2 * NP;
        double u[N];
#pragma unroll
        for (int k = 0; k < N; ++k) u[k] = heat ? st[k * 64 + tid] : st[k * 64 + tid] * sWb[k * 64 + tid] * rWs;
        __syncthreads();  // (the previous job is done with sU, sA, sB)
#pragma unroll
        for (int k = 0; k < N; ++k) sU[k * 64 + tid] = u[k];
        __syncthreads();
        double az[N];
        auto level = [&](auto K) {
            constexpr int k = decltype(K)::value;
            double gr, gs, gt;
            grad_level<k>(sU, t, i, j, u, gr, gs, gt);
            const double a = st[k * 64 + tid], b = st[NP + k * 64 + tid];
            const double y = heat ? 0.0 : a, c = heat ? b : Ws * b * sRw[k * 64 + tid];
            const double wq = wij * cW[k];
            // (both: minus the gradient flux; species: plus Y_k times the correction flux)
            const double jx = fma(y, sFx[k * 64 + tid], -(c * sx) * gr);
            const double jy = fma(y, sFy[k * 64 + tid], -(c * sy) * gs);
            const double jz = fma(y, sFz[k * 64 + tid], -(c * sz) * gt);
            sA[k * 64 + tid] = jx * (wq * sx);
            sB[k * 64 + tid] = jy * (wq * sy);
            az[k] = jz * (wq * sz);
        };
        for_levels(level);
        __syncthreads();
        double out[N];
        weak_div(sA, sB, t, i, j, az, out);
        if (live) {
            double *dst = heat ? dT : dY + (int64_t)s * n;
#pragma unroll
            for (int k = 0; k < N; ++k) dst[base + 64 * k] = out[k];
        }
    }
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
    const size_t smem = sizeof(double) * EPB * 12 * NP;
    if ((e = cudaFuncSetAttribute(sem_diffusion_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem)) != cudaSuccess) return e;
    sem_diffusion_kernel<<<(unsigned)((nel + EPB - 1) / EPB), 64 * EPB, smem, st>>>(m, h3, T, Wbar, Y, lam, rhoD, nel, dY, dT);
    crf_count_launch();
    return cudaGetLastError();
}
