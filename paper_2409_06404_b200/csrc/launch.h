// launch.h -- host-side launchers of the kernels (one per public call), private to libcrf.so.
#pragma once
#include "crf_internal.h"

void crf_count_launch();

// What one launch of the production-rates kernels reads and writes (device pointers).
//   mode 0  omega, qdot at (T, p, Y); optionally the thermodynamic by-products of the same pass (crf_rhs_pointwise)
//   mode 1  two states of the same points in one launch: (T, p, Y) -> omega, qdot and (T2, p2, Y2) -> omega2, qdot2
//   mode 2  difference quotient: second state = (T, p, Y) + (sigma T2, sigma_p p2, sigma Y2) formed in the kernel;
//           omega, qdot of the base state (may be null) and omega2, qdot2 = (f(second) - f(base)) (1/sigma)
struct RatesIO {
    const double *T, *p, *Y;
    const double *T2, *p2, *Y2;
    double sigma, sigma_p, inv_sigma;  // (sigma_p: the step applied to p2; 0 when the caller gave no dp)
    int mode;
    double *omega, *qdot;
    double *omega2, *qdot2;
    double *cp, *h, *cpk, *rho, *Wbar;  // mode 0 only, any may be null: mixture c_p, h; molar c_pk [Ns*n]; rho; Wbar
};
inline RatesIO rates_io(const double *T, const double *p, const double *Y, double *omega, double *qdot)
{
    RatesIO io{};
    io.T = T, io.p = p, io.Y = Y, io.omega = omega, io.qdot = qdot;
    io.T2 = T, io.p2 = p, io.Y2 = Y;  // (never null: the kernels form row pointers from them in every mode)
    return io;
}

cudaError_t launch_thermo(const DevTables &m, const double *T, const double *Y, int64_t n, double *cp, double *h,
                          cudaStream_t st);
cudaError_t launch_thermo_species(const DevTables &m, const double *T, int64_t n, double *cpk, double *hk, double *sk,
                                  cudaStream_t st);
cudaError_t launch_density(const DevTables &m, const double *T, const double *p, const double *Y, int64_t n, double *rho,
                           double *Wbar, cudaStream_t st);
cudaError_t launch_rates(const DevTables &m, const double *T, const double *p, const double *Y, int64_t n,
                         double *omega, double *qdot, cudaStream_t st);
cudaError_t launch_transport(const DevTables &m, const double *T, const double *p, const double *Y, int64_t n,
                             double *mu, double *lambda, double *rhoD, cudaStream_t st);
cudaError_t launch_transport_tiled(const DevTables &m, const double *T, const double *Y, int64_t n, double *mu,
                                   double *lambda, double *rhoD, cudaStream_t st);
cudaError_t launch_transport_small(const DevTables &m, const double *T, const double *Y, int64_t n, double *mu,
                                   double *lambda, double *rhoD, cudaStream_t st);
cudaError_t launch_rates_staged(const DevTables &m, const double *T, const double *p, const double *Y, int64_t n,
                                double *omega, double *qdot, cudaStream_t st);
cudaError_t launch_rates_smem(const DevTables &m, const double *T, const double *p, const double *Y, int64_t n,
                              double *omega, double *qdot, cudaStream_t st);
cudaError_t launch_rates_group(const DevTables &m, const RatesIO &io, int64_t n, cudaStream_t st);
bool rates_thread_tm_serves(const DevTables &m, const RatesIO &io);
cudaError_t launch_rates_thread_io(const DevTables &m, const RatesIO &io, int64_t n, cudaStream_t st);
cudaError_t launch_sem_diffusion(const DevTables &m, const double *h3, const double *T, const double *Wbar, const double *Y,
                                 const double *lam, const double *rhoD, int64_t nel, double *dY, double *dT, cudaStream_t st);
cudaError_t launch_fp64_probe(int iters, double *inst_per_s);
cudaError_t launch_f64_to_f32(const double *in, float *out, int64_t count, cudaStream_t st);
// dynamic shared memory per block of the kernel the plan selects (0 for the generic kernels' own sizing): crf_plan_info
size_t rates_dynamic_smem(const DevTables &m);
size_t transport_dynamic_smem(const DevTables &m);
size_t rates_smem_dynamic_smem(const DevTables &m);
size_t rates_group_dynamic_smem(const DevTables &m);
size_t rates_staged_dynamic_smem(const DevTables &m);
size_t transport_tiled_dynamic_smem(const DevTables &m);
size_t transport_small_dynamic_smem(const DevTables &m);
