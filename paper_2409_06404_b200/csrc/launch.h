// launch.h -- host-side launchers of the kernels (one per public call), private to libcrf.so.
#pragma once
#include "crf_internal.h"

void crf_count_launch();

cudaError_t launch_thermo(const DevTables &m, const double *T, const double *Y, int64_t n, double *cp, double *h,
                          cudaStream_t st);
cudaError_t launch_thermo_species(const DevTables &m, const double *T, int64_t n, double *cpk, double *hk, double *sk,
                                  cudaStream_t st);
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
cudaError_t launch_rates_group(const DevTables &m, const double *T, const double *p, const double *Y, int64_t n,
                               double *omega, double *qdot, cudaStream_t st);
cudaError_t launch_fp64_probe(int iters, double *inst_per_s);
// dynamic shared memory per block of the kernel the plan selects (0 for the generic kernels' own sizing): crf_plan_info
size_t rates_dynamic_smem(const DevTables &m);
size_t transport_dynamic_smem(const DevTables &m);
size_t rates_smem_dynamic_smem(const DevTables &m);
size_t rates_group_dynamic_smem(const DevTables &m);
size_t rates_staged_dynamic_smem(const DevTables &m);
size_t transport_tiled_dynamic_smem(const DevTables &m);
size_t transport_small_dynamic_smem(const DevTables &m);
