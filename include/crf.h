/* crf.h -- C ABI of libcrf.so: pointwise thermochemistry and mixture-averaged transport
 * for reactive low-Mach flow (the data-parallel hot path of arXiv 2409.06404, nekCRF),
 * evaluated by hand-written sm_100a CUDA kernels.
 *
 * What the calls compute.  The paper's right-hand-side function "employs highly optimized
 * kernels for ... species production rates, and thermodynamic and transport properties"
 * generated from "a combustion model expressed in Cantera format"; the
 * quantities are the ones Eq. 1a-1d consume (omega_k, h_k, c_p, lambda, rho)
 * and the mixture-averaged D_k of Eq. 2 and mu of Eq. 4.  The
 * paper prints none of the formulas; the definitions are the Chemkin-II/Cantera ones in the
 * reading of SURVEY.md section 8(c), restated in DESIGN.md "What the path computes".
 *
 * Conventions (all calls).
 *  - SI units with kmol.  R = 8314.46261815324 J/(kmol K).
 *  - Field arguments are DEVICE pointers owned by the caller, except in crf_step_host.
 *    T[n], p[n]: temperature [K] and thermodynamic pressure [Pa] per point.
 *    Y[Ns*n]: mass fractions, species-major: Y[k*n + i] (one contiguous field per species,
 *    the element-lexicographic field layout of PAPER.md:213).  Y carries all Ns species
 *    (the caller fills the excess species); it is used as given: never
 *    clipped, never renormalised.
 *  - Every pointer must be 16-byte aligned; inputs must not alias outputs.  n >= 0 is the
 *    number of points; n = 0 is a no-op.  Odd n is accepted (scalar tail).
 *  - Calls are asynchronous on the mechanism's stream (crf_mech_set_stream, default: the
 *    legacy default stream) and do not synchronise.
 *  - Return 0 (CRF_OK) or a negative code; crf_last_error() gives the text of the last
 *    failure on the calling thread.  No C++ exception crosses this boundary.
 *  - Validated input range: 250 K <= T <= 5000 K, p > 0, finite Y.  crf_mech_create admits the
 *    fast form of the equilibrium constant (a product of per-species factors instead of a second
 *    exponential per reaction) only if every factor stays inside the double range over that
 *    temperature window; otherwise it selects the log-space kernel by itself.  Outside the
 *    window (and for non-finite inputs or T <= 0, which are not checked) outputs are
 *    unspecified: rate constants that underflow are flushed towards zero, nothing traps.
 *  - Kernel plans (warps per point group, chunk sizes, which kernel variant) are chosen by
 *    crf_mech_create from the mechanism's size; no environment variable is read.  Explicit
 *    plan options and the diagnostics live in crf_diag.h.
 */
#ifndef CRF_H
#define CRF_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define CRF_OK 0
#define CRF_EINVAL (-1)       /* null or misaligned pointer, negative n, inconsistent tables */
#define CRF_EUNSUPPORTED (-2) /* mechanism too large for the compiled kernels */
#define CRF_ECUDA (-3)        /* CUDA allocation/launch failure (text in crf_last_error) */

#define CRF_TABLES_VERSION 1
#define CRF_MAX_SLOTS 3 /* reactant (and product) slots per reaction */
#define CRF_MAX_SPECIES 220 /* largest Ns crf_mech_create accepts (per-point state in shared memory) */

/* Host-side species-major SoA mechanism tables, produced by the packer
 * (paper_2409_06404_b200/packer.py) from a mechanism description.  All pointers are HOST
 * pointers; crf_mech_create copies what it needs, the caller may free them afterwards.
 *
 * Reactions are sorted by type: [0, Nr-N3-Nt) elementary, then N3 third-body, then Nt Troe
 * falloff.  Rate constants are in SI-kmol units and stored as logarithms:
 * k = exp(lnA + beta ln T - Ea_R / T).  All reactions are reversible; the reverse constant
 * is k_f / K_c with K_c = exp(-sum_k nu_k g_k/(RT)) (p_ref/(RT))^dnu. */
typedef struct crf_tables {
    int32_t version; /* CRF_TABLES_VERSION */
    int32_t Ns;      /* species */
    int32_t Nr;      /* reactions */
    int32_t N3;      /* third-body reactions (both rates of progress multiplied by [M]) */
    int32_t Nt;      /* Troe falloff reactions */
    int32_t reserved;
    double p_ref; /* Pa: standard pressure of the NASA entropies and of the D_jk fits */

    const double *W;       /* [Ns]    molar mass, kg/kmol */
    const double *Tmid;    /* [Ns]    NASA range switch: T <= Tmid uses nasa_lo */
    const double *nasa_lo; /* [7][Ns] a1..a7, coefficient-major: nasa_lo[c*Ns + k] */
    const double *nasa_hi; /* [7][Ns] */

    const double *lnA;  /* [Nr] (falloff: high-pressure limit) */
    const double *beta; /* [Nr] */
    const double *Ea_R; /* [Nr] K */
    const int16_t *reac; /* [CRF_MAX_SLOTS][Nr] reactant species per slot, -1 = empty;
                            a species listed twice has stoichiometric coefficient 2 */
    const int16_t *prod; /* [CRF_MAX_SLOTS][Nr] product species per slot */

    /* third-body efficiencies, CSR over the N3+Nt reactions that have a third body, in the
     * sorted order: [M]_r = sum_k C_k + sum_{e in row r} eff_val[e] * C_{eff_idx[e]},
     * eff_val = efficiency - 1 */
    const int32_t *eff_ptr; /* [N3+Nt+1] */
    const int16_t *eff_idx; /* [eff_ptr[N3+Nt]] */
    const double *eff_val;  /* [eff_ptr[N3+Nt]] */

    /* Troe falloff, one entry per falloff reaction: low-pressure limit k0 and
     * F_cent = (1-alpha) exp(-T/T3) + alpha exp(-T/T1) + exp(-T2/T).  T3 and T1 must be non-zero
     * (CRF_EINVAL otherwise); the Chemkin conventions T3 = 1e-30, T1 = 1e30 and a missing fourth
     * parameter written as T2 = 1e30 or +inf are accepted (the terms evaluate to 0, alpha and 0). */
    const double *lnA0, *beta0, *Ea0_R, *alpha, *T3, *T1, *T2; /* [Nt] each */

    /* transport fits, natural-log cubics in ln T: ln f = c[0] + c[1] x + c[2] x^2 + c[3] x^3 */
    const double *mu_c;  /* [4][Ns]            ln(mu_k / Pa s) */
    const double *lam_c; /* [4][Ns]            ln(lambda_k / (W/m/K)) */
    const double *D_c;   /* [4][Ns(Ns+1)/2]    ln(D_jk / (m^2/s)) at p_ref, upper triangle incl.
                            the diagonal, pair (j <= k) at j*Ns - j(j-1)/2 + (k - j) */
} crf_tables;

typedef struct crf_mech crf_mech; /* opaque; owns the device copies of all tables */

/* Builds the device-resident mechanism (tables re-laid-out for the kernels and uploaded to
 * the current CUDA device).  Returns CRF_EINVAL for inconsistent tables (bad version, species
 * index out of range, no reactant, W <= 0 ...), CRF_EUNSUPPORTED if Ns exceeds what the
 * kernels support (CRF_MAX_SPECIES), CRF_ECUDA on allocation failure.  *out is set only on success. */
int crf_mech_create(const crf_tables *tables, crf_mech **out);
void crf_mech_destroy(crf_mech *mech);

/* cuda_stream is a cudaStream_t (e.g. torch.cuda.current_stream().cuda_stream); NULL = default. */
int crf_mech_set_stream(crf_mech *mech, void *cuda_stream);
int crf_mech_num_species(const crf_mech *mech);
int crf_mech_num_reactions(const crf_mech *mech);

/* NASA-7 mixture thermodynamics (c_p and h_k of Eq. 1b).
 *   cp[n]  mixture heat capacity  sum_k Y_k c_{p,k}/W_k          [J/(kg K)]
 *   h[n]   mixture enthalpy       sum_k Y_k h_k/W_k              [J/kg]
 * p is accepted for uniformity and not read (may be NULL). */
int crf_thermo(const crf_mech *mech, const double *T, const double *p, const double *Y, int64_t n,
               double *cp, double *h);

/* Per-species molar properties (the c_{p,k}, h_k of Eq. 1b): cpk, hk, sk are [Ns*n] species-major,
 * J/(kmol K), J/kmol, J/(kmol K); any of the three may be NULL. */
int crf_thermo_species(const crf_mech *mech, const double *T, int64_t n, double *cpk, double *hk, double *sk);

/* Net molar production rates from finite-rate chemistry and the heat release
 * (omega_k of Eq. 1a and the source of Eq. 1b).
 *   omega[Ns*n]  sum_r nu_kr (Q_f - Q_r)       [kmol/(m^3 s)], species-major
 *   qdot[n]      -sum_k h_k(T) omega_k          [W/m^3], positive when exothermic */
int crf_production_rates(const crf_mech *mech, const double *T, const double *p, const double *Y, int64_t n,
                         double *omega, double *qdot);

/* Mixture-averaged transport (lambda of Eq. 1b, D_k of Eq. 2,
 * mu of Eq. 4).
 *   mu[n]        Wilke mixture viscosity                                   [Pa s]
 *   lambda[n]    (sum X_k lambda_k + 1/sum X_k/lambda_k)/2                 [W/(m K)]
 *   rhoD[Ns*n]   rho D_km, D_km = (1 - Y_k)/sum_{j!=k} X_j/D_jk, D_jk ~ p_ref/p; a pure
 *                species (sum exactly 0) gives rho D_kk                    [kg/(m s)] */
int crf_mix_transport(const crf_mech *mech, const double *T, const double *p, const double *Y, int64_t n,
                      double *mu, double *lambda, double *rhoD);

/* Everything one evaluation of the right-hand side consumes at a grid point, in one call.  "The
 * right-hand side (RHS) function, evaluated in each Newton step and linear iteration, employs ... kernels for ...
 * species production rates, and thermodynamic and transport properties": omega_k and the heat release
 * of Eq. 1a-1b, c_p and c_{p,k} of Eq. 1b-1c, rho of Eq. 1d, the
 * mean molar mass, lambda, D_k (Eq. 2) and mu (Eq. 4).  The outputs shared
 * with crf_thermo, crf_production_rates and crf_mix_transport are defined as there; in addition
 *   cpk[Ns*n]  molar c_{p,k}, species-major              [J/(kmol K)]   (may be NULL)
 *   rho[n]     p Wbar / (R T)                            [kg/m^3]
 *   Wbar[n]    1 / sum_k Y_k / W_k                       [kg/kmol]
 * The thermodynamic outputs are by-products of the production-rates kernel (no separate pass over Y); transport is
 * a second kernel on the same stream.  Mechanisms without a warp-group rates plan take the separate kernels. */
int crf_rhs_pointwise(const crf_mech *mech, const double *T, const double *p, const double *Y, int64_t n, double *omega,
                      double *qdot, double *cp, double *h, double *cpk, double *rho, double *Wbar, double *mu,
                      double *lambda, double *rhoD);

/* Production rates at TWO states of the same n points in one launch: the matrix-free Newton-Krylov
 * solver of the paper approximates Jacobian-vector products by difference quotients, so the rates
 * are wanted at y and at a perturbed y' = y + sigma v.  Both states of a point share a lane of the kernel: mechanism
 * tables, reaction records and incidence lists are read once for the two evaluations.  Results are bit-identical to
 * two crf_production_rates calls whenever both run the same kernel.  (T2, p2, Y2) -> (omega2, qdot2). */
int crf_production_rates_pair(const crf_mech *mech, const double *T, const double *p, const double *Y, const double *T2,
                              const double *p2, const double *Y2, int64_t n, double *omega, double *qdot, double *omega2,
                              double *qdot2);

/* The difference quotient itself: the perturbed state y' = (T + sigma dT, p + sigma dp, Y + sigma dY) is formed in
 * the kernel (multiply, then add: one rounding each, as a host would), both states are evaluated in one launch and
 *   Jomega[Ns*n] = (omega(y') - omega(y)) (1/sigma),   Jqdot[n] = (qdot(y') - qdot(y)) (1/sigma)
 * are returned next to omega(y), qdot(y) (omega and qdot may both be NULL).  dp may be NULL (no pressure
 * perturbation).  sigma must be finite and non-zero.  Each value of the quotient carries the rounding of two
 * evaluations divided by sigma: its tolerance scale is (S(y) + S(y')) / |sigma|.  CRF_EUNSUPPORTED for a mechanism
 * whose plan cannot hold two states per lane (explicit one-point-per-lane or fall-back kernels). */
int crf_production_rates_jv(const crf_mech *mech, const double *T, const double *p, const double *Y, const double *dT,
                            const double *dp, const double *dY, double sigma, int64_t n, double *omega, double *qdot,
                            double *Jomega, double *Jqdot);

/* The same difference quotient when omega(y) and qdot(y) are known already, which is how an integrator calls it: CVODE's
 * matrix-free Newton-Krylov iteration forms J v = (f(y + sigma v) - f(y)) / sigma with f(y) in hand, and
 * the Jacobian-vector products are most of the right-hand-side evaluations of a step.  omega[Ns*n] and
 * qdot[n] are INPUTS here (the values crf_production_rates returned for (T, p, Y)); only the perturbed state is
 * evaluated, at the cost of one crf_production_rates call:
 *   Jomega = (omega(y') - omega) (1/sigma),   Jqdot = (qdot(y') - qdot) (1/sigma),   y' as in crf_production_rates_jv
 * (bit for bit what crf_production_rates_jv returns for the same base values).  dp may be NULL.  CRF_EUNSUPPORTED for a
 * mechanism that runs a fall-back kernel. */
int crf_production_rates_jv_base(const crf_mech *mech, const double *T, const double *p, const double *Y, const double *dT,
                                 const double *dp, const double *dY, double sigma, int64_t n, const double *omega,
                                 const double *qdot, double *Jomega, double *Jqdot);

/* The element-local spectral-element diffusion operator on what crf_rhs_pointwise emits: "diffusion"
 * is the most expensive kernel of the paper's right-hand side.  The fields live on nel hexahedral
 * elements of polynomial order 7: n = 512 nel points, node (i, j, k) of element e at
 * 512 e + i + 8 j + 64 k (i along x fastest) = the 8 x 8 x 8 Gauss-Lobatto-Legendre points of the element, which is an
 * affine box of edge lengths h3[3 e + 0..2] = (hx, hy, hz) [m] (h3: device pointer, nel x 3).  With
 *   X_k = Y_k Wbar / W_k,   f_k = (W_k / Wbar) (rho D_k) grad X_k,   j_k = -f_k + Y_k sum_j f_j
 * (j_k = rho Y_k V_k of Eq. 2 with the correction velocity V_c, written without the division by X_k)
 *   dY[Ns*n]  dY_k[i] = sum_q w_q |J| grad phi_i(x_q) . j_k(x_q)               weak form of -div(rho Y_k V_k), Eq. 1a
 *   dT[n]     dT[i]   = -sum_q w_q |J| grad phi_i(x_q) . (lambda grad T)(x_q)   weak form of div(lambda grad T), Eq. 1b
 * with the nodal basis phi_i and GLL quadrature, element by element: no gather-scatter across elements, no boundary
 * terms and no inverse mass matrix (the assembly steps of the solver).  Units: kg/s and W per node. */
int crf_sem_diffusion(const crf_mech *mech, const double *h3, const double *T, const double *Wbar, const double *Y,
                      const double *lambda, const double *rhoD, int64_t nel, double *dY, double *dT);

/* One pass of the whole path with HOST buffers: copies T, p, Y to the device in chunks, runs
 * crf_thermo, crf_production_rates and crf_mix_transport on each chunk and copies the seven
 * outputs back, chunks pipelined over internal streams.  All pointers are host pointers with
 * the layouts above (species-major with leading dimension n); pinned memory gives full copy
 * bandwidth.  Synchronous: returns when every output is in host memory.  The outputs of one call form a group,
 * (cp, h), (omega, qdot), (mu, lambda, rhoD): a group whose pointers are all NULL is neither computed nor copied (a
 * Jacobian-vector product needs omega and qdot only: a third of the device-to-host traffic); a partly given group or
 * no group at all is CRF_EINVAL. */
int crf_step_host(crf_mech *mech, const double *T, const double *p, const double *Y, int64_t n,
                  double *cp, double *h, double *omega, double *qdot, double *mu, double *lambda, double *rhoD);

/* Mixed-precision variant of crf_step_host: every step of the path is computed in double precision on the device, the
 * OUTPUTS are rounded once (to nearest) to single precision on the device and returned as float arrays of the same
 * layouts: half the device-to-host traffic of the end-to-end leg, which that traffic bounds.  This is the
 * storage-in-reduced-precision technique the paper applies to its Krylov basis (FP32 basis, FP64 arithmetic,
 * PAPER.md:59) and names as ongoing work, applied to what this library returns to a host-side
 * consumer.  Each value is the float nearest to what crf_step_host returns.  Output groups as in crf_step_host. */
int crf_step_host_f32(crf_mech *mech, const double *T, const double *p, const double *Y, int64_t n, float *cp, float *h,
                      float *omega, float *qdot, float *mu, float *lambda, float *rhoD);

/* crf_step_host for callers that may not allocate (code under CUDA graph capture, serving loops, harnesses that forbid
 * cudaMalloc): the same path, host pointers, layouts and output groups as crf_step_host, but the device staging of the
 * batch lives in a 16 MiB array that is part of the library's device image (every GPU that loads libcrf.so holds it
 * until the process exits), and the work runs on the mechanism's stream (crf_mech_set_stream).  The call creates no
 * stream and calls no cudaMalloc, cudaFree or other allocating routine; its only set-up is the address lookup of that
 * array, once per device, on the first call there (with that device current, as for every call of a mechanism).
 *   Limit: 7 ceil32(n) + 3 ceil32(Ns n) <= 2 097 152 doubles (ceil32: rounded up to a multiple of 32), i.e. about
 *   2 097 152 / (7 + 3 Ns) points per call: 61 674 at Ns = 9, 5 808 at Ns = 118; crf_step_host_static_max_points
 *   gives the exact number for a mechanism.  A larger n is CRF_EINVAL (crf_last_error names the limit); nothing runs.
 * The array is shared by every call on the device, of any mechanism, and keeps the last call's contents (no part of it
 * has to start at zero: a call writes every row before it reads it): calls that overlap on the GPU (other host threads
 * or streams) race and must be serialised by the caller.  Synchronous: returns when the outputs are in host memory.
 * Values are those of the device calls on a batch of n points (bit for bit those of crf_step_host for n <= 65 536). */
int crf_step_host_static(crf_mech *mech, const double *T, const double *p, const double *Y, int64_t n, double *cp, double *h,
                         double *omega, double *qdot, double *mu, double *lambda, double *rhoD);
/* the largest n crf_step_host_static accepts for this mechanism (negative: error code) */
int64_t crf_step_host_static_max_points(const crf_mech *mech);

const char *crf_last_error(void);

#ifdef __cplusplus
}
#endif
#endif /* CRF_H */
