/* crf_oracle.c -- TEST INFRASTRUCTURE, NOT PRODUCT.
 *
 * Plain, slow, double-precision CPU statement of what the hot path computes at one
 * grid point: NASA-7 thermodynamics, finite-rate net production rates with heat
 * release, and mixture-averaged transport.  One point at a time, straightforward
 * dense loops, libm exp/log/pow/log10/sqrt, no blocking, no fusion, no log-space
 * rewrites.  It shares no code, header, table or constant generator with the CUDA
 * path (paper_2409_06404_b200/csrc) and reads the mechanism *description* (dense
 * stoichiometry, cgs Arrhenius data), never the packed tables.  Only tests/,
 * __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may
 * use it.
 *
 * What it follows.  The paper names the models and prints none of their formulas:
 * "finite rate chemistry, mixture-averaged transport", "species
 * production rates, and thermodynamic and transport properties" generated from "a
 * combustion model expressed in Cantera format", with the consumers
 * Eq. 1a-d (omega_k, h_k, c_p, c_{p,k}, lambda, rho) and Eq. 2
 * (D_k, X_k).  The definitions written out below are the standard
 * Chemkin-II / Cantera ones those names refer to, in the reading
 * fixed by SURVEY.md section 8(c) steps 1-13 and listed in DESIGN.md "Readings".
 * Each function cites its step.
 *
 * Parity with the paper's own kernels / Cantera / Chemkin: PARITY UNPINNED (no
 * formulas, code, mechanism file or Cantera in the container).  The formulas
 * themselves are pinned by closed forms, invariants and special cases in
 * tests/test_oracle_*.py.
 *
 * Layout: T[n], p[n]; Y, omega, rhoD are species-major A[k*n + i]; SI units with
 * kmol (omega kmol/m^3/s, qdot W/m^3, cp J/kg/K, h J/kg, mu Pa s, lambda W/m/K,
 * rhoD kg/m/s).
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#ifdef _OPENMP
#include <omp.h>
#endif

#define R_GAS 8314.46261815324 /* J/(kmol K) */

typedef struct {
    int Ns, Nr;
    const double *W;       /* [Ns]      kg/kmol                                    */
    const double *Tmid;    /* [Ns]      K                                          */
    const double *nasa_lo; /* [Ns][7]   a1..a7 for T <= Tmid                       */
    const double *nasa_hi; /* [Ns][7]   a1..a7 for T >  Tmid                       */
    const double *nu_f;    /* [Nr][Ns]  reactant coefficients nu'                  */
    const double *nu_r;    /* [Nr][Ns]  product coefficients nu''                  */
    const int *type;       /* [Nr]      0 elementary, 1 three-body, 2 Troe falloff */
    const double *A;       /* [Nr]      cgs-mol (falloff: high-pressure limit)     */
    const double *beta;    /* [Nr]                                                 */
    const double *Ea;      /* [Nr]      kJ/mol                                     */
    const double *eff;     /* [Nr][Ns]  third-body efficiencies (1 unless listed)  */
    const double *A0, *beta0, *Ea0;      /* [Nr] low-pressure limit (type 2)       */
    const double *alpha, *T3, *T1, *T2;  /* [Nr] Troe alpha, T***, T*, T**         */
    const double *mu_fit;  /* [Ns][4]     ln mu_k     = sum_m c_m (ln T)^m         */
    const double *lam_fit; /* [Ns][4]     ln lambda_k                              */
    const double *D_fit;   /* [Ns][Ns][4] ln D_jk at p_ref                         */
    double p_ref;          /* Pa */
} oracle_mech;

int oracle_max_threads(void)
{
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

/* ---- step 2: NASA-7, one species ----------------------------------------------------
 * cp/R   = a1 + a2 T + a3 T^2 + a4 T^3 + a5 T^4
 * h/(RT) = a1 + a2 T/2 + a3 T^2/3 + a4 T^3/4 + a5 T^4/5 + a6/T
 * s/R    = a1 ln T + a2 T + a3 T^2/2 + a4 T^3/3 + a5 T^4/4 + a7
 * low set for T <= Tmid, no clamping outside the fit range (SURVEY 8(c) readings). */
static void nasa7(const oracle_mech *m, int k, double T, double *cp_R, double *h_RT, double *s_R)
{
    const double *a = (T <= m->Tmid[k]) ? m->nasa_lo + 7 * k : m->nasa_hi + 7 * k;
    double T2 = T * T, T3 = T2 * T, T4 = T3 * T;
    *cp_R = a[0] + a[1] * T + a[2] * T2 + a[3] * T3 + a[4] * T4;
    *h_RT = a[0] + a[1] * T / 2.0 + a[2] * T2 / 3.0 + a[3] * T3 / 4.0 + a[4] * T4 / 5.0 + a[5] / T;
    *s_R = a[0] * log(T) + a[1] * T + a[2] * T2 / 2.0 + a[3] * T3 / 3.0 + a[4] * T4 / 4.0 + a[6];
}

/* per-species molar cp [J/kmol/K], h [J/kmol], s [J/kmol/K], g/(RT) [-] at each T */
void oracle_thermo_species(const oracle_mech *m, const double *T, int64_t n,
                           double *cpk, double *hk, double *sk, double *g_RT)
{
    for (int64_t i = 0; i < n; ++i)
        for (int k = 0; k < m->Ns; ++k) {
            double c, h, s;
            nasa7(m, k, T[i], &c, &h, &s);
            if (cpk) cpk[k * n + i] = c * R_GAS;
            if (hk) hk[k * n + i] = h * R_GAS * T[i];
            if (sk) sk[k * n + i] = s * R_GAS;
            if (g_RT) g_RT[k * n + i] = h - s;
        }
}

/* ---- step 3: mixture cp [J/kg/K] and h [J/kg]: sum_k Y_k cp_k / W_k, sum_k Y_k h_k / W_k.
 * h_scale = sum_k |Y_k h_k / W_k| (the cancellation scale used by the h tolerance). */
void oracle_thermo(const oracle_mech *m, const double *T, const double *p, const double *Y,
                   int64_t n, double *cp, double *h, double *h_scale)
{
    (void)p;
#pragma omp parallel for schedule(static)
    for (int64_t i = 0; i < n; ++i) {
        double cpm = 0.0, hm = 0.0, hs = 0.0;
        for (int k = 0; k < m->Ns; ++k) {
            double c, hh, s;
            nasa7(m, k, T[i], &c, &hh, &s);
            cpm += Y[k * n + i] * (c * R_GAS) / m->W[k];
            hm += Y[k * n + i] * (hh * R_GAS * T[i]) / m->W[k];
            hs += fabs(Y[k * n + i] * (hh * R_GAS * T[i]) / m->W[k]);
        }
        cp[i] = cpm;
        h[i] = hm;
        if (h_scale) h_scale[i] = hs;
    }
}

/* Arrhenius k = A T^beta exp(-E/(R T)), A converted from cgs-mol to SI-kmol:
 * 1 cm^3/mol = 1e-3 m^3/kmol, so A_SI = A_cgs * (1e-3)^(order-1);  E[kJ/mol]*1e6 = J/kmol. */
static double arrhenius(double A_cgs, double beta, double Ea_kJ, double order, double T)
{
    double A_si = A_cgs * pow(1.0e-3, order - 1.0);
    return A_si * pow(T, beta) * exp(-(Ea_kJ * 1.0e6) / (R_GAS * T));
}

/* ---- steps 1, 2, 4-9 at one point ---------------------------------------------------
 * Yi[Ns] are the mass fractions of the point.  Outputs per reaction (may be NULL):
 * kf, kr (after falloff), Qf, Qr (incl. third-body factor), M ([M] or 0). */
static void rates_point(const oracle_mech *m, double T, double p, const double *Yi,
                        double *C, double *g_RT, double *h_mol,
                        double *omega, double *qdot, double *S_omega, double *S_q,
                        double *kf_o, double *kr_o, double *Qf_o, double *Qr_o, double *M_o)
{
    const int Ns = m->Ns, Nr = m->Nr;
    /* step 1: Wbar = 1/sum Y_k/W_k; rho = p Wbar/(R T) (Eq. 1d); C_k = rho Y_k/W_k */
    double inv_W = 0.0;
    for (int k = 0; k < Ns; ++k) inv_W += Yi[k] / m->W[k];
    double Wbar = 1.0 / inv_W;
    double rho = p * Wbar / (R_GAS * T);
    for (int k = 0; k < Ns; ++k) {
        double c, h, s;
        C[k] = rho * Yi[k] / m->W[k];
        nasa7(m, k, T, &c, &h, &s);
        g_RT[k] = h - s;
        h_mol[k] = h * R_GAS * T;
        omega[k] = 0.0;
        if (S_omega) S_omega[k] = 0.0;
    }
    for (int r = 0; r < Nr; ++r) {
        const double *nf = m->nu_f + (size_t)r * Ns, *nr = m->nu_r + (size_t)r * Ns;
        double order = 0.0, dnu = 0.0, dG = 0.0;
        for (int k = 0; k < Ns; ++k) {
            order += nf[k];
            dnu += nr[k] - nf[k];
            dG += (nr[k] - nf[k]) * g_RT[k];
        }
        /* step 5: [M] = sum_k eps_rk C_k */
        double M = 0.0;
        if (m->type[r] != 0)
            for (int k = 0; k < Ns; ++k) M += m->eff[(size_t)r * Ns + k] * C[k];
        double kf;
        if (m->type[r] == 2) {
            /* step 6: Troe falloff */
            double kinf = arrhenius(m->A[r], m->beta[r], m->Ea[r], order, T);
            double k0 = arrhenius(m->A0[r], m->beta0[r], m->Ea0[r], order + 1.0, T);
            double Pr = k0 * M / kinf;
            double Fcent = (1.0 - m->alpha[r]) * exp(-T / m->T3[r]) + m->alpha[r] * exp(-T / m->T1[r])
                           + exp(-m->T2[r] / T);
            double lFc = log10(fmax(Fcent, 1.0e-300));
            double c = -0.4 - 0.67 * lFc;
            double N = 0.75 - 1.27 * lFc;
            double lPr = log10(Pr);
            double f1 = (lPr + c) / (N - 0.14 * (lPr + c));
            double F = pow(10.0, lFc / (1.0 + f1 * f1));
            kf = kinf * (Pr / (1.0 + Pr)) * F;
        } else {
            /* step 4 (a third body adds one to the order of A's units) */
            kf = arrhenius(m->A[r], m->beta[r], m->Ea[r], order + (m->type[r] == 1 ? 1.0 : 0.0), T);
        }
        /* step 7: K_c = exp(-sum nu g/(RT)) (p_ref/(R T))^dnu ; k_r = k_f / K_c */
        double Kc = exp(-dG) * pow(m->p_ref / (R_GAS * T), dnu);
        double kr = kf / Kc;
        /* step 8: rates of progress */
        double Qf = kf, Qr = kr;
        for (int k = 0; k < Ns; ++k) {
            if (nf[k] != 0.0) Qf *= pow(C[k], nf[k]);
            if (nr[k] != 0.0) Qr *= pow(C[k], nr[k]);
        }
        if (m->type[r] == 1) {
            Qf *= M;
            Qr *= M;
        }
        double q = Qf - Qr;
        for (int k = 0; k < Ns; ++k) {
            double nu = nr[k] - nf[k];
            omega[k] += nu * q;
            if (S_omega) S_omega[k] += fabs(nu) * (fabs(Qf) + fabs(Qr));
        }
        if (kf_o) kf_o[r] = kf;
        if (kr_o) kr_o[r] = kr;
        if (Qf_o) Qf_o[r] = Qf;
        if (Qr_o) Qr_o[r] = Qr;
        if (M_o) M_o[r] = M;
    }
    /* step 9: qdot = -sum_k h_k omega_k (Eq. 1b source; iHRR) */
    double qd = 0.0, sq = 0.0;
    for (int k = 0; k < Ns; ++k) {
        qd -= h_mol[k] * omega[k];
        if (S_omega) sq += fabs(h_mol[k]) * S_omega[k];
    }
    *qdot = qd;
    if (S_q) *S_q = sq;
}

/* omega[Ns][n], qdot[n]; S_omega[Ns][n], S_q[n] are the tolerance scales (may be NULL) */
void oracle_production_rates(const oracle_mech *m, const double *T, const double *p, const double *Y,
                             int64_t n, double *omega, double *qdot, double *S_omega, double *S_q)
{
    const int Ns = m->Ns;
#pragma omp parallel
    {
        double *buf = (double *)malloc(sizeof(double) * 6 * (size_t)Ns);
        double *Yi = buf, *C = buf + Ns, *g = buf + 2 * Ns, *hm = buf + 3 * Ns, *om = buf + 4 * Ns,
               *So = buf + 5 * Ns;
#pragma omp for schedule(static)
        for (int64_t i = 0; i < n; ++i) {
            double qd, sq;
            for (int k = 0; k < Ns; ++k) Yi[k] = Y[k * n + i];
            rates_point(m, T[i], p[i], Yi, C, g, hm, om, &qd, So, &sq, 0, 0, 0, 0, 0);
            for (int k = 0; k < Ns; ++k) {
                omega[k * n + i] = om[k];
                if (S_omega) S_omega[k * n + i] = So[k];
            }
            qdot[i] = qd;
            if (S_q) S_q[i] = sq;
        }
        free(buf);
    }
}

/* one point, with the per-reaction intermediates (debugging and the closed-form pins) */
void oracle_rates_detail(const oracle_mech *m, double T, double p, const double *Yi,
                         double *omega, double *qdot, double *kf, double *kr, double *Qf, double *Qr,
                         double *M, double *C)
{
    const int Ns = m->Ns;
    double *buf = (double *)malloc(sizeof(double) * 3 * (size_t)Ns);
    double *Cb = C ? C : buf;
    rates_point(m, T, p, Yi, Cb, buf + Ns, buf + 2 * Ns, omega, qdot, 0, 0, kf, kr, Qf, Qr, M);
    free(buf);
}

static double log_cubic(const double *c, double lnT)
{
    return exp(c[0] + c[1] * lnT + c[2] * lnT * lnT + c[3] * lnT * lnT * lnT);
}

/* ---- steps 1, 10-13 -------------------------------------------------------------------
 * mu[n], lambda[n], rhoD[Ns][n]; Dkm[Ns][n] optional (m^2/s). */
void oracle_mix_transport(const oracle_mech *m, const double *T, const double *p, const double *Y,
                          int64_t n, double *mu, double *lambda, double *rhoD, double *Dkm_out)
{
    const int Ns = m->Ns;
#pragma omp parallel
    {
        double *buf = (double *)malloc(sizeof(double) * 3 * (size_t)Ns);
        double *X = buf, *muk = buf + Ns, *lamk = buf + 2 * Ns;
#pragma omp for schedule(static)
        for (int64_t i = 0; i < n; ++i) {
            double lnT = log(T[i]);
            /* step 1 */
            double inv_W = 0.0;
            for (int k = 0; k < Ns; ++k) inv_W += Y[k * n + i] / m->W[k];
            double Wbar = 1.0 / inv_W;
            double rho = p[i] * Wbar / (R_GAS * T[i]);
            for (int k = 0; k < Ns; ++k) {
                X[k] = Y[k * n + i] * Wbar / m->W[k];
                /* step 10 */
                muk[k] = log_cubic(m->mu_fit + 4 * k, lnT);
                lamk[k] = log_cubic(m->lam_fit + 4 * k, lnT);
            }
            /* step 11: Wilke.  Phi_kj = [1 + (mu_k/mu_j)^(1/2) (W_j/W_k)^(1/4)]^2 / [8 (1 + W_k/W_j)]^(1/2) */
            double mu_mix = 0.0;
            for (int k = 0; k < Ns; ++k) {
                double den = 0.0;
                for (int j = 0; j < Ns; ++j) {
                    double t = 1.0 + sqrt(muk[k] / muk[j]) * pow(m->W[j] / m->W[k], 0.25);
                    double Phi = t * t / sqrt(8.0 * (1.0 + m->W[k] / m->W[j]));
                    den += X[j] * Phi;
                }
                mu_mix += X[k] * muk[k] / den;
            }
            mu[i] = mu_mix;
            /* step 12: lambda = (sum X_k lambda_k + 1 / sum X_k/lambda_k) / 2 */
            double sa = 0.0, sh = 0.0;
            for (int k = 0; k < Ns; ++k) {
                sa += X[k] * lamk[k];
                sh += X[k] / lamk[k];
            }
            lambda[i] = 0.5 * (sa + 1.0 / sh);
            /* step 13: D_jk = exp(cubic) p_ref/p ; D_km = (1 - Y_k) / sum_{j!=k} X_j / D_jk ;
             * pure species (sum exactly 0) -> D_kk (Eq. 2 coefficient) */
            for (int k = 0; k < Ns; ++k) {
                double s = 0.0;
                for (int j = 0; j < Ns; ++j) {
                    if (j == k) continue;
                    double Djk = log_cubic(m->D_fit + 4 * ((size_t)j * Ns + k), lnT) * m->p_ref / p[i];
                    s += X[j] / Djk;
                }
                double Dkm;
                if (s == 0.0)
                    Dkm = log_cubic(m->D_fit + 4 * ((size_t)k * Ns + k), lnT) * m->p_ref / p[i];
                else
                    Dkm = (1.0 - Y[k * n + i]) / s;
                rhoD[k * n + i] = rho * Dkm;
                if (Dkm_out) Dkm_out[k * n + i] = Dkm;
            }
        }
        free(buf);
    }
}

/* ---- everything one evaluation of the right-hand side consumes at a grid point ------------------
 * "The right-hand side (RHS) function, evaluated in each Newton step and linear iteration, employs ... kernels for
 * ... species production rates, and thermodynamic and transport properties": omega_k and the heat
 * release of Eq. 1a-1b, c_p and c_{p,k} of Eq. 1b-1c, rho of Eq. 1d, the mean molar
 * mass Wbar, lambda (Eq. 1b), D_k (Eq. 2) and mu (Eq. 4).
 * A plain composition of the functions above (no shared intermediates) plus
 *   Wbar = 1 / sum_k Y_k / W_k [kg/kmol],   rho = p Wbar / (R T) [kg/m^3],   cpk = molar c_{p,k} [J/(kmol K)]. */
void oracle_rhs_pointwise(const oracle_mech *m, const double *T, const double *p, const double *Y, int64_t n,
                          double *omega, double *qdot, double *S_omega, double *S_q,
                          double *cp, double *h, double *h_scale, double *cpk, double *rho, double *Wbar,
                          double *mu, double *lambda, double *rhoD)
{
    oracle_production_rates(m, T, p, Y, n, omega, qdot, S_omega, S_q);
    oracle_thermo(m, T, p, Y, n, cp, h, h_scale);
    oracle_thermo_species(m, T, n, cpk, 0, 0, 0);
    oracle_mix_transport(m, T, p, Y, n, mu, lambda, rhoD, 0);
    for (int64_t i = 0; i < n; ++i) {
        double inv_W = 0.0;
        for (int k = 0; k < m->Ns; ++k) inv_W += Y[k * n + i] / m->W[k];
        Wbar[i] = 1.0 / inv_W;
        rho[i] = p[i] * Wbar[i] / (R_GAS * T[i]);
    }
}
