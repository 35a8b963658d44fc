// crf_internal.h -- device-side mechanism tables and small device helpers shared by the kernels.
// Private to libcrf.so (the public boundary is include/crf.h).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#define CRF_R_GAS 8314.46261815324  // J/(kmol K)

// Device-resident tables, re-laid-out by crf_mech_create from crf_tables.
// All pointers are device pointers into one allocation owned by crf_mech.
struct DevTables {
    int Ns, Nr, Ne, N3, Nt;  // Ne = Nr - N3 - Nt elementary reactions come first
    int npair;               // Ns (Ns+1)/2
    double p_ref;

    const double *W;     // [Ns]
    const double *rW;    // [Ns]  1/W
    const double *Tmid;  // [Ns]
    // NASA-7 in the forms the kernels evaluate, [2][.][Ns] (range 0 = low, 1 = high):
    //   cpc[5]: cp/R   = c0 + T (c1 + T (c2 + T (c3 + T c4)))
    //   hc[6]:  h/(RT) = c0 + T (c1 + T (c2 + T (c3 + T c4))) + c5/T        (c_i = a_{i+1}/(i+1))
    //   gc[7]:  g/(RT) = c0 (1 - ln T) + T (c1 + T (c2 + T (c3 + T c4))) + c5/T + c6
    //                    (c1..c4 = -a2/2, -a3/6, -a4/12, -a5/20; c5 = a6; c6 = -a7)
    const double *cpc, *hc, *gc, *sc;  // sc[6]: s/R = c0 ln T + T(c1 + ...c4) + c5
    // reactions (sorted elementary | third-body | falloff)
    const double *lnA, *beta, *Ea_R, *dnu;  // [Nr]; dnu = sum nu'' - sum nu'
    const int16_t *reac, *prod;             // [3][Nr]
    const int32_t *eff_ptr;                 // [N3+Nt+1]
    const int16_t *eff_idx;
    const double *eff_val;
    const double *lnA0, *beta0, *Ea0_R, *alpha, *rT3, *rT1, *T2;  // [Nt]; rT3 = 1/T3, rT1 = 1/T1
    // transport
    const double *mu_c, *lam_c;  // [4][Ns]
    const double *nDc;           // [npair][4]  NEGATED D_jk fit, pair-major: exp gives 1/D_jk(p_ref)
    const double *wilke_c;       // [Ns][Ns]    c_kj = 1/sqrt(8 (1 + W_k/W_j))
    const double *wq;            // [Ns]        W_k^(-1/4)
};

__device__ __forceinline__ int crf_pair_index(int j, int k, int ns)
{  // j <= k
    return j * ns - (j * (j - 1)) / 2 + (k - j);
}
