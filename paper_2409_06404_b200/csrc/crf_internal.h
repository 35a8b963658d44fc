// crf_internal.h -- device-side mechanism tables and small device helpers shared by the kernels.
// Private to libcrf.so (the public boundary is include/crf.h).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#define CRF_R_GAS 8314.46261815324  // J/(kmol K)

// Plan of the tiled crf_mix_transport kernel (transport_tiled.cu): species padded to blocks of 8, the pair
// triangle cut into 8x8 (or 7x7) tiles.  W warps share 32 PPL points; tiles are dealt to them in rounds whose tiles
// touch disjoint species blocks (round-robin tournament over the blocks: a block's bye is its diagonal
// tile), so the warps update disjoint rows of S.  A round's coefficients are one contiguous block that the
// thread block copies global -> shared with cp.async while it works on the previous round.
struct TransportPlan {
    int W;         // warps per block (1, 2, 4 or 8); 0 = no plan (generic kernel)
    int PPL;       // points per lane (1 or 2)
    int NsP, nb;   // padded species count (rows of the state) and number of 8-blocks (Wilke phase)
    int TS;        // tile edge of the pair phase: species blocks of 7 or 8
    int n_wilke;   // stage blocks of the Wilke phase (they come first in `rounds`)
    int n_rounds;  // stage blocks (rounds) of the pair phase
    int stage_bytes;          // largest stage block (multiple of 16)
    const int4 *rounds;       // [n_wilke + n_rounds] stage blocks: x = byte offset in pair_coef, y = bytes;
                              //   Wilke blocks: z = first column block | pass << 8 | first panel << 16 |
                              //   last panel << 17, w = column blocks nJ
    const unsigned char *pair_coef;  // the stage blocks.  Block = header {int4 descriptor of the next block,
                              //   int2 sched[W] (pair rounds): x = kind | jb << 8 | kb << 16 (kind 0 idle, 1 off-diagonal,
                              //   2 diagonal), y = byte offset of the tile's coefficients in the block}, padded to 16 bytes;
                              //   payload: Wilke [W][8 rows][8 nJ] of c_kj, or per pair (c0,c1,c2,c3) of the
                              //   -log2(e) ln D_jk fit (0 for padding)
    const double *wilke_cP;   // [NsP][NsP] c_kj = 1/sqrt(8 (1 + W_k/W_j)), 0 in padded rows/columns
    const double *sp;         // [NsP][12]: 0-3 -log2(e) ln(mu_k)/2 cubic, 4-7 log2(e) ln(lambda_k) cubic, 8 W^1/4, 9 W^1/2,
                              //   10 1/W (0 for padding), 11 unused
    const double *Ddiag;      // [Ns][4] ln D_kk cubic (pure-species guard)
    // mechanisms with Ns <= 16 (W = 0): one table for transport_small.cu, small_n doubles:
    //   sp [Ns][12] as above | Ddiag [Ns][4] | c_kj [Ns][Ns] (+ pad to even) | pair fits [Ns(Ns-1)/2][4], j < k lexicographic, as pair_coef
    const double *small;
    int small_n;
};

// Plan of the staged crf_production_rates kernel (rates_staged.cu).
struct RatesPlan {
    int W;        // warps per block; 0 = no plan
    int Rc;       // reactions per chunk (q buffer rows)
    int n_chunks;
    const int4 *chunk;      // [n_chunks]: x = type (0 elementary, 1 third-body, 2 falloff), y = first reaction,
                            //   z = count, w = first row of the third-body/falloff tables
    const double *rc;       // [Nr][4]: log2(e) lnA, beta, -log2(e) Ea/R, dnu
    const int4 *rs;         // [Nr][2]: byte offsets into the (C,g) state of reactants (3) and products (3); -1 = empty
    const int *inc_ptr;     // [n_chunks][Ns+1] incidence lists of each chunk, species-major
    const double2 *inc;     // entries: x = nu_kr (signed), y = bit pattern of the q-row byte offset
    const double *troe;     // [Nt][8]: log2e lnA0, beta0, -log2e Ea0/R, alpha, -log2e/T3, -log2e/T1, -log2e T2, 0
    const double *gco;      // [Ns][16]: g/(RT) Horner sets, low range 0-6, high range 8-14, 7 = Tmid, 15 = 1/W
    const double *hco;      // [Ns][16]: h/(RT) sets, low 0-5, high 8-13
};

// Plan of the shared-memory-staged crf_production_rates kernel (rates_smem.cu): the reactions are cut into
// chunks of one kind; everything a chunk needs (reaction records, per-species incidence lists, third-body
// lists, Troe sets) is one contiguous block of `stage` that the thread block copies into shared memory
// with cp.async while it works on the previous chunk.  Layout of a chunk block (byte offsets from its start):
//   [0, 48 count)            reaction records: f64 log2(e) lnA, f64 beta, f64 -log2(e) Ea/R, u32 x0, u32 x1,
//                            u32 a0, a1, b0, b1 (byte offsets of the reactant/product rows in the state);
//                            x0, x1 = third reactant/product rows (generic kinds) or offset/count of the
//                            third-body list (kinds 1, 2)
//   [48 count, +(16 + 4 maxown) W)  per warp: u32 start of its incidence entries, 3 pad words, u32 end of the
//                            entries of each owned species k = warp + W slot (entries are warp-major, slot-major)
//   then                     Troe sets, 64 bytes per reaction (kind 2 only)
//   then                     incidence entries {f64 nu, u32 byte offset of q_r, u32 0} and third-body
//                            entries {f64 efficiency - 1, u32 state row offset, u32 0}
struct RatesSmemPlan {
    int W;            // warps sharing a point group; 0 = no plan
    int PPL;          // points per lane (1 or 2)
    int maxown;       // owned-species slots per warp the tables are laid out for (4, 8 or 16)
    int Rc;           // q buffer rows (max reactions per chunk)
    int n_chunks;
    int stage_bytes;  // largest chunk block, multiple of 16
    int tmem;         // thread kernel: the per-thread state lives in tensor memory (6 (Ns + 1) <= 512 columns)
    const int4 *chunk;           // [n_chunks]: x = kind (0 elementary, 1 third body, 2 falloff) | generic << 2,
                                 //   y = reactions, z = byte offset of the block in stage, w = block bytes
    const unsigned char *stage;
    const double *gco;  // [Ns][16]: log2(e) g/(RT) Horner sets, low range 0-6, high range 8-14, 7 = Tmid, 15 = 1/W
    const double *hco;  // [Ns][16]: h/(RT) sets, low 0-5, high 8-13, 7 = Tmid
};

// Plan of the warp-group crf_production_rates kernel (rates_group.cu).  W warps share 32 PPL points.  The reactions are
// cut into n_chunks chunks of at most Rc reactions; a chunk's reactions are dealt to the W warps (balanced by cost), its
// q_r go to a shared q buffer (row Rc stays zero), and each warp then sums q_r for the species it owns.  Everything a
// chunk needs is one contiguous block of `stage`, copied into shared memory by one bulk copy (cp.async.bulk + mbarrier)
// while the previous chunk is evaluated.  Block layout (byte offsets from its start):
//   [0, 32 W)      per warp: u32 records, u32 first q row (byte offset in the q buffer), u32 slot table, u32 Troe sets,
//                  u16 n[4] = reactions of kind elementary / elementary with three slots / third body / falloff
//   records        64 bytes per reaction, in the warp's processing order (the four kinds in that order; q rows are
//                  consecutive): f64 log2(e) lnA, f64 log2(e) beta, f64 -log2(e) Ea/R, u32 b0u, b1u, u32 a0d, a1d, a0u,
//                  a1u, u32 x0, x1, x0u, x1u.  *d = byte offset of the species' d row in the shared-memory state, *u =
//                  handle of its u row (tensor-memory column, or byte offset of the row in shared memory); a = reactants,
//                  b = products, x0/x0u = third reactant, x1u = third product (kind "three slots"), or x0/x1 = offset /
//                  count of the third-body list; empty slots point at the dummy species, row Ns
//   Troe sets      64 bytes per falloff reaction of the warp, in order
//   third-body     entries {f64 efficiency - 1, u32 d offset, u32 u handle}
//   slot table     per warp: u32 {end of the plus list, end of the minus list}[maxown], u32 start of the first list
//   entries        u32 = byte offset of the q row (a coefficient of +-2 is two entries); a list starts 8-byte aligned
//                  and has even length (padded with the zero row Rc)
// State: d_k = (p_ref/RT) exp(-g_k/RT) and u_k = C_k / d_k, rows of 256 PPL bytes [lane][PPL].  Shared memory: d rows
// [Ns + 1], then (tm_cols = 0) u rows [Ns + 1].  tm_cols > 0: u_k lives in tensor memory, columns [2 PPL k, 2 PPL (k + 1)).
struct RatesGroupPlan {
    int W;            // warps sharing a point group; 0 = no plan
    int PPL;          // points per lane (1 or 2)
    int maxown;       // owned-species slots per warp (4, 8 or 16)
    int Rc;           // largest chunk; q buffer row Rc is the zero row
    int q_rows;       // rows of the q buffer (>= Rc + 1; the prologue's scratch too)
    int tm_cols;      // tensor-memory columns a block allocates (power of two), 0 = U in shared memory
    int n_chunks;
    int stage_bytes;  // largest chunk block, multiple of 16
    double log2_c0;   // log2(p_ref / R)
    const int4 *chunk;           // [n_chunks]: x = byte offset of the block in stage, y = block bytes, z = reactions
    const unsigned char *stage;
    const double *gco;  // [Ns][16]: log2(e) g/(RT) Horner sets, low range 0-6, high range 8-14, 7 = Tmid, 15 = 1/W
    const double *hco;  // [Ns][16]: h/(RT) sets, low 0-5, high 8-13, 7 = Tmid
    const int *own;     // [W][maxown]: species owned by (warp, slot), -1 = none (balanced by incidence count)
};

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
    // crf_thermo (thermo.cu): [Ns][14] = {a1..a5, a6} / W_k of the low range, of the high range, then T_mid, pad
    const double *thermo_tab;
    int thermo_sets;  // 1: a lane reads the coefficient set of its range; 2: both sets at uniform addresses (thermo.cu)
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
    TransportPlan tp;
    RatesPlan rp;
    RatesSmemPlan rs;
    RatesGroupPlan rg;
};

__device__ __forceinline__ int crf_pair_index(int j, int k, int ns)
{  // j <= k
    return j * ns - (j * (j - 1)) / 2 + (k - j);
}
