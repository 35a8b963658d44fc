/* crf_diag.h -- diagnostics and explicit kernel-plan control of libcrf.so.
 *
 * Nothing here is part of the method (include/crf.h holds the calls that follow the paper's
 * statement of the problem).  These entry points exist for the benchmark (measured FP64 peak,
 * launch counter), for the tests (every kernel variant must meet the same tolerances, so the
 * tests must be able to select each one) and for tuning.  The library never reads an
 * environment variable: a plan is either chosen by crf_mech_create from the mechanism's size
 * or requested here, explicitly.
 */
#ifndef CRF_DIAG_H
#define CRF_DIAG_H

#include "crf.h"

#ifdef __cplusplus
extern "C" {
#endif

/* Which kernel variant a call dispatches to. */
#define CRF_RATES_AUTO 0
#define CRF_RATES_GENERIC 1 /* one thread per point, libm exponentials, any mechanism (rates.cu) */
#define CRF_RATES_STAGED 2  /* warp groups, log-space K_c: two exponentials per reaction (rates_staged.cu) */
#define CRF_RATES_GROUP 3   /* warp groups, activity form of K_c, u rows in tensor memory, chunk tables staged by bulk copies (rates_group.cu) */
#define CRF_RATES_THREAD 4  /* one thread per point, product form of K_c, small mechanisms (rates_smem.cu) */

#define CRF_TRANSPORT_AUTO 0
#define CRF_TRANSPORT_GENERIC 1 /* one thread per point, any Ns (transport.cu) */
#define CRF_TRANSPORT_SMALL 2   /* register-resident, 2 <= Ns <= 16 (transport_small.cu) */
#define CRF_TRANSPORT_TILED 3   /* warp groups, 8x8 species tiles, Ns >= 17 (transport_tiled.cu) */

/* Plan request.  Zero-initialise: 0 means "let crf_mech_create choose".  A request the
 * mechanism does not admit (e.g. CRF_RATES_GROUP when the product form of K_c leaves the double
 * range, CRF_TRANSPORT_SMALL with Ns > 16) makes crf_mech_create_ex fail with CRF_EUNSUPPORTED
 * rather than silently pick something else. */
typedef struct crf_plan_options {
    int32_t rates_kernel;     /* CRF_RATES_* */
    int32_t rates_W;          /* warps sharing a point group: 4, 8 or 16 (GROUP); 1, 2, 4 (STAGED) */
    int32_t rates_PPL;        /* points per lane: 1 or 2 (GROUP) */
    int32_t rates_Rc;         /* reactions per chunk (GROUP): upper bound, rounded to the kernel's granularity */
    int32_t transport_kernel; /* CRF_TRANSPORT_* */
    int32_t transport_W;      /* warps sharing a point group: 1, 2, 4 or 8 (TILED) */
    int32_t transport_PPL;    /* points per lane: 1 or 2 (TILED) */
    int32_t transport_panel;  /* column blocks per Wilke panel (TILED) */
    int32_t rates_tmem;       /* GROUP: 0 = u rows in tensor memory when they fit, 1 = in shared memory, 2 = require tensor memory */
    int32_t transport_TS;     /* species per block of the pair tiles (TILED): 7 or 8; 0 = whichever the plan's estimate prefers */
    int32_t thermo_sets;      /* crf_thermo: 2 = both NASA-7 sets of a species at warp-uniform addresses, the point's mass fraction
                               * routed to the set of its range (twelve FMAs per species and point; the default: 0.80-0.86 of
                               * the HBM roofline on every config); 1 = every lane reads the set of its own range (six FMAs;
                               * faster, 0.91-0.93, where the points of a warp share their ranges, as in spatially coherent
                               * fields, slower, 0.74, where they do not); 0 = default */
    int32_t reserved[5];      /* must be 0 */
} crf_plan_options;

/* What a mechanism will run. */
typedef struct crf_plan_info {
    int32_t rates_kernel; /* CRF_RATES_* (never AUTO) */
    int32_t rates_W, rates_PPL, rates_Rc, rates_chunks, rates_stage_bytes, rates_smem_bytes;
    int32_t transport_kernel; /* CRF_TRANSPORT_* (never AUTO) */
    int32_t transport_W, transport_PPL, transport_nb, transport_stage_blocks, transport_stage_bytes,
        transport_smem_bytes;
    int32_t rates_tmem_cols; /* tensor-memory columns a block of the GROUP kernel allocates (0: u rows in shared memory) */
    int32_t transport_TS;    /* species per block of the pair tiles (transport_nb counts these blocks) */
    int32_t thermo_sets;     /* 1 or 2 (crf_plan_options.thermo_sets) */
    int32_t reserved[5];
} crf_plan_info;

/* crf_mech_create with an explicit plan request (options may be NULL = all automatic). */
int crf_mech_create_ex(const crf_tables *tables, const crf_plan_options *options, crf_mech **out);
int crf_mech_plan_info(const crf_mech *mech, crf_plan_info *info);

/* Sustained FP64 pipe rate of the current device: runs a register-only kernel of `iters`
 * dependent-chain DFMA groups on every SM and returns the FP64 instructions per second it
 * reached in *inst_per_s (the measured denominator of the ALU roofline).  Synchronous. */
int crf_fp64_probe(int iters, double *inst_per_s);

/* How many kernel launches this library has issued in this process (for bench.py). */
int64_t crf_launch_count(void);

/* Host-only (no device needed): the tile schedule crf_mech_create lays out for crf_mix_transport on a
 * mechanism whose species fill nb blocks (of 8 or 7 species), dealt to W warps.  Writes up to `cap` tiles as
 * int32 quadruples {round, kind (1 off-diagonal, 2 diagonal), jb, kb} to out and returns the number of tiles
 * of the schedule (which may exceed cap), or CRF_EINVAL. */
int crf_transport_schedule(int nb, int W, int32_t *out, int cap);

#ifdef __cplusplus
}
#endif
#endif /* CRF_DIAG_H */
