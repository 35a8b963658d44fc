"""Algorithmic work and HBM bytes per grid point of the three calls.

"Algorithmic" = what the method as stated in DESIGN.md must do, independent of how a kernel
does it: FP64 pipe instructions ``I`` (one per DFMA/DADD/DMUL) and flops ``F`` (FMA = 2), with
the transcendentals at their sm_100a SASS fast-path cost (CUDA 12.9: exp 14 DFMA + 1 DADD,
log 16 DFMA + 4 DMUL + 8 DADD, divide 7 DFMA + 1 DMUL, reciprocal 5 DFMA, sqrt 5 DFMA + 3 DMUL;
MUFU seeds and integer work not counted).  Bytes = fields that must cross HBM once.

Peaks: HBM from MEASURED_PEAKS.json (fallback 6650 GB/s, B200_PROFILING.md); FP64 ALU from the
unit counts and clocks: 148 SM x 64 FP64 lanes x 1.965 GHz = 18.61e12 instr/s = 37.2 TFLOP/s
(FMA = 2).  bench.py also measures the sustained DFMA rate (crf_fp64_probe) and reports it.
"""
from __future__ import annotations

import json
import os

# (instructions, flops) of the fast paths
EXP = (15, 29)
LOG = (28, 44)
DIV = (8, 15)
RCP = (5, 10)
SQRT = (8, 13)
LOG10 = (29, 45)
EXP10 = (16, 30)

N_SM, FP64_LANES_PER_SM, SM_MAX_HZ = 148, 64, 1.965e9
FP64_PEAK_INST = N_SM * FP64_LANES_PER_SM * SM_MAX_HZ   # 1.861e13 instr/s
FP64_PEAK_TFLOPS = 2.0 * FP64_PEAK_INST / 1e12          # 37.2
HBM_FALLBACK_GBS = 6650.0


def _acc(*terms):
    """sum of count * (I, F) terms; a bare (I, F) has count 1"""
    i = f = 0.0
    for t in terms:
        c, (ti, tf) = t if isinstance(t[1], tuple) else (1, t)
        i += c * ti
        f += c * tf
    return i, f


FMA, OP = (1, 2), (1, 1)


def thermo_work(Ns: int):
    """rows a2-a3: per species 4 FMA (cp) + 5 FMA (h) + 1 MUL (Y/W) + 2 FMA (sums); 1/T, 3 scalings"""
    I, F = _acc((11 * Ns, FMA), (Ns, OP), RCP, (3, OP))
    return dict(I=I, F=F, B=8.0 * (Ns + 1) + 16.0)


def rates_work(Ns: int, Nr: int, N3: int, Nt: int, n_eff: int):
    """rows a1, a2, a4-a9.  Per species: 1 FMA (1/Wbar) + 2 MUL + 1 ADD (C_k, sum C) + 7 FMA
    (g/RT) + 6 FMA (h_k and the qdot sum).  Per reaction: 2 FMA (ln k_f) + exp + 3 ADD + 1 FMA
    (sum nu g - dnu ln c0) + exp + 1 MUL (k_r) + 2 MUL (products) + 1 MUL + 1 FMA (q) + 4 ADD
    (scatter) = 45.  Third body: one FMA per listed efficiency + 1 MUL.  Troe: ln k_0 (2 FMA),
    exp(P_r) + MUL, 3 exp + 3 MUL + 2 FMA (F_cent), 2 log10, 2 FMA, 2 FMA + divide (f1), FMA +
    divide + exp10, P_r/(1+P_r): ADD + divide, 2 MUL."""
    per_species = _acc((14, FMA), (3, OP))
    per_reaction = _acc((4, FMA), (2, EXP), (11, OP))
    troe = _acc((2, FMA), EXP, OP, (3, EXP), (3, OP), (2, FMA), (2, LOG10), (2, FMA), (2, FMA), DIV, FMA, DIV,
                EXP10, OP, DIV, (2, OP))
    base = _acc(LOG, RCP, DIV, (6, OP))
    I = base[0] + Ns * per_species[0] + Nr * per_reaction[0] + Nt * troe[0] + n_eff + N3
    F = base[1] + Ns * per_species[1] + Nr * per_reaction[1] + Nt * troe[1] + 2 * n_eff + N3
    return dict(I=I, F=F, B=8.0 * (2 * Ns + 3))


def transport_work(Ns: int):
    """rows a1, a10-a13.  Per species: 2 cubics (6 FMA) + 2 exp (mu_k, lambda_k) + sqrt + reciprocal
    (Wilke factors) + divide (X/lambda) + X_k (2 MUL) + 1/Wbar FMA + 3 FMA (sums) + the final
    (1 - Y_k)/S_k (ADD + divide + MUL) + mu term (MUL + divide).  Per unordered pair: cubic (3 FMA)
    + exp + 2 FMA (S_j, S_k).  Per ordered pair (Wilke): FMA, 2 MUL, FMA."""
    per_species = _acc((10, FMA), (2, EXP), SQRT, RCP, (3, DIV), (6, OP))
    per_upair = _acc((5, FMA), EXP)
    per_opair = _acc((2, FMA), (2, OP))
    base = _acc(LOG, (2, RCP), DIV, (6, OP))
    nu, no = Ns * (Ns - 1) // 2, Ns * Ns
    I = base[0] + Ns * per_species[0] + nu * per_upair[0] + no * per_opair[0]
    F = base[1] + Ns * per_species[1] + nu * per_upair[1] + no * per_opair[1]
    return dict(I=I, F=F, B=8.0 * (2 * Ns + 4))


def measured_peaks(repo_root: str) -> dict:
    """{'hbm_gbs': ..., 'source': 'measured'|'fallback'} from MEASURED_PEAKS.json (driver-written)."""
    path = os.path.join(repo_root, "MEASURED_PEAKS.json")
    try:
        with open(path) as f:
            d = json.load(f)
        return dict(hbm_gbs=float(d["hbm_gbs"]), source="measured")
    except (OSError, KeyError, ValueError):
        return dict(hbm_gbs=HBM_FALLBACK_GBS, source="fallback")
