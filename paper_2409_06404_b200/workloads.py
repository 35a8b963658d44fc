"""Seeded synthetic inputs: mechanism *descriptions* and thermochemical states.

This module is the only code shared by the CUDA path (via ``packer.py``) and the
CPU oracle (via ``oracle/crf_oracle.py``).  It holds none of the method's
arithmetic: it draws species, reactions, fit coefficients and (T, p, Y) fields
from seeded ``numpy`` generators and returns them as plain data.  The only
mathematics here is generic polynomial algebra (``numpy.polynomial``) used to
make the NASA-7 coefficient sets continuous at ``T_mid`` — it constructs inputs,
it evaluates nothing on the hot path.

Recipes follow BASELINE.json ``configs`` (called C1..C5, seeds 0..4) and
SURVEY.md §8(d); where the literal recipe is infeasible the construction used
is stated in the docstring of the function that does it.

Units of a description (the oracle and the packer each convert on their own):

* ``W``            kg/kmol (from atomic masses H 1.008, C 12.011, N 14.007, O 15.999)
* NASA-7           standard dimensionless a1..a7 (a6 in K), two ranges split at ``Tmid``
* ``A``            cgs-mol: (cm^3/mol)^(order-1)/s, order = number of reactant
                   molecules (+1 for a third body; the low-pressure limit of a
                   falloff reaction has one order more than its high-pressure limit)
* ``Ea``           kJ/mol
* transport fits   natural-log cubics in ln(T): ln mu [Pa s], ln lambda [W/m/K],
                   ln D_jk [m^2/s] at ``p_ref``
"""
from __future__ import annotations

import itertools
from collections import defaultdict

import numpy as np
from numpy.polynomial import polynomial as npoly

ATOMIC_MASS = {"H": 1.008, "C": 12.011, "N": 14.007, "O": 15.999}
P_REF = 101325.0
POINTS_PER_ELEMENT = 512  # (7+1)^3 GLL points, PAPER.md:92,102 ("p = 7")

# name -> (seed, elements, Ns, Nr, N3 third-body, Nt Troe, duplicate pairs, max atom count,
#          n_elements, state kind, Dirichlet alpha, trace fraction, p kind)
CONFIGS = {
    "C1": dict(seed=0, elements=("H", "O", "N"), Ns=9, Nr=21, N3=4, Nt=0, ndup=0, cmax=2,
               n_elem=1, state="uniform", alpha=0.5, trace=0.2, p="const", eff_all=True),
    "C2": dict(seed=1, elements=("H", "O", "N"), Ns=9, Nr=21, N3=4, Nt=0, ndup=0, cmax=2,
               n_elem=32768, state="flame", alpha=0.5, trace=0.2, p="const", eff_all=True),
    "C3": dict(seed=2, elements=("C", "H", "O", "N"), Ns=21, Nr=84, N3=12, Nt=6, ndup=0, cmax=2,
               n_elem=8192, state="uniform", alpha=0.5, trace=0.2, p="const", eff_all=False),
    "C4": dict(seed=3, elements=("C", "H", "O", "N"), Ns=53, Nr=325, N3=40, Nt=25, ndup=8, cmax=2,
               n_elem=8192, state="flame", alpha=0.5, trace=0.2, p="const", eff_all=False),
    "C5": dict(seed=4, elements=("C", "H", "O", "N"), Ns=118, Nr=720, N3=60, Nt=50, ndup=0, cmax=3,
               n_elem=4096, state="uniform", alpha=0.3, trace=0.3, p="range", eff_all=False),
}


def config_points(name: str) -> int:
    return CONFIGS[name]["n_elem"] * POINTS_PER_ELEMENT


# --------------------------------------------------------------------------------------
# species and reactions
# --------------------------------------------------------------------------------------
def _formula_name(elements, counts) -> str:
    return "".join(f"{e}{c}" for e, c in zip(elements, counts) if c > 0)


def _enumerate_balanced(comp: np.ndarray, reactive: list[int]):
    """All atom-balanced A+B<=>C+D and A+B<=>C over ``reactive`` with disjoint sides."""
    by_sum = defaultdict(list)
    for ia, a in enumerate(reactive):
        for b in reactive[ia:]:
            by_sum[tuple(comp[:, a] + comp[:, b])].append((a, b))
    single = defaultdict(list)
    for c in reactive:
        single[tuple(comp[:, c])].append(c)
    two_two, two_one = [], []
    for key, pairs in by_sum.items():
        for p, q in itertools.combinations(pairs, 2):
            if not (set(p) & set(q)):
                two_two.append((p, q))
        for c in single.get(key, ()):
            for p in pairs:
                if c not in p:
                    two_one.append((p, (c,)))
    return two_two, two_one


def _draw_species(rng, elements, n_reactive, cmax, need_22, need_21, tries=400):
    """Species set by rejection sampling over formula sets (BASELINE.json configs:
    'random atom counts, at least one atom each ... found by rejection sampling over
    species multisets with matching element totals').

    The inert (N2-like) species is the last one and takes part in no reaction.  A set is
    accepted when it admits enough distinct balanced stoichiometries.
    found that 8 independent draws over H,O,N never admit 21: after ``tries`` rejections
    the reactive species become the full count lattice of the first two elements
    (counts 0..cmax, zero vector removed), which admits 30 for cmax=2.
    """
    ne = len(elements)
    if "N" not in elements:
        raise ValueError("the inert species is N2: 'N' must be one of the elements")
    all_formulas = [c for c in itertools.product(range(cmax + 1), repeat=ne) if sum(c) > 0]
    inert = tuple(2 if e == "N" else 0 for e in elements)
    pool = [c for c in all_formulas if c != inert]
    for _ in range(tries):
        if n_reactive > len(pool):
            break
        idx = rng.choice(len(pool), size=n_reactive, replace=False)
        counts = [pool[i] for i in sorted(idx)]
        comp = np.array(counts + [inert], dtype=np.int64).T
        c22, c21 = _enumerate_balanced(comp, list(range(n_reactive)))
        if len(c21) >= need_21 and len(c22) + len(c21) >= need_22 + need_21:
            return comp, c22, c21
    lattice = [c for c in all_formulas if all(x == 0 for x in c[2:])]
    lattice = [c for c in lattice if c != inert]
    if len(lattice) != n_reactive:
        raise ValueError("no feasible species set: widen cmax or lower Nr")
    comp = np.array(lattice + [inert], dtype=np.int64).T
    c22, c21 = _enumerate_balanced(comp, list(range(n_reactive)))
    if len(c21) < need_21 or len(c22) + len(c21) < need_22 + need_21:
        raise ValueError("lattice species set admits too few balanced reactions")
    return comp, c22, c21


def _arrhenius(rng):
    return dict(A=float(10.0 ** rng.uniform(6.0, 14.0)), beta=float(rng.uniform(-1.5, 1.5)),
                Ea=float(rng.uniform(0.0, 150.0)))


def _efficiencies(rng, ns, eff_all):
    if eff_all:
        ks = np.arange(ns)
    else:
        ks = np.sort(rng.choice(ns, size=int(rng.integers(2, 7)), replace=False))
    return {int(k): float(rng.uniform(0.5, 3.0)) for k in ks}


def _draw_reactions(rng, cfg, c22, c21, ns):
    """Nr reversible reactions: Nt Troe falloff + N3 third-body + the rest elementary,
    ``ndup`` of the elementary ones duplicated (same stoichiometry, own Arrhenius set).

    Falloff reactions are association reactions A+B(+M)<=>C(+M); third-body reactions
    prefer A+B+M<=>C+M and take A+B+M<=>C+D+M when the set has too few associations.
    The low-pressure A0 is A_inf * 10^U[3,7] cm^3/mol so that the reduced pressure
    P_r = k0[M]/k_inf straddles 1 over the state range (SURVEY.md §8(c) falloff reading).
    Returned order is the draw order (types mixed); sorting by type is the packer's job.
    """
    nr, n3, nt, ndup = cfg["Nr"], cfg["N3"], cfg["Nt"], cfg["ndup"]
    n_distinct = nr - ndup
    c21 = [c21[i] for i in rng.permutation(len(c21))]
    c22 = [c22[i] for i in rng.permutation(len(c22))]
    n_assoc = min(len(c21), nt + n3)
    stoich = c21[:n_assoc]
    rest = c22 + c21[n_assoc:]
    rest = [rest[i] for i in rng.permutation(len(rest))]
    stoich = stoich + rest[: n_distinct - n_assoc]
    if len(stoich) < n_distinct:
        raise ValueError("too few balanced stoichiometries")
    kinds = ["falloff"] * nt + ["three_body"] * n3 + ["elementary"] * (n_distinct - nt - n3)
    reactions = []
    for (lhs, rhs), kind in zip(stoich, kinds):
        r = dict(reactants=_slots(lhs), products=_slots(rhs), type=kind, **_arrhenius(rng))
        if kind != "elementary":
            r["eff"] = _efficiencies(rng, ns, cfg["eff_all"])
        if kind == "falloff":
            r["troe"] = dict(
                A0=r["A"] * float(10.0 ** rng.uniform(3.0, 7.0)),
                beta0=float(rng.uniform(-1.5, 1.5)), Ea0=float(rng.uniform(0.0, 150.0)),
                alpha=float(rng.uniform(0.3, 0.9)),
                T3=float(10.0 ** rng.uniform(1.0, 4.0)), T1=float(10.0 ** rng.uniform(1.0, 4.0)),
                T2=float(10.0 ** rng.uniform(1.0, 4.0)))
        reactions.append(r)
    elem_idx = [i for i, r in enumerate(reactions) if r["type"] == "elementary"]
    for i in rng.choice(elem_idx, size=ndup, replace=False) if ndup else ():
        twin = dict(reactions[int(i)])
        twin.update(_arrhenius(rng))
        reactions.append(twin)
    order = rng.permutation(len(reactions))
    return [reactions[i] for i in order]


def _slots(side):
    """(species, coefficient) list; a repeated species becomes coefficient 2."""
    out = defaultdict(int)
    for k in side:
        out[int(k)] += 1
    return sorted(out.items())


# --------------------------------------------------------------------------------------
# NASA-7 and transport fits
# --------------------------------------------------------------------------------------
_T0 = 298.15


def _draw_nasa(rng, ns, comp, hf_mode):
    """Two-range NASA-7 sets with cp/R in [2.5, 8] on 200..3500 K, continuous cp, h, s at
    T_mid, h(298.15 K) ~ U[-300, 300] kJ/mol and s(298.15 K) ~ U[150, 250] J/mol/K.

    cp/R is a smooth rising curve lo + (hi-lo)*(1-exp(-T/theta)) sampled on each range and
    fitted by a quartic; the high-range quartic is shifted to meet the low one at T_mid
    and a6/a7 follow from the antiderivatives.  About a quarter of the species get a T_mid
    drawn in [800, 1400] K instead of 1000 K so that the range select is exercised.

    ``hf_mode`` "uniform" is the literal recipe (independent h_f per species; reaction
    enthalpies then reach +-1200 kJ/mol and equilibrium constants e^(+-480), so one
    reaction dominates each omega_k).  "group" draws h_f = sum_e a_ek eta_e + U[-40, 40]
    kJ/mol with per-element eta_e ~ U[-60, 60], clipped to the same +-300 range: atom
    balance cancels the element part, reaction enthalpies stay below 160 kJ/mol as in a
    real mechanism, and many reactions contribute comparably to each omega_k (the parity
    tests run both).
    """
    R_kJ = 8.31446261815324e-3  # kJ/mol/K, only to turn the h_f and s draws into a6, a7
    tmid = np.where(rng.random(ns) < 0.25, rng.uniform(800.0, 1400.0, ns), 1000.0)
    lo_set, hi_set = np.zeros((ns, 7)), np.zeros((ns, 7))
    eta = rng.uniform(-60.0, 60.0, comp.shape[0])
    for k in range(ns):
        c_lo = rng.uniform(2.5, 4.5)
        c_hi = rng.uniform(c_lo + 0.2, 7.8)
        theta = rng.uniform(500.0, 1500.0)
        curve = lambda T: c_lo + (c_hi - c_lo) * (1.0 - np.exp(-T / theta))  # noqa: E731
        coef = []
        for (ta, tb) in ((200.0, tmid[k]), (tmid[k], 3500.0)):
            t = np.linspace(ta, tb, 60)
            coef.append(npoly.polyfit(t / 1000.0, curve(t), 4) / 1000.0 ** np.arange(5))
        a_lo, a_hi = coef
        a_hi[0] += npoly.polyval(tmid[k], a_lo) - npoly.polyval(tmid[k], a_hi)
        # keep cp/R inside [2.5, 8] on each set's own range: contract both sets about the
        # mid value 5.25 by one common factor (continuity at T_mid is preserved)
        v = np.concatenate((npoly.polyval(np.linspace(200.0, tmid[k], 200), a_lo),
                            npoly.polyval(np.linspace(tmid[k], 3500.0, 200), a_hi)))
        f = min(1.0, 2.7 / max(np.abs(v - 5.25).max(), 1e-30))
        for a in (a_lo, a_hi):
            a *= f
            a[0] += 5.25 * (1.0 - f)
        # h/R = int cp/R dT + a6 ;  s/R = a1 ln T + int (cp/R - a1)/T dT + a7
        H = lambda a: npoly.polyint(a)  # noqa: E731
        S = lambda a: np.concatenate(([0.0], a[1:] / np.arange(1, 5)))  # noqa: E731
        h_f = rng.uniform(-300.0, 300.0)
        h_res = rng.uniform(-40.0, 40.0)
        if hf_mode == "group":
            h_f = float(np.clip(comp[:, k] @ eta + h_res, -300.0, 300.0))
        h_f /= R_kJ                                        # K
        s_0 = rng.uniform(150.0, 250.0) * 1e-3 / R_kJ      # dimensionless
        a6_lo = h_f - npoly.polyval(_T0, H(a_lo))
        a7_lo = s_0 - a_lo[0] * np.log(_T0) - npoly.polyval(_T0, S(a_lo))
        a6_hi = a6_lo + npoly.polyval(tmid[k], H(a_lo)) - npoly.polyval(tmid[k], H(a_hi))
        a7_hi = (a7_lo + (a_lo[0] - a_hi[0]) * np.log(tmid[k])
                 + npoly.polyval(tmid[k], S(a_lo)) - npoly.polyval(tmid[k], S(a_hi)))
        lo_set[k] = np.concatenate((a_lo, [a6_lo, a7_lo]))
        hi_set[k] = np.concatenate((a_hi, [a6_hi, a7_hi]))
    return tmid, lo_set, hi_set


def _log_cubic(rng, ln_ref, slope, shape):
    """Coefficients c0..c3 of ln f = sum c_m (ln T)^m, built as
    ln_ref + slope*x + q*x^2 + c*x^3 with x = ln(T/1000 K) and small q, c."""
    x0 = np.log(1000.0)
    q = rng.uniform(-0.05, 0.05, shape)
    c = rng.uniform(-0.01, 0.01, shape)
    out = np.zeros(tuple(np.atleast_1d(shape)) + (4,))
    out[..., 0] = ln_ref - slope * x0 + q * x0 ** 2 - c * x0 ** 3
    out[..., 1] = slope - 2.0 * q * x0 + 3.0 * c * x0 ** 2
    out[..., 2] = q - 3.0 * c * x0
    out[..., 3] = c
    return out


def _draw_transport(rng, ns):
    """mu_k ~ 1e-5..1e-4 Pa s, lambda_k ~ 0.03..0.3 W/m/K, D_jk ~ 1e-5..1e-3 m^2/s over
    300..2500 K (BASELINE.json configs), D_jk symmetric with its own diagonal."""
    mu = _log_cubic(rng, np.log(rng.uniform(2.5e-5, 6e-5, ns)), rng.uniform(0.6, 0.8, ns), ns)
    lam = _log_cubic(rng, np.log(rng.uniform(0.05, 0.2, ns)), rng.uniform(0.7, 0.9, ns), ns)
    iu = np.triu_indices(ns)
    npair = iu[0].size
    tri = _log_cubic(rng, np.log(rng.uniform(8e-5, 3e-4, npair)), rng.uniform(1.6, 1.8, npair), npair)
    D = np.zeros((ns, ns, 4))
    D[iu[0], iu[1]] = tri
    D[iu[1], iu[0]] = tri
    return mu, lam, D


# --------------------------------------------------------------------------------------
# public: mechanism description
# --------------------------------------------------------------------------------------
def make_mechanism(name: str | None = None, **override) -> dict:
    """Seeded synthetic mechanism description for config ``name`` (C1..C5)."""
    cfg = dict(CONFIGS[name]) if name else {}
    cfg.update(override)
    rng = np.random.default_rng([cfg["seed"], 0x6D656368])  # stream "mech"
    elements, ns = tuple(cfg["elements"]), cfg["Ns"]
    n_distinct = cfg["Nr"] - cfg["ndup"]
    need_21 = min(cfg["Nt"], n_distinct)
    comp, c22, c21 = _draw_species(rng, elements, ns - 1, cfg["cmax"], n_distinct - need_21, need_21)
    W = comp.T.astype(float) @ np.array([ATOMIC_MASS[e] for e in elements])
    tmid, lo, hi = _draw_nasa(rng, ns, comp, cfg.get("hf", "uniform"))
    mu, lam, D = _draw_transport(rng, ns)
    reactions = _draw_reactions(rng, cfg, c22, c21, ns)
    return dict(
        name=name or "custom", elements=list(elements),
        species=[_formula_name(elements, comp[:, k]) for k in range(ns)],
        comp=comp, W=W, nasa_Tmid=tmid, nasa_lo=lo, nasa_hi=hi,
        reactions=reactions, mu_fit=mu, lam_fit=lam, D_fit=D, p_ref=P_REF)


# --------------------------------------------------------------------------------------
# public: states
# --------------------------------------------------------------------------------------
def _dirichlet_with_traces(rng, ns, n, alpha, trace):
    """Y[ns, n]: Dirichlet(alpha) columns, a fraction ``trace`` of the entries set to 1e-20,
    then renormalised (the largest entry of a column is never made a trace)."""
    Y = rng.standard_gamma(alpha, size=(ns, n))
    Y = np.maximum(Y, 1e-300)
    mask = rng.random((ns, n)) < trace
    mask[np.argmax(Y, axis=0), np.arange(n)] = False
    Y /= Y.sum(axis=0, keepdims=True)
    Y[mask] = 1e-20
    Y /= Y.sum(axis=0, keepdims=True)
    return Y


def make_state(name: str, n: int | None = None, *, offset: int = 0, total: int | None = None,
               **override) -> dict:
    """Seeded state for config ``name``: dict(T[n], p[n], Y[Ns, n]) (species-major).

    ``n`` defaults to the config's full size.  For the flame configs the profile position
    of point i is x_i = (offset + i + 1/2)/total, so a shard (``offset``, ``n``) of a
    ``total``-point field is the same as that slice of the whole field's profile; the
    noise of a shard is drawn from a stream keyed by ``offset``.
    """
    cfg = dict(CONFIGS[name])
    cfg.update(override)
    ns = cfg["Ns"]
    n = config_points(name) if n is None else int(n)
    total = max(n, 1) if total is None else int(total)
    rng = np.random.default_rng([cfg["seed"], 0x73746174, offset])  # stream "stat"
    if cfg["state"] == "uniform":
        T = rng.uniform(300.0, 2500.0, n)
        Y = _dirichlet_with_traces(rng, ns, n, cfg["alpha"], cfg["trace"])
    else:
        ends = np.random.default_rng([cfg["seed"], 0x656E6473])  # same end states for every shard
        Yu = _dirichlet_with_traces(ends, ns, 1, cfg["alpha"], cfg["trace"])
        Yb = _dirichlet_with_traces(ends, ns, 1, cfg["alpha"], cfg["trace"])
        x0, delta = 0.5 + 0.05 * ends.uniform(-1, 1), 0.05
        x = (offset + np.arange(n) + 0.5) / total
        c = 0.5 * (1.0 + np.tanh((x - x0) / delta))
        T = (300.0 + 2100.0 * c) * (1.0 + 0.05 * rng.uniform(-1.0, 1.0, n))
        Y = (1.0 - c)[None, :] * Yu + c[None, :] * Yb
    p = rng.uniform(1e5, 4e6, n) if cfg["p"] == "range" else np.full(n, P_REF)
    return dict(T=np.ascontiguousarray(T), p=np.ascontiguousarray(p), Y=np.ascontiguousarray(Y))
