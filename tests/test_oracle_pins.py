"""Pins of the CPU oracle against what the mathematics fixes (SURVEY.md §8(c) "What pins each
part"): closed forms, conservation laws, thermodynamic equilibrium, limits that reduce to
textbook expressions, metamorphic relations, and a 50-digit re-evaluation for rounding.
CPU only.  A plausible slip in crf_oracle.c (dropped term, wrong sign/index, transposed
operand, wrong unit factor) fails at least one of these.
"""
import mpmath as mp
import numpy as np
import pytest

from paper_2409_06404_b200 import workloads as wl
from tests import mp_reference
from tests.helpers import (P_REF, R, R_KJ_MOL, col, const_cp_nasa, mass_from_mole, rxn, tiny_mech)


@pytest.fixture(scope="module")
def Oracle(oracle_mod):
    return oracle_mod.Oracle


SMALL = dict(seed=11, elements=("H", "O", "N"), Ns=14, Nr=40, N3=5, Nt=5, ndup=2, cmax=2,
             n_elem=1, state="uniform", alpha=0.5, trace=0.2, p="range", eff_all=False)


# ------------------------------------------------------------------ NASA-7 (step 2, 3)
def test_nasa_constant_cp_closed_form(Oracle):
    m = tiny_mech([2.0, 28.0], [], nasa=([const_cp_nasa(3.5, -1000.0, 4.0), const_cp_nasa(2.5, 25000.0, -1.0)],) * 2)
    T = np.array([300.0, 1000.0, 1000.0000001, 2500.0])
    s = Oracle(m).thermo_species(T)
    for k, (a1, a6, a7) in enumerate([(3.5, -1000.0, 4.0), (2.5, 25000.0, -1.0)]):
        np.testing.assert_allclose(s["cpk"][k], a1 * R * np.ones_like(T), rtol=1e-15)
        np.testing.assert_allclose(s["hk"][k], R * (a1 * T + a6), rtol=1e-15)
        np.testing.assert_allclose(s["sk"][k], R * (a1 * np.log(T) + a7), rtol=1e-15)
        np.testing.assert_allclose(s["g_RT"][k], (a1 * T + a6) / T - (a1 * np.log(T) + a7), rtol=1e-14)
    # mixture: mass-weighted, per kg  (cp = sum Y_k cp_k / W_k)
    Y = np.array([[0.25] * 4, [0.75] * 4])
    th = Oracle(m).thermo(T, np.full(4, P_REF), Y)
    np.testing.assert_allclose(th["cp"], 0.25 * 3.5 * R / 2.0 + 0.75 * 2.5 * R / 28.0, rtol=1e-15)
    np.testing.assert_allclose(th["h"], 0.25 * R * (3.5 * T - 1000.0) / 2.0 + 0.75 * R * (2.5 * T + 25000.0) / 28.0,
                               rtol=1e-14)


@pytest.mark.parametrize("cfg", ["C1", "C3", "C5"])
def test_nasa_calculus_identities(Oracle, cfg):
    """dh/dT = cp, ds/dT = cp/T (central differences), g = h - T s, continuity at T_mid."""
    m = wl.make_mechanism(cfg)
    o = Oracle(m)
    rng = np.random.default_rng(5)
    T = rng.uniform(250.0, 3200.0, 64)
    T = T[np.min(np.abs(T[None, :] - m["nasa_Tmid"][:, None]), axis=0) > 1.0]
    d = 0.01
    s0, sp, sm = o.thermo_species(T), o.thermo_species(T + d), o.thermo_species(T - d)
    np.testing.assert_allclose((sp["hk"] - sm["hk"]) / (2 * d), s0["cpk"], rtol=1e-7)
    np.testing.assert_allclose((sp["sk"] - sm["sk"]) / (2 * d), s0["cpk"] / T, rtol=1e-7)
    np.testing.assert_allclose(s0["g_RT"], s0["hk"] / (R * T) - s0["sk"] / R, rtol=1e-12, atol=1e-12)
    assert s0["cpk"].min() >= 2.5 * R * (1 - 1e-9) and s0["cpk"].max() <= 8.0 * R * (1 + 1e-9)
    for k in range(len(m["W"])):
        tm = m["nasa_Tmid"][k]
        a, b = o.thermo_species([tm]), o.thermo_species([np.nextafter(tm, 1e9)])
        for key in ("cpk", "hk", "sk"):
            assert abs(a[key][k, 0] - b[key][k, 0]) <= 1e-9 * abs(a[key][k, 0]) + 1e-3, (cfg, k, key)


def test_nasa_formation_anchor(Oracle):
    """generator recipe: h(298.15 K) in [-300, 300] kJ/mol, s(298.15 K) in [150, 250] J/mol/K"""
    m = wl.make_mechanism("C3")
    s = Oracle(m).thermo_species([298.15])
    assert np.all(np.abs(s["hk"]) <= 300.0e6 * (1 + 1e-12))
    assert np.all((s["sk"] >= 150.0e3 * (1 - 1e-12)) & (s["sk"] <= 250.0e3 * (1 + 1e-12)))


# ------------------------------------------------------------------ single reactions (steps 1, 4, 7, 8)
def _conc(X, T, p):
    return np.asarray(X) * p / (R * T)


def test_single_reaction_dnu0_closed_form(Oracle):
    """beta=0, E=0, identical NASA sets => K_c = 1, q = A (C_A C_B - C_C C_D); A 1e12 cm^3/mol/s = 1e9 m^3/kmol/s."""
    W = [2.0, 32.0, 17.0, 17.0, 28.0]
    m = tiny_mech(W, [rxn([(0, 1), (1, 1)], [(2, 1), (3, 1)], A=1.0e12)])
    X = np.array([0.2, 0.1, 0.15, 0.05, 0.5])
    T, p = 1234.5, 2.5e5
    d = Oracle(m).rates_detail(T, p, mass_from_mole(X, W))
    C = _conc(X, T, p)
    np.testing.assert_allclose(d["C"], C, rtol=1e-14)
    assert d["kf"][0] == pytest.approx(1.0e9, rel=1e-14)
    assert d["kr"][0] == pytest.approx(1.0e9, rel=1e-13)
    q = 1.0e9 * (C[0] * C[1] - C[2] * C[3])
    np.testing.assert_allclose(d["omega"], np.array([-q, -q, q, q, 0.0]), rtol=1e-12, atol=0)


def test_single_reaction_association_closed_form(Oracle):
    """A+B<=>C with constant-cp species: g/RT = a1 + a6/T - a1 ln T - a7 in closed form,
    K_c = exp(-(g_C - g_A - g_B)) (p_ref/RT)^(-1); with identical g sets k_r = A p_ref/(RT) e^{-g}."""
    W = [1.0, 16.0, 17.0]
    sets = [(3.5, -500.0, 3.0), (2.5, 1500.0, 6.0), (4.0, -4000.0, 8.0)]
    nasa = [const_cp_nasa(*s) for s in sets]
    m = tiny_mech(W, [rxn([(0, 1), (1, 1)], [(2, 1)], A=3.0e13, beta=0.0, Ea=0.0)], nasa=(nasa, nasa))
    X = np.array([0.3, 0.3, 0.4])
    T, p = 900.0, 3.0e5
    g = [a1 + a6 / T - a1 * np.log(T) - a7 for a1, a6, a7 in sets]
    Kc = np.exp(-(g[2] - g[0] - g[1])) * (R * T / P_REF)
    d = Oracle(m).rates_detail(T, p, mass_from_mole(X, W))
    C = _conc(X, T, p)
    assert d["kf"][0] == pytest.approx(3.0e10, rel=1e-14)
    assert d["kr"][0] == pytest.approx(3.0e10 / Kc, rel=1e-12)
    q = 3.0e10 * C[0] * C[1] - 3.0e10 / Kc * C[2]
    np.testing.assert_allclose(d["omega"], [-q, -q, q], rtol=1e-11)


def test_arrhenius_units_and_temperature_dependence(Oracle):
    """Ea = R*1500 K => exp(-1500/T); beta = 0.5 => sqrt(T); third-body A in cm^6/mol^2/s => 1e-6;
    2A <=> B uses C_A^2 and order 2."""
    W = [10.0, 20.0, 30.0]
    rx = [rxn([(0, 1), (1, 1)], [(2, 1)], A=2.0e10, beta=0.5, Ea=R_KJ_MOL * 1500.0),
          rxn([(0, 1), (1, 1)], [(2, 1)], A=5.0e15, beta=-1.0, Ea=0.0, type="three_body"),
          rxn([(0, 2)], [(1, 1)], A=7.0e11, beta=0.0, Ea=R_KJ_MOL * 300.0)]
    m = tiny_mech(W, rx)
    X = np.array([0.5, 0.2, 0.3])
    for T in (400.0, 1700.0):
        p = 1.7e5
        d = Oracle(m).rates_detail(T, p, mass_from_mole(X, W))
        C = _conc(X, T, p)
        assert d["kf"][0] == pytest.approx(2.0e7 * np.sqrt(T) * np.exp(-1500.0 / T), rel=1e-13)
        assert d["kf"][1] == pytest.approx(5.0e9 / T, rel=1e-13)
        assert d["M"][1] == pytest.approx(p / (R * T), rel=1e-14)
        assert d["Qf"][1] == pytest.approx(5.0e9 / T * C[0] * C[1] * p / (R * T), rel=1e-13)
        assert d["kf"][2] == pytest.approx(7.0e8 * np.exp(-300.0 / T), rel=1e-13)
        assert d["Qf"][2] == pytest.approx(7.0e8 * np.exp(-300.0 / T) * C[0] ** 2, rel=1e-13)
    # species 0 is consumed twice per event of reaction 2
    m2 = tiny_mech(W, [rx[2]])
    d = Oracle(m2).rates_detail(1000.0, 1e5, mass_from_mole(X, W))
    q = d["Qf"][0] - d["Qr"][0]
    np.testing.assert_allclose(d["omega"], [-2 * q, q, 0.0], rtol=1e-13)


# ------------------------------------------------------------------ equilibrium (step 7)
@pytest.mark.parametrize("products", [[(2, 1)], [(2, 1), (3, 1)]])
def test_zero_net_rate_at_gibbs_minimum(Oracle, products):
    """Independent principle: the composition minimising G(T,p) = sum n_k (g_k + RT ln(X_k p/p_ref))
    along the reaction coordinate (found with mpmath at 50 digits, no law of mass action typed)
    must give zero net rate: |q| <= 1e-10 (|Q_f| + |Q_r|).  Fixes the sign of Delta G, the
    (p_ref/RT)^dnu factor and the use of p_ref in K_c."""
    m = wl.make_mechanism(None, **SMALL)
    W = m["W"][:4]
    sub = tiny_mech(W, [rxn([(0, 1), (1, 1)], products, A=4.0e11, beta=0.3, Ea=40.0)],
                    nasa=(m["nasa_lo"][:4], m["nasa_hi"][:4]), Tmid=m["nasa_Tmid"][:4])
    o = Oracle(sub)
    for T, p in ((800.0, 1.0e5), (1500.0, 3.0e6), (2400.0, 2.0e4)):
        g = [mp.mpf(float(x)) for x in o.thermo_species([T])["g_RT"][:, 0]]
        inert = mp.mpf("0.7")

        def G(xi):
            n = [1 - xi, 1 - xi, mp.mpf(0), mp.mpf(0)]
            for k, _ in products:
                n[k] = xi
            if len(products) == 1:
                n[3] = inert
            tot = sum(n)
            return sum(nk * (g[k] + mp.log(nk / tot * mp.mpf(p) / mp.mpf(P_REF))) for k, nk in enumerate(n) if nk > 0)

        # golden-section style: solve dG/dxi = 0 by bisection on a numerical derivative
        f = lambda x: mp.diff(G, x)  # noqa: E731
        lo, hi = mp.mpf("1e-40"), 1 - mp.mpf("1e-40")
        for _ in range(200):
            mid = (lo + hi) / 2
            if f(mid) < 0:
                lo = mid
            else:
                hi = mid
        xi = (lo + hi) / 2
        n = [1 - xi, 1 - xi, mp.mpf(0), mp.mpf(0)]
        for k, _ in products:
            n[k] = xi
        if len(products) == 1:
            n[3] = inert
        X = np.array([float(x / sum(n)) for x in n])
        d = o.rates_detail(T, p, mass_from_mole(X, W))
        assert abs(d["Qf"][0] - d["Qr"][0]) <= 1e-10 * (abs(d["Qf"][0]) + abs(d["Qr"][0])), (T, p, xi)


def test_vant_hoff(Oracle):
    """d ln K_p / dT = Delta h / (R T^2) with K_p = (k_f/k_r) (RT/p_ref)^dnu: ties step 7 to step 2."""
    m = wl.make_mechanism(None, **SMALL)
    rx = [rxn([(0, 1), (1, 1)], [(2, 1)], A=1e12, beta=0.7, Ea=55.0),
          rxn([(3, 1), (4, 1)], [(5, 1), (6, 1)], A=1e10, beta=-0.4, Ea=12.0)]
    sub = dict(m, reactions=rx)
    o = Oracle(sub)
    Y = np.full(len(m["W"]), 1.0 / len(m["W"]))
    for T in (450.0, 1250.0, 2200.0):
        dT = 0.01
        lnKp = []
        for t in (T - dT, T + dT):
            d = o.rates_detail(t, 1e5, Y)
            lnKp.append(np.log(d["kf"] / d["kr"]) + np.array([-1.0, 0.0]) * np.log(R * t / P_REF))
        hk = o.thermo_species([T])["hk"][:, 0]
        dh = np.array([hk[2] - hk[0] - hk[1], hk[5] + hk[6] - hk[3] - hk[4]])
        np.testing.assert_allclose((lnKp[1] - lnKp[0]) / (2 * dT), dh / (R * T * T), rtol=2e-6)


# ------------------------------------------------------------------ third body, falloff (steps 5, 6)
def test_third_body_efficiencies(Oracle):
    W = [2.0, 32.0, 34.0, 28.0]
    X = np.array([0.2, 0.3, 0.1, 0.4])
    T, p = 1100.0, 2.0e5
    base = rxn([(0, 1), (1, 1)], [(2, 1)], A=1e16, type="three_body")
    d1 = Oracle(tiny_mech(W, [base])).rates_detail(T, p, mass_from_mole(X, W))
    assert d1["M"][0] == pytest.approx(p / (R * T), rel=1e-14)            # all eps = 1 -> [M] = C_tot
    scaled = rxn([(0, 1), (1, 1)], [(2, 1)], A=1e16, type="three_body", eff={k: 2.5 for k in range(4)})
    d2 = Oracle(tiny_mech(W, [scaled])).rates_detail(T, p, mass_from_mole(X, W))
    np.testing.assert_allclose(d2["omega"], 2.5 * d1["omega"], rtol=1e-13)
    one = rxn([(0, 1), (1, 1)], [(2, 1)], A=1e16, type="three_body", eff={3: 0.0, 1: 3.0})
    d3 = Oracle(tiny_mech(W, [one])).rates_detail(T, p, mass_from_mole(X, W))
    C = _conc(X, T, p)
    assert d3["M"][0] == pytest.approx(C[0] + 3.0 * C[1] + C[2], rel=1e-14)
    # k_f itself carries no [M]
    assert d3["kf"][0] == pytest.approx(d1["kf"][0], rel=1e-15)


def _falloff(A, A0, troe_extra, eff=None):
    troe = dict(A0=A0, beta0=0.0, Ea0=0.0, **troe_extra)
    return rxn([(0, 1), (1, 1)], [(2, 1)], A=A, type="falloff", eff=eff or {}, troe=troe)


def test_falloff_lindemann_limits(Oracle):
    """alpha=1, T*=T***=1e300, T**=1e300 => F_cent = 1 => F = 1: k = k_inf k0[M]/(k_inf + k0[M])
    (Lindemann); P_r -> 0 gives k0[M], P_r -> inf gives k_inf."""
    W = [2.0, 32.0, 34.0]
    X = np.array([0.3, 0.3, 0.4])
    T, p = 1000.0, 1.0e5
    lind = dict(alpha=1.0, T3=1e300, T1=1e300, T2=1e300)
    Mtot = p / (R * T)
    kinf = 1e13 * 1e-3
    for A0, expect in ((1e2, None), (1e40, None), (1e16 * 1.0, None)):
        d = Oracle(tiny_mech(W, [_falloff(1e13, A0, lind)])).rates_detail(T, p, mass_from_mole(X, W))
        k0M = A0 * 1e-6 * Mtot
        assert d["kf"][0] == pytest.approx(kinf * k0M / (kinf + k0M), rel=1e-13)
    d = Oracle(tiny_mech(W, [_falloff(1e13, 1e2, lind)])).rates_detail(T, p, mass_from_mole(X, W))
    assert d["kf"][0] == pytest.approx(1e2 * 1e-6 * Mtot, rel=1e-9)             # low-pressure limit
    d = Oracle(tiny_mech(W, [_falloff(1e13, 1e40, lind)])).rates_detail(T, p, mass_from_mole(X, W))
    assert d["kf"][0] == pytest.approx(kinf, rel=1e-9)                          # high-pressure limit
    # a falloff rate of progress has no extra [M] factor: Q_f = k_f C_A C_B
    C = _conc(X, T, p)
    assert d["Qf"][0] == pytest.approx(d["kf"][0] * C[0] * C[1], rel=1e-14)


def test_falloff_troe_centre_and_asymptote(Oracle):
    """At log10 P_r = -c (c = -0.4 - 0.67 log10 F_cent) the Troe exponent is 1: F = F_cent exactly.
    At log10 P_r + c = N/1.14 it is 1/2: F = sqrt(F_cent).  As P_r -> inf, f1 -> -1/0.14, so
    log10 F -> log10 F_cent / (1 + 1/0.14^2)."""
    W = [2.0, 32.0, 34.0]
    X = np.array([0.3, 0.3, 0.4])
    T, p = 1300.0, 1.0e5
    troe = dict(alpha=0.6, T3=200.0, T1=1500.0, T2=4000.0)
    Fc = 0.4 * np.exp(-T / 200.0) + 0.6 * np.exp(-T / 1500.0) + np.exp(-4000.0 / T)
    c = -0.4 - 0.67 * np.log10(Fc)
    Mtot = p / (R * T)
    kinf = 1e13 * 1e-3
    A0 = 10.0 ** (-c) * kinf / Mtot / 1e-6          # makes P_r = 10^-c
    d = Oracle(tiny_mech(W, [_falloff(1e13, A0, troe)])).rates_detail(T, p, mass_from_mole(X, W))
    Pr = 10.0 ** (-c)
    assert d["kf"][0] == pytest.approx(kinf * Pr / (1 + Pr) * Fc, rel=1e-11)
    # at log10 P_r + c = N/1.14 (N = 0.75 - 1.27 log10 F_cent) f1 = 1: F = sqrt(F_cent)
    N = 0.75 - 1.27 * np.log10(Fc)
    Pr = 10.0 ** (N / 1.14 - c)
    d = Oracle(tiny_mech(W, [_falloff(1e13, Pr * kinf / Mtot / 1e-6, troe)])).rates_detail(
        T, p, mass_from_mole(X, W))
    assert d["kf"][0] == pytest.approx(kinf * Pr / (1 + Pr) * np.sqrt(Fc), rel=1e-11)
    # far above the centre (log10 P_r ~ 240, the most a double allows) F is within 10 % of its limit
    d = Oracle(tiny_mech(W, [_falloff(1e13, 1e250, troe)])).rates_detail(T, p, mass_from_mole(X, W))
    assert np.log10(d["kf"][0] / kinf) == pytest.approx(np.log10(Fc) / (1 + 1 / 0.14 ** 2), rel=0.1)
    # efficiencies enter P_r: doubling every efficiency at small P_r doubles k_f (Lindemann part)
    lind = dict(alpha=1.0, T3=1e300, T1=1e300, T2=1e300)
    a = Oracle(tiny_mech(W, [_falloff(1e13, 1e3, lind)])).rates_detail(T, p, mass_from_mole(X, W))
    b = Oracle(tiny_mech(W, [_falloff(1e13, 1e3, lind, eff={0: 2.0, 1: 2.0, 2: 2.0})])).rates_detail(
        T, p, mass_from_mole(X, W))
    assert b["kf"][0] == pytest.approx(2.0 * a["kf"][0], rel=1e-8)


# ------------------------------------------------------------------ omega as a whole (steps 8, 9)
@pytest.mark.parametrize("cfg,hf", [("C1", "uniform"), ("C3", "uniform"), ("C3", "group"),
                                    ("C4", "group"), ("C5", "uniform")])
def test_mass_and_element_conservation(Oracle, cfg, hf):
    """sum_k W_k omega_k = 0 and sum_k a_ek omega_k = 0 for every element."""
    m = wl.make_mechanism(cfg, hf=hf)
    st = wl.make_state(cfg, n=96)
    r = Oracle(m).production_rates(**st)
    assert np.all(np.isfinite(r["omega"])) and np.all(np.isfinite(r["qdot"]))
    assert np.all(np.abs(m["W"] @ r["omega"]) <= 1e-12 * (m["W"] @ r["S_omega"]))
    assert np.all(np.abs(m["comp"] @ r["omega"]) <= 1e-12 * (m["comp"] @ r["S_omega"]) + 1e-300)
    assert np.all(r["omega"][-1] == 0.0)          # the inert species takes part in no reaction


def test_metamorphic_relations(Oracle):
    m = wl.make_mechanism(None, **SMALL)
    st = wl.make_state("C3", n=16, Ns=SMALL["Ns"], p="range")
    base = Oracle(m).production_rates(**st)
    tol = 1e-12 * base["S_omega"] + 1e-300
    # reaction order is immaterial
    perm = np.random.default_rng(3).permutation(len(m["reactions"]))
    r = Oracle(dict(m, reactions=[m["reactions"][i] for i in perm])).production_rates(**st)
    assert np.all(np.abs(r["omega"] - base["omega"]) <= tol)
    # splitting a reaction into two duplicates with A/2 each changes nothing
    rx = list(m["reactions"])
    i = next(i for i, x in enumerate(rx) if x["type"] == "elementary")
    half = dict(rx[i], A=rx[i]["A"] / 2)
    r = Oracle(dict(m, reactions=rx[:i] + [half, half] + rx[i + 1:])).production_rates(**st)
    assert np.all(np.abs(r["omega"] - base["omega"]) <= tol)
    # relabelling the species permutes the outputs
    sp = np.random.default_rng(4).permutation(len(m["W"]))
    inv = np.argsort(sp)
    pm = dict(m, W=m["W"][sp], nasa_Tmid=m["nasa_Tmid"][sp], nasa_lo=m["nasa_lo"][sp], nasa_hi=m["nasa_hi"][sp],
              comp=m["comp"][:, sp], mu_fit=m["mu_fit"][sp], lam_fit=m["lam_fit"][sp],
              D_fit=m["D_fit"][sp][:, sp],
              reactions=[dict(x, reactants=[(int(inv[k]), nu) for k, nu in x["reactants"]],
                              products=[(int(inv[k]), nu) for k, nu in x["products"]],
                              **({"eff": {int(inv[k]): e for k, e in x["eff"].items()}} if "eff" in x else {}))
                         for x in m["reactions"]])
    pst = dict(st, Y=st["Y"][sp])
    r = Oracle(pm).production_rates(**pst)
    assert np.all(np.abs(r["omega"] - base["omega"][sp]) <= tol[sp])
    np.testing.assert_allclose(r["qdot"], base["qdot"], rtol=0, atol=1e-12 * base["S_q"].max())
    t0, t1 = Oracle(m).mix_transport(**st), Oracle(pm).mix_transport(**pst)
    np.testing.assert_allclose(t1["mu"], t0["mu"], rtol=1e-13)
    np.testing.assert_allclose(t1["lam"], t0["lam"], rtol=1e-13)
    np.testing.assert_allclose(t1["rhoD"], t0["rhoD"][sp], rtol=1e-13)
    # doubling A of one reaction doubles its rate of progress and nothing else
    o = Oracle(m)
    d0 = o.rates_detail(st["T"][0], st["p"][0], st["Y"][:, 0])
    rx2 = list(m["reactions"])
    rx2[i] = dict(rx2[i], A=2 * rx2[i]["A"])
    d1 = Oracle(dict(m, reactions=rx2)).rates_detail(st["T"][0], st["p"][0], st["Y"][:, 0])
    ratio = np.ones(len(rx))
    ratio[i] = 2.0
    np.testing.assert_allclose(d1["Qf"], ratio * d0["Qf"], rtol=1e-14)
    np.testing.assert_allclose(d1["Qr"], ratio * d0["Qr"], rtol=1e-14)


def test_heat_release_identity(Oracle):
    """qdot = -sum_k h_k omega_k = -sum_r q_r Delta h_r"""
    m = wl.make_mechanism(None, **SMALL)
    st = wl.make_state("C3", n=8, Ns=SMALL["Ns"])
    o = Oracle(m)
    nu = o.nu
    for i in range(8):
        d = o.rates_detail(st["T"][i], st["p"][i], st["Y"][:, i])
        hk = o.thermo_species([st["T"][i]])["hk"][:, 0]
        dh = nu @ hk
        scale = np.sum(np.abs(nu) @ np.abs(hk) * (np.abs(d["Qf"]) + np.abs(d["Qr"])))
        assert abs(d["qdot"] + np.sum((d["Qf"] - d["Qr"]) * dh)) <= 1e-12 * scale
    r = o.production_rates(**st)
    assert r["qdot"][0] == pytest.approx(o.rates_detail(st["T"][0], st["p"][0], st["Y"][:, 0])["qdot"], rel=1e-15)


# ------------------------------------------------------------------ transport (steps 10-13)
def test_pure_species_limits(Oracle):
    """Y_k = 1 => mu = mu_k(T), lambda = lambda_k(T) (Phi_kk = 1), D_km = D_kk (guard), for fits
    evaluated here as exp(polyval)."""
    m = wl.make_mechanism("C3")
    o = Oracle(m)
    T = np.array([350.0, 1600.0])
    lnT = np.log(T)
    for k in (0, 7, 20):
        Y = np.zeros((21, 2))
        Y[k] = 1.0
        t = o.mix_transport(T, np.array([1e5, 7e5]), Y)
        fit = lambda c: np.exp(c[0] + c[1] * lnT + c[2] * lnT ** 2 + c[3] * lnT ** 3)  # noqa: E731
        np.testing.assert_allclose(t["mu"], fit(m["mu_fit"][k]), rtol=1e-13)
        np.testing.assert_allclose(t["lam"], fit(m["lam_fit"][k]), rtol=1e-13)
        np.testing.assert_allclose(t["Dkm"][k], fit(m["D_fit"][k, k]) * P_REF / np.array([1e5, 7e5]), rtol=1e-13)


def test_wilke_and_conductivity_special_cases(Oracle):
    # identical W and mu => mu_mix = mu whatever the composition (all Phi = 1)
    m = tiny_mech([20.0, 20.0, 20.0], [], mu=[3e-5] * 3, lam=[0.1, 0.1, 0.1])
    Y = col([0.2, 0.5, 0.3])
    t = Oracle(m).mix_transport([700.0], [1e5], Y)
    assert t["mu"][0] == pytest.approx(3e-5, rel=1e-14)
    assert t["lam"][0] == pytest.approx(0.1, rel=1e-14)
    # conductivity: half arithmetic plus half harmonic mole-fraction mean
    m = tiny_mech([20.0, 20.0], [], lam=[0.1, 0.3])
    t = Oracle(m).mix_transport([700.0], [1e5], col([0.5, 0.5]))
    assert t["lam"][0] == pytest.approx(0.5 * (0.2 + 1.0 / (0.5 / 0.1 + 0.5 / 0.3)), rel=1e-14)
    # Wilke, binary, equal masses, mu_1 = 4 mu_2: Phi_12 = (1+2)^2/4 = 9/4, Phi_21 = (1+1/2)^2/4 = 9/16
    m = tiny_mech([20.0, 20.0], [], mu=[4e-5, 1e-5])
    t = Oracle(m).mix_transport([700.0], [1e5], col([0.5, 0.5]))
    expect = 0.5 * 4e-5 / (0.5 + 0.5 * 9 / 4) + 0.5 * 1e-5 / (0.5 + 0.5 * 9 / 16)
    assert t["mu"][0] == pytest.approx(expect, rel=1e-14)
    # Wilke, equal viscosities, W_1 = 16 W_2 (fourth root exact): Phi_12 = (1 + 1/2)^2/sqrt(8*17),
    # Phi_21 = (1 + 2)^2/sqrt(8*(1+1/16))
    m = tiny_mech([32.0, 2.0], [], mu=[2e-5, 2e-5])
    X = np.array([0.25, 0.75])
    t = Oracle(m).mix_transport([700.0], [1e5], col(mass_from_mole(X, [32.0, 2.0])))
    P12, P21 = 1.5 ** 2 / np.sqrt(8 * 17.0), 3.0 ** 2 / np.sqrt(8 * (1 + 1 / 16.0))
    expect = X[0] * 2e-5 / (X[0] + X[1] * P12) + X[1] * 2e-5 / (X[1] + X[0] * P21)
    assert t["mu"][0] == pytest.approx(expect, rel=1e-13)


def test_mixture_averaged_diffusion_special_cases(Oracle):
    # binary: D_1m = D_12 (1 - Y_1)/X_2, equal masses => D_12
    D = np.array([[5e-5, 2e-4], [2e-4, 7e-5]])
    t = Oracle(tiny_mech([20.0, 20.0], [], D=D)).mix_transport([900.0], [P_REF], col([0.3, 0.7]))
    np.testing.assert_allclose(t["Dkm"][:, 0], [2e-4, 2e-4], rtol=1e-14)
    W = [4.0, 40.0]
    X = np.array([0.6, 0.4])
    Y = mass_from_mole(X, W)
    t = Oracle(tiny_mech(W, [], D=D)).mix_transport([900.0], [P_REF], col(Y))
    np.testing.assert_allclose(t["Dkm"][:, 0], [2e-4 * (1 - Y[0]) / X[1], 2e-4 * (1 - Y[1]) / X[0]], rtol=1e-14)
    # all D_jk = D0 and equal masses => D_km = D0 ; D ~ p_ref/p
    t = Oracle(tiny_mech([20.0] * 4, [], D=np.full((4, 4), 3e-4))).mix_transport(
        [900.0, 900.0], [P_REF, 4 * P_REF], np.array([[0.1, 0.1], [0.2, 0.2], [0.3, 0.3], [0.4, 0.4]]))
    np.testing.assert_allclose(t["Dkm"][:, 0], 3e-4, rtol=1e-14)
    np.testing.assert_allclose(t["Dkm"][:, 1], 0.75e-4, rtol=1e-14)
    # rho = p Wbar/(R T)
    assert t["rhoD"][0, 0] == pytest.approx(P_REF * 20.0 / (R * 900.0) * 3e-4, rel=1e-14)


def test_transport_pressure_independence(Oracle):
    """mu, lambda and rho*D_km do not depend on p (rho ~ p, D ~ 1/p)."""
    m = wl.make_mechanism("C3")
    st = wl.make_state("C3", n=32)
    o = Oracle(m)
    a = o.mix_transport(st["T"], st["p"], st["Y"])
    b = o.mix_transport(st["T"], 13.7 * st["p"], st["Y"])
    np.testing.assert_allclose(b["mu"], a["mu"], rtol=1e-15)
    np.testing.assert_allclose(b["lam"], a["lam"], rtol=1e-15)
    np.testing.assert_allclose(b["rhoD"], a["rhoD"], rtol=1e-14)
    np.testing.assert_allclose(b["Dkm"] * 13.7, a["Dkm"], rtol=1e-14)


# ------------------------------------------------------------------ rounding (all steps)
@pytest.mark.parametrize("which", ["C1", "small"])
def test_against_mpmath(Oracle, which):
    if which == "C1":
        m, st = wl.make_mechanism("C1"), wl.make_state("C1", n=6)
    else:
        m = wl.make_mechanism(None, hf="group", **SMALL)
        st = wl.make_state("C3", n=5, Ns=SMALL["Ns"], p="range")
    o = Oracle(m)
    th, r, t = o.thermo(**st), o.production_rates(**st), o.mix_transport(**st)
    for i in range(st["T"].size):
        ref = mp_reference.evaluate(m, st["T"][i], st["p"][i], st["Y"][:, i])
        assert abs(th["cp"][i] - ref["cp"]) <= 1e-14 * abs(ref["cp"])
        # the two tolerance scales the GPU parity tests divide by (tests/parity.py) are themselves pinned
        assert abs(th["h_scale"][i] - ref["h_scale"]) <= 1e-12 * ref["h_scale"]
        assert abs(r["S_q"][i] - ref["S_q"]) <= 1e-12 * ref["S_q"]
        assert abs(th["h"][i] - ref["h"]) <= 1e-14 * ref["h_scale"]
        for k in range(len(m["W"])):
            assert abs(r["omega"][k, i] - ref["omega"][k]) <= 2e-13 * ref["S_omega"][k] + 1e-300, (i, k)
            assert abs(r["S_omega"][k, i] - ref["S_omega"][k]) <= 1e-12 * ref["S_omega"][k]
            assert abs(t["rhoD"][k, i] - ref["rhoD"][k]) <= 1e-13 * ref["rhoD"][k]
        assert abs(r["qdot"][i] - ref["qdot"]) <= 2e-13 * ref["S_q"]
        assert abs(t["mu"][i] - ref["mu"]) <= 1e-13 * ref["mu"]
        assert abs(t["lam"][i] - ref["lam"]) <= 1e-13 * ref["lam"]
