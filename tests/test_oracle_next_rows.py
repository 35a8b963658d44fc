"""Pins of the oracle functions behind SURVEY.md 8(f) rows 1 and 2 (the fused right-hand-side evaluation and the
difference quotient of the Jacobian-vector product): closed forms and identities the mathematics fixes.  CPU only."""
import numpy as np
import pytest

from paper_2409_06404_b200 import workloads as wl
from tests.helpers import P_REF, R, col, rxn, tiny_mech


@pytest.fixture(scope="module")
def Oracle(oracle_mod):
    return oracle_mod.Oracle


def test_rhs_density_and_mean_molar_mass_closed_form(Oracle):
    """rho = p Wbar / (R T) (Eq. 1d) and Wbar = 1 / sum Y_k / W_k by hand: a pure species has
    Wbar = W_k; a 50/50 mass mixture of W = 2 and W = 32 has Wbar = 1 / (0.25 + 0.015625); air-like numbers give the
    textbook density 1.177 kg/m^3 at 300 K, 1 atm for W = 28.97."""
    m = tiny_mech([2.0, 32.0, 28.97], [])
    T = np.array([300.0, 300.0, 1500.0, 300.0])
    p = np.array([P_REF, P_REF, 5.0 * P_REF, P_REF])
    Y = np.array([[1.0, 0.5, 0.5, 0.0], [0.0, 0.5, 0.5, 0.0], [0.0, 0.0, 0.0, 1.0]])
    r = Oracle(m).rhs_pointwise(T, p, Y)
    Wb = np.array([2.0, 1.0 / (0.25 + 0.015625), 1.0 / (0.25 + 0.015625), 28.97])
    np.testing.assert_allclose(r["Wbar"], Wb, rtol=1e-15)
    np.testing.assert_allclose(r["rho"], p * Wb / (R * T), rtol=1e-15)
    assert abs(r["rho"][3] - 1.1769) < 2e-4  # (the ideal-gas density of air at 300 K, 1 atm)
    # rho scales with p and 1/T, and sum_k C_k = p / (R T) whatever the composition
    assert r["rho"][2] / r["rho"][1] == pytest.approx(5.0 * 300.0 / 1500.0, rel=1e-15)


@pytest.mark.parametrize("cfg", ["C1", "C3"])
def test_rhs_is_the_three_calls_plus_species_heat_capacities(Oracle, cfg):
    """oracle_rhs_pointwise is a composition: every shared output is bit-identical to the separate calls, cpk is the
    molar heat capacity of thermo_species, and c_p = sum_k Y_k cpk / W_k ties cpk to the mixture value."""
    m = wl.make_mechanism(cfg)
    st = wl.make_state(cfg, n=96, total=96)
    o = Oracle(m)
    r = o.rhs_pointwise(**st)
    th, ra, tr, sp = o.thermo(**st), o.production_rates(**st), o.mix_transport(**st), o.thermo_species(st["T"])
    for k in ("cp", "h", "h_scale"):
        assert np.array_equal(r[k], th[k]), k
    for k in ("omega", "qdot", "S_omega", "S_q"):
        assert np.array_equal(r[k], ra[k]), k
    for k in ("mu", "lam", "rhoD"):
        assert np.array_equal(r[k], tr[k]), k
    assert np.array_equal(r["cpk"], sp["cpk"])
    np.testing.assert_allclose(np.sum(st["Y"] * r["cpk"] / m["W"][:, None], axis=0), r["cp"], rtol=1e-13)
    # rho ties the transport output to D_km: rhoD = rho D_km
    np.testing.assert_allclose(r["rhoD"], r["rho"][None, :] * tr["Dkm"], rtol=1e-14)


def test_jv_quotient_closed_form(Oracle):
    """A + B <=> C + D with beta = 0, E = 0, identical NASA sets and equal molar masses: q = A (C_A C_B - C_C C_D) with
    C_k = rho Y_k / W linear in Y_k as long as sum dY = 0 (rho is then unchanged), so the difference quotient along
    (dT, dp) = 0 is the polynomial  A (rho/W)^2 [Y_A dY_B + dY_A Y_B - Y_C dY_D - dY_C Y_D + sigma (dY_A dY_B - dY_C dY_D)]
    exactly: this fixes the order of the subtraction, the 1/sigma and which state is perturbed."""
    A_cgs = 3.0e12
    m = tiny_mech([20.0] * 4, [rxn([(0, 1), (1, 1)], [(2, 1), (3, 1)], A=A_cgs)])
    T, p = np.array([1200.0]), np.array([2.0 * P_REF])
    Y = col([0.4, 0.3, 0.2, 0.1])
    dY = col([0.5, -1.0, 0.25, 0.25])
    for sigma in (1e-3, -2e-4, 1e-7):
        r = Oracle(m).production_rates_jv(T, p, Y, np.zeros(1), np.zeros(1), dY, sigma)
        c = p[0] * 20.0 / (R * T[0]) / 20.0  # rho / W = p / (R T)
        A_si = A_cgs * 1e-3
        lin = Y[0, 0] * dY[1, 0] + dY[0, 0] * Y[1, 0] - Y[2, 0] * dY[3, 0] - dY[2, 0] * Y[3, 0]
        quad = dY[0, 0] * dY[1, 0] - dY[2, 0] * dY[3, 0]
        Jq = A_si * c * c * (lin + sigma * quad)
        tol = 4e-16 * A_si * c * c / abs(sigma)  # two roundings of O(q) divided by sigma
        np.testing.assert_allclose(r["Jomega"][:, 0], np.array([-1.0, -1.0, 1.0, 1.0]) * Jq, rtol=0, atol=tol)
        assert r["S_Jomega"][0, 0] == pytest.approx((r["S_omega"][0, 0] + r["S_omega2"][0, 0]) / abs(sigma), rel=1e-15)


def test_jv_converges_to_the_temperature_derivative(Oracle):
    """Along v = (dT, 0, 0) the quotient tends to d omega / dT: a single reaction k = A T^beta exp(-E/RT) with identical
    NASA sets and Delta nu = 0 has d ln q / dT = beta/T + E/(R T^2) - 2/T (C_k ~ 1/T each) in closed form."""
    beta, Ea = 1.3, 40.0  # kJ/mol
    m = tiny_mech([20.0] * 4, [rxn([(0, 1), (1, 1)], [(2, 1), (3, 1)], A=1e10, beta=beta, Ea=Ea)])
    T, p = np.array([1500.0]), np.array([P_REF])
    Y = col([0.4, 0.3, 0.2, 0.1])
    o = Oracle(m)
    base = o.production_rates(T, p, Y)
    r = o.production_rates_jv(T, p, Y, np.ones(1), np.zeros(1), np.zeros((4, 1)), 1e-4)
    dlnq = beta / T[0] + Ea * 1e6 / (R * T[0] ** 2) - 2.0 / T[0]
    np.testing.assert_allclose(r["Jomega"][:, 0], base["omega"][:, 0] * dlnq, rtol=1e-6)
    assert np.array_equal(r["omega"], base["omega"]) and np.array_equal(r["qdot"], base["qdot"])


def test_pair_is_two_plain_calls(Oracle):
    m = wl.make_mechanism("C3")
    a, b = wl.make_state("C3", n=40, total=80), wl.make_state("C3", n=40, offset=40, total=80)
    o = Oracle(m)
    r = o.production_rates_pair(a["T"], a["p"], a["Y"], b["T"], b["p"], b["Y"])
    ra, rb = o.production_rates(**a), o.production_rates(**b)
    assert np.array_equal(r["omega"], ra["omega"]) and np.array_equal(r["omega2"], rb["omega"])
    assert np.array_equal(r["qdot"], ra["qdot"]) and np.array_equal(r["qdot2"], rb["qdot"])
