"""Cantera-format YAML ingestion ("a combustion model expressed in Cantera format"):
the hand-written fixture tests/golden/toy_mechanism.yaml -> description -> packer -> oracle / GPU.  The expected
description is typed by hand below (species order, stoichiometry, cgs-mol pre-exponential factors, kJ/mol
activation energies), so a slip in the equation parser or in a unit factor fails here before any kernel runs."""
import os

import numpy as np
import pytest

from paper_2409_06404_b200 import cantera_yaml, packer

HERE = os.path.dirname(os.path.abspath(__file__))
TOY = os.path.join(HERE, "golden", "toy_mechanism.yaml")
CAL = 4.184e-3  # kJ per cal


def test_toy_mechanism_description_typed_by_hand():
    m = cantera_yaml.load(TOY)
    assert m["species"] == ["X", "X2", "Z", "XZ", "X2Z", "I2"] and m["elements"] == ["H", "O", "N"]
    np.testing.assert_array_equal(m["comp"], [[1, 2, 0, 1, 2, 0], [0, 0, 1, 1, 1, 0], [0, 0, 0, 0, 0, 2]])
    np.testing.assert_allclose(m["W"], [1.008, 2.016, 15.999, 17.007, 18.015, 28.014], rtol=1e-15)
    np.testing.assert_array_equal(m["nasa_Tmid"], [1000.0, 1000.0, 900.0, 1200.0, 1000.0, 5000.0])
    np.testing.assert_array_equal(m["nasa_lo"][2], [2.95, -1.6e-03, 2.4e-06, -1.6e-09, 3.9e-13, 29150.0, 3.0])
    np.testing.assert_array_equal(m["nasa_hi"][2], [2.55, -3.0e-05, -3.0e-09, 4.5e-12, -4.0e-16, 29230.0, 4.9])
    np.testing.assert_array_equal(m["nasa_lo"][5], m["nasa_hi"][5])  # a single range serves both
    r = m["reactions"]
    assert len(r) == 5
    assert (r[0]["type"], sorted(r[0]["reactants"]), sorted(r[0]["products"])) == ("elementary", [(1, 1), (2, 1)], [(0, 1), (3, 1)])
    assert (r[0]["A"], r[0]["beta"]) == (5.0e4, 2.7) and r[0]["Ea"] == pytest.approx(6290.0 * CAL, rel=1e-15)
    assert (r[1]["type"], sorted(r[1]["reactants"]), r[1]["products"]) == ("three_body", [(0, 1), (3, 1)], [(4, 1)])
    assert (r[1]["A"], r[1]["beta"], r[1]["Ea"]) == (4.0e22, -2.0, 0.0) and r[1]["eff"] == {1: 2.5, 4: 12.0, 5: 1.0}
    assert (r[2]["type"], r[2]["reactants"], r[2]["products"]) == ("falloff", [(0, 2)], [(1, 1)])
    assert (r[2]["A"], r[2]["beta"]) == (1.5e12, 0.6) and r[2]["eff"] == {1: 2.0, 4: 11.0}
    assert r[2]["troe"] == dict(A0=6.0e19, beta0=-1.4, Ea0=0.0, alpha=0.8, T3=1e-30, T1=1e30, T2=1e300)
    for k in (3, 4):
        assert (r[k]["type"], r[k]["reactants"], sorted(r[k]["products"]), r[k]["duplicate"]) == \
            ("elementary", [(3, 2)], [(2, 1), (4, 1)], True)
    assert r[3]["Ea"] == pytest.approx(-2110.0 * CAL, rel=1e-15) and r[4]["A"] == 1.2e10
    np.testing.assert_array_equal(m["mu_fit"][4], [-21.0, 2.70, -0.210, 0.0075])
    np.testing.assert_array_equal(m["D_fit"][1, 4], [-20.3, 2.26, -0.053, 0.0021])
    np.testing.assert_array_equal(m["D_fit"], np.transpose(m["D_fit"], (1, 0, 2)))
    packer.pack(m)  # the packer takes it as it takes the synthetic descriptions


def test_units_block_si_gives_the_same_description():
    """The same file in Cantera's default units (m, kmol, J/kmol): A scales by (1e-3 m^3/kmol per cm^3/mol)^(order-1)."""
    text = open(TOY).read()
    si = (text.replace("units: {length: cm, quantity: mol, activation-energy: cal/mol}", "")
          .replace("{A: 5.0e+04, b: 2.7, Ea: 6290.0}", "{A: 5.0e+01, b: 2.7, Ea: 26317360.0}")
          .replace("{A: 4.0e+22, b: -2.0, Ea: 0.0}", "{A: 4.0e+16, b: -2.0, Ea: 0.0}")
          .replace("{A: 6.0e+19, b: -1.4, Ea: 0.0}", "{A: 6.0e+13, b: -1.4, Ea: 0.0}")
          .replace("{A: 1.5e+12, b: 0.6, Ea: 0.0}", "{A: 1.5e+09, b: 0.6, Ea: 0.0}")
          .replace("{A: 3.6e+04, b: 2.4, Ea: -2110.0}", "{A: 3.6e+01, b: 2.4, Ea: -8828240.0}")
          .replace("{A: 1.2e+10, b: 0.9, Ea: 17000.0}", "{A: 1.2e+07, b: 0.9, Ea: 71128000.0}"))
    a, b = cantera_yaml.load(TOY), cantera_yaml.load(si)
    for ra, rb in zip(a["reactions"], b["reactions"]):
        assert rb["A"] == pytest.approx(ra["A"], rel=1e-13) and rb["Ea"] == pytest.approx(ra["Ea"], rel=1e-13, abs=0)
        if ra["type"] == "falloff":
            assert rb["troe"]["A0"] == pytest.approx(ra["troe"]["A0"], rel=1e-13)


@pytest.mark.parametrize("bad, msg", [
    ("equation: X2 + Z <=> XZ + X  ", None),
    ("equation: X2 + Z => XZ + X", "irreversible"),
    ("equation: X2 + Q <=> XZ + X", "unknown species"),
    ("equation: X2 + Z <=> XZ + XZ", "not balanced"),
    ("equation: 3 X <=> X2 + X", "> 2"),
    ("equation: X2 + Z (+ X2Z) <=> XZ + X (+ X2Z)", "collider"),
])
def test_rejects_what_the_tables_cannot_hold(bad, msg):
    text = open(TOY).read().replace("equation: X2 + Z <=> XZ + X  ", bad, 1)
    if msg is None:
        cantera_yaml.load(text)
        return
    with pytest.raises(ValueError, match=msg):
        cantera_yaml.load(text)


def test_missing_transport_fits_are_reported():
    text = open(TOY).read().split("crf-transport-fits:")[0]
    with pytest.raises(ValueError, match="Lennard-Jones"):
        cantera_yaml.load(text)


def test_oracle_runs_the_toy_mechanism_and_conserves_atoms(oracle_mod):
    m = cantera_yaml.load(TOY)
    o = oracle_mod.Oracle(m)
    rng = np.random.default_rng(3)
    n = 64
    Y = rng.dirichlet(np.ones(6), n).T
    T, p = rng.uniform(400.0, 2500.0, n), rng.uniform(5e4, 2e6, n)
    r = o.production_rates(T, p, Y)
    scale = np.sum(m["W"][:, None] * r["S_omega"], axis=0)
    assert np.all(np.abs(np.sum(m["W"][:, None] * r["omega"], axis=0)) <= 1e-12 * scale)
    for e in range(3):
        assert np.all(np.abs(m["comp"][e] @ r["omega"]) <= 1e-12 * (np.abs(m["comp"][e]) @ r["S_omega"]) + 1e-300)
    # the Troe set with T3 = 1e-30, T1 = 1e30 and no T2 has F_cent = alpha: the falloff reaction is finite and active
    d = o.rates_detail(1500.0, 1e5, Y[:, 0])
    assert np.isfinite(d["kf"]).all() and d["kf"][2] > 0.0 and d["M"][2] > 0.0


@pytest.mark.gpu
def test_gpu_parity_on_the_toy_mechanism(oracle_mod):
    import torch

    from paper_2409_06404_b200 import binding
    from tests import parity
    m = cantera_yaml.load(TOY)
    gm, om = binding.Mechanism(m), oracle_mod.Oracle(m)
    rng = np.random.default_rng(4)
    n = 2049
    st = dict(T=rng.uniform(300.0, 2800.0, n), p=rng.uniform(5e4, 3e6, n), Y=np.ascontiguousarray(rng.dirichlet(0.5 * np.ones(6), n).T))
    parity.assert_parity(parity.run_gpu(gm, st), parity.run_oracle(om, st), "toy yaml")
    d = parity.to_dev(st)
    out = {k: (v.cpu().numpy() if v is not None else None) for k, v in gm.rhs_pointwise(d["T"], d["p"], d["Y"]).items()}
    parity.assert_parity(out, om.rhs_pointwise(**st), "toy yaml rhs")
    for kernel in ("group", "staged", "generic", "thread"):
        g2 = binding.Mechanism(m, options=dict(rates_kernel=kernel))
        parity.assert_parity(parity.run_gpu(g2, st), parity.run_oracle(om, st), f"toy yaml {kernel}")
    torch.cuda.synchronize()
