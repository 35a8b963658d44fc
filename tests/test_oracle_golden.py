"""Regression guard: the oracle and the seeded generator still give the stored C1 values
(tests/golden/oracle_C1.json, written by tests/golden/make_golden.py from oracle/ only)."""
import json
import os

import numpy as np

from paper_2409_06404_b200 import workloads as wl


def test_oracle_matches_stored_C1(oracle_mod):
    with open(os.path.join(os.path.dirname(__file__), "golden", "oracle_C1.json")) as f:
        g = json.load(f)
    mech, st = wl.make_mechanism("C1"), wl.make_state("C1", n=8)
    np.testing.assert_array_equal(st["T"], g["T"])          # the generator is bit-reproducible
    np.testing.assert_array_equal(st["Y"], g["Y"])
    o = oracle_mod.Oracle(mech)
    th, r, t = o.thermo(**st), o.production_rates(**st), o.mix_transport(**st)
    np.testing.assert_allclose(th["cp"], g["cp"], rtol=1e-13)
    np.testing.assert_allclose(th["h"], g["h"], rtol=1e-12)
    assert np.all(np.abs(r["omega"] - np.array(g["omega"])) <= 1e-12 * np.array(g["S_omega"]))
    assert np.all(np.abs(r["qdot"] - np.array(g["qdot"])) <= 1e-12 * np.array(g["S_q"]))
    np.testing.assert_allclose(t["mu"], g["mu"], rtol=1e-13)
    np.testing.assert_allclose(t["lam"], g["lam"], rtol=1e-13)
    np.testing.assert_allclose(t["rhoD"], g["rhoD"], rtol=1e-13)
