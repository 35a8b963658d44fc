"""Writes tests/golden/oracle_C1.json: the oracle's outputs on the first 8 points of C1.

Calls only oracle/ and the seeded input generator -- never the CUDA path.  The paper prints
no value for this path (PAPER.md gives S_L, delta_f and an ignition-delay error, all of which
need the Li et al. mechanism and a flow solver), so this fixture is a regression guard for the
oracle itself, not a citation.  Run:  python tests/golden/make_golden.py
"""
import json
import os
import sys

ROOT = os.path.dirname(os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
sys.path.insert(0, ROOT)

from oracle import crf_oracle  # noqa: E402
from paper_2409_06404_b200 import workloads as wl  # noqa: E402


def main():
    mech, st = wl.make_mechanism("C1"), wl.make_state("C1", n=8)
    o = crf_oracle.Oracle(mech)
    th, r, t = o.thermo(**st), o.production_rates(**st), o.mix_transport(**st)
    out = dict(source="oracle/crf_oracle.c on workloads.make_mechanism('C1'), make_state('C1', n=8)",
               T=st["T"].tolist(), p=st["p"].tolist(), Y=st["Y"].tolist(),
               cp=th["cp"].tolist(), h=th["h"].tolist(), omega=r["omega"].tolist(), qdot=r["qdot"].tolist(),
               S_omega=r["S_omega"].tolist(), S_q=r["S_q"].tolist(),
               mu=t["mu"].tolist(), lam=t["lam"].tolist(), rhoD=t["rhoD"].tolist())
    with open(os.path.join(os.path.dirname(os.path.abspath(__file__)), "oracle_C1.json"), "w") as f:
        json.dump(out, f, indent=1)


if __name__ == "__main__":
    main()
