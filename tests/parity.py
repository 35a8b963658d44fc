"""GPU-vs-oracle comparison with the tolerances of BASELINE.json ``north_star``:

* omega_k:  |gpu - ref| <= 1e-10 * S_k + 1e-30,  S_k = sum_r |nu_kr| (|Q_f| + |Q_r|)
* qdot:     |gpu - ref| <= 1e-10 * S_q + 1e-30,  S_q = sum_k |h_k| S_k   (SURVEY 8(c) reading)
* cp, mu, lambda, rhoD: 1e-12 relative
* h: 1e-12 relative to max(|h|, 1e-3 * sum_k |Y_k h_k / W_k|) (SURVEY 8(c) reading: the mixture
  enthalpy passes through zero; the strict |h| form is returned too for reporting)

The scales S_k, S_q and the h scale come from the oracle (they are part of the tolerance
definition, not of the result).  Test infrastructure: imports oracle/ and the binding.
"""
import numpy as np
import torch

RTOL = 1e-12
RATE_TOL = 1e-10


def to_dev(st, device="cuda"):
    return {k: torch.from_numpy(np.ascontiguousarray(v)).to(device) for k, v in st.items()}


def run_gpu(mech_gpu, st):
    """All three calls on device tensors made from the numpy state; numpy results."""
    d = to_dev(st)
    cp, h = mech_gpu.thermo(d["T"], d["p"], d["Y"])
    omega, qdot = mech_gpu.production_rates(d["T"], d["p"], d["Y"])
    mu, lam, rhoD = mech_gpu.mix_transport(d["T"], d["p"], d["Y"])
    torch.cuda.synchronize()
    return {k: v.cpu().numpy() for k, v in dict(cp=cp, h=h, omega=omega, qdot=qdot, mu=mu, lam=lam, rhoD=rhoD).items()}


def run_oracle(oracle, st):
    th, r, t = oracle.thermo(**st), oracle.production_rates(**st), oracle.mix_transport(**st)
    return dict(cp=th["cp"], h=th["h"], h_scale=th["h_scale"], omega=r["omega"], qdot=r["qdot"],
                S_omega=r["S_omega"], S_q=r["S_q"], mu=t["mu"], lam=t["lam"], rhoD=t["rhoD"])


def _rel(a, b, scale=None):
    scale = np.abs(b) if scale is None else scale
    with np.errstate(divide="ignore", invalid="ignore"):
        e = np.abs(a - b) / scale
    e[(a == b)] = 0.0
    return e


def errors(gpu, ref):
    """Worst error of each output in units of its tolerance (<= 1 passes), plus raw maxima."""
    out = {}
    for key in ("cp", "mu", "lam", "rhoD"):
        out[key] = float(np.max(_rel(gpu[key], ref[key]), initial=0.0)) / RTOL
    hs = np.maximum(np.abs(ref["h"]), 1e-3 * ref["h_scale"])
    out["h"] = float(np.max(_rel(gpu["h"], ref["h"], hs), initial=0.0)) / RTOL
    out["h_strict"] = float(np.max(_rel(gpu["h"], ref["h"]), initial=0.0)) / RTOL
    out["omega"] = float(np.max(np.abs(gpu["omega"] - ref["omega"]) / (RATE_TOL * ref["S_omega"] + 1e-30),
                                initial=0.0))
    out["qdot"] = float(np.max(np.abs(gpu["qdot"] - ref["qdot"]) / (RATE_TOL * ref["S_q"] + 1e-30), initial=0.0))
    return out


def assert_parity(gpu, ref, what=""):
    for key in ("cp", "h", "omega", "qdot", "mu", "lam", "rhoD"):
        assert np.all(np.isfinite(gpu[key])), f"{what}: non-finite {key}"
    e = errors(gpu, ref)
    bad = {k: v for k, v in e.items() if k != "h_strict" and not v <= 1.0}
    assert not bad, f"{what}: outside tolerance (units of the tolerance): {bad}  all: {e}"
    return e
