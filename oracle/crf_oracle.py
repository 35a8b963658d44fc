"""ctypes front end of the CPU oracle (crf_oracle.c) -- TEST INFRASTRUCTURE, NOT PRODUCT.

Only tests/, ``__graft_entry__.smoke()`` and bench.py's ``cpu_baseline`` /
``--impl reference`` legs may import this.  It imports nothing from the product
package: a mechanism arrives as the plain description dict documented in
``paper_2409_06404_b200/workloads.py`` (hand-written ones in the tests have the same
keys) and is expanded here into the dense arrays crf_oracle.c reads.  No arithmetic of
the method happens in this file.

Parity with the paper's own kernels: PARITY UNPINNED (see crf_oracle.c header).
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "crf_oracle.c")
_LIB = os.path.join(_HERE, "liboracle.so")
_lib = None

TYPE_CODE = {"elementary": 0, "three_body": 1, "falloff": 2}


def build(force: bool = False) -> str:
    """gcc -O2 (no -ffast-math), OpenMP for the timed baseline."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        subprocess.check_call(["gcc", "-O2", "-std=c99", "-fPIC", "-shared", "-fopenmp",
                               "-ffp-contract=off", "-o", _LIB, _SRC, "-lm"])
    return _LIB


class _Mech(C.Structure):
    _fields_ = [("Ns", C.c_int), ("Nr", C.c_int)] + [
        (nm, C.c_void_p) for nm in
        ("W", "Tmid", "nasa_lo", "nasa_hi", "nu_f", "nu_r", "type", "A", "beta", "Ea", "eff",
         "A0", "beta0", "Ea0", "alpha", "T3", "T1", "T2", "mu_fit", "lam_fit", "D_fit")
    ] + [("p_ref", C.c_double)]


def _load():
    global _lib
    if _lib is None:
        _lib = C.CDLL(build())
        _lib.oracle_max_threads.restype = C.c_int
    return _lib


def max_threads() -> int:
    return int(_load().oracle_max_threads())


def _f64(a):
    return np.ascontiguousarray(a, dtype=np.float64)


def _ptr(a):
    return None if a is None else a.ctypes.data_as(C.c_void_p)


class Oracle:
    """The oracle bound to one mechanism description."""

    def __init__(self, mech: dict):
        _load()
        ns = len(mech["W"])
        rx = mech["reactions"]
        nr = len(rx)
        self.Ns, self.Nr = ns, nr
        a = self._arrays = {}
        a["W"] = _f64(mech["W"])
        a["Tmid"] = _f64(mech["nasa_Tmid"])
        a["nasa_lo"] = _f64(mech["nasa_lo"]).reshape(ns, 7)
        a["nasa_hi"] = _f64(mech["nasa_hi"]).reshape(ns, 7)
        nu_f, nu_r = np.zeros((nr, ns)), np.zeros((nr, ns))
        eff = np.ones((nr, ns))
        typ = np.zeros(nr, dtype=np.int32)
        per = {k: np.zeros(nr) for k in ("A", "beta", "Ea", "A0", "beta0", "Ea0", "alpha", "T3", "T1", "T2")}
        for r, rxn in enumerate(rx):
            for k, nu in rxn["reactants"]:
                nu_f[r, k] += nu
            for k, nu in rxn["products"]:
                nu_r[r, k] += nu
            typ[r] = TYPE_CODE[rxn["type"]]
            for key in ("A", "beta", "Ea"):
                per[key][r] = rxn[key]
            for k, e in rxn.get("eff", {}).items():
                eff[r, int(k)] = e
            if rxn["type"] == "falloff":
                for key in ("A0", "beta0", "Ea0", "alpha", "T3", "T1", "T2"):
                    per[key][r] = rxn["troe"][key]
        a["nu_f"], a["nu_r"], a["eff"], a["type"] = nu_f, nu_r, eff, typ
        a.update(per)
        a["mu_fit"] = _f64(mech["mu_fit"]).reshape(ns, 4)
        a["lam_fit"] = _f64(mech["lam_fit"]).reshape(ns, 4)
        a["D_fit"] = _f64(mech["D_fit"]).reshape(ns, ns, 4)
        self.nu = nu_r - nu_f
        self._m = _Mech(Ns=ns, Nr=nr, p_ref=float(mech["p_ref"]),
                        **{k: _ptr(v) for k, v in a.items()})

    def _state(self, T, p, Y):
        T, p, Y = _f64(T).ravel(), _f64(p).ravel(), _f64(Y)
        n = T.size
        assert p.size == n and Y.shape == (self.Ns, n), (Y.shape, self.Ns, n)
        return T, p, Y, n

    def thermo(self, T, p, Y):
        """dict(cp[n] J/kg/K, h[n] J/kg, h_scale[n])"""
        T, p, Y, n = self._state(T, p, Y)
        cp, h, hs = np.empty(n), np.empty(n), np.empty(n)
        _lib.oracle_thermo(C.byref(self._m), _ptr(T), _ptr(p), _ptr(Y), C.c_int64(n),
                           _ptr(cp), _ptr(h), _ptr(hs))
        return dict(cp=cp, h=h, h_scale=hs)

    def thermo_species(self, T):
        """dict(cpk, hk, sk [Ns,n] molar J/kmol(/K), g_RT [Ns,n])"""
        T = _f64(T).ravel()
        n = T.size
        out = {k: np.empty((self.Ns, n)) for k in ("cpk", "hk", "sk", "g_RT")}
        _lib.oracle_thermo_species(C.byref(self._m), _ptr(T), C.c_int64(n),
                                   *[_ptr(out[k]) for k in ("cpk", "hk", "sk", "g_RT")])
        return out

    def production_rates(self, T, p, Y):
        """dict(omega[Ns,n] kmol/m^3/s, qdot[n] W/m^3, S_omega[Ns,n], S_q[n])"""
        T, p, Y, n = self._state(T, p, Y)
        om, So = np.empty((self.Ns, n)), np.empty((self.Ns, n))
        qd, Sq = np.empty(n), np.empty(n)
        _lib.oracle_production_rates(C.byref(self._m), _ptr(T), _ptr(p), _ptr(Y), C.c_int64(n),
                                     _ptr(om), _ptr(qd), _ptr(So), _ptr(Sq))
        return dict(omega=om, qdot=qd, S_omega=So, S_q=Sq)

    def rates_detail(self, T, p, Yi):
        """One point: dict(omega, qdot, kf, kr, Qf, Qr, M, C) (per-reaction intermediates)."""
        Yi = _f64(Yi).ravel()
        assert Yi.size == self.Ns
        om, Cc = np.empty(self.Ns), np.empty(self.Ns)
        qd = C.c_double()
        per = {k: np.empty(self.Nr) for k in ("kf", "kr", "Qf", "Qr", "M")}
        _lib.oracle_rates_detail(C.byref(self._m), C.c_double(float(T)), C.c_double(float(p)), _ptr(Yi),
                                 _ptr(om), C.byref(qd), *[_ptr(per[k]) for k in ("kf", "kr", "Qf", "Qr", "M")],
                                 _ptr(Cc))
        return dict(omega=om, qdot=qd.value, C=Cc, **per)

    def mix_transport(self, T, p, Y):
        """dict(mu[n] Pa s, lam[n] W/m/K, rhoD[Ns,n] kg/m/s, Dkm[Ns,n] m^2/s)"""
        T, p, Y, n = self._state(T, p, Y)
        mu, lam = np.empty(n), np.empty(n)
        rhoD, Dkm = np.empty((self.Ns, n)), np.empty((self.Ns, n))
        _lib.oracle_mix_transport(C.byref(self._m), _ptr(T), _ptr(p), _ptr(Y), C.c_int64(n),
                                  _ptr(mu), _ptr(lam), _ptr(rhoD), _ptr(Dkm))
        return dict(mu=mu, lam=lam, rhoD=rhoD, Dkm=Dkm)

    def rhs_pointwise(self, T, p, Y):
        """dict of everything one right-hand-side evaluation consumes (oracle_rhs_pointwise):
        omega, qdot, S_omega, S_q, cp, h, h_scale, cpk [Ns,n] J/kmol/K, rho [n] kg/m^3, Wbar [n] kg/kmol, mu, lam, rhoD."""
        T, p, Y, n = self._state(T, p, Y)
        o = {k: np.empty((self.Ns, n)) for k in ("omega", "S_omega", "cpk", "rhoD")}
        o.update({k: np.empty(n) for k in ("qdot", "S_q", "cp", "h", "h_scale", "rho", "Wbar", "mu", "lam")})
        order = ("omega", "qdot", "S_omega", "S_q", "cp", "h", "h_scale", "cpk", "rho", "Wbar", "mu", "lam", "rhoD")
        _lib.oracle_rhs_pointwise(C.byref(self._m), _ptr(T), _ptr(p), _ptr(Y), C.c_int64(n), *[_ptr(o[k]) for k in order])
        return o

    def production_rates_pair(self, T, p, Y, T2, p2, Y2):
        """omega and qdot at two states of the same points: two plain calls."""
        a, b = self.production_rates(T, p, Y), self.production_rates(T2, p2, Y2)
        return dict(omega=a["omega"], qdot=a["qdot"], S_omega=a["S_omega"], S_q=a["S_q"],
                    omega2=b["omega"], qdot2=b["qdot"], S_omega2=b["S_omega"], S_q2=b["S_q"])

    def production_rates_jv(self, T, p, Y, dT, dp, dY, sigma):
        """the difference quotient behind the matrix-free Jacobian-vector product:
        J v ~ (omega(y + sigma v) - omega(y)) / sigma with y = (T, p, Y), v = (dT, dp, dY).  The perturbed state is
        formed in double with one rounding per operation (multiply, then add); then two plain calls and the quotient.
        The tolerance scale of the quotient is (S(y) + S(y + sigma v)) / sigma."""
        T, p, Y, n = self._state(T, p, Y)
        dT, dp, dY, _ = self._state(dT, dp, dY)
        sigma = float(sigma)
        T2, p2, Y2 = T + sigma * dT, p + sigma * dp, Y + sigma * dY
        r = self.production_rates_pair(T, p, Y, T2, p2, Y2)
        r["Jomega"] = (r["omega2"] - r["omega"]) / sigma
        r["Jqdot"] = (r["qdot2"] - r["qdot"]) / sigma
        r["S_Jomega"] = (r["S_omega"] + r["S_omega2"]) / abs(sigma)
        r["S_Jqdot"] = (r["S_q"] + r["S_q2"]) / abs(sigma)
        return r
