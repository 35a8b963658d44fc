"""Hand-built mechanism descriptions for the pins (same keys as workloads.make_mechanism)."""
import numpy as np

R = 8314.46261815324          # J/(kmol K)
R_KJ_MOL = 8.31446261815324e-3  # kJ/(mol K)
P_REF = 101325.0


def const_cp_nasa(a1, a6, a7):
    """NASA-7 set with a2..a5 = 0 (constant cp)."""
    return np.array([a1, 0.0, 0.0, 0.0, 0.0, a6, a7])


def log_const(value):
    """cubic-in-lnT fit that is the constant ``value``"""
    return np.array([np.log(value), 0.0, 0.0, 0.0])


def tiny_mech(W, reactions, nasa=None, mu=None, lam=None, D=None, Tmid=None):
    """Species with constant cp unless ``nasa`` = (lo[Ns,7], hi[Ns,7]) is given; transport fits
    constant in T: mu[Ns], lam[Ns], D[Ns,Ns] values (defaults 2e-5, 0.05, 1e-4)."""
    W = np.asarray(W, dtype=float)
    ns = W.size
    if nasa is None:
        lo = np.array([const_cp_nasa(3.5, 0.0, 5.0) for _ in range(ns)])
        hi = lo.copy()
    else:
        lo, hi = (np.array(x, dtype=float) for x in nasa)
    mu = np.full(ns, 2e-5) if mu is None else np.asarray(mu, dtype=float)
    lam = np.full(ns, 0.05) if lam is None else np.asarray(lam, dtype=float)
    D = np.full((ns, ns), 1e-4) if D is None else np.asarray(D, dtype=float)
    return dict(
        name="tiny", elements=[], species=[f"S{k}" for k in range(ns)],
        comp=np.zeros((0, ns), dtype=np.int64), W=W,
        nasa_Tmid=np.full(ns, 1000.0) if Tmid is None else np.asarray(Tmid, dtype=float),
        nasa_lo=lo, nasa_hi=hi, reactions=reactions,
        mu_fit=np.array([log_const(v) for v in mu]),
        lam_fit=np.array([log_const(v) for v in lam]),
        D_fit=np.array([[log_const(D[j, k]) for k in range(ns)] for j in range(ns)]),
        p_ref=P_REF)


def rxn(reactants, products, A=1.0, beta=0.0, Ea=0.0, type="elementary", eff=None, troe=None):
    r = dict(reactants=list(reactants), products=list(products), type=type, A=A, beta=beta, Ea=Ea)
    if type != "elementary":
        r["eff"] = dict(eff or {})
    if troe is not None:
        r["troe"] = dict(troe)
    return r


def mass_from_mole(X, W):
    X, W = np.asarray(X, dtype=float), np.asarray(W, dtype=float)
    return X * W / np.sum(X * W)


def col(v):
    """[Ns] -> [Ns,1] species-major single point"""
    return np.asarray(v, dtype=float).reshape(-1, 1)
