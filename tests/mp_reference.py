"""50-digit mpmath evaluation of SURVEY.md §8(c) steps 1-13 at one point.

Pins the *rounding* of oracle/crf_oracle.c (not its choice of formulas: those are pinned by
the closed forms and invariants in test_oracle_pins.py).  Written from the description dict,
sparse loops, its own unit conversion -- shares nothing with the oracle or the CUDA path.
"""
import mpmath as mp

mp.mp.dps = 50
R = mp.mpf("8314.46261815324")


def _nasa(mech, k, T):
    a = mech["nasa_lo"][k] if T <= mp.mpf(float(mech["nasa_Tmid"][k])) else mech["nasa_hi"][k]
    a = [mp.mpf(float(x)) for x in a]
    cp = sum(a[i] * T ** i for i in range(5))
    h = sum(a[i] * T ** i / (i + 1) for i in range(5)) + a[5] / T
    s = a[0] * mp.log(T) + sum(a[i] * T ** i / i for i in range(1, 5)) + a[6]
    return cp, h, s


def _arr(A, beta, Ea, order, T):
    return mp.mpf(float(A)) * mp.mpf(10) ** (-3 * (order - 1)) * T ** mp.mpf(float(beta)) \
        * mp.exp(-mp.mpf(float(Ea)) * 10 ** 6 / (R * T))


def evaluate(mech, T, p, Y):
    T, p = mp.mpf(float(T)), mp.mpf(float(p))
    W = [mp.mpf(float(w)) for w in mech["W"]]
    Y = [mp.mpf(float(y)) for y in Y]
    ns = len(W)
    Wbar = 1 / sum(Y[k] / W[k] for k in range(ns))
    rho = p * Wbar / (R * T)
    C = [rho * Y[k] / W[k] for k in range(ns)]
    X = [Y[k] * Wbar / W[k] for k in range(ns)]
    th = [_nasa(mech, k, T) for k in range(ns)]
    g = [t[1] - t[2] for t in th]
    hmol = [t[1] * R * T for t in th]
    out = dict(cp=sum(Y[k] * th[k][0] * R / W[k] for k in range(ns)),
               h=sum(Y[k] * hmol[k] / W[k] for k in range(ns)),
               h_scale=sum(abs(Y[k] * hmol[k] / W[k]) for k in range(ns)),
               rho=rho, Wbar=Wbar, cpk=[t[0] * R for t in th], hk=hmol)
    omega = [mp.mpf(0)] * ns
    S = [mp.mpf(0)] * ns
    pref = mp.mpf(float(mech["p_ref"]))
    for rx in mech["reactions"]:
        order = sum(nu for _, nu in rx["reactants"])
        M = None
        if rx["type"] != "elementary":
            M = sum(mp.mpf(float(rx["eff"].get(k, 1.0))) * C[k] for k in range(ns))
        if rx["type"] == "falloff":
            t = rx["troe"]
            kinf = _arr(rx["A"], rx["beta"], rx["Ea"], order, T)
            k0 = _arr(t["A0"], t["beta0"], t["Ea0"], order + 1, T)
            Pr = k0 * M / kinf
            al = mp.mpf(float(t["alpha"]))
            Fc = (1 - al) * mp.exp(-T / mp.mpf(float(t["T3"]))) + al * mp.exp(-T / mp.mpf(float(t["T1"]))) \
                + mp.exp(-mp.mpf(float(t["T2"])) / T)
            lFc = mp.log10(Fc)
            c = mp.mpf("-0.4") - mp.mpf("0.67") * lFc
            N = mp.mpf("0.75") - mp.mpf("1.27") * lFc
            f1 = (mp.log10(Pr) + c) / (N - mp.mpf("0.14") * (mp.log10(Pr) + c))
            kf = kinf * Pr / (1 + Pr) * mp.mpf(10) ** (lFc / (1 + f1 * f1))
        else:
            kf = _arr(rx["A"], rx["beta"], rx["Ea"], order + (1 if rx["type"] == "three_body" else 0), T)
        dnu = sum(nu for _, nu in rx["products"]) - order
        dG = sum(nu * g[k] for k, nu in rx["products"]) - sum(nu * g[k] for k, nu in rx["reactants"])
        Kc = mp.exp(-dG) * (pref / (R * T)) ** dnu
        Qf, Qr = kf, kf / Kc
        for k, nu in rx["reactants"]:
            Qf *= C[k] ** nu
        for k, nu in rx["products"]:
            Qr *= C[k] ** nu
        if rx["type"] == "three_body":
            Qf, Qr = Qf * M, Qr * M
        for k, nu in rx["reactants"]:
            omega[k] -= nu * (Qf - Qr)
            S[k] += nu * (abs(Qf) + abs(Qr))
        for k, nu in rx["products"]:
            omega[k] += nu * (Qf - Qr)
            S[k] += nu * (abs(Qf) + abs(Qr))
    out.update(omega=omega, S_omega=S, qdot=-sum(hmol[k] * omega[k] for k in range(ns)),
               S_q=sum(abs(hmol[k]) * S[k] for k in range(ns)))
    lnT = mp.log(T)

    def fit(c):
        return mp.exp(sum(mp.mpf(float(c[i])) * lnT ** i for i in range(4)))
    muk = [fit(mech["mu_fit"][k]) for k in range(ns)]
    lamk = [fit(mech["lam_fit"][k]) for k in range(ns)]
    mu = mp.mpf(0)
    for k in range(ns):
        den = sum(X[j] * (1 + mp.sqrt(muk[k] / muk[j]) * (W[j] / W[k]) ** mp.mpf("0.25")) ** 2
                  / mp.sqrt(8 * (1 + W[k] / W[j])) for j in range(ns))
        mu += X[k] * muk[k] / den
    lam = (sum(X[k] * lamk[k] for k in range(ns)) + 1 / sum(X[k] / lamk[k] for k in range(ns))) / 2
    rhoD = []
    for k in range(ns):
        s = sum(X[j] / (fit(mech["D_fit"][j][k]) * pref / p) for j in range(ns) if j != k)
        rhoD.append(rho * (1 - Y[k]) / s)
    out.update(mu=mu, lam=lam, rhoD=rhoD)
    return out
