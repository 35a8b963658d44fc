"""Pins of the spectral-element diffusion oracle (oracle/sem_oracle.py): textbook quadrature values,
exact differentiation of polynomials, conservation identities of the weak form and of the correction velocity, a
closed form for linear fields, and a brute-force assembly with explicitly differentiated Lagrange polynomials."""
import numpy as np
import pytest
from numpy.polynomial import polynomial as npoly

from oracle import sem_oracle as so


def test_gll_textbook_values_and_exactness():
    x, w = so.gll(3)
    np.testing.assert_allclose(x, [-1.0, 0.0, 1.0], atol=1e-15)
    np.testing.assert_allclose(w, [1 / 3, 4 / 3, 1 / 3], rtol=1e-15)
    x, w = so.gll(4)
    np.testing.assert_allclose(x, [-1.0, -1 / np.sqrt(5), 1 / np.sqrt(5), 1.0], atol=1e-15)
    np.testing.assert_allclose(w, [1 / 6, 5 / 6, 5 / 6, 1 / 6], rtol=1e-14)
    x, w = so.gll(8)  # p = 7, the paper's order: exact for polynomials up to degree 2p - 1 = 13
    assert np.allclose(x, -x[::-1], atol=1e-15) and abs(w.sum() - 2.0) < 1e-14
    for m in range(14):
        assert abs(np.sum(w * x ** m) - (0.0 if m % 2 else 2.0 / (m + 1))) < 1e-14
    D = so.deriv_matrix(x)
    for m in range(8):
        np.testing.assert_allclose(D @ x ** m, m * x ** max(m - 1, 0) if m else np.zeros(8), atol=2e-13)


def _fields(rng, nel, ns, N, Y_sum_one=True):
    n = nel * N ** 3
    Y = rng.dirichlet(np.ones(ns), n).T if Y_sum_one else rng.uniform(0.1, 1.0, (ns, n))
    W = rng.uniform(2.0, 44.0, ns)
    Wbar = 1.0 / np.sum(Y / W[:, None], axis=0)
    return dict(W=W, h3=rng.uniform(0.5e-3, 2e-3, (nel, 3)), T=rng.uniform(300.0, 2000.0, n), Wbar=Wbar, Y=Y,
                lam=rng.uniform(0.02, 0.2, n), rhoD=rng.uniform(1e-5, 1e-4, (ns, n)))


@pytest.mark.parametrize("N", [3, 5, 8])
def test_conservation_identities(N):
    """sum_i grad phi_i = 0 (partition of unity): every local residual sums to zero over the element; and the
    correction velocity makes the species fluxes sum to zero (sum_k j_k = 0 when sum_k Y_k = 1)."""
    rng = np.random.default_rng(N)
    f = _fields(rng, 3, 4, N)
    r = so.sem_diffusion(N=N, **f)
    scale = np.abs(r["dY"]).max()
    assert np.abs(r["dY"].reshape(4, 3, -1).sum(axis=2)).max() <= 1e-13 * scale * N ** 3
    assert np.abs(r["dT"].reshape(3, -1).sum(axis=1)).max() <= 1e-13 * np.abs(r["dT"]).max() * N ** 3
    assert np.abs(r["dY"].sum(axis=0)).max() <= 1e-13 * scale * 4


def test_linear_temperature_constant_conductivity_closed_form():
    """T = a . x, lambda = const: the flux is constant, so dT[i] = -lambda a . int grad phi_i = -lambda a . (boundary
    integral of phi_i n): zero at interior nodes, -+lambda a_x w_j w_k hy hz / 4 on the faces x = -+hx/2, etc."""
    N, lam0 = 8, 0.07
    hx, hy, hz = 1.0e-3, 2.0e-3, 0.5e-3
    a = np.array([300.0, -120.0, 50.0]) * 1e3
    x, w = so.gll(N)
    X, Yc, Z = np.meshgrid(x * hx / 2, x * hy / 2, x * hz / 2, indexing="ij")  # [i, j, k]
    T = (1000.0 + a[0] * X + a[1] * Yc + a[2] * Z).transpose(2, 1, 0).reshape(-1)  # node index i + N j + N^2 k
    n = N ** 3
    r = so.sem_diffusion(W=np.array([28.0]), h3=np.array([[hx, hy, hz]]), T=T, Wbar=np.full(n, 28.0), Y=np.ones((1, n)),
                         lam=np.full(n, lam0), rhoD=np.full((1, n), 1e-5), N=N)
    dT = r["dT"].reshape(N, N, N)  # [k, j, i]
    exp = np.zeros((N, N, N))
    for sgn, idx in ((-1.0, 0), (1.0, N - 1)):
        exp[:, :, idx] += -lam0 * a[0] * sgn * np.outer(w, w) * hy * hz / 4   # [k, j]
        exp[:, idx, :] += -lam0 * a[1] * sgn * np.outer(w, w) * hx * hz / 4   # [k, i]
        exp[idx, :, :] += -lam0 * a[2] * sgn * np.outer(w, w) * hx * hy / 4   # [j, i]
    np.testing.assert_allclose(dT, exp, atol=1e-12 * np.abs(exp).max())
    assert np.abs(r["dY"]).max() == 0.0  # a pure species does not diffuse


def _lagrange_derivs(x):
    """l_m'(x_i) by differentiating the Lagrange polynomials explicitly (an independent route to D)."""
    N = x.size
    D = np.zeros((N, N))
    for m in range(N):
        c = npoly.polyfromroots(np.delete(x, m))
        c = c / npoly.polyval(x[m], c)
        D[:, m] = npoly.polyval(x, npoly.polyder(c))
    return D


@pytest.mark.parametrize("N", [3, 4])
def test_against_brute_force_assembly(N):
    """Every entry of dY and dT from plain loops over test functions, quadrature points, directions and species."""
    rng = np.random.default_rng(10 + N)
    ns = 3
    f = _fields(rng, 1, ns, N, Y_sum_one=False)
    r = so.sem_diffusion(N=N, **f)
    x, w = so.gll(N)
    Dl = _lagrange_derivs(x)
    h = f["h3"][0]
    idx = lambda i, j, k: i + N * j + N * N * k  # noqa: E731
    Xk = f["Y"] * f["Wbar"] / f["W"][:, None]

    def grad(u, i, j, k):
        return np.array([sum(Dl[i, m] * u[idx(m, j, k)] for m in range(N)) * 2 / h[0],
                         sum(Dl[j, m] * u[idx(i, m, k)] for m in range(N)) * 2 / h[1],
                         sum(Dl[k, m] * u[idx(i, j, m)] for m in range(N)) * 2 / h[2]])
    dY, dT = np.zeros((ns, N ** 3)), np.zeros(N ** 3)
    for qi in range(N):
        for qj in range(N):
            for qk in range(N):
                q = idx(qi, qj, qk)
                wq = w[qi] * w[qj] * w[qk] * h.prod() / 8
                fk = [f["W"][s] / f["Wbar"][q] * f["rhoD"][s, q] * grad(Xk[s], qi, qj, qk) for s in range(ns)]
                fc = sum(fk)
                heat = f["lam"][q] * grad(f["T"], qi, qj, qk)
                for ti in range(N):
                    for tj in range(N):
                        for tk in range(N):
                            # grad phi_t at the quadrature point: the basis is a tensor product of Lagrange polynomials
                            gphi = np.array([Dl[qi, ti] * (tj == qj) * (tk == qk) * 2 / h[0],
                                             (ti == qi) * Dl[qj, tj] * (tk == qk) * 2 / h[1],
                                             (ti == qi) * (tj == qj) * Dl[qk, tk] * 2 / h[2]])
                            t = idx(ti, tj, tk)
                            dT[t] -= wq * gphi @ heat
                            for s in range(ns):
                                dY[s, t] += wq * gphi @ (-fk[s] + f["Y"][s, q] * fc)
    np.testing.assert_allclose(r["dY"], dY, atol=1e-13 * np.abs(dY).max())
    np.testing.assert_allclose(r["dT"], dT, atol=1e-13 * np.abs(dT).max())


def test_heat_operator_is_symmetric_and_negative():
    """With a fixed lambda field, T -> dT is linear, symmetric and negative semi-definite (the stiffness matrix)."""
    N = 5
    rng = np.random.default_rng(7)
    f = _fields(rng, 2, 2, N)
    n = 2 * N ** 3

    def A(u):
        return so.sem_diffusion(N=N, **{**f, "T": u})["dT"]
    u, v = rng.standard_normal(n), rng.standard_normal(n)
    assert abs(u @ A(v) - v @ A(u)) <= 1e-12 * abs(u @ A(v))
    assert u @ A(u) < 0.0 and np.abs(A(np.ones(n))).max() <= 1e-12 * np.abs(A(u)).max()


def test_gross_scale_bounds_the_result():
    """sem_diffusion_scale sums the magnitudes of the products sem_diffusion sums: it bounds the result entry by entry,
    and for a field that is constant over the element (the result is exactly a rounding residue) it stays at the size
    of the cancelling terms."""
    rng = np.random.default_rng(21)
    f = _fields(rng, 2, 3, 8)
    r, s = so.sem_diffusion(**f), so.sem_diffusion_scale(**f)
    assert np.all(np.abs(r["dY"]) <= s["dY"] * (1 + 1e-12)) and np.all(np.abs(r["dT"]) <= s["dT"] * (1 + 1e-12))
    f["T"] = np.full_like(f["T"], 1234.5)
    r, s = so.sem_diffusion(**f), so.sem_diffusion_scale(**f)
    assert np.abs(r["dT"]).max() <= 1e-13 * s["dT"].max() and s["dT"].min() > 0.0
