"""CPU oracle of the element-local spectral-element diffusion operator -- TEST INFRASTRUCTURE, NOT
PRODUCT.  Plain numpy (einsum as the library contraction), double precision, any polynomial order; shares no code with
the CUDA path (which computes its own quadrature nodes and derivative matrix in csrc/sem_diffusion.cu).

What it follows.  The species equation (1a) has the diffusion term  -div(rho Y_k V_k)  with the mixture-averaged
diffusion velocity of Eq. 2,  V_k = -(D_k / X_k) grad X_k + V_c,  V_c = -sum_k Y_k V_k, and the
temperature equation (1b) has  div(lambda grad T).  "nekRS ... based on the spectral element method
... matrix-free ... tensor-product", polynomial order p = 7 in the paper's runs.
The paper prints neither the discrete operator nor its geometry; the reading is the standard Galerkin
weak form on Gauss-Lobatto-Legendre (GLL) points with GLL quadrature, element-local (no gather-scatter, no boundary
terms: those belong to the assembly the paper does in its QQ^T kernel), on affine box elements (hx, hy, hz):

  X_k = Y_k Wbar / W_k                                   mole fractions
  f_k = (W_k / Wbar) (rho D_k) grad X_k                  = rho Y_k (D_k / X_k) grad X_k  without the division by X_k
  j_k = -f_k + Y_k sum_j f_j                             = rho Y_k V_k with the correction velocity (sum_k j_k = 0)
  dY_k[i] = sum_q w_q |J| grad phi_i(x_q) . j_k(x_q)     weak form of  -div j_k  tested with the nodal basis phi_i
  dT[i]   = -sum_q w_q |J| grad phi_i(x_q) . (lambda grad T)(x_q)     weak form of  div(lambda grad T)

Layout: a field is [n] with n = nel N^3, node (i, j, k) of element e at e N^3 + i + N j + N^2 k (i along x fastest);
Y, rhoD, dY are species-major [Ns, n]; h3 is [nel, 3] = (hx, hy, hz).
Parity with the paper's own diffusion kernel: PARITY UNPINNED (no formulas or code for it in the container); the
operator is pinned by exactness on polynomials, conservation identities and a brute-force assembly (tests/).
"""
from __future__ import annotations

import numpy as np
from numpy.polynomial import legendre as npleg


def gll(N: int):
    """N Gauss-Lobatto-Legendre nodes on [-1, 1] (ends and the roots of P'_{N-1}) and weights 2/(p (p+1) P_p(x)^2)."""
    p = N - 1
    c = np.zeros(N)
    c[p] = 1.0
    x = np.concatenate(([-1.0], np.sort(npleg.legroots(npleg.legder(c))), [1.0]))
    w = 2.0 / (p * (p + 1) * npleg.legval(x, c) ** 2)
    return x, w


def deriv_matrix(x: np.ndarray) -> np.ndarray:
    """D[i, m] = l_m'(x_i) for the Lagrange basis on the nodes x (barycentric form; rows sum to zero)."""
    N = x.size
    b = np.array([1.0 / np.prod([x[m] - x[q] for q in range(N) if q != m]) for m in range(N)])
    D = np.zeros((N, N))
    for i in range(N):
        for m in range(N):
            if i != m:
                D[i, m] = (b[m] / b[i]) / (x[i] - x[m])
        D[i, i] = -np.sum(D[i, :])
    return D


def _grad(D, u, h3):
    """u [nel, N, N, N] indexed [e, k, j, i] -> (du/dx, du/dy, du/dz)"""
    gx = np.einsum("im,ekjm->ekji", D, u) * (2.0 / h3[:, 0])[:, None, None, None]
    gy = np.einsum("jm,ekmi->ekji", D, u) * (2.0 / h3[:, 1])[:, None, None, None]
    gz = np.einsum("km,emji->ekji", D, u) * (2.0 / h3[:, 2])[:, None, None, None]
    return gx, gy, gz


def _weak_div(D, w, fx, fy, fz, h3):
    """sum_q w_q |J| grad phi_i . f  for the nodal basis: D^T applied along each direction to the weighted flux"""
    jw = (w[None, :, None, None] * w[None, None, :, None] * w[None, None, None, :]) * (np.prod(h3, axis=1) / 8.0)[:, None, None, None]
    ax = fx * jw * (2.0 / h3[:, 0])[:, None, None, None]
    ay = fy * jw * (2.0 / h3[:, 1])[:, None, None, None]
    az = fz * jw * (2.0 / h3[:, 2])[:, None, None, None]
    return (np.einsum("mi,ekjm->ekji", D, ax) + np.einsum("mj,ekmi->ekji", D, ay) + np.einsum("mk,emji->ekji", D, az))


def sem_diffusion(W, h3, T, Wbar, Y, lam, rhoD, N: int = 8):
    """dict(dY [Ns, n], dT [n]): the element-local weak-form diffusion terms defined in the module docstring."""
    W, h3 = np.asarray(W, dtype=np.float64), np.asarray(h3, dtype=np.float64)
    nel, ns = h3.shape[0], W.size
    sh = (nel, N, N, N)
    T, Wbar, lam = (np.asarray(a, dtype=np.float64).reshape(sh) for a in (T, Wbar, lam))
    Y = np.asarray(Y, dtype=np.float64).reshape((ns,) + sh)
    rhoD = np.asarray(rhoD, dtype=np.float64).reshape((ns,) + sh)
    x, w = gll(N)
    D = deriv_matrix(x)
    f = []
    for k in range(ns):
        gx, gy, gz = _grad(D, Y[k] * Wbar / W[k], h3)
        c = (W[k] / Wbar) * rhoD[k]
        f.append((c * gx, c * gy, c * gz))
    fc = [sum(fk[d] for fk in f) for d in range(3)]
    dY = np.empty((ns, nel * N ** 3))
    for k in range(ns):
        j = [-f[k][d] + Y[k] * fc[d] for d in range(3)]
        dY[k] = _weak_div(D, w, j[0], j[1], j[2], h3).reshape(-1)
    gx, gy, gz = _grad(D, T, h3)
    dT = -_weak_div(D, w, lam * gx, lam * gy, lam * gz, h3).reshape(-1)
    return dict(dY=dY, dT=dT)


def sem_diffusion_scale(W, h3, T, Wbar, Y, lam, rhoD, N: int = 8):
    """dict(dY [Ns, n], dT [n]): the GROSS sums behind sem_diffusion -- the same contractions with |D_im| and the
    magnitudes of every factor, i.e. the sum of the absolute values of all the products that cancel in dY and dT.
    The operator differentiates: where a field is nearly constant over an element its result is a small difference
    of large terms, so a tolerance relative to the result itself would ask for more digits than the inputs carry;
    this is the scale the parity tolerance is relative to (the analogue of S_k for omega_k)."""
    W, h3 = np.asarray(W, dtype=np.float64), np.asarray(h3, dtype=np.float64)
    nel, ns = h3.shape[0], W.size
    sh = (nel, N, N, N)
    T, Wbar, lam = (np.abs(np.asarray(a, dtype=np.float64)).reshape(sh) for a in (T, Wbar, lam))
    Y = np.abs(np.asarray(Y, dtype=np.float64)).reshape((ns,) + sh)
    rhoD = np.abs(np.asarray(rhoD, dtype=np.float64)).reshape((ns,) + sh)
    x, w = gll(N)
    D = np.abs(deriv_matrix(x))
    f = []
    for k in range(ns):
        gx, gy, gz = _grad(D, Y[k] * Wbar / W[k], h3)
        c = (W[k] / Wbar) * rhoD[k]
        f.append((c * gx, c * gy, c * gz))
    fc = [sum(fk[d] for fk in f) for d in range(3)]
    dY = np.empty((ns, nel * N ** 3))
    for k in range(ns):
        j = [f[k][d] + Y[k] * fc[d] for d in range(3)]
        dY[k] = _weak_div(D, w, j[0], j[1], j[2], h3).reshape(-1)
    gx, gy, gz = _grad(D, T, h3)
    dT = _weak_div(D, w, lam * gx, lam * gy, lam * gz, h3).reshape(-1)
    return dict(dY=dY, dT=dT)
