"""Closed-form spacetimes used to pin the oracle (tests only). Built with sympy so that no
Z4c formula of the oracle is retyped here: the Ricci tensor comes from the textbook definition
d_k Gam^k_ij - d_j Gam^k_ik + Gam^k_kl Gam^l_ij - Gam^k_jl Gam^l_ik, conformal variables from their
definitions (chi = det(gamma)^(-1/3), gt = chi gamma, At = chi (K_ij - gamma_ij K/3),
Gamt^i = -d_j gt^ij for det gt = 1)."""
from __future__ import annotations

import functools

import numpy as np
import sympy as sp

x, y, z = sp.symbols("x y z", real=True)
X = [x, y, z]
PAIRS = [(0, 0), (0, 1), (0, 2), (1, 1), (1, 2), (2, 2)]


def _christoffel(G, Gi):
    return [[[sum(Gi[k, l] * (sp.diff(G[l, i], X[j]) + sp.diff(G[l, j], X[i]) - sp.diff(G[i, j], X[l]))
                  for l in range(3)) / 2 for j in range(3)] for i in range(3)] for k in range(3)]


def _ricci(Gam):
    R = sp.zeros(3, 3)
    for i in range(3):
        for j in range(i, 3):
            R[i, j] = (sum(sp.diff(Gam[k][i][j], X[k]) - sp.diff(Gam[k][i][k], X[j]) for k in range(3))
                       + sum(Gam[k][k][l] * Gam[l][i][j] - Gam[k][j][l] * Gam[l][i][k]
                             for k in range(3) for l in range(3)))
            R[j, i] = R[i, j]
    return R


@functools.lru_cache(maxsize=None)
def unimodular_metric():
    """A smooth non-diagonal metric with det = 1 exactly: g = L D L^T, L unit lower triangular,
    D = diag(e^f, e^g, e^(-f-g)). Returns fn(x,y,z) -> (g[6], Ricci[6], Gam_d[3])."""
    f = sp.Rational(3, 10) * sp.sin(x + 2 * y) + sp.Rational(1, 10) * sp.cos(z)
    g = sp.Rational(1, 5) * sp.cos(y - z) * sp.sin(x)
    p_ = sp.Rational(1, 4) * sp.sin(x - z)
    q_ = sp.Rational(1, 5) * sp.cos(y + x)
    r_ = sp.Rational(3, 20) * sp.sin(z + y)
    L = sp.Matrix([[1, 0, 0], [p_, 1, 0], [q_, r_, 1]])
    G = L * sp.diag(sp.exp(f), sp.exp(g), sp.exp(-f - g)) * L.T
    Gi = G.inv()
    Gam = _christoffel(G, Gi)
    Ric = _ricci(Gam)
    Gd = [sum(Gi[i, j] * Gam[k][i][j] for i in range(3) for j in range(3)) for k in range(3)]
    exprs = [G[i, j] for i, j in PAIRS] + [Ric[i, j] for i, j in PAIRS] + Gd
    fn = sp.lambdify((x, y, z), exprs, "numpy", cse=True)

    def ev(xx, yy, zz):
        out = [np.broadcast_to(np.asarray(o, dtype=np.float64), np.broadcast(xx, yy, zz).shape)
               for o in fn(xx, yy, zz)]
        return np.stack(out[0:6]), np.stack(out[6:12]), np.stack(out[12:15])
    return ev


@functools.lru_cache(maxsize=None)
def kerr_schild(M=1):
    """Schwarzschild in Kerr-Schild coordinates: gamma_ij = delta_ij + 2H l_i l_j, H = M/r, l_i = x_i/r,
    alpha = (1+2H)^(-1/2), beta^i = 2H l^i/(1+2H), K_ij = (2H alpha/r)[delta_ij - (2+H) l_i l_j].
    Returns fn(x,y,z) -> dict of the 22 conformal fields plus analytic advective gauge terms."""
    r = sp.sqrt(x * x + y * y + z * z)
    H = M / r
    l = [x / r, y / r, z / r]
    gam = sp.Matrix(3, 3, lambda i, j: (1 if i == j else 0) + 2 * H * l[i] * l[j])
    alpha = 1 / sp.sqrt(1 + 2 * H)
    beta = [2 * H * l[i] / (1 + 2 * H) for i in range(3)]
    Kij = sp.Matrix(3, 3, lambda i, j: (2 * H * alpha / r) * ((1 if i == j else 0) - (2 + H) * l[i] * l[j]))
    det = 1 + 2 * H                     # det(delta + 2H l l^T) with |l| = 1
    gami = sp.Matrix(3, 3, lambda i, j: (1 if i == j else 0) - 2 * H * l[i] * l[j] / (1 + 2 * H))
    chi = det ** sp.Rational(-1, 3)
    gt = chi * gam
    gti = gami / chi
    K = sum(gami[i, j] * Kij[i, j] for i in range(3) for j in range(3))
    At = chi * (Kij - gam * K / 3)
    Gamt = [-sum(sp.diff(gti[i, j], X[j]) for j in range(3)) for i in range(3)]
    adv_alpha = sum(beta[k] * sp.diff(alpha, X[k]) for k in range(3))
    adv_beta = [sum(beta[k] * sp.diff(beta[i], X[k]) for k in range(3)) for i in range(3)]
    exprs = ([chi] + [gt[i, j] for i, j in PAIRS] + [K] + [At[i, j] for i, j in PAIRS] + Gamt
             + [sp.Integer(0), alpha] + beta + [adv_alpha] + adv_beta)
    fn = sp.lambdify((x, y, z), exprs, "numpy", cse=True)

    def ev(xx, yy, zz):
        shape = np.broadcast(xx, yy, zz).shape
        out = [np.broadcast_to(np.asarray(o, dtype=np.float64), shape) for o in fn(xx, yy, zz)]
        return np.stack(out[:22]).copy(), out[22], np.stack(out[23:26])
    return ev
