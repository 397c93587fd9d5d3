"""WENO5-Z built from its definition (test helper; no oracle code, no GPU code).

Nothing here is typed from a coefficient table: every number is derived at import time from the
definitions that Jiang & Shu / Borges et al. give in words ("[18]", G1):

* candidate k (k = 0, 1, 2) is the parabola p_k whose cell averages over the three cells
  i-2+k .. i+k equal the data; its face value is q_k = p_k(x_{i+1/2});
* smoothness indicator  beta_k = sum_{l=1,2} dx^(2l-1) * integral over cell i of (d^l p_k / dx^l)^2 dx;
* ideal weights d_k: the combination sum_k d_k q_k that equals the face value of the quartic whose cell
  averages match all five cells;
* WENO-Z (power 1): tau = |beta_0 - beta_2|, alpha_k = d_k (1 + tau / (beta_k + eps)), value = sum alpha_k q_k / sum alpha_k.

With dx = 1 and cell i = [-1/2, 1/2] the parabolas, integrals and the quartic are evaluated with
numpy.polynomial; `wenoz` then applies them to (arrays of) stencil values.
"""
import numpy as np
from numpy.polynomial import Polynomial

EPS = 1e-40


def _avg_matrix(cells, degree):
    """A[r, m] = average of x^m over cell cells[r] = [c - 1/2, c + 1/2]."""
    A = np.empty((len(cells), degree + 1))
    for r, c in enumerate(cells):
        for m in range(degree + 1):
            A[r, m] = ((c + 0.5) ** (m + 1) - (c - 0.5) ** (m + 1)) / (m + 1)
    return A


def _derive():
    face = 0.5
    Q = np.zeros((3, 3))          # q_k = Q[k] . (stencil values of candidate k)
    M = np.zeros((3, 3, 3))       # beta_k = v^T M[k] v
    for k in range(3):
        cells = [-2 + k, -1 + k, k]
        coef = np.linalg.solve(_avg_matrix(cells, 2), np.eye(3))    # column j: parabola for data e_j
        polys = [Polynomial(coef[:, j]) for j in range(3)]
        for a in range(3):
            Q[k, a] = polys[a](face)
            for b in range(3):
                integrand = polys[a].deriv(1) * polys[b].deriv(1) + polys[a].deriv(2) * polys[b].deriv(2)
                I = integrand.integ()
                M[k, a, b] = I(0.5) - I(-0.5)
    # quartic through all five cell averages, evaluated at the face: a row of 5 coefficients
    coef5 = np.linalg.solve(_avg_matrix([-2, -1, 0, 1, 2], 4), np.eye(5))
    row5 = np.array([Polynomial(coef5[:, j])(face) for j in range(5)])
    # ideal weights: sum_k d_k (Q[k] embedded at columns k..k+2) = row5
    A = np.zeros((5, 3))
    for k in range(3):
        A[k:k + 3, k] = Q[k]
    d, res, _, _ = np.linalg.lstsq(A, row5, rcond=None)
    assert np.abs(A @ d - row5).max() < 1e-14          # the system is consistent
    return Q, M, d


Q, M, D = _derive()


def betas(a, b, c, d, e):
    v = (a, b, c, d, e)
    out = []
    for k in range(3):
        s = 0.0
        for x in range(3):
            for y in range(3):
                s = s + M[k, x, y] * v[k + x] * v[k + y]
        out.append(s)
    return out


def candidates(a, b, c, d, e):
    v = (a, b, c, d, e)
    return [Q[k, 0] * v[k] + Q[k, 1] * v[k + 1] + Q[k, 2] * v[k + 2] for k in range(3)]


def wenoz(a, b, c, d, e, eps=EPS):
    """Face value at i+1/2 from cell averages q[i-2..i+2]; scalars or numpy arrays.  eps is a parameter so that
    tests can show which values of it the data can tell apart (tests/test_oracle_eps_pin.py)."""
    be = betas(a, b, c, d, e)
    q = candidates(a, b, c, d, e)
    tau = np.abs(be[0] - be[2])
    al = [D[k] * (1.0 + tau / (be[k] + eps)) for k in range(3)]
    return (al[0] * q[0] + al[1] * q[1] + al[2] * q[2]) / (al[0] + al[1] + al[2])
