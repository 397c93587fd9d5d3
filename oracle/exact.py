"""ORACLE — TEST INFRASTRUCTURE, NOT THE PRODUCT.

Closed-form references the oracle's time stepper is pinned against (BASELINE.json north_star):
  * exact solution of the Riemann problem for the ideal-gas Euler equations (Sod, LeBlanc),
  * the Sedov-Taylor point-blast similarity constant xi0 (shock radius),
  * the paper's L1 metric with cell averages of the analytic solution by 10-node Gauss-Legendre
    quadrature (eq.19).
These are textbook definitions written out directly; tests pin them to the textbook numbers.
"""
from __future__ import annotations

import numpy as np


# ----------------------------------------------------------------------------- exact Riemann
def _fK(p, rhoK, pK, g):
    """Pressure function of one side and its derivative (shock branch p>pK, else rarefaction)."""
    cK = np.sqrt(g * pK / rhoK)
    if p > pK:
        A = 2.0 / ((g + 1.0) * rhoK)
        B = (g - 1.0) / (g + 1.0) * pK
        s = np.sqrt(A / (p + B))
        return (p - pK) * s, s * (1.0 - 0.5 * (p - pK) / (p + B))
    pr = p / pK
    return 2.0 * cK / (g - 1.0) * (pr ** ((g - 1.0) / (2.0 * g)) - 1.0), (1.0 / (rhoK * cK)) * pr ** (-(g + 1.0) / (2.0 * g))


def riemann_star(rhoL, uL, pL, rhoR, uR, pR, g):
    """Star-region pressure and velocity by Newton iteration on f_L(p)+f_R(p)+uR-uL = 0."""
    cL, cR = np.sqrt(g * pL / rhoL), np.sqrt(g * pR / rhoR)
    # two-rarefaction guess: always positive, good for strong rarefactions (LeBlanc)
    z = (g - 1.0) / (2.0 * g)
    p = ((cL + cR - 0.5 * (g - 1.0) * (uR - uL)) / (cL / pL ** z + cR / pR ** z)) ** (1.0 / z)
    for _ in range(200):
        fL, dL = _fK(p, rhoL, pL, g)
        fR, dR = _fK(p, rhoR, pR, g)
        dp = (fL + fR + (uR - uL)) / (dL + dR)
        pn = p - dp
        if pn <= 0.0:
            pn = 0.5 * p
        if abs(pn - p) <= 1e-15 * (pn + p):
            p = pn
            break
        p = pn
    fL, _ = _fK(p, rhoL, pL, g)
    fR, _ = _fK(p, rhoR, pR, g)
    return p, 0.5 * (uL + uR) + 0.5 * (fR - fL)


def riemann_sample(xi, rhoL, uL, pL, rhoR, uR, pR, g):
    """(rho, u, p) of the exact solution at similarity coordinates xi = (x - x0)/t (array)."""
    xi = np.asarray(xi, dtype=np.float64)
    ps, us = riemann_star(rhoL, uL, pL, rhoR, uR, pR, g)
    cL, cR = np.sqrt(g * pL / rhoL), np.sqrt(g * pR / rhoR)
    gm, gp = g - 1.0, g + 1.0
    rho = np.empty_like(xi)
    u = np.empty_like(xi)
    p = np.empty_like(xi)
    left = xi <= us
    # ---- left of the contact
    if ps > pL:  # left shock
        SL = uL - cL * np.sqrt(gp / (2 * g) * ps / pL + gm / (2 * g))
        rs = rhoL * (ps / pL + gm / gp) / (gm / gp * ps / pL + 1.0)
        m0 = left & (xi < SL)
        m1 = left & ~m0
        rho[m0], u[m0], p[m0] = rhoL, uL, pL
        rho[m1], u[m1], p[m1] = rs, us, ps
    else:  # left rarefaction
        rs = rhoL * (ps / pL) ** (1.0 / g)
        cs = cL * (ps / pL) ** (gm / (2 * g))
        head, tail = uL - cL, us - cs
        m0 = left & (xi < head)
        m2 = left & (xi > tail)
        m1 = left & ~m0 & ~m2
        rho[m0], u[m0], p[m0] = rhoL, uL, pL
        rho[m2], u[m2], p[m2] = rs, us, ps
        f = 2.0 / gp + gm / (gp * cL) * (uL - xi[m1])
        rho[m1] = rhoL * f ** (2.0 / gm)
        u[m1] = 2.0 / gp * (cL + 0.5 * gm * uL + xi[m1])
        p[m1] = pL * f ** (2.0 * g / gm)
    # ---- right of the contact
    right = ~left
    if ps > pR:  # right shock
        SR = uR + cR * np.sqrt(gp / (2 * g) * ps / pR + gm / (2 * g))
        rs = rhoR * (ps / pR + gm / gp) / (gm / gp * ps / pR + 1.0)
        m0 = right & (xi > SR)
        m1 = right & ~m0
        rho[m0], u[m0], p[m0] = rhoR, uR, pR
        rho[m1], u[m1], p[m1] = rs, us, ps
    else:
        rs = rhoR * (ps / pR) ** (1.0 / g)
        cs = cR * (ps / pR) ** (gm / (2 * g))
        head, tail = uR + cR, us + cs
        m0 = right & (xi > head)
        m2 = right & (xi < tail)
        m1 = right & ~m0 & ~m2
        rho[m0], u[m0], p[m0] = rhoR, uR, pR
        rho[m2], u[m2], p[m2] = rs, us, ps
        f = 2.0 / gp - gm / (gp * cR) * (uR - xi[m1])
        rho[m1] = rhoR * f ** (2.0 / gm)
        u[m1] = 2.0 / gp * (-cR + 0.5 * gm * uR + xi[m1])
        p[m1] = pR * f ** (2.0 * g / gm)
    return rho, u, p


def riemann_waves(rhoL, uL, pL, rhoR, uR, pR, g):
    """Dictionary of star values and wave speeds (left rarefaction / right shock layout assumed
    only for the keys that exist)."""
    ps, us = riemann_star(rhoL, uL, pL, rhoR, uR, pR, g)
    cL, cR = np.sqrt(g * pL / rhoL), np.sqrt(g * pR / rhoR)
    gm, gp = g - 1.0, g + 1.0
    out = {"p_star": ps, "u_star": us}
    if ps <= pL:
        out["rho_star_L"] = rhoL * (ps / pL) ** (1.0 / g)
        out["head_L"] = uL - cL
        out["tail_L"] = us - cL * (ps / pL) ** (gm / (2 * g))
    else:
        out["rho_star_L"] = rhoL * (ps / pL + gm / gp) / (gm / gp * ps / pL + 1.0)
        out["shock_L"] = uL - cL * np.sqrt(gp / (2 * g) * ps / pL + gm / (2 * g))
    if ps > pR:
        out["rho_star_R"] = rhoR * (ps / pR + gm / gp) / (gm / gp * ps / pR + 1.0)
        out["shock_R"] = uR + cR * np.sqrt(gp / (2 * g) * ps / pR + gm / (2 * g))
    else:
        out["rho_star_R"] = rhoR * (ps / pR) ** (1.0 / g)
        out["head_R"] = uR + cR
        out["tail_R"] = us + cR * (ps / pR) ** (gm / (2 * g))
    return out


# ----------------------------------------------------------------------------- L1 metric (eq.19)
_GL_X, _GL_W = np.polynomial.legendre.leggauss(10)


def cell_average_1d(fn, x_lo, dx, n):
    """<A(x_i)> over each of n cells [x_lo + i dx, x_lo + (i+1) dx] by 10-node Gauss-Legendre."""
    centres = x_lo + (np.arange(n) + 0.5) * dx
    pts = centres[:, None] + 0.5 * dx * _GL_X[None, :]
    vals = fn(pts.ravel()).reshape(n, 10)
    return 0.5 * (vals * _GL_W[None, :]).sum(axis=1)


def l1_error(numerical, analytic_avg, dV):
    """L1 = dV * sum |N_i - <A(x_i)>|  (eq.19)."""
    return dV * np.abs(np.asarray(numerical) - np.asarray(analytic_avg)).sum()


def riemann_l1_density(rho_num, x_lo, dx, x0, t, left, right, g):
    n = len(rho_num)
    fn = lambda x: riemann_sample((x - x0) / t, *left, *right, g)[0]
    return l1_error(rho_num, cell_average_1d(fn, x_lo, dx, n), dx)


# ----------------------------------------------------------------------------- Sedov-Taylor
def sedov_profiles(V, g):
    """Closed-form spherical (nu=3) similarity solution parametrised by V in (1/g, 2/(g+1)]:
    returns (xi/xi0, G = rho/rho0, Z) with u = (2/5)(r/t) V, c^2 = (2/5)^2 (r/t)^2 Z."""
    nu1 = -(13.0 * g * g - 7.0 * g + 12.0) / ((3.0 * g - 1.0) * (2.0 * g + 1.0))
    nu2 = 5.0 * (g - 1.0) / (2.0 * g + 1.0)
    nu3 = 3.0 / (2.0 * g + 1.0)
    nu4 = -nu1 / (2.0 - g)
    nu5 = -2.0 / (2.0 - g)
    a = 0.5 * (g + 1.0) * V
    b = (g + 1.0) / (7.0 - g) * (5.0 - (3.0 * g - 1.0) * V)
    c = (g + 1.0) / (g - 1.0) * (g * V - 1.0)
    d = (g + 1.0) / (g - 1.0) * (1.0 - V)
    lam5 = a ** -2.0 * b ** nu1 * c ** nu2
    G = (g + 1.0) / (g - 1.0) * c ** nu3 * b ** nu4 * d ** nu5
    Z = g * (g - 1.0) * (1.0 - V) * V * V / (2.0 * (g * V - 1.0))
    return lam5 ** 0.2, G, Z


def sedov_xi0(g, n=200001):
    """xi0 with R(t) = xi0 (E0 t^2 / rho0)^(1/5): energy integral of the similarity solution,
    E0 = int (rho u^2/2 + p/(g-1)) 4 pi r^2 dr  =>  xi0^5 (16 pi/25) int_0^1 G (V^2/2 + Z/(g(g-1))) l^4 dl = 1."""
    V0, V1 = 1.0 / g, 2.0 / (g + 1.0)
    # cluster points towards V0 where lambda -> 0 slowly
    s = np.linspace(0.0, 1.0, n)[1:]
    V = V0 + (V1 - V0) * s ** 2
    lam, G, Z = sedov_profiles(V, g)
    f = G * (0.5 * V * V + Z / (g * (g - 1.0))) * lam ** 4
    lam = np.concatenate([[0.0], lam])
    f = np.concatenate([[0.0], f])
    integral = np.sum(0.5 * (f[1:] + f[:-1]) * np.diff(lam))
    return (25.0 / (16.0 * np.pi * integral)) ** 0.2


def sedov_radius(t, E0, rho0, g):
    return sedov_xi0(g) * (E0 * t * t / rho0) ** 0.2
