"""Pins for the oracle's building blocks (CPU only).  Each test checks the oracle against something
the paper or the mathematics fixes — never against itself."""
import itertools
import os

import numpy as np
import pytest

import oracle
from oracle import exact

GOLD = os.path.join(os.path.dirname(__file__), "golden")


def _rows(name):
    out = []
    for line in open(os.path.join(GOLD, name)):
        if line.strip() and not line.startswith("#"):
            out.append([float(x) for x in line.split()])
    return out


# ------------------------------------------------------------------ sum3sym (G8)
def test_sum3sym_permutation_and_sign():
    rng = np.random.default_rng(1)
    for _ in range(200):
        a, b, c = rng.standard_normal(3) * 10.0 ** rng.integers(-8, 8, 3)
        ref = oracle.sum3sym(a, b, c)
        for p in itertools.permutations((a, b, c)):
            assert oracle.sum3sym(*p) == ref
        assert oracle.sum3sym(-a, -b, -c) == -ref
        assert abs(ref - (a + b + c)) <= 4e-16 * (abs(a) + abs(b) + abs(c))
    assert oracle.sum3sym(1e-30, 5.0, -5.0) == 1e-30
    assert oracle.sum3sym(0.0, 0.0, 3.5) == 3.5
    assert oracle.sum3sym(2.0, -2.0, 2.0) == 2.0


# ------------------------------------------------------------------ WENO5-Z (G1)
def _cell_avg_poly(coef, i):
    """exact average over cell [i-1/2, i+1/2] of sum coef[k] x^k"""
    P = np.polynomial.Polynomial(coef).integ()
    return P(i + 0.5) - P(i - 0.5)


def test_wenoz_exact_for_polynomials_up_to_degree_two():
    # every one of the three candidate stencils reproduces a polynomial of degree <= 2 exactly from its cell
    # averages, so any convex combination (whatever the nonlinear weights) gives the exact face value
    for coef in ([1.0], [0.3, -2.0], [1.0, 0.5, -0.7]):
        avg = [_cell_avg_poly(coef, i) for i in range(-2, 3)]
        exact_face = np.polynomial.Polynomial(coef)(0.5)
        assert oracle.wenoz(*avg) == pytest.approx(exact_face, rel=0, abs=2e-15)
        exact_face_m = np.polynomial.Polynomial(coef)(-0.5)
        assert oracle.wenoz(*avg[::-1]) == pytest.approx(exact_face_m, rel=0, abs=2e-15)


def test_wenoz_smooth_limit_matches_fifth_order_linear_scheme():
    # On smooth data WENO-Z weights tend to (1/10, 6/10, 3/10) and the value to the classical
    # fifth-order upwind-biased interpolant (2a - 13b + 47c + 27d - 3e)/60; the difference must
    # shrink like h^5 or faster (Borges et al.: weights are within O(h^3..h^4) of linear ones,
    # candidates within O(h^3) of each other).
    errs = []
    for h in (0.1, 0.05, 0.025):
        f = lambda x: np.sin(1.0 + x) + 0.3 * x
        F = lambda x: -np.cos(1.0 + x) + 0.15 * x * x
        avg = [(F((i + 0.5) * h) - F((i - 0.5) * h)) / h for i in range(-2, 3)]
        a, b, c, d, e = avg
        lin = (2 * a - 13 * b + 47 * c + 27 * d - 3 * e) / 60.0
        errs.append(abs(oracle.wenoz(*avg) - lin))
        assert abs(oracle.wenoz(*avg) - f(0.5 * h)) < 2.0 * h ** 5
    assert errs[1] < errs[0] / 16 and errs[2] < errs[1] / 16


def test_wenoz_discontinuity_picks_smooth_stencil():
    # step between c and d: only candidate 0 (a,b,c) is smooth => value ~ c side extrapolation
    v = oracle.wenoz(1.0, 1.0, 1.0, 0.0, 0.0)
    assert abs(v - 1.0) < 1e-12
    v = oracle.wenoz(0.0, 0.0, 1.0, 1.0, 1.0)   # step between b and c: candidate 2 (c,d,e) smooth
    assert abs(v - 1.0) < 1e-12
    # odd symmetry and translation: wenoz(-q) = -wenoz(q) exactly
    rng = np.random.default_rng(3)
    for _ in range(100):
        q = rng.standard_normal(5)
        assert oracle.wenoz(*(-q)) == -oracle.wenoz(*q)


def test_wenoz_bounded_by_weights_convexity():
    rng = np.random.default_rng(4)
    for _ in range(200):
        a, b, c, d, e = rng.standard_normal(5)
        q0 = (2 * a - 7 * b + 11 * c) / 6
        q1 = (-b + 5 * c + 2 * d) / 6
        q2 = (2 * c + 5 * d - e) / 6
        v = oracle.wenoz(a, b, c, d, e)
        assert min(q0, q1, q2) - 1e-14 <= v <= max(q0, q1, q2) + 1e-14


# ------------------------------------------------------------------ minmod
def test_minmod_definition():
    assert oracle.minmod(1.0, 2.0) == 1.0
    assert oracle.minmod(3.0, 2.0) == 2.0
    assert oracle.minmod(-1.0, -2.0) == -1.0
    assert oracle.minmod(-1.0, 2.0) == 0.0
    assert oracle.minmod(0.0, 2.0) == 0.0
    assert oracle.minmod(1e-300, 1e-300) == 1e-300      # no product underflow


# ------------------------------------------------------------------ EOS / prim
def test_cons_to_prim_roundtrip():
    g = 1.4
    rho, u, v, w, p = 0.7, 0.3, -1.2, 2.0, 0.45
    E = p / (g - 1) + 0.5 * rho * (u * u + v * v + w * w)
    W = oracle.cons_to_prim([rho, rho * u, rho * v, rho * w, E], g)
    assert np.allclose(W, [rho, u, v, w, p], rtol=1e-14, atol=0)


# ------------------------------------------------------------------ Riemann fluxes
def _physical_flux(W, d, g):
    rho, vel, p = W[0], W[1:4], W[4]
    E = p / (g - 1) + 0.5 * rho * np.dot(vel, vel)
    F = np.empty(5)
    F[0] = rho * vel[d]
    F[1:4] = rho * vel * vel[d]
    F[1 + d] += p
    F[4] = (E + p) * vel[d]
    return F


@pytest.mark.parametrize("scheme", [0, 1])
def test_riemann_consistency(scheme):
    # F*(W, W) = F(W) of eq.3, sub- and supersonic in both directions, all three normals
    g = 1.4
    for W in ([1.0, 0.3, -0.2, 0.1, 1.0], [1.0, 3.0, 0.5, -0.4, 1.0], [0.5, -3.0, 0.2, 4.0, 0.7],
              [2.0, 0.0, 0.0, 0.0, 3.0]):
        for d in range(3):
            F = oracle.riemann(scheme, W, W, d, g)
            assert np.allclose(F, _physical_flux(np.array(W), d, g), rtol=1e-13, atol=1e-14)


@pytest.mark.parametrize("scheme", [0, 1])
def test_riemann_supersonic_upwinding(scheme):
    g = 1.4
    WL, WR = [1.0, 5.0, 0.1, 0.2, 1.0], [0.5, 4.0, -0.3, 0.0, 0.8]
    assert np.array_equal(oracle.riemann(scheme, WL, WR, 0, g), _physical_flux(np.array(WL), 0, g)) or \
        np.allclose(oracle.riemann(scheme, WL, WR, 0, g), _physical_flux(np.array(WL), 0, g), rtol=1e-15)
    WL2, WR2 = [1.0, -5.0, 0.1, 0.2, 1.0], [0.5, -4.0, -0.3, 0.0, 0.8]
    assert np.allclose(oracle.riemann(scheme, WL2, WR2, 0, g), _physical_flux(np.array(WR2), 0, g), rtol=1e-15)


@pytest.mark.parametrize("scheme", [0, 1])
def test_riemann_mirror_bitwise(scheme):
    # x -> -x: swap sides, negate normal velocity; mass/energy/tangential-momentum flux flip sign,
    # normal-momentum flux is even.  Must hold bit for bit (G5, G8).
    rng = np.random.default_rng(7)
    g = 5.0 / 3.0
    for _ in range(300):
        WL = np.array([rng.uniform(0.1, 2), *rng.uniform(-2, 2, 3), rng.uniform(0.1, 2)])
        WR = np.array([rng.uniform(0.1, 2), *rng.uniform(-2, 2, 3), rng.uniform(0.1, 2)])
        for d in range(3):
            F = oracle.riemann(scheme, WL, WR, d, g)
            ML, MR = WR.copy(), WL.copy()
            ML[1 + d] *= -1
            MR[1 + d] *= -1
            Fm = oracle.riemann(scheme, ML, MR, d, g)
            sign = -np.ones(5)
            sign[1 + d] = 1.0
            assert np.array_equal(Fm, sign * F)


@pytest.mark.parametrize("scheme", [0, 1])
def test_riemann_axis_relabelling_bitwise(scheme):
    rng = np.random.default_rng(8)
    g = 1.4
    for _ in range(100):
        WL = np.array([rng.uniform(0.1, 2), *rng.uniform(-2, 2, 3), rng.uniform(0.1, 2)])
        WR = np.array([rng.uniform(0.1, 2), *rng.uniform(-2, 2, 3), rng.uniform(0.1, 2)])
        F0 = oracle.riemann(scheme, WL, WR, 0, g)
        for perm in itertools.permutations(range(3)):
            # new axis a carries old axis perm[a]; normal x (old 0) becomes new axis perm.index(0)
            PL, PR = WL.copy(), WR.copy()
            for a in range(3):
                PL[1 + a] = WL[1 + perm[a]]
                PR[1 + a] = WR[1 + perm[a]]
            d = perm.index(0)
            F = oracle.riemann(scheme, PL, PR, d, g)
            assert F[0] == F0[0] and F[4] == F0[4]
            for a in range(3):
                assert F[1 + a] == F0[1 + perm[a]]


def test_hllc_resolves_stationary_contact_exactly():
    # u = 0, uniform p, density jump: HLLC returns (0, p, 0, 0, 0) exactly; HLL smears (mass flux != 0)
    g = 1.4
    WL, WR = [1.0, 0.0, 0.0, 0.0, 0.7], [0.125, 0.0, 0.0, 0.0, 0.7]
    F = oracle.riemann(1, WL, WR, 0, g)
    assert np.array_equal(F, [0.0, 0.7, 0.0, 0.0, 0.0])
    assert oracle.riemann(0, WL, WR, 0, g)[0] != 0.0


def test_hll_matches_textbook_formula_on_subsonic_case():
    # Davis bounds + HLL average, typed out with numbers (independent arithmetic in numpy)
    g = 1.4
    WL, WR = np.array([1.0, 0.1, 0.2, -0.1, 1.0]), np.array([0.8, -0.2, 0.0, 0.3, 0.9])
    cL, cR = np.sqrt(g * WL[4] / WL[0]), np.sqrt(g * WR[4] / WR[0])
    SL, SR = min(WL[1] - cL, WR[1] - cR), max(WL[1] + cL, WR[1] + cR)

    def cons(W):
        return np.array([W[0], W[0] * W[1], W[0] * W[2], W[0] * W[3],
                         W[4] / (g - 1) + 0.5 * W[0] * np.dot(W[1:4], W[1:4])])
    ref = (SR * _physical_flux(WL, 0, g) - SL * _physical_flux(WR, 0, g) + SL * SR * (cons(WR) - cons(WL))) / (SR - SL)
    assert np.allclose(oracle.riemann(0, WL, WR, 0, g), ref, rtol=1e-14)


def test_hllc_matches_star_state_form():
    # the classical HLLC form F_K + S_K (U*_K - U_K) (Toro) agrees with the averaged-pressure form
    g = 1.4
    WL, WR = np.array([1.0, 0.1, 0.2, -0.1, 1.0]), np.array([0.8, -0.2, 0.0, 0.3, 0.9])
    cL, cR = np.sqrt(g * WL[4] / WL[0]), np.sqrt(g * WR[4] / WR[0])
    SL, SR = min(WL[1] - cL, WR[1] - cR), max(WL[1] + cL, WR[1] + cR)
    Ss = (WR[4] - WL[4] + WL[0] * WL[1] * (SL - WL[1]) - WR[0] * WR[1] * (SR - WR[1])) / \
        (WL[0] * (SL - WL[1]) - WR[0] * (SR - WR[1]))
    W, S = (WL, SL) if Ss >= 0 else (WR, SR)
    E = W[4] / (g - 1) + 0.5 * W[0] * np.dot(W[1:4], W[1:4])
    fac = W[0] * (S - W[1]) / (S - Ss)
    Us = fac * np.array([1.0, Ss, W[2], W[3], E / W[0] + (Ss - W[1]) * (Ss + W[4] / (W[0] * (S - W[1])))])
    U = np.array([W[0], W[0] * W[1], W[0] * W[2], W[0] * W[3], E])
    ref = _physical_flux(W, 0, g) + S * (Us - U)
    assert np.allclose(oracle.riemann(1, WL, WR, 0, g), ref, rtol=1e-13, atol=1e-15)


# ------------------------------------------------------------------ exact solutions used as pins
def test_exact_riemann_matches_textbook_sod():
    ps, us, rl, rr = _rows("sod_star_textbook.txt")[0]
    w = exact.riemann_waves(1.0, 0.0, 1.0, 0.125, 0.0, 0.1, 1.4)
    assert w["p_star"] == pytest.approx(ps, abs=5e-6)
    assert w["u_star"] == pytest.approx(us, abs=5e-6)
    assert w["rho_star_L"] == pytest.approx(rl, abs=5e-6)
    assert w["rho_star_R"] == pytest.approx(rr, abs=5e-6)
    # Rankine-Hugoniot across the right shock, independent of the solver's own formulas
    S = w["shock_R"]
    assert 0.125 * (0.0 - S) == pytest.approx(w["rho_star_R"] * (w["u_star"] - S), rel=1e-12)
    assert 0.1 + 0.125 * S * S == pytest.approx(w["p_star"] + w["rho_star_R"] * (w["u_star"] - S) ** 2, rel=1e-12)


def test_exact_riemann_leblanc_jump_conditions():
    g = 5.0 / 3.0
    pL, pR = (g - 1) * 0.1, (g - 1) * 1e-3 * 1e-7
    w = exact.riemann_waves(1.0, 0.0, pL, 1e-3, 0.0, pR, g)
    S = w["shock_R"]
    assert 1e-3 * (0.0 - S) == pytest.approx(w["rho_star_R"] * (w["u_star"] - S), rel=1e-12)
    assert pR + 1e-3 * S * S == pytest.approx(w["p_star"] + w["rho_star_R"] * (w["u_star"] - S) ** 2, rel=1e-10)
    # isentropic left rarefaction: p / rho^gamma constant, Riemann invariant u + 2c/(g-1) constant
    assert w["p_star"] / w["rho_star_L"] ** g == pytest.approx(pL, rel=1e-12)
    cs = np.sqrt(g * w["p_star"] / w["rho_star_L"])
    assert w["u_star"] + 2 * cs / (g - 1) == pytest.approx(2 * np.sqrt(g * pL) / (g - 1), rel=1e-12)
    assert 3.0 + 6.0 * S == pytest.approx(7.97471, abs=1e-4)


def test_sedov_constant_matches_textbook():
    for g, xi0, tol in _rows("sedov_xi0_textbook.txt"):
        assert exact.sedov_xi0(g) == pytest.approx(xi0, abs=tol)
    # the similarity profile satisfies the strong-shock jump conditions at V = 2/(g+1) and
    # conserves the swept-up mass: int_0^1 G lambda^2 dlambda = 1/3
    g = 1.4
    lam, G, Z = exact.sedov_profiles(np.array([2.0 / (g + 1.0)]), g)
    assert lam[0] == pytest.approx(1.0) and G[0] == pytest.approx((g + 1) / (g - 1))
    assert Z[0] == pytest.approx(2 * g * (g - 1) / (g + 1) ** 2)
    V = 1 / g + (2 / (g + 1) - 1 / g) * np.linspace(0, 1, 200001)[1:] ** 2
    lam, G, Z = exact.sedov_profiles(V, g)
    f = G * lam ** 2
    mass = np.sum(0.5 * (f[1:] + f[:-1]) * np.diff(lam))
    assert 3 * mass == pytest.approx(1.0, abs=1e-6)


def test_gauss_legendre_cell_average_exact_for_degree_19():
    coef = np.arange(1, 21, dtype=float) / 7.0
    P = np.polynomial.Polynomial(coef)
    avg = exact.cell_average_1d(P, 0.25, 0.5, 3)
    I = P.integ()
    ref = [(I(0.25 + 0.5 * (i + 1)) - I(0.25 + 0.5 * i)) / 0.5 for i in range(3)]
    assert np.allclose(avg, ref, rtol=1e-13)
