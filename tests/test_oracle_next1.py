"""NEXT-1: the radiation energy density as a sixth advected field, d_t E + d_j(E v^j) = 0
(eq.2 fourth row, eq.14 left-hand side), same reconstruction as the other variables and
the local Lax-Friedrichs (Rusanov) flux; reading G19.  Pins of the oracle's implementation."""
import math

import numpy as np
import pytest

import oracle
from paper_2509_08971_b200 import workloads as wl


def _run(state, er, n, bc, scheme, sp, nsteps=1, cfl=0.4, dt=None, gamma=1.4):
    o = oracle.Oracle(*n, gamma, bc, scheme=scheme, spacing=sp, radiation=True)
    o.set_state(*state)
    o.set_rad_energy(er)
    if dt is None:
        o.step(cfl, nsteps)
    else:
        o.step_dt(dt, nsteps)
    out, eo = o.get_state(), o.get_rad_energy()
    o.close()
    return out, eo


def _rand_er(n, seed):
    return 1.0 + 0.5 * np.random.default_rng(seed).random(n[::-1])


def test_rusanov_flux_definition():
    g = 1.4
    WL, WR = np.array([1.0, 0.3, -0.2, 0.1, 1.0]), np.array([0.8, -0.5, 0.4, 0.2, 0.9])
    for d in range(3):
        # consistency: F(E, E; W, W) = E u_d   (eq.14 LHS flux E v^j)
        assert oracle.rusanov(2.5, 2.5, WL, WL, d, g) == pytest.approx(2.5 * WL[1 + d], rel=1e-15)
        # the definition with numbers typed out
        cL, cR = math.sqrt(g * WL[4] / WL[0]), math.sqrt(g * WR[4] / WR[0])
        al = max(abs(WL[1 + d]) + cL, abs(WR[1 + d]) + cR)
        ref = 0.5 * (2.0 * WL[1 + d] + 3.0 * WR[1 + d]) - 0.5 * al * (3.0 - 2.0)
        assert oracle.rusanov(2.0, 3.0, WL, WR, d, g) == pytest.approx(ref, rel=1e-15)
        # mirror image: swap sides, negate the normal velocity -> flux changes sign, bit for bit
        ML, MR = WR.copy(), WL.copy()
        ML[1 + d] *= -1
        MR[1 + d] *= -1
        assert oracle.rusanov(3.0, 2.0, ML, MR, d, g) == -oracle.rusanov(2.0, 3.0, WL, WR, d, g)


@pytest.mark.parametrize("scheme", [0, 1])
def test_hydro_fields_do_not_see_the_radiation_field(scheme):
    n = (9, 8, 7)
    sp = (0.1, 0.07, 0.13)
    st = wl.random_state(n, seed=41)
    out6, _ = _run(st, _rand_er(n, 1), n, wl.BC_PERIODIC, scheme, sp, nsteps=3)
    o = oracle.Oracle(*n, 1.4, wl.BC_PERIODIC, scheme=scheme, spacing=sp)
    o.set_state(*st)
    o.step(0.4, 3)
    out5 = o.get_state()
    for f in range(5):
        assert np.array_equal(out6[f], out5[f])


@pytest.mark.parametrize("scheme", [0, 1])
def test_radiation_energy_conserved_and_uniform_flow_preserved(scheme):
    n = (10, 9, 8)
    sp = (0.1, 0.07, 0.13)
    st = wl.random_state(n, seed=42)
    er = _rand_er(n, 2)
    _, eo = _run(st, er, n, wl.BC_PERIODIC, scheme, sp, nsteps=10)
    ref = math.fsum(er.ravel().tolist())
    assert abs(math.fsum(eo.ravel().tolist()) - ref) <= 1e-13 * ref
    assert not np.array_equal(eo, er)
    g = 1.4
    vals = (1.3, 1.3 * 0.37, 1.3 * -0.21, 1.3 * 0.11, 0.9 / (g - 1) + 0.5 * 1.3 * (0.37 ** 2 + 0.21 ** 2 + 0.11 ** 2))
    uni = [np.full(n[::-1], v) for v in vals]
    out, eo = _run(uni, np.full(n[::-1], 2.75), n, wl.BC_PERIODIC, scheme, sp, nsteps=5)
    assert np.array_equal(eo, np.full(n[::-1], 2.75))
    for f in range(5):
        assert np.array_equal(out[f], uni[f])


@pytest.mark.parametrize("scheme", [0, 1])
@pytest.mark.parametrize("axis", [0, 1, 2])
def test_mirror_symmetry_with_radiation_bitwise(scheme, axis):
    n = (9, 8, 7)
    sp = (0.1, 0.07, 0.13)
    st, er = wl.random_state(n, seed=43), _rand_er(n, 3)
    out, eo = _run(st, er, n, wl.BC_OUTFLOW, scheme, sp, nsteps=3)
    ax_np = 2 - axis
    stm = [np.flip(a, ax_np).copy() for a in st]
    stm[1 + axis] = -stm[1 + axis]
    outm, eom = _run(stm, np.flip(er, ax_np).copy(), n, wl.BC_OUTFLOW, scheme, sp, nsteps=3)
    assert np.array_equal(np.flip(eom, ax_np), eo)
    assert np.array_equal(np.flip(outm[0], ax_np), out[0])


def _wz(a, b, c, d, e):
    b0 = 13 / 12 * (a - 2 * b + c) ** 2 + 0.25 * (a - 4 * b + 3 * c) ** 2
    b1 = 13 / 12 * (b - 2 * c + d) ** 2 + 0.25 * (b - d) ** 2
    b2 = 13 / 12 * (c - 2 * d + e) ** 2 + 0.25 * (3 * c - 4 * d + e) ** 2
    tau = np.abs(b0 - b2)
    al = [0.1 * (1 + tau / (b0 + 1e-40)), 0.6 * (1 + tau / (b1 + 1e-40)), 0.3 * (1 + tau / (b2 + 1e-40))]
    q = [(2 * a - 7 * b + 11 * c) / 6, (-b + 5 * c + 2 * d) / 6, (2 * c + 5 * d - e) / 6]
    return (al[0] * q[0] + al[1] * q[1] + al[2] * q[2]) / (al[0] + al[1] + al[2])


def test_bruteforce_scalar_advection_in_uniform_flow():
    """With a uniform fluid the face states are the constants themselves, so the E_rad update is linear scalar
    advection with WENO5-Z + Rusanov, alpha_d = |u_d| + c: restated here on whole arrays with np.roll."""
    g = 1.4
    n = (7, 6, 5)
    sp = (0.25, 0.2, 0.3)
    rho, vel, p = 1.3, (0.37, -0.21, 0.11), 0.9
    E = p / (g - 1) + 0.5 * rho * sum(v * v for v in vel)
    uni = [np.full(n[::-1], v) for v in (rho, rho * vel[0], rho * vel[1], rho * vel[2], E)]
    er = _rand_er(n, 5)
    dt = 0.03
    c = math.sqrt(g * p / rho)

    def L(e):
        out = np.zeros_like(e)
        for d in range(3):
            ax = 2 - d
            sh = lambda a, s: np.roll(a, -s, axis=ax)
            eL = _wz(sh(e, -2), sh(e, -1), e, sh(e, 1), sh(e, 2))                       # plus of cell i
            eR = sh(_wz(sh(e, 2), sh(e, 1), e, sh(e, -1), sh(e, -2)), 1)                # minus of cell i+1
            F = 0.5 * vel[d] * (eL + eR) - 0.5 * (abs(vel[d]) + c) * (eR - eL)
            out -= (F - sh(F, -1)) / sp[d]
        return out
    e1 = er + dt * L(er)
    ref = 0.5 * er + 0.5 * (e1 + dt * L(e1))
    _, eo = _run(uni, er, n, wl.BC_PERIODIC, 0, sp, dt=dt)
    assert np.abs(eo - ref).max() <= 1e-14 * np.abs(ref).max()
    assert np.abs(eo - er).max() > 1e-3


@pytest.mark.parametrize("scheme", [0, 1])
def test_advected_profile_returns_after_one_period(scheme):
    """Uniform flow u: E_rad(x, t) = E_rad(x - u t, 0); after one period the profile is back, error order -> 2."""
    g, u = 1.4, 0.8
    errs = []
    ns = [16, 32, 64, 128]
    for n in ns:
        dx = 1.0 / n
        x = (np.arange(n) + 0.5) * dx
        s = (np.cos(2 * np.pi * (x - 0.5 * dx)) - np.cos(2 * np.pi * (x + 0.5 * dx))) / (2 * np.pi * dx)
        er = 1.0 + 0.3 * s
        one = np.ones(n)
        st = [a.reshape(1, 1, n) for a in (one, u * one, 0 * one, 0 * one, 1.0 / (g - 1) + 0.5 * u * u * one)]
        o = oracle.Oracle(n, 1, 1, g, wl.BC_PERIODIC, scheme=scheme, spacing=(dx, 1, 1), radiation=True)
        o.set_state(*st)
        o.set_rad_energy(er.reshape(1, 1, n))
        o.run_to(1.0 / u, 0.4)
        errs.append(np.abs(o.get_rad_energy().ravel() - er).sum() * dx)
        o.close()
    pair = np.log2(np.array(errs[:-1]) / np.array(errs[1:]))
    assert pair[-1] >= (1.9 if scheme == 0 else 1.6) and errs[-1] < errs[0] / 20
